"""GPU parity: the CUDA path (through the C ABI) against the fp64 oracle, element by element, on the same
seeded fp32 inputs.  Tolerances are north_star's: per element |x - ref| / max(1, |ref|) <= 1e-4 for FK poses
and Jacobians, <= 1e-3 for RNEA torques and CRBA entries (the per-element reading)."""
import numpy as np
import pytest

import oracle
import manifold
from paper_2605_31481_b200 import binding, workloads as W

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

TOL_KIN, TOL_DYN = 1e-4, 1e-3


def nerr(x, ref):
    return float(np.max(np.abs(x.astype(np.float64) - ref) / np.maximum(1.0, np.abs(ref)))) if ref.size else 0.0


class Gpu:
    def __init__(self, desc):
        assert torch.cuda.is_available(), "GPU tests need CUDA; there is no CPU fallback"
        self.m = binding.Model(desc, device=0)
        self.o = oracle.Oracle(desc)
        self.dev = torch.device("cuda:0")

    def run(self, q, qd, qdd):
        m, dev = self.m, self.dev
        B = q.shape[1]
        tq, tqd, tqdd = (torch.from_numpy(np.ascontiguousarray(a)).to(dev) for a in (q, qd, qdd))
        # NaN-filled outputs: every element must be overwritten by the kernels
        pose = torch.full((m.nb, 12, B), float("nan"), device=dev)
        J = torch.full((m.nframes, 6, m.nv, B), float("nan"), device=dev)
        tau = torch.full((m.nv, B), float("nan"), device=dev)
        M = torch.full((m.nv, m.nv, B), float("nan"), device=dev)
        s = torch.cuda.current_stream().cuda_stream
        m.fk(B, tq, pose, s)
        m.jacobian(B, tq, J, s)
        m.rnea(B, tq, tqd, tqdd, tau, s)
        m.crba(B, tq, M, s)
        torch.cuda.synchronize()
        return pose.cpu().numpy(), J.cpu().numpy(), tau.cpu().numpy(), M.cpu().numpy()

    def check(self, q, qd, qdd):
        pose, J, tau, M = self.run(q, qd, qdd)
        q64, qd64, qdd64 = (a.astype(np.float64) for a in (q, qd, qdd))
        for a in (pose, J, tau, M):
            assert np.isfinite(a).all()
        errs = {
            "fk": nerr(pose, self.o.fk(q64)),
            "jac": nerr(J, self.o.jacobian(q64)) if self.m.nframes else 0.0,
            "rnea": nerr(tau, self.o.rnea(q64, qd64, qdd64)),
            "crba": nerr(M, self.o.crba(q64)),
        }
        assert errs["fk"] <= TOL_KIN, errs
        assert errs["jac"] <= TOL_KIN, errs
        assert errs["rnea"] <= TOL_DYN, errs
        assert errs["crba"] <= TOL_DYN, errs
        assert np.array_equal(M, np.swapaxes(M, 0, 1))      # written symmetric, bit for bit
        return errs


# B = 1000: several CTAs plus a ragged tail (not a multiple of 32, 64 or 128)
@pytest.mark.parametrize("cfg", [0, 1, 2, 3])
@pytest.mark.parametrize("B", [1, 37, 1000])
def test_configs(cfg, B):
    desc = W.config_robot(cfg)
    q, qd, qdd = W.config_states(cfg, B)
    Gpu(desc).check(q, qd, qdd)


@pytest.mark.parametrize("cfg", [0, 1, 2, 3])
def test_configs_B4096(cfg):
    desc = W.config_robot(cfg)
    q, qd, qdd = W.config_states(cfg, 4096)
    Gpu(desc).check(q, qd, qdd)


@pytest.mark.parametrize("seed", range(10))
def test_random_trees_all_joint_types(seed):
    """prismatic / fixed / free joints, non-identity T_post, general axes, full inertias, frame offsets, forests."""
    shape = ["random", "chain", "star", "unbalanced"][seed % 4]
    desc = W.random_tree(300 + seed, nb=2 + 3 * seed, shape=shape, free_root=(seed % 2 == 0), nframes=3)
    q, qd, qdd = W.sample_states(desc, 200, seed=77 + seed)
    Gpu(desc).check(q, qd, qdd)


def massless_fixed_links(seed, nb=9, free_root=False):
    """A tree whose FIXED-joint bodies are massless frames (URDF base / tool / sensor links), incl. a massless leaf."""
    desc = W.random_tree(seed, nb=nb, joint_types=(W.REVOLUTE, W.FIXED, W.PRISMATIC), free_root=free_root, nframes=3)
    jt = desc.joint_type.copy()
    jt[nb - 1] = W.FIXED                                # a massless tool frame at a leaf
    if not free_root:
        jt[0] = W.FIXED                                 # a massless base link
    desc.joint_type = jt
    for i in range(nb):
        if int(jt[i]) == W.FIXED:
            desc.mass[i] = 0.0
            desc.com[i] = 0.0
            desc.inertia[i] = 0.0
    return desc


@pytest.mark.parametrize("seed", range(4))
def test_massless_fixed_links(seed):
    """bodies with mass 0 (frames behind fixed joints) are legal for FK, Jacobian, RNEA and CRBA."""
    desc = massless_fixed_links(820 + seed, free_root=(seed % 2 == 1))
    q, qd, qdd = W.sample_states(desc, 300, seed=3 + seed)
    g = Gpu(desc)
    g.check(q, qd, qdd)
    g.m.set_option("spec_min_b", 0)
    g.m.specialize(("fk", "jacobian", "rnea", "crba"))
    g.check(q, qd, qdd)


def test_max_size_tree():
    desc = W.random_tree(4242, nb=64, shape="random", nframes=16)
    q, qd, qdd = W.sample_states(desc, 96, seed=5)
    Gpu(desc).check(q, qd, qdd)


def test_single_fixed_body_and_no_frames():
    desc = W.build_robot("one_fixed", [-1], [W.FIXED], seed=1)
    q, qd, qdd = W.sample_states(desc, 8, seed=1)
    g = Gpu(desc)
    pose, J, tau, M = g.run(q, qd, qdd)
    assert nerr(pose, g.o.fk(q.astype(np.float64))) <= TOL_KIN
    assert J.size == 0 and tau.size == 0 and M.size == 0


def test_empty_batch_is_ok():
    desc = W.config_robot(0)
    m = binding.Model(desc, device=0)
    m.fk(0, None, None)
    m.rnea(0, None, None, None, None)
    m.crba(0, None, None)
    m.jacobian(0, None, None)


def test_unnormalised_quaternion_is_normalised_inside():
    desc = W.config_robot(1)
    q, qd, qdd = W.config_states(1, 64)
    q = q.copy()
    q[3:7] *= 3.0
    Gpu(desc).check(q, qd, qdd)


def test_euler_rollout_config2():
    """config 2: 24 consecutive steps, q advanced by explicit Euler from random qdd; all four operators per step."""
    desc = W.config_robot(2)
    g = Gpu(desc)
    for q, qd, qdd in manifold.euler_rollout(2, 256, steps=24):
        g.check(q, qd, qdd)


def test_non_default_stream_and_launch_count():
    desc = W.config_robot(3)
    g = Gpu(desc)
    q, qd, qdd = W.config_states(3, 512)
    n0 = binding.launch_count()
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        g.check(q, qd, qdd)
    assert binding.launch_count() - n0 == 4


@pytest.mark.parametrize("cfg,B", [(3, 65536), (0, 1048576)])
def test_full_size_sampled(cfg, B):
    """Full bench sizes: compare a strided sample of environments against the oracle (the oracle evaluates
    envs one by one, so any subset is computable)."""
    desc = W.config_robot(cfg)
    q, qd, qdd = W.config_states(cfg, B)
    g = Gpu(desc)
    pose, J, tau, M = g.run(q, qd, qdd)
    idx = np.unique(np.concatenate([np.arange(0, B, max(1, B // 997)), [B - 1, B - 2, 127, 128, B // 2]]))
    q64, qd64, qdd64 = (np.ascontiguousarray(a[:, idx].astype(np.float64)) for a in (q, qd, qdd))
    assert nerr(pose[..., idx], g.o.fk(q64)) <= TOL_KIN
    assert nerr(J[..., idx], g.o.jacobian(q64)) <= TOL_KIN
    assert nerr(tau[..., idx], g.o.rnea(q64, qd64, qdd64)) <= TOL_DYN
    assert nerr(M[..., idx], g.o.crba(q64)) <= TOL_DYN
    for a in (pose, J, tau, M):
        assert np.isfinite(a).all()


@pytest.mark.parametrize("knobs", [{"pack": 2}, {"pack": 1}, {"pack": 2, "BARD_FORCE_GENERAL": "1"},
                                   {"BARD_TEAM_WARPS": "1"}, {"BARD_TEAM_WARPS": "8", "pack": 2},
                                   {"teams": 1}])
@pytest.mark.parametrize("cfg", [0, 1, 2, 3])
def test_every_kernel_instantiation(cfg, knobs, monkeypatch):
    """The launch heuristics pick (environments per lane, SIMPLE/general kernels, team width) from B and the
    model; the test knobs force each instantiation on every config, at a size with several tiles and a ragged tail.
    Launch knobs are model options; the two that shape the model's constant tables (team width, general kernels)
    are read from the environment once, by bard_model_create."""
    for k, v in knobs.items():
        if k.startswith("BARD_"):
            monkeypatch.setenv(k, v)
    desc = W.config_robot(cfg)
    for B in (1000, 130):
        q, qd, qdd = W.config_states(cfg, B)
        g = Gpu(desc)
        for k, v in knobs.items():
            if not k.startswith("BARD_"):
                g.m.set_option(k, v)
        g.check(q, qd, qdd)


def test_odd_batch_and_misaligned_views():
    """Odd B and output/input pointers that are only 4-byte aligned must take the scalar paths, never fault."""
    desc = W.config_robot(1)
    B = 777
    q, qd, qdd = W.config_states(1, B)
    g = Gpu(desc)
    m, dev = g.m, g.dev
    def off(a):                                    # a tensor whose data pointer is 4 (mod 16)
        buf = torch.empty(a.size + 1, device=dev)
        v = buf[1:].view(a.shape)
        v.copy_(torch.from_numpy(a))
        return v
    tq, tqd, tqdd = off(q), off(qd), off(qdd)
    pose = off(np.full((m.nb, 12, B), np.nan, np.float32)); J = off(np.full((m.nframes, 6, m.nv, B), np.nan, np.float32))
    tau = off(np.full((m.nv, B), np.nan, np.float32)); M = off(np.full((m.nv, m.nv, B), np.nan, np.float32))
    s = torch.cuda.current_stream().cuda_stream
    m.fk(B, tq, pose, s); m.jacobian(B, tq, J, s); m.rnea(B, tq, tqd, tqdd, tau, s); m.crba(B, tq, M, s)
    torch.cuda.synchronize()
    q64, qd64, qdd64 = (a.astype(np.float64) for a in (q, qd, qdd))
    assert nerr(pose.cpu().numpy(), g.o.fk(q64)) <= TOL_KIN
    assert nerr(J.cpu().numpy(), g.o.jacobian(q64)) <= TOL_KIN
    assert nerr(tau.cpu().numpy(), g.o.rnea(q64, qd64, qdd64)) <= TOL_DYN
    assert nerr(M.cpu().numpy(), g.o.crba(q64)) <= TOL_DYN


def test_too_many_elements_is_refused_not_wrapped():
    """Outputs of 2^32 elements or more are refused (32-bit element indices in the kernels)."""
    desc = W.config_robot(3)
    m = binding.Model(desc, device=0)
    t = torch.empty(16, device="cuda:0")
    with pytest.raises(binding.BardError) as e:
        m.crba(1 << 23, t, t)                      # 841 * 2^23 > 2^32: refused before any launch
    assert e.value.code == 3


@pytest.mark.parametrize("cfg", [1, 3])
def test_repeated_launches_are_bit_identical(cfg):
    """No atomics, fixed child order (DESIGN reading 7): every launch must reproduce the same bits.  A race
    between a team's warps (barriers, shared-memory rows that are reused) would show up here as noise."""
    desc = W.config_robot(cfg)
    g = Gpu(desc)
    q, qd, qdd = W.config_states(cfg, 4096 + 32)
    ref = g.run(q, qd, qdd)
    for _ in range(5):
        out = g.run(q, qd, qdd)
        for a, b in zip(ref, out):
            assert np.array_equal(a, b)
