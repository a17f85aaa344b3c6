"""Model-specialised kernels (bard_model_specialize): host-side generation + NVRTC compilation on CPU, and GPU
parity of the generated FK / Jacobian / RNEA / CRBA against the fp64 oracle and against the level-parallel
team kernels."""
import os
import re

import numpy as np
import pytest

import oracle
from paper_2605_31481_b200 import binding, workloads as W

TOL_KIN, TOL_DYN = 1e-4, 1e-3
ALL = ("fk", "jacobian", "rnea", "crba")
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def nerr(x, ref):
    return float(np.max(np.abs(x.astype(np.float64) - ref) / np.maximum(1.0, np.abs(ref)))) if ref.size else 0.0


def _robots():
    out = [W.config_robot(c) for c in range(4)]
    for seed in range(6):
        shape = ["random", "chain", "star", "unbalanced"][seed % 4]
        out.append(W.random_tree(500 + seed, nb=2 + 4 * seed, shape=shape, free_root=(seed % 2 == 0), nframes=3))
    return out


# ------------------------------------------------------------------------------------------- CPU (no GPU needed)
@pytest.mark.parametrize("idx", range(10))
def test_generated_source_compiles_on_host(idx):
    """A host-only model: the source is generated and NVRTC-compiled for sm_100a, nothing is loaded."""
    desc = _robots()[idx]
    m = binding.Model(desc, device=-1)
    m.specialize(ALL + ("fused",))
    for op in ALL:
        assert 'extern "C" __global__' in m.specialized_source(op) and f"bard_{op}_n1" in m.specialized_source(op)
    if m.nv > 0 and m.nframes > 0:
        assert "bard_step_n1" in m.specialized_source("fused")       # written even where it is not worth building
    # FK: 12 rows per body; CRBA / Jacobian: every output row stored exactly once (fill + structural zeros)
    for op, arr, n in (("fk", "pose", 12 * m.nb), ("crba", "Mo", m.nv * m.nv), ("jacobian", "J", 6 * m.nframes * m.nv)):
        rows = sorted(int(r) for r in re.findall(r"STROW\(%s, (\d+)u," % arr, m.specialized_source(op)))
        assert rows == list(range(n)), op
    src = m.specialized_source("rnea")
    # one outward and one inward section per body, every tau row stored exactly once
    assert len(re.findall(r"// ---- body \d+ \(outward\)", src)) == m.nb
    assert len(re.findall(r"// ---- body \d+ \(inward\)", src)) == m.nb
    rows = sorted(int(r) for r in re.findall(r"STROW\(tau, (\d+)u,", src))
    assert rows == list(range(m.nv))
    # every input row is loaded exactly once
    for arr, n in (("q", m.nq), ("qd", m.nv), ("qdd", m.nv)):
        got = sorted(int(r) for r in re.findall(r"LDROW\(%s, (\d+)u\)" % arr, src))
        assert got == list(range(n)), arr


def test_parked_rows_follow_the_path_not_the_body_count():
    """Depth-first order: parked state is bounded by the deepest root-to-leaf path (8 rows per body on it plus
    12 per branch point), not by nb -- the star has many bodies and almost no parked state."""
    def rows(desc):
        m = binding.Model(desc, device=-1)
        m.specialize(("rnea",))
        return int(re.search(r"#define ROWS (\d+)", m.specialized_source("rnea")).group(1))
    chain = W.random_tree(1, nb=20, shape="chain", joint_types=(W.REVOLUTE,))
    star = W.random_tree(1, nb=20, shape="star", joint_types=(W.REVOLUTE,))
    assert rows(chain) <= 8 * 20 + 1
    assert rows(star) <= 8 + 12 + 8 + 1
    assert rows(W.config_robot(3)) <= 8 * 7 + 12 * 2 + 1          # humanoid: depth 7, two branch points on a path


def test_unknown_operator_bits_are_refused_and_set_frames_drops_the_jacobian():
    m = binding.Model(W.config_robot(0), device=-1)
    assert binding.lib().bard_model_specialize(m._h, 1 << 7) == 1  # BARD_ERR_INVALID_ARG
    with pytest.raises(binding.BardError):
        m.specialized_source("rnea")                              # not specialised yet
    m.specialize(("jacobian",))
    assert "frame 0 on body 6" in m.specialized_source("jacobian")
    m.set_frames([2])                                             # the generated code was for the old frame
    with pytest.raises(binding.BardError):
        m.specialized_source("jacobian")
    m.specialize(("jacobian",))
    assert "frame 0 on body 2" in m.specialized_source("jacobian")


def _single_root_and_branches(desc):
    parent = [int(p) for p in desc.parent]
    nchild = [parent.count(i) for i in range(len(parent))]
    return parent.count(-1) == 1 and any(n >= 2 for n in nchild)


def test_limb_role_source_on_a_host_only_model():
    """The limb-role RNEA kernel is generated where a single-rooted tree branches, one `if (role == r)` stretch per
    role, forces handed over through park_to and one named barrier; never for a chain."""
    for roles in (2, 3):
        m = binding.Model(W.config_robot(3), device=-1)
        m.set_option("spec_roles", roles)
        m.specialize(("rnea",))
        src = m.specialized_source("rnea_roles")
        for r in range(roles):
            assert f"if (role == {r}u)" in src
        assert f"if (role == {roles}u)" not in src
        assert "park_to<T, N, R>(le," in src and "bar.sync 15" in src and "bar.arrive 15" in src
    m = binding.Model(W.config_robot(0), device=-1)
    m.specialize(("rnea",))
    with pytest.raises(binding.BardError):
        m.specialized_source("rnea_roles")


def test_rnea_source_has_a_variant_without_l2_prefetch():
    """RNEA is generated twice by default: with the up-front L2 prefetch (grids of one wave) and without it
    (`_np`, larger grids); BARD_SPEC_L2PF = 1 / 0 generate one kernel; the other operators always one."""
    m = binding.Model(W.config_robot(1), device=-1)
    m.specialize(("rnea", "fk"))
    src = m.specialized_source("rnea")
    assert "bard_rnea_n1_np(" in src and "bard_rnea_n1(" in src and "if (PF) {" in src
    assert "_np(" not in m.specialized_source("fk")
    for v in ("0", "1"):
        m = binding.Model(W.config_robot(1), device=-1)
        m.set_option("spec_l2pf", int(v))
        m.specialize(("rnea",))
        src = m.specialized_source("rnea")
        assert "_np(" not in src and ("PFROW(q" in src) == (v == "1")


# ------------------------------------------------------------------------------------------- GPU
torch = pytest.importorskip("torch")


class Spec:
    def __init__(self, desc, ops=ALL, **opts):
        """`opts`: knobs of THIS model, set through bard_model_set_option before the kernels are generated."""
        assert torch.cuda.is_available(), "GPU tests need CUDA; there is no CPU fallback"
        self.m = binding.Model(desc, device=0)
        for k, v in opts.items():
            self.m.set_option(k, v)
        self.m.specialize(ops)
        self.o = oracle.Oracle(desc)
        self.dev = torch.device("cuda:0")

    def run_dev(self, q, qd, qdd):
        """As run(), but the outputs stay on the device (full bench sizes: gigabytes)."""
        m, B, dev = self.m, q.shape[1], self.dev
        tq, tqd, tqdd = (torch.from_numpy(np.ascontiguousarray(a)).to(dev) for a in (q, qd, qdd))
        outs = [torch.full(sh, float("nan"), device=dev) for sh in ((m.nb, 12, B), (m.nframes, 6, m.nv, B), (m.nv, B), (m.nv, m.nv, B))]
        s = torch.cuda.current_stream().cuda_stream
        m.fk(B, tq, outs[0], s)
        m.jacobian(B, tq, outs[1], s)
        m.rnea(B, tq, tqd, tqdd, outs[2], s)
        m.crba(B, tq, outs[3], s)
        torch.cuda.synchronize()
        return outs

    def run(self, q, qd, qdd):
        """All four operators, NaN-filled outputs (every element must be overwritten), one launch each."""
        m, B, dev = self.m, q.shape[1], self.dev
        tq, tqd, tqdd = (torch.from_numpy(np.ascontiguousarray(a)).to(dev) for a in (q, qd, qdd))
        pose = torch.full((m.nb, 12, B), float("nan"), device=dev)
        J = torch.full((m.nframes, 6, m.nv, B), float("nan"), device=dev)
        tau = torch.full((m.nv, B), float("nan"), device=dev)
        M = torch.full((m.nv, m.nv, B), float("nan"), device=dev)
        s = torch.cuda.current_stream().cuda_stream
        n0 = binding.launch_count()
        m.fk(B, tq, pose, s)
        m.jacobian(B, tq, J, s)
        m.rnea(B, tq, tqd, tqdd, tau, s)
        m.crba(B, tq, M, s)
        torch.cuda.synchronize()
        assert binding.launch_count() - n0 == 4 or m.nv == 0 or m.nframes == 0   # one launch per operator
        return pose.cpu().numpy(), J.cpu().numpy(), tau.cpu().numpy(), M.cpu().numpy()

    def refs(self, q, qd, qdd):
        q64, qd64, qdd64 = (np.ascontiguousarray(a.astype(np.float64)) for a in (q, qd, qdd))
        J = self.o.jacobian(q64) if self.m.nframes else np.zeros((0, 6, self.m.nv, q.shape[1]))
        return self.o.fk(q64), J, self.o.rnea(q64, qd64, qdd64), self.o.crba(q64)

    def check(self, out, ref):
        for a in out:
            assert np.isfinite(a).all()
        for a, r, tol in zip(out, ref, (TOL_KIN, TOL_KIN, TOL_DYN, TOL_DYN)):
            assert nerr(a, r) <= tol
        assert np.array_equal(out[3], np.swapaxes(out[3], 0, 1))   # M written symmetric, bit for bit


@pytest.mark.gpu
@pytest.mark.parametrize("idx", range(10))
@pytest.mark.parametrize("B", [1, 37, 1000])
def test_specialized_operators_match_oracle(idx, B):
    desc = _robots()[idx]
    s = Spec(desc, spec_min_b=0)                                  # the specialised kernels at every batch size
    q, qd, qdd = W.sample_states(desc, B, seed=900 + idx)
    out = s.run(q, qd, qdd)
    ref = s.refs(q, qd, qdd)
    s.check(out, ref)                                             # RNEA here: limb roles where the tree branches
    s.m.set_option("spec_roles_max_b", 0)                         # RNEA and CRBA: one thread per environment
    s.m.set_option("spec_crba_roles_max_b", 0)
    out = s.run(q, qd, qdd)
    s.check(out, ref)
    # and the team kernels on the same inputs: same arithmetic up to the folded zeros
    s.m.set_option("spec_min_b", 1 << 30)
    team = s.run(q, qd, qdd)
    for a, b in zip(out, team):
        assert nerr(a, b.astype(np.float64)) <= 1e-4


@pytest.mark.gpu
@pytest.mark.parametrize("block", [0, 32, 96, 512])
@pytest.mark.parametrize("roles_max_b", [None, 0])
def test_specialized_block_sizes_and_ragged_tail(block, roles_max_b):
    """Any block size (a run-time value) and a batch that ends in the middle of a warp; RNEA with limb roles
    (the default at this batch size) and without."""
    opts = {"spec_min_b": 0, "spec_block": block}
    if roles_max_b is not None:
        opts.update(spec_roles_max_b=roles_max_b, spec_crba_roles_max_b=roles_max_b)
    desc = W.config_robot(3)
    s = Spec(desc, **opts)
    q, qd, qdd = W.config_states(3, 5000 + 13)
    s.check(s.run(q, qd, qdd), s.refs(q, qd, qdd))


@pytest.mark.gpu
@pytest.mark.parametrize("roles", [2, 3, 4])
@pytest.mark.parametrize("idx", range(10))
def test_limb_role_rnea_matches_oracle(roles, idx):
    """RNEA with the subtrees below the first branching body dealt to `roles` groups of warps: against the oracle,
    below the specialised regime too (its own rule), and it never runs above its batch limit."""
    desc = _robots()[idx]
    s = Spec(desc, ops=("rnea",), spec_roles=roles, spec_min_b=1 << 30)   # roles have their own regime
    dev = torch.device("cuda:0")
    try:
        branching = "role == 1u" in s.m.specialized_source("rnea_roles")
    except binding.BardError:
        branching = False                                         # a chain or a forest: no limb-role kernel
    assert branching == _single_root_and_branches(desc)
    for B in (1, 45, 700):
        q, qd, qdd = W.sample_states(desc, B, seed=1700 + idx)
        tq, tqd, tqdd = (torch.from_numpy(np.ascontiguousarray(a)).to(dev) for a in (q, qd, qdd))
        ref = s.o.rnea(*(np.ascontiguousarray(a.astype(np.float64)) for a in (q, qd, qdd)))
        got = {}
        for mx in (None, 0):
            s.m.set_option("spec_roles_max_b", -1 if mx is None else mx)   # -1: the library's own rule
            tau = torch.full((s.m.nv, B), float("nan"), device=dev)
            s.m.rnea(B, tq, tqd, tqdd, tau, torch.cuda.current_stream().cuda_stream)
            torch.cuda.synchronize()
            got[mx] = tau.cpu().numpy()
            assert np.isfinite(got[mx]).all()
            assert nerr(got[mx], ref) <= TOL_DYN
        if not branching:                                         # a chain: both calls ran the team kernel
            assert np.array_equal(got[None], got[0])


@pytest.mark.gpu
@pytest.mark.parametrize("roles", [2, 3])
@pytest.mark.parametrize("idx", range(10))
def test_limb_role_crba_matches_oracle(roles, idx):
    """CRBA with limb roles (composite inertias of the other roles' subtrees handed over in the world frame, rows of a
    subtree's DOFs against the trunk filled by the subtree's role): every entry of M written, symmetric bit for bit,
    against the oracle and against the one-thread-per-environment kernel."""
    desc = _robots()[idx]
    s = Spec(desc, ops=("crba",), spec_roles=roles, spec_min_b=0)
    dev = torch.device("cuda:0")
    try:
        branching = "role == 1u" in s.m.specialized_source("crba_roles")
    except binding.BardError:
        branching = False
    assert branching == _single_root_and_branches(desc)
    for B in (1, 45, 700):
        q, _, _ = W.sample_states(desc, B, seed=2700 + idx)
        tq = torch.from_numpy(np.ascontiguousarray(q)).to(dev)
        ref = s.o.crba(np.ascontiguousarray(q.astype(np.float64)))
        got = {}
        for mx in (1 << 30, 0):
            s.m.set_option("spec_crba_roles_max_b", mx)
            s.m.set_option("spec_crba_roles_min_b", 0)
            Mo = torch.full((s.m.nv, s.m.nv, B), float("nan"), device=dev)
            s.m.crba(B, tq, Mo, torch.cuda.current_stream().cuda_stream)
            torch.cuda.synchronize()
            got[mx] = Mo.cpu().numpy()
            assert np.isfinite(got[mx]).all()
            assert nerr(got[mx], ref) <= TOL_DYN
            assert np.array_equal(got[mx], np.swapaxes(got[mx], 0, 1))
        assert nerr(got[1 << 30], got[0].astype(np.float64)) <= 1e-4
        if not branching:
            assert np.array_equal(got[1 << 30], got[0])


@pytest.mark.gpu
@pytest.mark.parametrize("idx", [0, 1, 2, 4, 5, 7, 9])
def test_fused_step_matches_oracle_and_the_four_calls(idx):
    """bard_step: one fused kernel where it is built (small parked state), else the four operators; both against
    the oracle, and the fused outputs against the four specialised kernels bit for bit (same generated arithmetic)."""
    desc = _robots()[idx]
    s = Spec(desc, spec_min_b=0, spec_fused_max_rows=100000, step_mode=2)   # build the fused kernel for every robot here, use it at every B
    s.m.specialize(("fused",))
    q, qd, qdd = W.sample_states(desc, 700, seed=40 + idx)
    four = s.run(q, qd, qdd)
    m, B, dev = s.m, 700, s.dev
    tq, tqd, tqdd = (torch.from_numpy(np.ascontiguousarray(a)).to(dev) for a in (q, qd, qdd))
    outs = [torch.full(sh, float("nan"), device=dev) for sh in ((m.nb, 12, B), (m.nframes, 6, m.nv, B), (m.nv, B), (m.nv, m.nv, B))]
    n0 = binding.launch_count()
    m.step(B, tq, tqd, tqdd, *outs, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    assert binding.launch_count() - n0 == (1 if m.nv > 0 and m.nframes > 0 else 4) or m.nv == 0
    fused = [t.cpu().numpy() for t in outs]
    s.check(fused, s.refs(q, qd, qdd))
    for a, b in zip(fused, four):
        assert nerr(a, b.astype(np.float64)) <= 1e-5


@pytest.mark.gpu
@pytest.mark.parametrize("cfg,B", [(3, 1000), (2, 777), (3, 65536)])
def test_side_by_side_step_is_one_launch_and_bit_equal_to_the_four_kernels(cfg, B):
    """Where the fused kernel does not pay, bard_step is ONE launch of the four specialised operators side by side
    (blockIdx.y = operator): the same generated code, so the same bits as the four separate launches."""
    desc = W.config_robot(cfg)
    # never the fused kernel, at any batch size; build the side-by-side kernel for every robot here
    s = Spec(desc, spec_min_b=0, spec_fused_max_rows=0, spec_fused_small_b=0, spec_step4_max_rows=100000, spec_kin_min_b=1 << 40, step_mode=2)
    s.m.specialize(("fused",))
    q, qd, qdd = W.config_states(cfg, B)
    four = s.run(q, qd, qdd)
    m, dev = s.m, s.dev
    tq, tqd, tqdd = (torch.from_numpy(np.ascontiguousarray(a)).to(dev) for a in (q, qd, qdd))
    outs = [torch.full(sh, float("nan"), device=dev) for sh in ((m.nb, 12, B), (m.nframes, 6, m.nv, B), (m.nv, B), (m.nv, m.nv, B))]
    n0 = binding.launch_count()
    m.step(B, tq, tqd, tqdd, *outs, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    assert binding.launch_count() - n0 == 1
    for t, ref in zip(outs, four):
        assert np.array_equal(t.cpu().numpy(), ref)


@pytest.mark.gpu
@pytest.mark.parametrize("cfg,B", [(3, 1000), (2, 777), (1, 300), (3, 65536)])
@pytest.mark.parametrize("kin_fork", [1, 0])
def test_kinematics_fused_step_matches_oracle_and_the_four_kernels(cfg, B, kin_fork):
    """bard_step on the robots without a full fused kernel: FK + Jacobian + CRBA in ONE walk (they share q, poses and
    screws) + bard_rnea (on a side stream or after it): two launches, every output against the oracle and against the four
    separate specialised kernels (same generated expressions: equal to a few ulp)."""
    desc = W.config_robot(cfg)
    # never the full fused kernel / side-by-side grid; the kinematics kernel at every batch size
    s = Spec(desc, spec_min_b=0, spec_fused_max_rows=0, spec_fused_small_b=0, spec_step4=0, spec_kin_min_b=0, step_fork_max_b=0,
             step_kin_fork=kin_fork, spec_roles_max_b=0, spec_crba_roles_max_b=0)
    s.m.specialize(("fused",))
    assert "bard_kin_n1" in s.m.specialized_source("kin")
    q, qd, qdd = W.config_states(cfg, B)
    four = s.run(q, qd, qdd)
    m, dev = s.m, s.dev
    tq, tqd, tqdd = (torch.from_numpy(np.ascontiguousarray(a)).to(dev) for a in (q, qd, qdd))
    outs = [torch.full(sh, float("nan"), device=dev) for sh in ((m.nb, 12, B), (m.nframes, 6, m.nv, B), (m.nv, B), (m.nv, m.nv, B))]
    n0 = binding.launch_count()
    m.step(B, tq, tqd, tqdd, *outs, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    assert binding.launch_count() - n0 == 2
    got = [t.cpu().numpy() for t in outs]
    idx = np.arange(0, B, max(1, B // 500))
    ref = s.refs(*(a[:, idx] for a in (q, qd, qdd)))
    for a, r, tol in zip(got, ref, (TOL_KIN, TOL_KIN, TOL_DYN, TOL_DYN)):
        assert np.isfinite(a).all()
        assert nerr(a[..., idx], r) <= tol
    assert np.array_equal(got[3], np.swapaxes(got[3], 0, 1))
    for a, b in zip(got, four):
        assert nerr(a, b.astype(np.float64)) <= 1e-5
    assert np.array_equal(got[2], four[2])                         # tau: the very same RNEA kernel


@pytest.mark.gpu
def test_step_fork_regime_is_measured_at_specialisation():
    """Where bard_step stops forking: 256 x SMs without generated kernels; bard_model_specialize(BARD_OP_FUSED) then times
    both forms at B = 4096 on the device (margins on these two robots: 2x) -- or applies the static rule when told not to
    measure; an explicit step_fork_max_b always wins; bard_model_set_frames drops the measurement with the kernels."""
    sms = 148
    for cfg, want in ((3, 128 * sms), (0, 3072)):
        desc = W.config_robot(cfg)
        m = binding.Model(desc, device=0)
        assert m.get_option("step_fork_regime") == 256 * sms
        m.specialize(ALL + ("fused",))
        # measured: the humanoid's two-launch step loses by 2x at 4096 (never 3072) and by ~20 % at 16 384 (18 944; 8192 if a noisy box flips it)
        assert m.get_option("step_fork_regime") in ((want,) if cfg == 0 else (want, 8192))
        assert m.get_option("step_fork_regime_captured") >= max(8192, m.get_option("step_fork_regime"))
        m.set_option("step_fork_max_b", 1234)
        assert m.get_option("step_fork_regime") == 1234
        m.set_option("step_fork_max_b", -1)
        m.set_frames(desc.frame_body, desc.frame_offset)
        assert m.get_option("step_fork_regime") in (256 * sms, 128 * sms, 3072)       # the static rule on what is left
        m2 = binding.Model(desc, device=0)
        m2.set_option("step_calibrate", 0)
        m2.specialize(ALL + ("fused",))
        assert m2.get_option("step_fork_regime") == want                                # the static rule agrees on the BASELINE robots


@pytest.mark.gpu
@pytest.mark.parametrize("cfg,B,specialised", [(3, 65536, True), (3, 1000, True), (1, 300, False), (2, 40000, True), (2, 5000, True), (2, 3000, True),
                                               (3, 20000, True), (3, 10000, True)])
def test_bard_kinematics_matches_oracle(cfg, B, specialised):
    """bard_kinematics: pose, J and M of one batch -- one launch of the kinematics-fused kernel where it exists and the
    batch is in its regime, bard_fk + bard_jacobian + bard_crba otherwise; either way the three operators' results."""
    desc = W.config_robot(cfg)
    m = binding.Model(desc, device=0)
    if specialised:
        m.specialize(ALL + ("fused",))
    o = oracle.Oracle(desc)
    dev = torch.device("cuda:0")
    q, _, _ = W.config_states(cfg, B)
    tq = torch.from_numpy(q).to(dev)
    outs = [torch.full(sh, float("nan"), device=dev) for sh in ((m.nb, 12, B), (m.nframes, 6, m.nv, B), (m.nv, m.nv, B))]
    n0 = binding.launch_count()
    m.kinematics(B, tq, *outs, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    # one launch above bard_step's fork regime (measured at specialisation: 3072 for the spined quadruped, 128 x SMs for the humanoid)
    one = specialised and cfg != 1 and B > m.get_option("step_fork_regime") and "bard_kin_n1" in m.specialized_source("kin")
    if specialised and cfg in (2, 3):
        assert m.get_option("step_fork_regime") in (3072, 8192, 128 * 148)
    assert binding.launch_count() - n0 == (1 if one else 3)
    idx = np.unique(np.concatenate([np.arange(0, B, max(1, B // 400)), [B - 1]]))
    q64 = np.ascontiguousarray(q[:, idx].astype(np.float64))
    for t, r, tol in zip(outs, (o.fk(q64), o.jacobian(q64), o.crba(q64)), (TOL_KIN, TOL_KIN, TOL_DYN)):
        a = t.cpu().numpy()
        assert np.isfinite(a).all()
        assert nerr(a[..., idx], r) <= tol


@pytest.mark.gpu
def test_step_without_specialisation_is_the_four_team_kernels():
    desc = W.config_robot(1)
    m = binding.Model(desc, device=0)
    o = oracle.Oracle(desc)
    B = 300
    q, qd, qdd = W.config_states(1, B)
    dev = torch.device("cuda:0")
    tq, tqd, tqdd = (torch.from_numpy(a).to(dev) for a in (q, qd, qdd))
    outs = [torch.full(sh, float("nan"), device=dev) for sh in ((m.nb, 12, B), (m.nframes, 6, m.nv, B), (m.nv, B), (m.nv, m.nv, B))]
    n0 = binding.launch_count()
    m.step(B, tq, tqd, tqdd, *outs, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    assert binding.launch_count() - n0 == 4
    q64, qd64, qdd64 = (a.astype(np.float64) for a in (q, qd, qdd))
    for t, r, tol in zip(outs, (o.fk(q64), o.jacobian(q64), o.rnea(q64, qd64, qdd64), o.crba(q64)), (TOL_KIN, TOL_KIN, TOL_DYN, TOL_DYN)):
        assert nerr(t.cpu().numpy(), r) <= tol


@pytest.mark.gpu
def test_specialized_max_size_tree_and_single_fixed_body():
    """The compiled limits (64 bodies, 16 frames) and the degenerate model (one fixed body: no q, no DOF)."""
    desc = W.random_tree(4242, nb=64, shape="random", nframes=16)
    s = Spec(desc, spec_min_b=0)
    q, qd, qdd = W.sample_states(desc, 96, seed=5)
    s.check(s.run(q, qd, qdd), s.refs(q, qd, qdd))
    one = W.build_robot("one_fixed", [-1], [W.FIXED], seed=1)
    m = binding.Model(one, device=0)
    m.set_option("spec_min_b", 0)
    m.specialize(ALL + ("fused",))
    pose = torch.full((1, 12, 8), float("nan"), device="cuda:0")
    n0 = binding.launch_count()
    m.fk(8, None, pose, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    assert binding.launch_count() - n0 == 1
    assert nerr(pose.cpu().numpy(), oracle.Oracle(one).fk(np.zeros((0, 8)))) <= TOL_KIN


@pytest.mark.gpu
def test_specialized_jacobian_follows_set_frames():
    desc = W.config_robot(3)
    s = Spec(desc, spec_min_b=0)
    q, qd, qdd = W.config_states(3, 257)
    s.check(s.run(q, qd, qdd), s.refs(q, qd, qdd))
    desc.frame_body = [5, 23, 14]                                  # new frames: team kernel until specialised again
    desc.frame_offset = [[0.1, 0.0, -0.2], [0.0, 0.0, 0.0], [0.0, 0.3, 0.0]]
    s.m.set_frames(desc.frame_body, desc.frame_offset)
    s.o = oracle.Oracle(desc)
    s.check(s.run(q, qd, qdd), s.refs(q, qd, qdd))
    s.m.specialize(("jacobian",))
    assert "frame 2 on body 14" in s.m.specialized_source("jacobian")
    s.check(s.run(q, qd, qdd), s.refs(q, qd, qdd))


@pytest.mark.gpu
@pytest.mark.parametrize("cfg,B", [(3, 65536), (1, 65536), (2, 65536), (0, 1048576), (3, 262144), (3, 1048576), (1, 1048576),
                                   (2, 1048576), (0, 65536), (0, 262144)])
def test_specialized_full_size_sampled(cfg, B):
    """bench.py's launch configuration (default knobs, every size of BASELINE.json's sweep from 65 536 up, where the
    launch rule changes: one wave of 448-thread CTAs -> multi-wave 256-thread CTAs and the RNEA variant without L2
    prefetch): a strided sample of environments against the oracle, every output element finite, repeat bit-identical.
    The outputs stay on the device (7.7 GB for the humanoid at 1 Mi); only the sampled columns come to the host."""
    desc = W.config_robot(cfg)
    s = Spec(desc)
    q, qd, qdd = W.config_states(cfg, B)
    out = s.run_dev(q, qd, qdd)
    # the sample: a stride that is coprime to the warp / CTA sizes, the ragged ends, CTA boundaries of both launch shapes
    idx = np.unique(np.concatenate([np.arange(0, B, max(1, B // 997)), [B - 1, B - 2, 127, 128, 255, 256, 447, 448, B // 2]]))
    ref = s.refs(*(a[:, idx] for a in (q, qd, qdd)))
    tidx = torch.from_numpy(idx).to(s.dev)
    for a in out:
        assert bool(torch.isfinite(a).all())
    for a, r, tol in zip(out, ref, (TOL_KIN, TOL_KIN, TOL_DYN, TOL_DYN)):
        assert nerr(a.index_select(a.dim() - 1, tidx).cpu().numpy(), r) <= tol
    assert bool(torch.equal(out[3], out[3].transpose(0, 1)))       # M symmetric bit for bit, all B environments
    cs = [a.view(torch.int32).sum(dtype=torch.int64).item() for a in out]   # bit pattern checksums: a repeat must match
    again = s.run_dev(q, qd, qdd)
    for a, b, c in zip(out, again, cs):
        assert b.view(torch.int32).sum(dtype=torch.int64).item() == c   # no atomics, fixed child order
        if a.numel() < (1 << 28):
            assert bool(torch.equal(a, b))


def wide_states(desc, B, seed):
    """Revolute angles far outside (-pi, pi) (continuous joints wind up): U(-200 pi, 200 pi), and in the first
    environments exact multiples of pi/2, +-1e4 rad, +-1e5 rad -- the range reduction of the kernels' own sincos
    runs with every quadrant and large k (reading 16)."""
    q, qd, qdd = W.sample_states(desc, B, seed=seed)
    rng = np.random.default_rng(seed + 1)
    special = np.array([0.0, np.pi / 2, -np.pi / 2, np.pi, -np.pi, 1.5 * np.pi, 2 * np.pi, 100 * np.pi, -99.5 * np.pi, 1e4, -1e4, 1e5, -1e5,
                        12345.678, -54321.0, 200 * np.pi], np.float64)
    qo = desc.q_off
    for i, t in enumerate(desc.joint_type):
        if int(t) == W.REVOLUTE:
            row = rng.uniform(-200 * np.pi, 200 * np.pi, size=B)
            k = min(B, len(special))
            row[:k] = np.roll(special, i)[:k]
            q[qo[i]] = row.astype(np.float32)
    return q, qd, qdd


@pytest.mark.gpu
@pytest.mark.parametrize("idx", range(10))
def test_wide_angles_both_kernel_families(idx):
    """every other parity input is U(-pi, pi); here the hand-written sincos (3-step Cody-Waite
    reduction) sees |q| up to 1e5 in the team kernels, the specialised kernels and the limb-role kernels."""
    desc = _robots()[idx]
    s = Spec(desc, spec_min_b=0)
    for B in (1000, 37):
        q, qd, qdd = wide_states(desc, B, seed=5100 + idx)
        ref = s.refs(q, qd, qdd)
        s.m.set_option("spec_min_b", 0)
        s.m.set_option("spec_roles_max_b", -1)
        s.m.set_option("spec_crba_roles_max_b", -1)
        s.check(s.run(q, qd, qdd), ref)                            # specialised, limb roles where the tree branches
        s.m.set_option("spec_roles_max_b", 0)
        s.m.set_option("spec_crba_roles_max_b", 0)
        s.check(s.run(q, qd, qdd), ref)                            # specialised, one thread per environment
        s.m.set_option("spec_min_b", 1 << 30)
        s.check(s.run(q, qd, qdd), ref)                            # team kernels
        s.m.set_option("pack", 2)
        s.check(s.run(q, qd, qdd), ref)                            # team kernels, two environments per lane (packed sincos)
        s.m.set_option("pack", 0)


@pytest.mark.gpu
@pytest.mark.parametrize("family", ["team", "team_pack2", "specialised"])
def test_sincos_of_the_kernels_against_fp64(family):
    """The kernels' own sincos, isolated: FK of ONE revolute joint about z with T_pre = I gives R = Rz(q), so
    pose[3] = R10 = 0 + sin q * 1 is the kernel's sine bit for bit and pose[0] = R00 = 1 - (1 - cos q) its cosine after
    two roundings of at most half an ulp of 1 each (6e-8 + 6e-8).  Claim (reading 16): |error| <= 9.4e-8 for
    |q| <= 1e6 rad.  Checked over 2 Mi angles: uniform in +-1e5, log-uniform magnitudes down to 1e-6, and a comb around
    every multiple of pi/2 up to 2000 pi (where a wrong reduction constant shows first)."""
    B = 1 << 21
    rng = np.random.default_rng(99)
    n = B // 4
    comb = (np.arange(n) % 4001 - 2000)[:, None] * (np.pi / 2) + rng.uniform(-1e-3, 1e-3, size=(n, 1))
    q = np.concatenate([rng.uniform(-1e5, 1e5, size=n), rng.uniform(-np.pi, np.pi, size=n),
                        np.sign(rng.normal(size=n)) * 10.0 ** rng.uniform(-6, 6, size=n), comb[:, 0]]).astype(np.float32)[None, :]
    T = np.zeros((1, 12)); T[0, 0] = T[0, 5] = T[0, 10] = 1.0
    desc = W.RobotDesc(name="rz", parent=np.array([-1], np.int32), joint_type=np.array([W.REVOLUTE], np.int32),
                       axis=np.array([[0.0, 0.0, 1.0]]), T_pre=T, T_post=None, mass=np.array([1.0]), com=np.zeros((1, 3)),
                       inertia=np.array([[1.0, 0, 0, 1.0, 0, 1.0]]))
    m = binding.Model(desc, device=0)
    if family == "specialised":
        m.set_option("spec_min_b", 0)
        m.specialize(("fk",))
    elif family == "team_pack2":
        m.set_option("pack", 2)
    dev = torch.device("cuda:0")
    pose = torch.full((1, 12, B), float("nan"), device=dev)
    m.fk(B, torch.from_numpy(q).to(dev), pose, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    p = pose.cpu().numpy().astype(np.float64)[0]
    q64 = q[0].astype(np.float64)
    assert np.max(np.abs(p[3] - np.sin(q64))) <= 9.4e-8            # R10 = sin q
    assert np.max(np.abs(p[1] + np.sin(q64))) <= 9.4e-8            # R01 = -sin q
    assert np.max(np.abs(p[0] - np.cos(q64))) <= 9.4e-8 + 1.2e-7   # R00 = 1 - (1 - cos q)
    assert np.max(np.abs(p[4] - np.cos(q64))) <= 9.4e-8 + 1.2e-7
    assert np.array_equal(p[8], np.ones(B)) and not p[[2, 5, 6, 7, 9, 10, 11]].any()


@pytest.mark.gpu
@pytest.mark.parametrize("cfg", [1, 3])
def test_rnea_variant_without_l2_prefetch_matches(cfg):
    """Grids beyond two CTAs per SM run the RNEA variant without the L2 prefetch (here forced with 32-thread CTAs):
    same arithmetic, so bit-identical to the prefetching variant, and within tolerance of the oracle."""
    desc = W.config_robot(cfg)
    s = Spec(desc, ops=("rnea",), spec_min_b=0, spec_roles_max_b=0)
    B = 32 * 2 * 148 + 32 * 40 + 7                                 # > 2 x SMs CTAs of 32 threads, ragged tail
    q, qd, qdd = W.sample_states(desc, B, seed=4242 + cfg)
    o = s.o
    ref = o.rnea(q.astype(np.float64), qd.astype(np.float64), qdd.astype(np.float64))
    tq, tqd, tqdd = (torch.from_numpy(np.ascontiguousarray(a)).to(s.dev) for a in (q, qd, qdd))
    taus = []
    for block in (32, 512):                                        # 337 CTAs (no prefetch) / 22 CTAs (prefetch)
        s.m.set_option("spec_block", block)
        tau = torch.full((s.m.nv, B), float("nan"), device=s.dev)
        s.m.rnea(B, tq, tqd, tqdd, tau, torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
        taus.append(tau.cpu().numpy())
        assert nerr(taus[-1], ref) <= TOL_DYN
    assert np.array_equal(taus[0], taus[1])


def test_cubin_disk_cache_round_trip(tmp_path, monkeypatch):
    """NVRTC output is cached on disk under $BARD_CACHE_DIR, keyed by hashes of (register cap, source): a second process
    loads the file instead of compiling; a corrupt file is ignored (compiled again); BARD_CACHE=0 writes nothing."""
    import subprocess
    import sys
    import time
    code = ("import time, sys; sys.path.insert(0, %r)\n"
            "from paper_2605_31481_b200 import binding, workloads as W\n"
            "m = binding.Model(W.config_robot(1), device=-1)\n"
            "t = time.perf_counter(); m.specialize(('crba',)); print(time.perf_counter() - t)\n") % ROOT
    env = dict(os.environ, BARD_CACHE="1", BARD_CACHE_DIR=str(tmp_path / "c"))
    t1 = float(subprocess.run([sys.executable, "-c", code], env=env, capture_output=True, text=True, check=True).stdout.split()[-1])
    files = sorted((tmp_path / "c").glob("*.cubin"))
    assert len(files) >= 1
    t2 = float(subprocess.run([sys.executable, "-c", code], env=env, capture_output=True, text=True, check=True).stdout.split()[-1])
    assert t2 < 0.5 * t1                                           # no NVRTC run the second time
    for f in files:
        f.write_bytes(b"garbage")                                  # a damaged file: compile again, replace it
    subprocess.run([sys.executable, "-c", code], env=env, capture_output=True, text=True, check=True)
    assert all(f.stat().st_size > 1000 for f in (tmp_path / "c").glob("*.cubin"))
    env0 = dict(env, BARD_CACHE="0", BARD_CACHE_DIR=str(tmp_path / "off"))
    subprocess.run([sys.executable, "-c", code], env=env0, capture_output=True, text=True, check=True)
    assert not (tmp_path / "off").exists()
