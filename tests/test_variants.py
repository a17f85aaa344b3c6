"""the fp64 instantiation and the batch-first (AoS) adaptor of the four operators (bard_*_v).

fp64: the generated kernels typed on double with the builder's unrounded constants -- held to <= 1e-11 against the fp64
oracle on the BASELINE robots, the paper's own way of validating (Table 1: 1000 random configurations
per robot, max |delta| between two fp64 implementations).  AoS: the paper's batch-first layout, served by
tiled transposes around the SoA kernels -- bit-equal to the SoA call after a transpose, for every kernel family."""
import re

import numpy as np
import pytest

import oracle
from paper_2605_31481_b200 import binding, workloads as W

ALL = ("fk", "jacobian", "rnea", "crba")
VARIANTS = [("f64", "soa"), ("f64", "aos"), ("f32", "aos")]


def nerr(x, ref):
    return float(np.max(np.abs(x.astype(np.float64) - ref) / np.maximum(1.0, np.abs(ref)))) if ref.size else 0.0


def _robots():
    out = [W.config_robot(c) for c in range(4)]
    for seed in range(4):
        shape = ["random", "chain", "star", "unbalanced"][seed % 4]
        out.append(W.random_tree(900 + seed, nb=3 + 4 * seed, shape=shape, free_root=(seed % 2 == 0), nframes=3))
    return out


# ------------------------------------------------------------------------------------------- CPU
@pytest.mark.parametrize("idx", [0, 3, 5, 6])
def test_fp64_sources_compile_on_host_and_cover_every_row(idx):
    desc = _robots()[idx]
    m = binding.Model(desc, device=-1)
    m.specialize_variant(ALL, "f64", "soa")
    for op, arr, n in (("fk", "pose", 12 * m.nb), ("crba", "Mo", m.nv * m.nv), ("jacobian", "J", 6 * m.nframes * m.nv), ("rnea", "tau", m.nv)):
        src = m.variant_source(op, "f64", "soa")
        assert "typedef double real;" in src and "#define REAL_F64 1" in src
        rows = sorted(int(r) for r in re.findall(r"STROW\(%s, (\d+)u," % arr, src))
        assert rows == list(range(n)), op
        body = src[src.index("op_body_"):]                       # no float literal may survive in an fp64 kernel body
        assert not re.search(r"\d\.\d+(e[-+]?\d+)?f\b", body.replace("T(0.0f)", "").replace("T(1.0f)", ""))
    with pytest.raises(binding.BardError):
        m.specialize_variant(("aba",), "f64", "soa")             # only the four operators have variants
    with pytest.raises(binding.BardError):
        m.fk_v("f64", "soa", 4, 1, 1)                            # host-only model: operators refuse to run
    assert m.variant_workspace_bytes("crba", "f64", "soa", 100) == 0
    assert m.variant_workspace_bytes("crba", "f64", "aos", 100) >= 8 * 100 * (m.nq + m.nv * m.nv)
    assert m.variant_workspace_bytes("rnea", "f32", "aos", 100) >= 4 * 100 * (m.nq + 3 * m.nv)


def test_set_frames_and_set_inertial_params_drop_the_dependent_variants():
    m = binding.Model(W.config_robot(0), device=-1)
    m.specialize_variant(ALL, "f64", "soa")
    m.set_frames([2])
    with pytest.raises(binding.BardError):
        m.variant_source("jacobian", "f64", "soa")
    m.variant_source("rnea", "f64", "soa")
    m.set_inertial_params(m.inertial_params() * 1.1)
    with pytest.raises(binding.BardError):
        m.variant_source("rnea", "f64", "soa")
    m.variant_source("fk", "f64", "soa")                         # kinematics do not depend on either


# ------------------------------------------------------------------------------------------- GPU
torch = pytest.importorskip("torch")


class Var:
    def __init__(self, desc, dtype, layout, specialise=False):
        assert torch.cuda.is_available(), "GPU tests need CUDA; there is no CPU fallback"
        self.m = binding.Model(desc, device=0)
        if dtype == "f64" or specialise:
            self.m.set_option("spec_min_b", 0)
            self.m.specialize_variant(ALL, dtype, layout)
        self.dtype, self.layout = dtype, layout
        self.td = torch.float64 if dtype == "f64" else torch.float32
        self.dev = torch.device("cuda:0")

    def run(self, q, qd, qdd):
        """Inputs SoA numpy [rows, B]; returns SoA numpy outputs whatever the device layout was."""
        m, B, dev, td = self.m, q.shape[1], self.dev, self.td
        aos = self.layout == "aos"

        def up(a):
            t = torch.from_numpy(np.ascontiguousarray(a)).to(dev).to(td)
            return t.t().contiguous() if aos else t

        tq, tqd, tqdd = up(q), up(qd), up(qdd)
        shapes = ((m.nb, 12), (m.nframes, 6, m.nv), (m.nv,), (m.nv, m.nv))
        outs = [torch.full(((B,) + sh) if aos else (sh + (B,)), float("nan"), device=dev, dtype=td) for sh in shapes]
        s = torch.cuda.current_stream().cuda_stream
        ws = torch.full((max(m.variant_workspace_bytes(op, self.dtype, self.layout, B) for op in ALL) // 8 + 1,), float("nan"),
                        device=dev, dtype=torch.float64)
        n0 = binding.launch_count()
        m.fk_v(self.dtype, self.layout, B, tq, outs[0], ws, s)
        m.jacobian_v(self.dtype, self.layout, B, tq, outs[1], ws, s)
        m.rnea_v(self.dtype, self.layout, B, tq, tqd, tqdd, outs[2], ws, s)
        m.crba_v(self.dtype, self.layout, B, tq, outs[3], ws, s)
        torch.cuda.synchronize()
        # SoA: one launch per operator; AoS: + one transpose per input array and one for the output
        assert binding.launch_count() - n0 == (4 + 6 + 4 if aos else 4) or m.nv == 0 or m.nframes == 0 or m.nq == 0
        res = []
        for t in outs:
            a = t.cpu().numpy()
            res.append(np.moveaxis(a, 0, -1) if aos else a)
        return res


def refs(o, q, qd, qdd):
    q64, qd64, qdd64 = (np.ascontiguousarray(a.astype(np.float64)) for a in (q, qd, qdd))
    J = o.jacobian(q64) if o.nframes else np.zeros((0, 6, o.nv, q.shape[1]))
    return o.fk(q64), J, o.rnea(q64, qd64, qdd64), o.crba(q64)


@pytest.mark.gpu
@pytest.mark.parametrize("layout", ["soa", "aos"])
@pytest.mark.parametrize("idx", range(8))
def test_fp64_kernels_against_the_oracle(idx, layout):
    """fp64 GPU vs fp64 oracle: two correct double implementations agree to 1e-15 ... 5e-13 in the paper's Table 1
    (PAPER.md:109-114); the bar here is 1e-11 per element, normalised -- 10^7 times sharper than the fp32 tolerances."""
    desc = _robots()[idx]
    v = Var(desc, "f64", layout)
    o = oracle.Oracle(desc)
    for B in (1, 37, 1000):
        q, qd, qdd = W.sample_states(desc, B, seed=600 + idx, dtype=np.float64)
        out = v.run(q, qd, qdd)
        for a, r in zip(out, refs(o, q, qd, qdd)):
            assert np.isfinite(a).all()
            assert nerr(a, r) <= 1e-11
        assert np.array_equal(out[3], np.swapaxes(out[3], 0, 1))


@pytest.mark.gpu
@pytest.mark.parametrize("cfg", [0, 1, 2, 3])
def test_table1_style_fp64_agreement(cfg):
    """The paper's protocol: 1000 random configurations per robot, fp64, max absolute discrepancy per
    operator -- against our oracle instead of Pinocchio.  Bars: the paper's own Table 1 rows (FK 1.3e-15, Jacobian
    3.1e-15, RNEA 5.1e-13, CRBA 1.4e-14, tests/golden/paper_table1.txt) times 20, to allow for different robots."""
    desc = W.config_robot(cfg)
    v = Var(desc, "f64", "soa")
    o = oracle.Oracle(desc)
    q, qd, qdd = W.sample_states(desc, 1000, seed=1234 + cfg, dtype=np.float64)
    out = v.run(q, qd, qdd)
    ref = refs(o, q, qd, qdd)
    d = [float(np.max(np.abs(a - r))) for a, r in zip(out, ref)]
    print(f"config {cfg}: max |delta| FK {d[0]:.2e} Jacobian {d[1]:.2e} RNEA {d[2]:.2e} CRBA {d[3]:.2e}")
    assert d[0] <= 20 * 1.3e-15 and d[1] <= 20 * 3.1e-15 and d[2] <= 20 * 5.1e-13 and d[3] <= 20 * 1.4e-14


@pytest.mark.gpu
@pytest.mark.parametrize("specialise", [False, True])
@pytest.mark.parametrize("idx", range(8))
def test_aos_fp32_matches_oracle_and_is_bit_equal_to_soa(idx, specialise):
    """The batch-first layout needs no kernels of its own: team kernels (no NVRTC) and specialised kernels alike."""
    desc = _robots()[idx]
    v = Var(desc, "f32", "aos", specialise=specialise)
    o = oracle.Oracle(desc)
    dev = torch.device("cuda:0")
    for B in (1, 45, 1000 + 7):
        q, qd, qdd = W.sample_states(desc, B, seed=640 + idx)
        out = v.run(q, qd, qdd)
        for a, r, tol in zip(out, refs(o, q, qd, qdd), (1e-4, 1e-4, 1e-3, 1e-3)):
            assert np.isfinite(a).all()
            assert nerr(a, r) <= tol
        tq, tqd, tqdd = (torch.from_numpy(a).to(dev) for a in (q, qd, qdd))
        m = v.m
        ref = [torch.empty(sh + (B,), device=dev) for sh in ((m.nb, 12), (m.nframes, 6, m.nv), (m.nv,), (m.nv, m.nv))]
        s = torch.cuda.current_stream().cuda_stream
        m.fk(B, tq, ref[0], s); m.jacobian(B, tq, ref[1], s); m.rnea(B, tq, tqd, tqdd, ref[2], s); m.crba(B, tq, ref[3], s)
        torch.cuda.synchronize()
        for a, r in zip(out, ref):
            assert np.array_equal(a, r.cpu().numpy())              # the same kernels behind two transposes


@pytest.mark.gpu
@pytest.mark.parametrize("dtype,layout", VARIANTS)
def test_variants_at_bench_size_sampled(dtype, layout):
    """Humanoid at B = 65 536 through every variant: a strided sample against the oracle, every element finite."""
    desc = W.config_robot(3)
    B = 65536
    v = Var(desc, dtype, layout, specialise=True)
    o = oracle.Oracle(desc)
    q, qd, qdd = W.sample_states(desc, B, seed=2003, dtype=np.float64 if dtype == "f64" else np.float32)
    out = v.run(q, qd, qdd)
    idx = np.unique(np.concatenate([np.arange(0, B, B // 499), [B - 1, 255, 256]]))
    tols = (1e-11,) * 4 if dtype == "f64" else (1e-4, 1e-4, 1e-3, 1e-3)
    for a, r, tol in zip(out, refs(o, q[:, idx], qd[:, idx], qdd[:, idx]), tols):
        assert np.isfinite(a).all()
        assert nerr(a[..., idx], r) <= tol


@pytest.mark.gpu
def test_variant_call_without_its_kernel_is_refused():
    m = binding.Model(W.config_robot(0), device=0)
    t = torch.zeros(64, device="cuda:0", dtype=torch.float64)
    with pytest.raises(binding.BardError) as e:
        m.fk_v("f64", "soa", 4, t, t)
    assert e.value.code == 3
    with pytest.raises(binding.BardError) as e:
        m.fk_v("f32", "aos", 4, t, t)                            # AoS without a workspace
    assert e.value.code == 1
