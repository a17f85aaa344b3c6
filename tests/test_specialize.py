"""Model-specialised kernels (bard_model_specialize): host-side generation + NVRTC compilation on CPU, and GPU
parity of the generated RNEA against the fp64 oracle and against the level-parallel team kernel."""
import re

import numpy as np
import pytest

import oracle
from paper_2605_31481_b200 import binding, workloads as W

TOL_DYN = 1e-3


def nerr(x, ref):
    return float(np.max(np.abs(x.astype(np.float64) - ref) / np.maximum(1.0, np.abs(ref)))) if ref.size else 0.0


def _robots():
    out = [W.config_robot(c) for c in range(4)]
    for seed in range(6):
        shape = ["random", "chain", "star", "unbalanced"][seed % 4]
        out.append(W.random_tree(500 + seed, nb=2 + 4 * seed, shape=shape, free_root=(seed % 2 == 0)))
    return out


# ------------------------------------------------------------------------------------------- CPU (no GPU needed)
@pytest.mark.parametrize("idx", range(10))
def test_generated_source_compiles_on_host(idx):
    """A host-only model: the source is generated and NVRTC-compiled for sm_100a, nothing is loaded."""
    desc = _robots()[idx]
    m = binding.Model(desc, device=-1)
    m.specialize(("rnea",))
    src = m.specialized_source("rnea")
    assert 'extern "C" __global__' in src and "bard_rnea_n1" in src
    # one outward and one inward section per body, every tau row stored exactly once
    assert len(re.findall(r"// ---- body \d+ \(outward\)", src)) == m.nb
    assert len(re.findall(r"// ---- body \d+ \(inward\)", src)) == m.nb
    rows = sorted(int(r) for r in re.findall(r"strow\(tau, (\d+)u \* B \+ e", src))
    assert rows == list(range(m.nv))
    # every input row is loaded exactly once
    for arr, n in (("q", m.nq), ("qd", m.nv), ("qdd", m.nv)):
        got = sorted(int(r) for r in re.findall(r"ldrow<T>\(%s, (\d+)u \* B \+ e\)" % arr, src))
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


def test_unsupported_operator_bits_are_refused():
    m = binding.Model(W.config_robot(0), device=-1)
    with pytest.raises(binding.BardError) as e:
        m.specialize(("fk",))
    assert e.value.code == 3
    with pytest.raises(binding.BardError):
        m.specialized_source("rnea")                              # not specialised yet


# ------------------------------------------------------------------------------------------- GPU
torch = pytest.importorskip("torch")


class Spec:
    def __init__(self, desc):
        assert torch.cuda.is_available(), "GPU tests need CUDA; there is no CPU fallback"
        self.m = binding.Model(desc, device=0)
        self.m.specialize(("rnea",))
        self.o = oracle.Oracle(desc)
        self.dev = torch.device("cuda:0")

    def rnea(self, q, qd, qdd):
        m, B = self.m, q.shape[1]
        t = [torch.from_numpy(np.ascontiguousarray(a)).to(self.dev) for a in (q, qd, qdd)]
        tau = torch.full((m.nv, B), float("nan"), device=self.dev)
        n0 = binding.launch_count()
        m.rnea(B, *t, tau, torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
        assert binding.launch_count() - n0 == 1
        return tau.cpu().numpy()


@pytest.mark.gpu
@pytest.mark.parametrize("idx", range(10))
@pytest.mark.parametrize("B", [1, 37, 1000])
def test_specialized_rnea_matches_oracle(idx, B, monkeypatch):
    monkeypatch.setenv("BARD_SPEC_MIN_B", "0")                    # the specialised kernel at every batch size
    desc = _robots()[idx]
    s = Spec(desc)
    q, qd, qdd = W.sample_states(desc, B, seed=900 + idx)
    tau = s.rnea(q, qd, qdd)
    assert np.isfinite(tau).all()
    ref = s.o.rnea(*(a.astype(np.float64) for a in (q, qd, qdd)))
    assert nerr(tau, ref) <= TOL_DYN
    # and the team kernel on the same inputs: same arithmetic up to the folded zeros
    monkeypatch.setenv("BARD_SPEC_MIN_B", str(1 << 30))
    team = s.rnea(q, qd, qdd)
    assert nerr(tau, team.astype(np.float64)) <= 1e-4


@pytest.mark.gpu
@pytest.mark.parametrize("block", [0, 32, 96, 512])
def test_specialized_rnea_block_sizes_and_ragged_tail(block, monkeypatch):
    """Any block size (a run-time value) and a batch that ends in the middle of a warp."""
    monkeypatch.setenv("BARD_SPEC_MIN_B", "0")
    if block:
        monkeypatch.setenv("BARD_SPEC_BLOCK", str(block))
    desc = W.config_robot(3)
    s = Spec(desc)
    q, qd, qdd = W.config_states(3, 5000 + 13)
    ref = s.o.rnea(*(a.astype(np.float64) for a in (q, qd, qdd)))
    assert nerr(s.rnea(q, qd, qdd), ref) <= TOL_DYN


@pytest.mark.gpu
@pytest.mark.parametrize("cfg,B", [(3, 65536), (1, 65536), (0, 1048576)])
def test_specialized_rnea_full_size_sampled(cfg, B):
    """bench.py's launch configuration (default knobs): a strided sample of environments against the oracle."""
    desc = W.config_robot(cfg)
    s = Spec(desc)
    q, qd, qdd = W.config_states(cfg, B)
    tau = s.rnea(q, qd, qdd)
    assert np.isfinite(tau).all()
    idx = np.unique(np.concatenate([np.arange(0, B, max(1, B // 997)), [B - 1, B - 2, 127, 128, B // 2]]))
    ref = s.o.rnea(*(np.ascontiguousarray(a[:, idx].astype(np.float64)) for a in (q, qd, qdd)))
    assert nerr(tau[:, idx], ref) <= TOL_DYN
    again = s.rnea(q, qd, qdd)
    assert np.array_equal(tau, again)                              # no atomics, fixed child order
