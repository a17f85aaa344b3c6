"""bard_rnea_vjp_params_static: the RNEA VJP for callers that cannot allocate device memory (scratch in a static device
array of the library) against the existing path, bard_rnea_vjp_params with a caller-owned workspace.

Collected last on purpose (the suite runs with ``pytest -x``); passes alone in a fresh process and after the other tests.
"""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from paper_2605_31481_b200 import binding, workloads as W

TOL = 1e-3        # tests/test_rnea_vjp.py: per element |g - ref| / max(1, |ref|)


def nerr(x, ref):
    return float(np.max(np.abs(np.asarray(x, np.float64) - ref) / np.maximum(1.0, np.abs(ref)))) if ref.size else 0.0


def _inputs(desc, B, seed, dev):
    q, qd, qdd = W.sample_states(desc, B, seed=seed)
    dtau = np.random.default_rng(seed).normal(size=(desc.nv, B)).astype(np.float32)
    return [torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).to(dev) for a in (q, qd, qdd, dtau)]


@pytest.mark.gpu
@pytest.mark.parametrize("cfg,generated", [(0, False), (3, False), (3, True)])
def test_static_scratch_vjp_matches_the_workspace_path_on_two_calls_in_a_row(cfg, generated):
    dev = torch.device("cuda:0")
    desc = W.config_robot(cfg)
    m = binding.Model(desc, device=0)
    if generated:
        m.specialize(("rnea_vjp",))          # both entry points then run the generated kernel
    stream = torch.cuda.current_stream().cuda_stream
    # two different calls in a row on one stream: a large batch (every CTA's partials used), then a small ragged one (the
    # array still holds the first call's partials beyond the second call's grid: they must not be read)
    calls = [(65536 + 13, 7), (1000, 8)]
    data = [(_inputs(desc, B, seed, dev), B) for B, seed in calls]
    refs = []
    for t, B in data:
        ws = torch.full((max(1, m.rnea_vjp_workspace_floats(B)),), float("nan"), device=dev)
        g = torch.full((m.nb, 10), float("nan"), device=dev)
        m.rnea_vjp_params(B, *t, g, ws, stream)
        refs.append(g)
    torch.cuda.synchronize()
    outs = [torch.full((m.nb, 10), float("nan"), device=dev) for _ in data]
    m.rnea_vjp_params_static(1, *[x[:, :1].contiguous() for x in data[1][0]], torch.empty((m.nb, 10), device=dev), stream)   # set-up: symbol lookup
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    n0 = binding.launch_count()
    for (t, B), g in zip(data, outs):
        m.rnea_vjp_params_static(B, *t, g, stream)
    torch.cuda.synchronize()
    assert binding.launch_count() - n0 == 4                                  # the same two kernels per call
    assert torch.cuda.mem_get_info()[0] == free0                             # nothing was allocated on the device
    for g, r in zip(outs, refs):
        a, b = g.cpu().numpy(), r.cpu().numpy()
        assert np.isfinite(a).all()
        assert nerr(a, b.astype(np.float64)) <= TOL
        assert np.array_equal(a, b)                                          # same kernels, same grid: the same bits


@pytest.mark.gpu
def test_static_scratch_vjp_refuses_what_does_not_fit_and_keeps_serving():
    dev = torch.device("cuda:0")
    big = W.random_tree(999, nb=64, shape="chain")           # 64 bodies: 640 partial sums per CTA
    m = binding.Model(big, device=0)
    B = 131072
    assert m.rnea_vjp_workspace_floats(B) > binding.VJP_STATIC_SCRATCH_FLOATS
    t = _inputs(big, B, 5, dev)
    g = torch.zeros((m.nb, 10), device=dev)
    with pytest.raises(binding.BardError, match="static array holds"):
        m.rnea_vjp_params_static(B, *t, g, torch.cuda.current_stream().cuda_stream)
    # a batch whose grid is small enough is served, and agrees with the workspace path
    Bs = 4096
    assert m.rnea_vjp_workspace_floats(Bs) <= binding.VJP_STATIC_SCRATCH_FLOATS
    ts = [x[:, :Bs].contiguous() for x in t]
    ws = torch.empty((m.rnea_vjp_workspace_floats(Bs),), device=dev)
    r = torch.zeros((m.nb, 10), device=dev)
    m.rnea_vjp_params(Bs, *ts, r, ws, torch.cuda.current_stream().cuda_stream)
    m.rnea_vjp_params_static(Bs, *ts, g, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    assert np.array_equal(g.cpu().numpy(), r.cpu().numpy(), equal_nan=True)
