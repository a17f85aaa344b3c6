"""SURVEY 8(b) "Execution": every operator call only enqueues work on the caller's stream, allocates nothing and never
synchronises -- so a sequence of calls can be captured into a CUDA graph (bench.py times its trains and the config-2
rollout that way).  Each entry point is captured once, the graph is replayed on NEW input contents, and the replayed
results must equal the eager results on the same inputs bit for bit (at batches where the captured and the plain call
take the same form of bard_step; the last test covers the batches where they do not): the forked bard_step (side streams joining the
capture), the one-launch and the two-launch bard_step, the single operators of both kernel families, the Euler steps,
ABA, the RNEA VJP (table-driven, generated, and the static-scratch entry point)."""
import numpy as np
import pytest

from paper_2605_31481_b200 import binding, workloads as W

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


def _state(cfg, B, step, dev):
    return [torch.from_numpy(a).to(dev) for a in W.config_states(cfg, B, step=step)]


def _capture(fn):
    """Warm up on a side stream (first-call set-up: function attributes, symbol look-ups), capture, return the graph."""
    st = torch.cuda.Stream()
    st.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(st):
        fn(st.cuda_stream)
    st.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=st):
        fn(torch.cuda.current_stream().cuda_stream)
    return g


@pytest.mark.parametrize("cfg,B,specialised", [(3, 4096, False), (3, 4096, True), (1, 70000, True), (3, 70000, True), (0, 1000, True)])
def test_step_and_single_operators_replay_bit_equal(cfg, B, specialised):
    dev = torch.device("cuda:0")
    desc = W.config_robot(cfg)
    m = binding.Model(desc, device=0)
    if specialised:
        m.specialize(("fk", "jacobian", "rnea", "crba", "fused"))
    q, qd, qdd = _state(cfg, B, 0, dev)
    shapes = ((m.nb, 12, B), (m.nframes, 6, m.nv, B), (m.nv, B), (m.nv, m.nv, B))
    step_out = [torch.zeros(s, device=dev) for s in shapes]
    single_out = [torch.zeros(s, device=dev) for s in shapes]
    kin_out = [torch.zeros(s, device=dev) for s in (shapes[0], shapes[1], shapes[3])]

    def work(s):
        m.step(B, q, qd, qdd, *step_out, s)
        m.fk(B, q, single_out[0], s)
        m.jacobian(B, q, single_out[1], s)
        m.rnea(B, q, qd, qdd, single_out[2], s)
        m.crba(B, q, single_out[3], s)
        m.kinematics(B, q, *kin_out, s)

    g = _capture(work)
    for step in (1, 2):                                     # new contents in the captured buffers
        for dst, src in zip((q, qd, qdd), _state(cfg, B, step, dev)):
            dst.copy_(src)
        for o in step_out + single_out + kin_out:
            o.fill_(float("nan"))
        g.replay()
        torch.cuda.synchronize()
        got = [o.clone() for o in step_out + single_out + kin_out]
        for o in step_out + single_out + kin_out:
            o.fill_(float("nan"))
        work(torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
        for a, b in zip(got, step_out + single_out + kin_out):
            assert torch.isfinite(a).all()
            assert torch.equal(a, b)


@pytest.mark.parametrize("generated", [False, True])
def test_dynamics_extras_replay_bit_equal(generated):
    """bard_euler_step / _to, bard_aba, bard_rnea_vjp_params and bard_rnea_vjp_params_static in one captured graph."""
    dev = torch.device("cuda:0")
    cfg, B = 2, 5000
    desc = W.config_robot(cfg)
    m = binding.Model(desc, device=0)
    if generated:
        m.specialize(("aba", "rnea_vjp"))
    q, qd, qdd = _state(cfg, B, 0, dev)
    dtau = torch.randn((m.nv, B), device=dev, generator=torch.Generator(device=dev).manual_seed(3))
    q2, qd2 = torch.zeros_like(q), torch.zeros_like(qd)
    q3, qd3 = torch.zeros_like(q), torch.zeros_like(qd)
    acc = torch.zeros((m.nv, B), device=dev)
    g1, g2 = torch.zeros((m.nb, 10), device=dev), torch.zeros((m.nb, 10), device=dev)
    ws_aba = torch.empty(m.aba_workspace_floats(B), device=dev)
    ws_vjp = torch.empty(max(1, m.rnea_vjp_workspace_floats(B)), device=dev)
    outs = (q2, qd2, q3, qd3, acc, g1, g2)

    def work(s):
        m.euler_step_to(B, 0.005, q, qd, qdd, q2, qd2, s)
        q3.copy_(q, non_blocking=True)
        qd3.copy_(qd, non_blocking=True)
        m.euler_step(B, 0.005, q3, qd3, qdd, s)
        m.aba(B, q, qd, qdd, acc, ws_aba, s)                 # qdd stands in for tau
        m.rnea_vjp_params(B, q, qd, qdd, dtau, g1, ws_vjp, s)
        m.rnea_vjp_params_static(B, q, qd, qdd, dtau, g2, s)

    st = torch.cuda.Stream()
    st.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(st):
        work(st.cuda_stream)
    st.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=st):
        work(torch.cuda.current_stream().cuda_stream)
    for step in (1, 2):
        for dst, src in zip((q, qd, qdd), _state(cfg, B, step, dev)):
            dst.copy_(src)
        for o in outs:
            o.fill_(float("nan"))
        g.replay()
        torch.cuda.synchronize()
        got = [o.clone() for o in outs]
        for o in outs:
            o.fill_(float("nan"))
        with torch.cuda.stream(st):
            work(st.cuda_stream)
        st.synchronize()
        for a, b in zip(got, outs):
            assert torch.isfinite(a).all()
            assert torch.equal(a, b)
        assert torch.equal(got[0], got[2]) and torch.equal(got[1], got[3])       # in place == out of place
        assert torch.equal(got[5], got[6])                                       # static scratch == caller workspace


@pytest.mark.parametrize("cfg", [0, 2])
def test_captured_step_may_take_another_form_than_the_plain_call_and_both_match_the_oracle(cfg):
    """Between the two fork regimes (plain calls: measured, 3072 on these robots; captured calls: at least 8192) a captured
    bard_step forks the four operators while the plain call is one launch: both are held to the oracle, and they agree to
    rounding (include/bard.h)."""
    import oracle
    dev = torch.device("cuda:0")
    desc = W.config_robot(cfg)
    m = binding.Model(desc, device=0)
    m.specialize(("fk", "jacobian", "rnea", "crba", "fused"))
    plain, captured = m.get_option("step_fork_regime"), m.get_option("step_fork_regime_captured")
    assert captured >= max(plain, 8192)
    B = 5000
    q, qd, qdd = _state(cfg, B, 0, dev)
    shapes = ((m.nb, 12, B), (m.nframes, 6, m.nv, B), (m.nv, B), (m.nv, m.nv, B))
    out = [torch.zeros(s, device=dev) for s in shapes]
    n0 = binding.launch_count()
    m.step(B, q, qd, qdd, *out, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    n_plain = binding.launch_count() - n0
    eager = [o.clone() for o in out]
    g = _capture(lambda s: m.step(B, q, qd, qdd, *out, s))
    n0 = binding.launch_count()
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        gg = torch.cuda.CUDAGraph()
        with torch.cuda.graph(gg, stream=st):
            m.step(B, q, qd, qdd, *out, torch.cuda.current_stream().cuda_stream)
    n_captured = binding.launch_count() - n0
    assert n_plain == (4 if B <= plain else n_plain) and n_captured == (4 if B <= captured else n_captured)
    for o in out:
        o.fill_(float("nan"))
    g.replay()
    torch.cuda.synchronize()
    o64 = oracle.Oracle(desc)
    idx = np.arange(0, B, 25)
    q64, qd64, qdd64 = (np.ascontiguousarray(t.cpu().numpy()[:, idx].astype(np.float64)) for t in (q, qd, qdd))
    refs = (o64.fk(q64), o64.jacobian(q64), o64.rnea(q64, qd64, qdd64), o64.crba(q64))

    def nerr(x, ref):
        return float(np.max(np.abs(np.asarray(x, np.float64) - ref) / np.maximum(1.0, np.abs(ref)))) if ref.size else 0.0
    for got, e, r, tol in zip(out, eager, refs, (1e-4, 1e-4, 1e-3, 1e-3)):
        a, b = got.cpu().numpy(), e.cpu().numpy()
        assert np.isfinite(a).all()
        assert nerr(a[..., idx], r) <= tol and nerr(b[..., idx], r) <= tol
        assert nerr(a, b.astype(np.float64)) <= 2 * tol
