"""SURVEY 8(b) "Execution": every operator call only enqueues work on the caller's stream, allocates nothing and never
synchronises -- so a sequence of calls can be captured into a CUDA graph (bench.py times its trains and the config-2
rollout that way).  Each entry point is captured once, the graph is replayed on NEW input contents, and the replayed
results must equal the eager results on the same inputs bit for bit: the forked bard_step (side streams joining the
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
