"""SURVEY 8(b) "Execution": concurrent operator calls on different streams of one model are legal.  Two host threads
issue bard_step (forked regime: the four operators over the model's side streams) and single operators on two
non-blocking streams of ONE model; every result must be bit-equal to the serial run.  And bard_model_set_frames after
work was enqueued on a non-blocking stream, with no host synchronisation in between."""
import threading

import numpy as np
import pytest

import oracle
from paper_2605_31481_b200 import binding, workloads as W

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


def _outs(m, B, dev):
    return [torch.full(sh, float("nan"), device=dev) for sh in ((m.nb, 12, B), (m.nframes, 6, m.nv, B), (m.nv, B), (m.nv, m.nv, B))]


@pytest.mark.parametrize("cfg,specialised", [(3, False), (3, True), (1, True)])
def test_two_threads_two_streams_one_model(cfg, specialised):
    desc = W.config_robot(cfg)
    dev = torch.device("cuda:0")
    m = binding.Model(desc, device=0)
    if specialised:
        m.specialize(("fk", "jacobian", "rnea", "crba", "fused"))
    sizes = (4096, 1000)                                   # both inside bard_step's fork regime (B <= 16384)
    ins, serial, serial_single = {}, {}, {}
    for t, B in enumerate(sizes):
        q, qd, qdd = W.config_states(cfg, B, step=t)
        ins[t] = [torch.from_numpy(a).to(dev) for a in (q, qd, qdd)]
        o = _outs(m, B, dev)
        s0 = torch.cuda.current_stream().cuda_stream
        m.step(B, *ins[t], *o, s0)
        torch.cuda.synchronize()
        serial[t] = [x.clone() for x in o]
        o = _outs(m, B, dev)                               # (a fused bard_step kernel rounds differently from the four operators)
        m.fk(B, ins[t][0], o[0], s0)
        m.jacobian(B, ins[t][0], o[1], s0)
        m.rnea(B, *ins[t], o[2], s0)
        m.crba(B, ins[t][0], o[3], s0)
        torch.cuda.synchronize()
        serial_single[t] = o
    rounds = 40
    results, errors = {}, []

    def worker(t):
        try:
            torch.cuda.set_device(0)
            B = sizes[t]
            st = torch.cuda.Stream()                       # non-blocking
            outs = [_outs(m, B, dev) for _ in range(rounds)]
            single = _outs(m, B, dev)
            with torch.cuda.stream(st):
                for r in range(rounds):
                    m.step(B, *ins[t], *outs[r], st.cuda_stream)
                    if r % 4 == t:                         # single operators interleaved on the same stream
                        m.fk(B, ins[t][0], single[0], st.cuda_stream)
                        m.jacobian(B, ins[t][0], single[1], st.cuda_stream)
                        m.rnea(B, *ins[t], single[2], st.cuda_stream)
                        m.crba(B, ins[t][0], single[3], st.cuda_stream)
            st.synchronize()
            results[t] = (outs, single)
        except Exception as ex:                            # pragma: no cover
            errors.append(ex)

    th = [threading.Thread(target=worker, args=(t,)) for t in range(2)]
    for x in th:
        x.start()
    for x in th:
        x.join()
    assert not errors, errors
    torch.cuda.synchronize()
    for t in range(2):
        outs, single = results[t]
        for r in range(rounds):
            for a, b in zip(outs[r], serial[t]):
                assert torch.equal(a, b), (t, r)
        for a, b in zip(single, serial_single[t]):
            assert torch.equal(a, b)


def test_set_frames_after_enqueued_work_without_host_sync():
    """bard_model_set_frames synchronises the device itself: a long train of bard_step / bard_jacobian calls on a
    non-blocking stream may still be running when it is called; they must finish with the OLD frames' results and the
    next call must see the new frames."""
    desc = W.config_robot(3)
    dev = torch.device("cuda:0")
    m = binding.Model(desc, device=0)
    m.specialize(("fk", "jacobian", "rnea", "crba", "fused"))
    B = 65536
    q, qd, qdd = W.config_states(3, B)
    tq, tqd, tqdd = (torch.from_numpy(a).to(dev) for a in (q, qd, qdd))
    st = torch.cuda.Stream()
    outs = _outs(m, B, dev)
    small = 4096
    outs_s = _outs(m, small, dev)
    with torch.cuda.stream(st):
        for _ in range(30):
            m.step(B, tq, tqd, tqdd, *outs, st.cuda_stream)
        m.step(small, tq[:, :small].contiguous(), tqd[:, :small].contiguous(), tqdd[:, :small].contiguous(), *outs_s, st.cuda_stream)
    new_frames = [5, 23]
    m.set_frames(new_frames, [[0.1, 0.0, -0.2], [0.0, 0.0, 0.05]])          # no host sync before this call
    idx = np.arange(0, B, 257)
    o_old = oracle.Oracle(desc)
    ref_old = o_old.jacobian(q[:, idx].astype(np.float64))
    got_old = outs[1].cpu().numpy()[..., idx]
    assert np.max(np.abs(got_old - ref_old) / np.maximum(1.0, np.abs(ref_old))) <= 1e-4
    desc.frame_body = new_frames
    desc.frame_offset = [[0.1, 0.0, -0.2], [0.0, 0.0, 0.05]]
    o_new = oracle.Oracle(desc)
    for spec in (False, True):
        if spec:
            m.specialize(("jacobian",))
        J = torch.full((2, 6, m.nv, B), float("nan"), device=dev)
        m.jacobian(B, tq, J, st.cuda_stream)
        st.synchronize()
        ref = o_new.jacobian(q[:, idx].astype(np.float64))
        got = J.cpu().numpy()[..., idx]
        assert np.isfinite(got).all()
        assert np.max(np.abs(got - ref) / np.maximum(1.0, np.abs(ref))) <= 1e-4
