"""Out-of-bounds writes (compute-sanitizer is not available on the GPU pool): every output array sits between two
guard bands filled with a sentinel; after each path has run -- team kernels, specialised kernels, fused / side-by-side
bard_step, forked bard_step, Euler step -- the guards must be untouched and the inputs unchanged."""
import numpy as np
import pytest

from paper_2605_31481_b200 import binding, workloads as W

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu
GUARD, SENT = 512, 12345.0


class Banded:
    """Arrays carved out of one buffer, each between guard bands."""

    def __init__(self, shapes, dev):
        n = sum(int(np.prod(s)) + 2 * GUARD for s in shapes)
        self.buf = torch.full((n,), SENT, device=dev)
        self.views, self.guards, o = [], [], 0
        for s in shapes:
            k = int(np.prod(s))
            self.guards.append((o, o + GUARD))
            self.views.append(self.buf[o + GUARD:o + GUARD + k].view(s))
            self.guards.append((o + GUARD + k, o + 2 * GUARD + k))
            o += k + 2 * GUARD

    def intact(self):
        return all(bool((self.buf[a:b] == SENT).all()) for a, b in self.guards)


@pytest.mark.parametrize("cfg,B", [(3, 1000 + 13), (1, 97), (0, 4096 + 1), (2, 33)])
@pytest.mark.parametrize("path", ["team", "specialised", "fused", "side_by_side", "kin"])
def test_no_write_outside_the_outputs(cfg, B, path):
    desc = W.config_robot(cfg)
    dev = torch.device("cuda:0")
    m = binding.Model(desc, device=0)
    m.set_option("spec_min_b", (1 << 30) if path == "team" else 0)
    if path == "kin":                                        # kinematics-fused kernel + RNEA at every batch size
        for k, v in (("spec_fused_max_rows", 0), ("spec_fused_small_b", 0), ("spec_step4", 0), ("spec_kin_min_b", 0), ("step_fork_max_b", 0)):
            m.set_option(k, v)
    if path in ("fused", "side_by_side"):
        m.set_option("step_mode", 2)                         # the one-launch forms at every batch size
    if path == "fused":
        m.set_option("spec_fused_max_rows", 100000)
    if path == "side_by_side":
        m.set_option("spec_fused_max_rows", 0)
        m.set_option("spec_fused_small_b", 0)
        m.set_option("spec_step4_max_rows", 100000)
        m.set_option("spec_kin_min_b", 1 << 40)
    if path != "team":
        m.specialize(("fk", "jacobian", "rnea", "crba") + (("fused",) if path != "specialised" else ()))
    q, qd, qdd = W.config_states(cfg, B)
    ins = Banded([q.shape, qd.shape, qdd.shape], dev)
    for v, a in zip(ins.views, (q, qd, qdd)):
        v.copy_(torch.from_numpy(a))
    out = Banded([(m.nb, 12, B), (m.nframes, 6, m.nv, B), (m.nv, B), (m.nv, m.nv, B)], dev)
    tq, tqd, tqdd = ins.views
    pose, J, tau, M = out.views
    s = torch.cuda.current_stream().cuda_stream
    m.fk(B, tq, pose, s); m.jacobian(B, tq, J, s); m.rnea(B, tq, tqd, tqdd, tau, s); m.crba(B, tq, M, s)
    m.step(B, tq, tqd, tqdd, pose, J, tau, M, s)
    torch.cuda.synchronize()
    assert out.intact() and ins.intact()
    for v, a in zip(ins.views, (q, qd, qdd)):
        assert torch.equal(v.cpu(), torch.from_numpy(a))          # the operators never write their inputs
    for v in out.views:
        assert bool(torch.isfinite(v).all())
    m.euler_step(B, 0.005, tq, tqd, tqdd, s)
    torch.cuda.synchronize()
    assert ins.intact() and torch.equal(tqdd.cpu(), torch.from_numpy(qdd))
