"""The explicit Euler step of BASELINE.json's config 2 (q advanced from random qdd, readings 1 and 15):
oracle pins on CPU, GPU parity of bard_euler_step, and the 24-step rollout with all four operators per step."""
import numpy as np
import pytest
from scipy.spatial.transform import Rotation

import oracle
import manifold
from paper_2605_31481_b200 import binding, workloads as W


def nerr(x, ref):
    return float(np.max(np.abs(x.astype(np.float64) - ref) / np.maximum(1.0, np.abs(ref)))) if ref.size else 0.0


# ------------------------------------------------------------------------------------------- oracle pins (CPU)
@pytest.mark.parametrize("cfg", [0, 1, 2, 3])
def test_oracle_step_agrees_with_the_independent_numpy_formulation(cfg):
    """oracle (C, rotation from the FK routine's quaternion matrix) vs tests/manifold.py manifold_step (numpy, written
    separately for the finite-difference stencils): two formulations of the same step."""
    desc = W.config_robot(cfg)
    o = oracle.Oracle(desc)
    q, qd, qdd = W.sample_states(desc, 64, seed=11 + cfg, dtype=np.float64)
    q1, qd1 = o.euler_step(0.005, q, qd, qdd)
    qd2 = qd + 0.005 * qdd
    q2 = manifold.manifold_step(desc, q, 0.005 * qd2)
    assert np.abs(qd1 - qd2).max() == 0.0
    assert np.abs(q1 - q2).max() <= 1e-15


def test_oracle_free_body_step_against_the_exponential_map():
    """Single free body, constant body-frame twist: one small step must agree with the exact flow
    R(dt) = R0 exp([omega] dt), p(dt) = p0 + R0 v dt + O(dt^2) to second order in dt."""
    desc = W.build_robot("free1", [-1], [W.FREE], seed=5)
    o = oracle.Oracle(desc)
    rng = np.random.default_rng(0)
    B, dt = 16, 1e-4
    q, qd, _ = W.sample_states(desc, B, seed=3, dtype=np.float64)
    q[3:7] *= 1.7                                   # not normalised on input: the step normalises
    qdd = np.zeros_like(qd)
    q1, qd1 = o.euler_step(dt, q, qd, qdd)
    assert np.array_equal(qd1, qd)
    assert np.abs(np.linalg.norm(q1[3:7], axis=0) - 1.0).max() <= 1e-15
    R0 = Rotation.from_quat(q[3:7].T)               # scipy: xyzw, normalises
    R1 = R0 * Rotation.from_rotvec((qd[3:6] * dt).T)
    ang = (Rotation.from_quat(q1[3:7].T).inv() * R1).magnitude()
    assert ang.max() <= 10 * dt ** 2 * np.abs(qd[3:6]).max() ** 2 + 1e-12
    p1 = q[0:3] + dt * np.einsum("bij,jb->ib", R0.as_matrix(), qd[0:3])
    assert np.abs(q1[0:3] - p1).max() <= 1e-14


def test_oracle_zero_velocity_is_a_fixed_point_and_revolute_is_plain_euler():
    desc = W.random_tree(77, nb=9, free_root=True)
    o = oracle.Oracle(desc)
    q, qd, qdd = W.sample_states(desc, 8, seed=1, dtype=np.float64)
    q0, _ = o.euler_step(0.01, q, np.zeros_like(qd), np.zeros_like(qdd))
    qn = q.copy()
    qn[3:7] /= np.linalg.norm(q[3:7], axis=0)
    assert np.abs(q0 - qn).max() <= 1e-15
    q1, qd1 = o.euler_step(0.01, q, qd, qdd)
    for i, t in enumerate(desc.joint_type):
        if int(t) in (W.REVOLUTE, W.PRISMATIC):
            a, v = desc.q_off[i], desc.v_off[i]
            assert np.allclose(q1[a], q[a] + 0.01 * (qd[v] + 0.01 * qdd[v]), rtol=0, atol=1e-15)


# ------------------------------------------------------------------------------------------- GPU
torch = pytest.importorskip("torch")


def _robots():
    return [W.config_robot(c) for c in range(4)] + [W.random_tree(60 + s, nb=3 + 5 * s, free_root=(s % 2 == 0)) for s in range(4)]


@pytest.mark.gpu
@pytest.mark.parametrize("idx", range(8))
@pytest.mark.parametrize("B", [1, 77, 4099])
def test_gpu_euler_step_matches_oracle(idx, B):
    desc = _robots()[idx]
    m = binding.Model(desc, device=0)
    o = oracle.Oracle(desc)
    q, qd, qdd = W.sample_states(desc, B, seed=21 + idx)
    dev = torch.device("cuda:0")
    tq, tqd, tqdd = (torch.from_numpy(a.copy()).to(dev) for a in (q, qd, qdd))
    n0 = binding.launch_count()
    m.euler_step(B, 0.005, tq, tqd, tqdd, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    assert binding.launch_count() - n0 == (1 if m.nq else 0)
    q1, qd1 = o.euler_step(np.float32(0.005), *(a.astype(np.float64) for a in (q, qd, qdd)))
    assert nerr(tq.cpu().numpy(), q1) <= 1e-6
    assert nerr(tqd.cpu().numpy(), qd1) <= 1e-6
    assert torch.equal(tqdd.cpu(), torch.from_numpy(qdd))          # qdd is read only


@pytest.mark.gpu
def test_config2_rollout_on_the_device():
    """config 2 as BASELINE.json states it: 24 consecutive steps, all four operators per step (bard_step), q
    advanced on the DEVICE by bard_euler_step from seeded qdd; the oracle integrates the same qdd in fp64.  The
    operators are compared at every step on the device trajectory (rounded to the oracle's input), and the two
    trajectories must stay together (fp32 drift only)."""
    cfg, B, dt = 2, 512, 0.005
    desc = W.config_robot(cfg)
    m = binding.Model(desc, device=0)
    m.set_option("spec_min_b", 0)
    m.specialize(("fk", "jacobian", "rnea", "crba", "fused"))
    o = oracle.Oracle(desc)
    dev = torch.device("cuda:0")
    q, qd, _ = W.sample_states(desc, B, seed=2000 + cfg)
    tq, tqd = torch.from_numpy(q).to(dev), torch.from_numpy(qd).to(dev)
    oq, oqd = q.astype(np.float64), qd.astype(np.float64)
    outs = [torch.empty(sh, device=dev) for sh in ((m.nb, 12, B), (m.nframes, 6, m.nv, B), (m.nv, B), (m.nv, m.nv, B))]
    s = torch.cuda.current_stream().cuda_stream
    for step in range(24):
        qdd = np.random.default_rng(2000 + cfg + 100 * (step + 1)).normal(size=(desc.nv, B)).astype(np.float32)
        tqdd = torch.from_numpy(qdd).to(dev)
        m.step(B, tq, tqd, tqdd, *outs, s)
        torch.cuda.synchronize()
        hq, hqd = tq.cpu().numpy().astype(np.float64), tqd.cpu().numpy().astype(np.float64)
        ref = (o.fk(hq), o.jacobian(hq), o.rnea(hq, hqd, qdd.astype(np.float64)), o.crba(hq))
        for t, r, tol in zip(outs, ref, (1e-4, 1e-4, 1e-3, 1e-3)):
            assert nerr(t.cpu().numpy(), r) <= tol, step
        m.euler_step(B, dt, tq, tqd, tqdd, s)
        oq, oqd = o.euler_step(np.float32(dt), oq, oqd, qdd.astype(np.float64))
        torch.cuda.synchronize()
        # the quaternion sign is free (q and -q are the same pose): compare poses through FK, velocities directly
        assert nerr(tqd.cpu().numpy(), oqd) <= 1e-5 * (step + 1)
        assert nerr(o.fk(tq.cpu().numpy().astype(np.float64)), o.fk(oq)) <= 1e-5 * (step + 1)


@pytest.mark.gpu
@pytest.mark.parametrize("cfg", [0, 2, 3])
def test_out_of_place_euler_step_equals_the_in_place_one(cfg):
    """bard_euler_step_to: same bits as bard_euler_step, inputs untouched, outputs fully written."""
    desc = W.config_robot(cfg)
    m = binding.Model(desc, device=0)
    dev = torch.device("cuda:0")
    B = 1000 + 13
    q, qd, qdd = W.config_states(cfg, B)
    tq, tqd, tqdd = (torch.from_numpy(a).to(dev) for a in (q, qd, qdd))
    q2, qd2 = torch.full_like(tq, float("nan")), torch.full_like(tqd, float("nan"))
    s = torch.cuda.current_stream().cuda_stream
    m.euler_step_to(B, 0.005, tq, tqd, tqdd, q2, qd2, s)
    torch.cuda.synchronize()
    assert torch.equal(tq.cpu(), torch.from_numpy(q)) and torch.equal(tqd.cpu(), torch.from_numpy(qd))
    m.euler_step(B, 0.005, tq, tqd, tqdd, s)
    torch.cuda.synchronize()
    assert torch.equal(q2, tq) and torch.equal(qd2, tqd)
