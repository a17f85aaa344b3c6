"""RNEA as a function of the inertial parameters and its vector-Jacobian product (the paper's
differentiability claim: link masses identified through RNEA, Table 2 at 164-174).

CPU part (-m "not gpu"): pins of the oracle's bard_oracle_rnea_params / bard_oracle_rnea_vjp_params against things other
than themselves -- the pinned bard_oracle_rnea, linearity in the parameters, the pendulum closed form, central finite
differences through the ORIGINAL description (mass, COM, inertia about the COM).  GPU part: bard_rnea_vjp_params against
the oracle, and a synthetic system identification on config 0 (the paper's KUKA iiwa data is not available: torques from
our own RNEA + 5 % noise)."""
import copy

import numpy as np
import pytest

import oracle
from paper_2605_31481_b200 import binding, workloads as W

G = 9.81


def _robots():
    out = [W.config_robot(c) for c in range(4)]
    for seed in range(4):
        shape = ["random", "chain", "star", "unbalanced"][seed % 4]
        out.append(W.random_tree(700 + seed, nb=3 + 3 * seed, shape=shape, free_root=(seed % 2 == 0), nframes=1))
    return out


def theta_of(desc):
    """(m, m c, Ic + m (|c|^2 1 - c c^T)) written out in numpy from the description: the map whose chain rule the
    finite-difference pins need.  Independent of the oracle's C code."""
    m, c, Ic = np.asarray(desc.mass, float), np.asarray(desc.com, float), np.asarray(desc.inertia, float)
    th = np.zeros((len(m), 10))
    th[:, 0] = m
    th[:, 1:4] = m[:, None] * c
    c2 = (c * c).sum(1)
    th[:, 4] = Ic[:, 0] + m * (c2 - c[:, 0] ** 2)
    th[:, 5] = Ic[:, 1] - m * c[:, 0] * c[:, 1]
    th[:, 6] = Ic[:, 2] - m * c[:, 0] * c[:, 2]
    th[:, 7] = Ic[:, 3] + m * (c2 - c[:, 1] ** 2)
    th[:, 8] = Ic[:, 4] - m * c[:, 1] * c[:, 2]
    th[:, 9] = Ic[:, 5] + m * (c2 - c[:, 2] ** 2)
    return th


@pytest.mark.parametrize("idx", range(8))
def test_params_entry_reproduces_the_pinned_rnea(idx):
    desc = _robots()[idx]
    o = oracle.Oracle(desc)
    q, qd, qdd = W.sample_states(desc, 16, seed=11 + idx, dtype=np.float64)
    th = o.inertial_params()
    np.testing.assert_allclose(th, theta_of(desc), rtol=0, atol=1e-14)          # layout and definition of the ten parameters
    ref = o.rnea(q, qd, qdd)
    np.testing.assert_allclose(o.rnea_params(q, qd, qdd, th), ref, rtol=0, atol=1e-12 * max(1.0, np.abs(ref).max()))


@pytest.mark.parametrize("idx", range(8))
def test_tau_is_linear_in_the_parameters(idx):
    desc = _robots()[idx]
    o = oracle.Oracle(desc)
    rng = np.random.default_rng(idx)
    q, qd, qdd = W.sample_states(desc, 8, seed=21 + idx, dtype=np.float64)
    t1, t2 = rng.normal(size=(o.nb, 10)), rng.normal(size=(o.nb, 10))       # any vectors, physical or not
    a, b = o.rnea_params(q, qd, qdd, t1), o.rnea_params(q, qd, qdd, t2)
    s = o.rnea_params(q, qd, qdd, 0.7 * t1 - 2.5 * t2)
    np.testing.assert_allclose(s, 0.7 * a - 2.5 * b, rtol=0, atol=1e-11 * max(1.0, np.abs(a).max(), np.abs(b).max()))
    assert not o.rnea_params(q, qd, qdd, np.zeros((o.nb, 10))).any()         # tau(0) = 0: gravity enters through the inertia


def test_pendulum_closed_form_gradient():
    """One revolute joint about y at the world origin, gravity -z: tau = Io_yy qdd - g h_x cos q - g h_z sin q in the ten
    parameters (potential U = g (h_z cos q - h_x sin q)), so the VJP has three non-zero entries with closed forms."""
    T = np.zeros((1, 12)); T[0, 0] = T[0, 5] = T[0, 10] = 1.0
    desc = W.RobotDesc(name="pendulum", parent=np.array([-1], np.int32), joint_type=np.array([W.REVOLUTE], np.int32),
                       axis=np.array([[0.0, 1.0, 0.0]]), T_pre=T, T_post=None, mass=np.array([1.3]), com=np.array([[0.05, 0.02, -0.4]]),
                       inertia=np.array([[0.02, 0.001, -0.002, 0.03, 0.0005, 0.01]]))
    o = oracle.Oracle(desc)
    rng = np.random.default_rng(5)
    B = 64
    q, qd, qdd, dtau = rng.uniform(-3, 3, (1, B)), rng.normal(size=(1, B)), rng.normal(size=(1, B)), rng.normal(size=(1, B))
    g = o.rnea_vjp_params(q, qd, qdd, dtau)
    want = np.zeros((1, 10))
    want[0, 7] = (dtau * qdd).sum()                       # d tau / d Io_yy = qdd
    want[0, 1] = (dtau * (-G * np.cos(q))).sum()          # d tau / d h_x
    want[0, 3] = (dtau * (-G * np.sin(q))).sum()          # d tau / d h_z
    np.testing.assert_allclose(g, want, rtol=0, atol=1e-11)
    th = o.inertial_params()
    tau = o.rnea(q, qd, qdd)
    np.testing.assert_allclose(tau, th[0, 7] * qdd - G * th[0, 1] * np.cos(q) - G * th[0, 3] * np.sin(q), rtol=0, atol=1e-12)


@pytest.mark.parametrize("idx", range(8))
def test_vjp_against_finite_differences_through_the_description(idx):
    """L(desc) = sum dtau . tau(desc) through the pinned bard_oracle_rnea, differentiated by central differences in the
    description's own mass / COM / inertia; the VJP in the ten parameters chained through theta_of() must match."""
    desc = _robots()[idx]
    o = oracle.Oracle(desc)
    rng = np.random.default_rng(100 + idx)
    B = 12
    q, qd, qdd = W.sample_states(desc, B, seed=31 + idx, dtype=np.float64)
    dtau = rng.normal(size=(o.nv, B))
    g = o.rnea_vjp_params(q, qd, qdd, dtau)                # [nb, 10]

    def L(d):
        return float((dtau * oracle.Oracle(d).rnea(q, qd, qdd)).sum())

    def fd(field, i, k, h):
        dp, dm = copy.deepcopy(desc), copy.deepcopy(desc)
        getattr(dp, field)[(i, k) if k is not None else i] += h
        getattr(dm, field)[(i, k) if k is not None else i] -= h
        return (L(dp) - L(dm)) / (2 * h), (theta_of(dp) - theta_of(dm))[i] / (2 * h)

    scale = max(1.0, np.abs(g).max())
    for i in rng.choice(o.nb, size=min(o.nb, 4), replace=False):
        for field, ks, h in (("mass", [None], 1e-4), ("com", [0, 1, 2], 1e-5), ("inertia", range(6), 1e-4)):
            for k in ks:
                num, dth = fd(field, int(i), k, h)
                np.testing.assert_allclose(float(g[i] @ dth), num, rtol=0, atol=2e-7 * scale)


def test_vjp_is_the_transpose_of_the_regressor():
    """dparams . dtheta = dtau . (tau(theta + dtheta) - tau(theta)) for ANY dtheta (exactly, by linearity)."""
    desc = W.config_robot(2)
    o = oracle.Oracle(desc)
    rng = np.random.default_rng(3)
    q, qd, qdd = W.sample_states(desc, 20, seed=41, dtype=np.float64)
    dtau, dth = rng.normal(size=(o.nv, 20)), rng.normal(size=(o.nb, 10))
    g = o.rnea_vjp_params(q, qd, qdd, dtau)
    lhs = float((g * dth).sum())
    rhs = float((dtau * o.rnea_params(q, qd, qdd, dth)).sum())
    assert abs(lhs - rhs) <= 1e-10 * max(1.0, abs(rhs))


# ------------------------------------------------------------------------------------------- GPU
torch = pytest.importorskip("torch")
TOL = 1e-3        # as for RNEA itself (north_star): per element |g - ref| / max(1, |ref|)


def nerr(x, ref):
    return float(np.max(np.abs(np.asarray(x, np.float64) - ref) / np.maximum(1.0, np.abs(ref)))) if ref.size else 0.0


def gpu_vjp(m, q, qd, qdd, dtau, repeat=1):
    dev = torch.device("cuda:0")
    B = q.shape[1]
    t = [torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).to(dev) for a in (q, qd, qdd, dtau)]
    ws = torch.full((max(1, m.rnea_vjp_workspace_floats(B)),), float("nan"), device=dev)
    outs = []
    for _ in range(repeat):
        g = torch.full((m.nb, 10), float("nan"), device=dev)
        m.rnea_vjp_params(B, *t, g, ws, torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
        outs.append(g.cpu().numpy())
    return outs if repeat > 1 else outs[0]


@pytest.mark.gpu
@pytest.mark.parametrize("idx", range(8))
@pytest.mark.parametrize("B", [1, 37, 1000, 4096 + 17])
def test_gpu_vjp_matches_oracle(idx, B):
    desc = _robots()[idx]
    m = binding.Model(desc, device=0)
    o = oracle.Oracle(desc)
    np.testing.assert_allclose(m.inertial_params(), o.inertial_params(), rtol=0, atol=1e-14)
    q, qd, qdd = W.sample_states(desc, B, seed=51 + idx)
    dtau = np.random.default_rng(idx).normal(size=(desc.nv, B)).astype(np.float32)
    g1, g2 = gpu_vjp(m, q, qd, qdd, dtau, repeat=2)
    assert np.isfinite(g1).all()
    assert np.array_equal(g1, g2)                                            # deterministic batch reduction
    ref = o.rnea_vjp_params(*(a.astype(np.float64) for a in (q, qd, qdd, dtau)))
    assert nerr(g1, ref) <= TOL


@pytest.mark.gpu
@pytest.mark.parametrize("idx", range(8))
@pytest.mark.parametrize("B", [1, 37, 1000, 4096 + 17, 200003])
def test_gpu_generated_vjp_matches_oracle_and_table_kernel(idx, B):
    """bard_model_specialize(BARD_OP_RNEA_VJP): the generated kernel (one tile per CTA up to one wave, a grid-stride loop
    over tiles beyond: 200 003, ragged) against the oracle, against the table-driven kernel, and bit-identical on a repeat."""
    desc = _robots()[idx]
    m = binding.Model(desc, device=0)
    o = oracle.Oracle(desc)
    q, qd, qdd = W.sample_states(desc, B, seed=151 + idx)
    dtau = np.random.default_rng(idx).normal(size=(desc.nv, B)).astype(np.float32)
    g_table = gpu_vjp(m, q, qd, qdd, dtau)
    m.specialize(("rnea_vjp",))
    assert "bard_rnea_vjp_n1" in m.specialized_source("rnea_vjp")
    n0 = binding.launch_count()
    g1, g2 = gpu_vjp(m, q, qd, qdd, dtau, repeat=2)
    assert binding.launch_count() - n0 == 4                                  # the generated kernel + the sum over its CTAs, twice
    assert np.isfinite(g1).all()
    assert np.array_equal(g1, g2)
    if B <= 5000:                                                            # the oracle needs nb * 10 RNEAs per environment
        ref = o.rnea_vjp_params(*(a.astype(np.float64) for a in (q, qd, qdd, dtau)))
        assert nerr(g1, ref) <= TOL
    else:                                                                    # the whole batch: against the table-driven kernel (itself held to the oracle)
        scale = np.maximum(1.0, np.abs(g_table.astype(np.float64)))
        assert float(np.max(np.abs(g1.astype(np.float64) - g_table) / scale)) <= TOL * max(1.0, np.sqrt(B / 4096.0))
    m.set_option("spec_vjp_min_b", 1 << 40)                                  # the table-driven kernel again
    assert np.array_equal(gpu_vjp(m, q, qd, qdd, dtau), g_table)


@pytest.mark.gpu
def test_gpu_vjp_full_size_and_adjoint_identity():
    """Humanoid at B = 65 536 (bench size): against the oracle's definition (240 RNEA evaluations per environment on the
    host cores), and the adjoint identity dparams . dtheta = sum dtau . tau(dtheta) with tau(dtheta) from the GPU's own
    bard_rnea after bard_model_set_inertial_params(dtheta) -- the VJP is the transpose of what bard_rnea computes."""
    desc = W.config_robot(3)
    B = 65536
    m = binding.Model(desc, device=0)
    o = oracle.Oracle(desc)
    q, qd, qdd = W.config_states(3, B)
    rng = np.random.default_rng(8)
    dtau = rng.normal(size=(desc.nv, B)).astype(np.float32)
    g = gpu_vjp(m, q, qd, qdd, dtau)
    ref = o.rnea_vjp_params(*(a.astype(np.float64) for a in (q, qd, qdd, dtau)))
    assert nerr(g, ref) <= TOL
    dth = o.inertial_params() * (1.0 + 0.3 * rng.normal(size=(desc.nb, 10)))   # a direction of physical magnitude
    m.set_inertial_params(dth)
    dev = torch.device("cuda:0")
    tq, tqd, tqdd = (torch.from_numpy(a).to(dev) for a in (q, qd, qdd))
    tau = torch.empty((desc.nv, B), device=dev)
    m.rnea(B, tq, tqd, tqdd, tau, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    rhs = float((tau.double().cpu().numpy() * dtau.astype(np.float64)).sum())
    lhs = float((g.astype(np.float64) * dth).sum())
    scale = float(np.abs(g.astype(np.float64) * dth).sum())
    assert abs(lhs - rhs) <= 1e-4 * scale


@pytest.mark.gpu
def test_set_inertial_params_reaches_every_kernel_family():
    """After bard_model_set_inertial_params the team kernels read the new constants at once and the generated RNEA / CRBA
    are dropped (they had the old parameters as literals) until the model is specialised again."""
    desc = W.config_robot(1)
    m = binding.Model(desc, device=0)
    m.set_option("spec_min_b", 0)
    m.specialize(("rnea", "crba"))
    rng = np.random.default_rng(2)
    new = copy.deepcopy(desc)
    new.mass = desc.mass * rng.uniform(0.5, 2.0, size=desc.nb)
    new.com = desc.com + rng.uniform(-0.02, 0.02, size=desc.com.shape)
    m.set_inertial_params(theta_of(new))
    with pytest.raises(binding.BardError):
        m.specialized_source("rnea")
    o = oracle.Oracle(new)
    B = 500
    q, qd, qdd = W.config_states(1, B)
    dev = torch.device("cuda:0")
    tq, tqd, tqdd = (torch.from_numpy(a).to(dev) for a in (q, qd, qdd))
    q64, qd64, qdd64 = (a.astype(np.float64) for a in (q, qd, qdd))
    for spec in (False, True):
        if spec:
            m.specialize(("rnea", "crba"))
        tau = torch.full((desc.nv, B), float("nan"), device=dev)
        M = torch.full((desc.nv, desc.nv, B), float("nan"), device=dev)
        s = torch.cuda.current_stream().cuda_stream
        m.rnea(B, tq, tqd, tqdd, tau, s)
        m.crba(B, tq, M, s)
        torch.cuda.synchronize()
        assert nerr(tau.cpu().numpy(), o.rnea(q64, qd64, qdd64)) <= 1e-3
        assert nerr(M.cpu().numpy(), o.crba(q64)) <= 1e-3


@pytest.mark.gpu
def test_synthetic_system_identification_of_link_masses():
    """The paper's experiment (Table 2) on a stand-in: its KUKA iiwa data and Pinocchio ground truth are
    not available, so config 0 (7-DOF chain) plays the arm, the "measured" torques are our own bard_rnea at the true
    masses with 5 % multiplicative noise, and L-BFGS recovers the seven link masses from a 2x-off start through
    loss = 1/2B sum |tau(m) - tau_meas|^2, gradient = bard_rnea_vjp_params chained to the masses (COM and inertia about
    the COM held fixed).  The loss is quadratic in m, so the optimum is also available in closed form from the oracle's
    regressor: L-BFGS through the GPU gradient must land on it."""
    from scipy.optimize import minimize
    desc = W.config_robot(0)
    B = 4096
    dev = torch.device("cuda:0")
    m = binding.Model(desc, device=0)
    q, qd, qdd = W.sample_states(desc, B, seed=77)
    tq, tqd, tqdd = (torch.from_numpy(a).to(dev) for a in (q, qd, qdd))
    s = torch.cuda.current_stream().cuda_stream
    tau = torch.empty((desc.nv, B), device=dev)
    m.rnea(B, tq, tqd, tqdd, tau, s)
    torch.cuda.synchronize()
    rng = np.random.default_rng(0)
    meas = tau * torch.from_numpy((1 + 0.05 * rng.normal(size=(desc.nv, B))).astype(np.float32)).to(dev)
    ws = torch.empty(m.rnea_vjp_workspace_floats(B), device=dev)
    g = torch.empty((desc.nb, 10), device=dev)

    def theta(mass):
        d = copy.deepcopy(desc)
        d.mass = np.asarray(mass, float)
        return theta_of(d)

    c = desc.com
    dth_dm = np.zeros((desc.nb, 10))                                           # d theta_i / d m_i with c, Ic fixed
    dth_dm[:, 0] = 1.0
    dth_dm[:, 1:4] = c
    c2 = (c * c).sum(1)
    dth_dm[:, 4], dth_dm[:, 7], dth_dm[:, 9] = c2 - c[:, 0] ** 2, c2 - c[:, 1] ** 2, c2 - c[:, 2] ** 2
    dth_dm[:, 5], dth_dm[:, 6], dth_dm[:, 8] = -c[:, 0] * c[:, 1], -c[:, 0] * c[:, 2], -c[:, 1] * c[:, 2]

    def loss_and_grad(mass):
        m.set_inertial_params(theta(mass))
        m.rnea(B, tq, tqd, tqdd, tau, s)
        r = (tau - meas) / B
        m.rnea_vjp_params(B, tq, tqd, tqdd, r, g, ws, s)
        torch.cuda.synchronize()
        loss = 0.5 * B * float((r.double() ** 2).sum())
        return loss, (g.double().cpu().numpy() * dth_dm).sum(1)

    m0 = desc.mass * np.where(np.arange(desc.nb) % 2 == 0, 2.0, 0.5)
    l0, _ = loss_and_grad(m0)
    res = minimize(loss_and_grad, m0, jac=True, method="L-BFGS-B", options={"maxiter": 200, "ftol": 1e-14, "gtol": 1e-9})
    # closed-form optimum from the oracle (fp64 regressor in the masses)
    o = oracle.Oracle(desc)
    q64, qd64, qdd64 = (a.astype(np.float64) for a in (q, qd, qdd))
    t0 = o.rnea_params(q64, qd64, qdd64, theta(np.zeros(desc.nb)))
    Y = np.stack([(o.rnea_params(q64, qd64, qdd64, theta(np.eye(desc.nb)[i])) - t0).ravel() for i in range(desc.nb)], 1)
    best = np.linalg.lstsq(Y, (meas.double().cpu().numpy() - t0).ravel(), rcond=None)[0]
    assert res.fun < 0.05 * l0
    np.testing.assert_allclose(res.x, best, rtol=5e-3, atol=1e-3)               # the optimiser reached the least-squares optimum
    assert np.max(np.abs(res.x - desc.mass) / desc.mass) < 0.15                 # and the masses are recovered (5 % torque noise)
