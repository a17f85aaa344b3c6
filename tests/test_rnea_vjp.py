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
