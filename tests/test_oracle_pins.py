"""Pins for the fp64 oracle (CPU only): closed forms, brute force, second formulations, invariants.

Each test ties ``oracle/`` to something other than itself (north_star's list; SURVEY.md section 8(c)
"What pins the oracle"): textbook closed forms of the pendulum / double pendulum / free rigid body /
planar arm, finite differences of FK for the Jacobian, the unit-acceleration construction of M, energy
and symmetry invariants, scipy's rotation routines for the Rodrigues / quaternion conventions.
"""
import numpy as np
import pytest
from scipy.spatial.transform import Rotation

import oracle
import manifold
from paper_2605_31481_b200 import workloads as W

G = 9.81
I12 = np.array([1, 0, 0, 0, 0, 1, 0, 0, 0, 0, 1, 0], float)


def Rt12(R, t):
    return np.concatenate([np.asarray(R, float), np.asarray(t, float).reshape(3, 1)], axis=1).reshape(12)


def make(parent, jt, axis, T_pre, mass, com, inertia, T_post=None, gravity=(0, 0, -G), frames=(), offs=None):
    nb = len(parent)
    return W.RobotDesc("t", np.asarray(parent, np.int32), np.asarray(jt, np.int32), np.asarray(axis, float).reshape(nb, 3),
                       np.asarray(T_pre, float).reshape(nb, 12), None if T_post is None else np.asarray(T_post, float).reshape(nb, 12),
                       np.asarray(mass, float), np.asarray(com, float).reshape(nb, 3), np.asarray(inertia, float).reshape(nb, 6),
                       np.asarray(gravity, float), np.asarray(frames, np.int32), offs)


# ----------------------------------------------------------------------------- closed forms

def test_single_pendulum_closed_form():
    """tau = (Iyy + m l^2) qdd + m g l sin q ; M = Iyy + m l^2 (revolute about y, COM at (0,0,-l))."""
    rng = np.random.default_rng(1)
    m, l = 1.7, 0.43
    inertia = [0.05, 0.011, -0.007, 0.031, 0.004, 0.02]  # off-diagonals must not matter for a y rotation
    d = make([-1], [W.REVOLUTE], [[0, 1, 0]], [I12], [m], [[0, 0, -l]], [inertia])
    o = oracle.Oracle(d)
    q, qd, qdd = rng.uniform(-np.pi, np.pi, (1, 64)), rng.normal(size=(1, 64)), rng.normal(size=(1, 64))
    Iyy = inertia[3]
    np.testing.assert_allclose(o.crba(q)[0, 0], np.full(64, Iyy + m * l * l), rtol=0, atol=1e-14)
    np.testing.assert_allclose(o.rnea(q, qd, qdd)[0], (Iyy + m * l * l) * qdd[0] + m * G * l * np.sin(q[0]), rtol=0, atol=1e-13)


def test_double_pendulum_closed_form():
    """Planar double pendulum (both axes y): M, Coriolis and gravity terms (SURVEY 8(c) pins)."""
    rng = np.random.default_rng(2)
    m1, m2, l1, lc1, lc2, I1, I2 = 1.3, 0.8, 0.5, 0.21, 0.33, 0.04, 0.025
    d = make([-1, 0], [W.REVOLUTE] * 2, [[0, 1, 0]] * 2, [I12, Rt12(np.eye(3), [0, 0, -l1])], [m1, m2],
             [[0, 0, -lc1], [0, 0, -lc2]], [[0.01, 0, 0, I1, 0, 0.02], [0.03, 0, 0, I2, 0, 0.015]])
    o = oracle.Oracle(d)
    B = 50
    q, qd, qdd = rng.uniform(-np.pi, np.pi, (2, B)), rng.normal(size=(2, B)), rng.normal(size=(2, B))
    c2 = np.cos(q[1])
    M11 = I1 + I2 + m1 * lc1 ** 2 + m2 * (l1 ** 2 + lc2 ** 2 + 2 * l1 * lc2 * c2)
    M12 = I2 + m2 * (lc2 ** 2 + l1 * lc2 * c2)
    M22 = np.full(B, I2 + m2 * lc2 ** 2)
    M = o.crba(q)
    np.testing.assert_allclose(M[0, 0], M11, atol=1e-14)
    np.testing.assert_allclose(M[0, 1], M12, atol=1e-14)
    np.testing.assert_allclose(M[1, 0], M12, atol=1e-14)
    np.testing.assert_allclose(M[1, 1], M22, atol=1e-14)
    h = m2 * l1 * lc2 * np.sin(q[1])
    c = np.stack([-h * (2 * qd[0] * qd[1] + qd[1] ** 2), h * qd[0] ** 2])
    g = np.stack([(m1 * lc1 + m2 * l1) * G * np.sin(q[0]) + m2 * lc2 * G * np.sin(q[0] + q[1]), m2 * lc2 * G * np.sin(q[0] + q[1])])
    tau_ref = np.stack([M11 * qdd[0] + M12 * qdd[1], M12 * qdd[0] + M22 * qdd[1]]) + c + g
    np.testing.assert_allclose(o.rnea(q, qd, qdd), tau_ref, atol=2e-13)


def test_free_body_newton_euler_closed_form():
    """Single free body: M = spatial inertia for every q; tau = [F; N] from Newton-Euler about the COM."""
    rng = np.random.default_rng(3)
    m, c = 2.3, np.array([0.03, -0.07, 0.11])
    A = rng.normal(size=(3, 3))
    Ic = A @ A.T * 0.02 + 0.01 * np.eye(3)
    inertia = [Ic[0, 0], Ic[0, 1], Ic[0, 2], Ic[1, 1], Ic[1, 2], Ic[2, 2]]
    grav = np.array([0.4, -1.1, -9.0])
    d = make([-1], [W.FREE], [[0, 0, 0]], [I12], [m], [c], [inertia], gravity=grav)
    o = oracle.Oracle(d)
    B = 40
    q, qd, qdd = W.sample_states(d, B, seed=5, dtype=np.float64)
    q[3:7] *= rng.uniform(0.5, 2.0, size=B)  # un-normalised quaternion: the operators normalise inside
    cx = np.array([[0, -c[2], c[1]], [c[2], 0, -c[0]], [-c[1], c[0], 0]])
    Mref = np.block([[m * np.eye(3), m * cx.T], [m * cx, Ic + m * cx @ cx.T]])
    M = o.crba(q)
    for b in range(B):
        np.testing.assert_allclose(M[:, :, b], Mref, atol=1e-14)
    np.testing.assert_allclose(o.spatial_inertia(0), Mref, atol=1e-15)
    tau = o.rnea(q, qd, qdd)
    for b in range(B):
        R = Rotation.from_quat(q[3:7, b]).as_matrix()  # scipy: scalar-last (x, y, z, w), normalises
        v, w, vd, wd = qd[:3, b], qd[3:, b], qdd[:3, b], qdd[3:, b]
        F = m * (vd + np.cross(w, v) - R.T @ grav + np.cross(wd, c) + np.cross(w, np.cross(w, c)))
        N = Ic @ wd + np.cross(w, Ic @ w) + np.cross(c, F)
        np.testing.assert_allclose(tau[:, b], np.concatenate([F, N]), atol=1e-12)


def test_planar_arm_fk_and_jacobian_closed_form():
    """Planar 3R arm about z with link lengths along x: textbook tip position, orientation and Jacobian."""
    rng = np.random.default_rng(4)
    L = [0.4, 0.3, 0.2]
    T_pre = [I12, Rt12(np.eye(3), [L[0], 0, 0]), Rt12(np.eye(3), [L[1], 0, 0])]
    d = make([-1, 0, 1], [W.REVOLUTE] * 3, [[0, 0, 1]] * 3, T_pre, [1, 1, 1], np.zeros((3, 3)), np.tile([.01, 0, 0, .01, 0, .01], (3, 1)),
             frames=[2], offs=np.array([[L[2], 0, 0.0]]))
    o = oracle.Oracle(d)
    q = rng.uniform(-np.pi, np.pi, (3, 32))
    a1, a12, a123 = q[0], q[0] + q[1], q[0] + q[1] + q[2]
    P = o.fk(q)
    np.testing.assert_allclose(P[2, 9], L[0] * np.cos(a1) + L[1] * np.cos(a12), atol=1e-14)   # p_x of body 2
    np.testing.assert_allclose(P[2, 10], L[0] * np.sin(a1) + L[1] * np.sin(a12), atol=1e-14)  # p_y
    np.testing.assert_allclose(P[2, 0], np.cos(a123), atol=1e-14)    # R00
    np.testing.assert_allclose(P[2, 1], -np.sin(a123), atol=1e-14)   # R01 (row-major: child -> world)
    np.testing.assert_allclose(P[2, 3], np.sin(a123), atol=1e-14)    # R10
    J = o.jacobian(q)[0]  # [6, nv, B]: tip at L2 along x of body 2
    s1, s12, s123, c1, c12, c123 = np.sin(a1), np.sin(a12), np.sin(a123), np.cos(a1), np.cos(a12), np.cos(a123)
    np.testing.assert_allclose(J[0, 0], -L[0] * s1 - L[1] * s12 - L[2] * s123, atol=1e-14)
    np.testing.assert_allclose(J[0, 1], -L[1] * s12 - L[2] * s123, atol=1e-14)
    np.testing.assert_allclose(J[0, 2], -L[2] * s123, atol=1e-14)
    np.testing.assert_allclose(J[1, 0], L[0] * c1 + L[1] * c12 + L[2] * c123, atol=1e-14)
    np.testing.assert_allclose(J[1, 2], L[2] * c123, atol=1e-14)
    np.testing.assert_allclose(J[5], np.ones((3, 32)), atol=1e-15)   # angular z row
    np.testing.assert_allclose(J[2:5], 0, atol=1e-15)


def test_revolute_matches_scipy_rotvec_and_prismatic_translation():
    """T_pc = T_pre T_J(q) T_post against scipy's axis-angle rotation (library routine for Rodrigues)."""
    rng = np.random.default_rng(5)
    ax = rng.normal(size=3)
    Rpre, Rpost = Rotation.random(random_state=1).as_matrix(), Rotation.random(random_state=2).as_matrix()
    tpre, tpost = rng.normal(size=3), rng.normal(size=3)
    for jt in (W.REVOLUTE, W.PRISMATIC, W.FIXED):
        d = make([-1], [jt], [ax], [Rt12(Rpre, tpre)], [1], [[0, 0, 0]], [[1, 0, 0, 1, 0, 1]], T_post=[Rt12(Rpost, tpost)])
        o = oracle.Oracle(d)
        q = rng.uniform(-np.pi, np.pi, (o.nq, 16))
        P = o.fk(q)
        for b in range(16):
            n = ax / np.linalg.norm(ax)
            RJ = Rotation.from_rotvec(n * q[0, b]).as_matrix() if jt == W.REVOLUTE else np.eye(3)
            tJ = n * q[0, b] if jt == W.PRISMATIC else np.zeros(3)
            R = Rpre @ RJ @ Rpost
            t = Rpre @ (RJ @ tpost + tJ) + tpre
            np.testing.assert_allclose(P[0, :9, b].reshape(3, 3), R, atol=1e-14)
            np.testing.assert_allclose(P[0, 9:, b], t, atol=1e-14)


# ----------------------------------------------------------------------------- brute force: finite-difference Jacobians

def fd_jacobian(o, d, q, h=1e-6):
    """Central differences of the oracle's own FK under the manifold step (free: p += R v h, quat (x)= exp)."""
    B = q.shape[1]
    J = np.zeros((o.nframes, 6, o.nv, B))
    offs = np.zeros((o.nframes, 3)) if d.frame_offset is None else d.frame_offset
    for k in range(o.nv):
        dv = np.zeros((o.nv, B))
        dv[k] = h
        Pp, Pm = o.fk(manifold.manifold_step(d, q, dv)), o.fk(manifold.manifold_step(d, q, -dv))
        for f, body in enumerate(d.frame_body):
            Rp, Rm = Pp[body, :9].reshape(3, 3, B), Pm[body, :9].reshape(3, 3, B)
            pe_p = Pp[body, 9:] + np.einsum("ijb,j->ib", Rp, offs[f])
            pe_m = Pm[body, 9:] + np.einsum("ijb,j->ib", Rm, offs[f])
            J[f, :3, k] = (pe_p - pe_m) / (2 * h)
            dR = np.einsum("ijb,kjb->ikb", Rp, Rm)  # R+ R-^T ~ exp([2 h w]x)
            J[f, 3, k] = (dR[2, 1] - dR[1, 2]) / (4 * h)
            J[f, 4, k] = (dR[0, 2] - dR[2, 0]) / (4 * h)
            J[f, 5, k] = (dR[1, 0] - dR[0, 1]) / (4 * h)
    return J


@pytest.mark.parametrize("n", [1, 2, 3, 4])
def test_jacobian_finite_difference_chains(n):
    d = W.random_tree(seed=10 + n, nb=n, shape="chain", joint_types=(W.REVOLUTE, W.PRISMATIC), nframes=1)
    d.frame_body = np.array([n - 1], np.int32)
    o = oracle.Oracle(d)
    q, _, _ = W.sample_states(d, 8, seed=n, dtype=np.float64)
    np.testing.assert_allclose(o.jacobian(q), fd_jacobian(o, d, q), atol=3e-9)


def test_jacobian_finite_difference_tree_all_joint_types():
    parent = [-1, 0, 1, 1, 3, 0, 5]
    jt = [W.FREE, W.REVOLUTE, W.FIXED, W.PRISMATIC, W.REVOLUTE, W.REVOLUTE, W.FREE]  # a second free joint mid-tree too
    d = W.build_robot("mixed", parent, jt, seed=77, frames=[2, 4, 6], random_T_post=True, random_frame_offsets=True, full_inertia=True)
    o = oracle.Oracle(d)
    q, _, _ = W.sample_states(d, 6, seed=9, dtype=np.float64)
    Ja, Jf = o.jacobian(q), fd_jacobian(o, d, q)
    np.testing.assert_allclose(Ja, Jf, atol=3e-9)
    # structural zeros: columns of bodies that are not ancestors of the frame's body
    anc = o.table("ANC_MASK")
    dof_body = o.table("DOF_BODY")
    for f, body in enumerate(d.frame_body):
        for k in range(o.nv):
            if not (int(anc[body]) >> int(dof_body[k])) & 1:
                assert np.all(Ja[f, :, k] == 0.0)


# ----------------------------------------------------------------------------- second formulations

TREES = [dict(seed=21, nb=9, free_root=True), dict(seed=22, nb=12, free_root=False), dict(seed=23, nb=6, shape="star", free_root=True),
         dict(seed=24, nb=10, shape="unbalanced"), dict(seed=25, nb=5, shape="chain", joint_types=(W.REVOLUTE,))]


@pytest.mark.parametrize("kw", TREES)
def test_fk_rodrigues_constants_match_4x4_products(kw):
    """eq. (2)-(5) (Rodrigues constants) reproduce eq. (1) (explicit products) to rounding."""
    d = W.random_tree(**kw)
    o = oracle.Oracle(d)
    q, _, _ = W.sample_states(d, 16, seed=kw["seed"], dtype=np.float64)
    np.testing.assert_allclose(o.fk_rodrigues(q), o.fk(q), atol=5e-15)


@pytest.mark.parametrize("kw", TREES)
def test_crba_equals_unit_acceleration_rnea(kw):
    """Column k of M = RNEA(q, 0, e_k) with zero gravity (unit-acceleration method)."""
    d = W.random_tree(**kw)
    d.gravity = np.zeros(3)
    o = oracle.Oracle(d)
    B = 5
    q, _, _ = W.sample_states(d, B, seed=kw["seed"] + 1, dtype=np.float64)
    M = o.crba(q)
    for k in range(o.nv):
        e = np.zeros((o.nv, B))
        e[k] = 1.0
        np.testing.assert_allclose(M[:, k], o.rnea(q, np.zeros((o.nv, B)), e), atol=1e-12)


# ----------------------------------------------------------------------------- invariants

ROBOTS = [W.chain7, W.quadruped12, W.spined_quadruped11, W.humanoid23] + [lambda kw=kw: W.random_tree(**kw) for kw in TREES]


@pytest.mark.parametrize("mk", ROBOTS)
def test_mass_matrix_invariants(mk):
    d = mk()
    o = oracle.Oracle(d)
    B = 12
    q, qd, qdd = W.sample_states(d, B, seed=31, dtype=np.float64)
    M = o.crba(q)
    np.testing.assert_allclose(M, M.transpose(1, 0, 2), atol=1e-13)
    for b in range(B):
        assert np.linalg.eigvalsh(M[:, :, b]).min() > 0
    # RNEA(q, qd, qdd) - RNEA(q, qd, 0) = M qdd
    Mqdd = np.einsum("ijb,jb->ib", M, qdd)
    scale = max(1.0, np.abs(Mqdd).max())
    np.testing.assert_allclose(o.rnea(q, qd, qdd) - o.rnea(q, qd, 0 * qdd), Mqdd, atol=2e-12 * scale)
    # zero gravity, zero velocity: RNEA = M qdd
    d0 = mk()
    d0.gravity = np.zeros(3)
    o0 = oracle.Oracle(d0)
    np.testing.assert_allclose(o0.rnea(q, 0 * qd, qdd), Mqdd, atol=2e-12 * scale)
    # kinetic energy: 1/2 qd^T M qd = sum_i 1/2 v_i^T I_i v_i
    V = o.body_velocity(q, qd)
    T_bodies = sum(0.5 * np.einsum("ib,ij,jb->b", V[i], o.spatial_inertia(i), V[i]) for i in range(o.nb))
    T_M = 0.5 * np.einsum("ib,ijb,jb->b", qd, M, qd)
    np.testing.assert_allclose(T_M, T_bodies, rtol=1e-12)


@pytest.mark.parametrize("mk", [W.quadruped12, W.spined_quadruped11, W.humanoid23])
def test_floating_base_total_mass_block(mk):
    d = mk()
    o = oracle.Oracle(d)
    q, _, _ = W.sample_states(d, 4, seed=3, dtype=np.float64)
    M = o.crba(q)
    for b in range(4):
        np.testing.assert_allclose(M[:3, :3, b], d.mass.sum() * np.eye(3), atol=1e-12)


@pytest.mark.parametrize("mk", ROBOTS)
def test_frame_velocity_equals_jacobian_times_qd(mk):
    """J qd (world axes, at the frame origin) = world-rotated body twist from the RNEA velocity recursion."""
    d = mk()
    o = oracle.Oracle(d)
    B = 7
    q, qd, _ = W.sample_states(d, B, seed=41, dtype=np.float64)
    J, P, V = o.jacobian(q), o.fk(q), o.body_velocity(q, qd)
    offs = np.zeros((o.nframes, 3)) if d.frame_offset is None else d.frame_offset
    for f, body in enumerate(d.frame_body):
        R = P[body, :9].reshape(3, 3, B)
        v_lin_body = V[body, :3] + np.cross(V[body, 3:], offs[f][:, None], axis=0)  # velocity of the offset point
        ref = np.concatenate([np.einsum("ijb,jb->ib", R, v_lin_body), np.einsum("ijb,jb->ib", R, V[body, 3:])])
        np.testing.assert_allclose(np.einsum("rkb,kb->rb", J[f], qd), ref, atol=1e-12)


def test_rnea_gravity_only_equals_potential_gradient():
    """Static torques = d(sum_i m_i g . c_i^world)/dq by finite differences (fixed-base tree)."""
    d = W.random_tree(seed=51, nb=7, joint_types=(W.REVOLUTE, W.PRISMATIC, W.FIXED))
    o = oracle.Oracle(d)
    B = 6
    q, _, _ = W.sample_states(d, B, seed=2, dtype=np.float64)

    def U(qq):
        P = o.fk(qq)
        u = np.zeros(B)
        for i in range(o.nb):
            cw = P[i, 9:] + np.einsum("ijb,j->ib", P[i, :9].reshape(3, 3, B), d.com[i])
            u += -d.mass[i] * (d.gravity @ cw)
        return u

    z = np.zeros((o.nv, B))
    tau = o.rnea(q, z, z)
    h = 1e-6
    for k in range(o.nv):
        dv = np.zeros((o.nv, B))
        dv[k] = h
        np.testing.assert_allclose(tau[k], (U(manifold.manifold_step(d, q, dv)) - U(manifold.manifold_step(d, q, -dv))) / (2 * h), atol=2e-8)


# ----------------------------------------------------------------------------- tables: brute force

def brute_tables(parent, jt):
    nb = len(parent)
    level = []
    for i in range(nb):
        l, j = 0, parent[i]
        while j >= 0:
            l, j = l + 1, parent[j]
        level.append(l)
    order = sorted(range(nb), key=lambda i: (level[i], i))
    nlev = max(level) + 1
    ptr = [sum(1 for l in level if l < k) for k in range(nlev + 1)]
    pslot = [(-1 if parent[i] < 0 else order.index(parent[i])) for i in order]
    nq = {0: 1, 1: 1, 2: 0, 3: 7}
    nv = {0: 1, 1: 1, 2: 0, 3: 6}
    qoff = [sum(nq[t] for t in jt[:i]) for i in range(nb + 1)]
    voff = [sum(nv[t] for t in jt[:i]) for i in range(nb + 1)]
    dofb = [i for i in range(nb) for _ in range(nv[jt[i]])]
    anc = []
    for i in range(nb):
        m, j = 0, i
        while j >= 0:
            m, j = m | (1 << j), parent[j]
        anc.append(m)
    return dict(LEVEL_PTR=ptr, LEVEL_BODY=order, BODY_LEVEL=level, PARENT_SLOT=pslot, Q_OFF=qoff, V_OFF=voff, DOF_BODY=dofb, ANC_MASK=anc)


@pytest.mark.parametrize("seed,nb,shape", [(1, 1, "random"), (2, 5, "chain"), (3, 9, "star"), (4, 17, "unbalanced"), (5, 33, "random"),
                                           (6, 58, "random"), (7, 58, "chain")])
def test_level_tables_brute_force(seed, nb, shape):
    d = W.random_tree(seed=seed, nb=nb, shape=shape, joint_types=(W.REVOLUTE, W.PRISMATIC, W.FIXED), general=False)
    o = oracle.Oracle(d)
    ref = brute_tables([int(p) for p in d.parent], [int(t) for t in d.joint_type])
    for name, val in ref.items():
        got = o.table(name)
        assert [int(x) for x in got] == [int(x) for x in val], name


@pytest.mark.parametrize("mk", ROBOTS)
def test_coriolis_power_equals_kinetic_energy_rate(mk):
    """With qdd = 0: qd^T (RNEA(q,qd,0) - RNEA(q,0,0)) = d/dt (1/2 qd^T M(q) qd), by central differences
    of M along the manifold step q (+) h qd (pins every velocity-product term of RNEA on general trees)."""
    d = mk()
    o = oracle.Oracle(d)
    B = 5
    q, qd, _ = W.sample_states(d, B, seed=61, dtype=np.float64)
    z = np.zeros_like(qd)
    power = np.einsum("ib,ib->b", qd, o.rnea(q, qd, z) - o.rnea(q, z, z))
    h = 1e-6
    T = lambda qq: 0.5 * np.einsum("ib,ijb,jb->b", qd, o.crba(qq), qd)
    dT = (T(manifold.manifold_step(d, q, h * qd)) - T(manifold.manifold_step(d, q, -h * qd))) / (2 * h)
    np.testing.assert_allclose(power, dT, atol=1e-7 * max(1.0, np.abs(dT).max()))


def test_oracle_under_asan_ubsan(tmp_path):
    """SURVEY section 5 (sanitizers row): every entry point of the oracle under AddressSanitizer + UBSan on a small tree
    with all four joint types (tests/oracle_asan_driver.c).  A report aborts the driver with a non-zero exit code."""
    import os
    import subprocess
    here = os.path.dirname(os.path.abspath(__file__))
    exe = str(tmp_path / "oracle_asan")
    subprocess.run(["gcc", "-std=c99", "-O1", "-g", "-fopenmp", "-fsanitize=address,undefined", "-fno-sanitize-recover=all",
                    "-fno-omit-frame-pointer", "-o", exe, os.path.join(here, "oracle_asan_driver.c"),
                    os.path.join(here, "..", "oracle", "bard_oracle.c"), "-lm"], check=True)
    r = subprocess.run([exe], capture_output=True, text=True, env=dict(os.environ, ASAN_OPTIONS="detect_leaks=1"))
    assert r.returncode == 0, r.stdout + r.stderr
    assert "rc 0" in r.stdout and "ERROR" not in r.stderr and "runtime error" not in r.stderr
