"""Seeded synthetic robots and states (the ONLY module shared by the CUDA path's tests/bench and the oracle's).

It holds none of the method's arithmetic: no kinematics, no dynamics, no integrator, no level schedule.  It only
draws the inputs both sides consume -- robot descriptions (topology, joint types/axes, fixed offsets, inertial
parameters) and batches of (q, qd, qdd) -- with ``numpy.random.default_rng`` (PCG64), following the recipe
of BASELINE.json ``configs`` as restated in SURVEY.md section 8(d) and DESIGN.md "Input recipe".  (The one formula
here, ``_quat_to_R``, turns a drawn unit quaternion into the rotation part of a FIXED offset of the description;
the numpy manifold step the tests use as a finite-difference stencil lives in ``tests/manifold.py``.)

These robots stand in for the paper's URDF models (xArm7 / SPARC / Go2 / G1), which are not
available; only their shapes (DOF count, tree topology, depth) are taken.

Layouts: every batched array is structure-of-arrays, batch last (= batch fastest in memory):
``q[nq, B]``, ``qd[nv, B]``, ``qdd[nv, B]``.  Free joint: q = [p(3), quat x,y,z,w], qd = body-frame twist
[v_lin(3), omega(3)].
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Optional

import numpy as np

REVOLUTE, PRISMATIC, FIXED, FREE = 0, 1, 2, 3
_NQ = {REVOLUTE: 1, PRISMATIC: 1, FIXED: 0, FREE: 7}
_NV = {REVOLUTE: 1, PRISMATIC: 1, FIXED: 0, FREE: 6}


@dataclass
class RobotDesc:
    name: str
    parent: np.ndarray        # int32 [nb]
    joint_type: np.ndarray    # int32 [nb]
    axis: np.ndarray          # f64 [nb,3]
    T_pre: np.ndarray         # f64 [nb,12] rows (R|t)
    T_post: Optional[np.ndarray]  # f64 [nb,12] or None (= identity)
    mass: np.ndarray          # f64 [nb]
    com: np.ndarray           # f64 [nb,3]
    inertia: np.ndarray       # f64 [nb,6] xx,xy,xz,yy,yz,zz about the COM
    gravity: np.ndarray = field(default_factory=lambda: np.array([0.0, 0.0, -9.81]))
    frame_body: np.ndarray = field(default_factory=lambda: np.zeros(0, np.int32))
    frame_offset: Optional[np.ndarray] = None  # f64 [nframes,3] or None (= zeros)

    @property
    def nb(self) -> int:
        return int(len(self.parent))

    @property
    def nq(self) -> int:
        return int(sum(_NQ[int(t)] for t in self.joint_type))

    @property
    def nv(self) -> int:
        return int(sum(_NV[int(t)] for t in self.joint_type))

    @property
    def q_off(self) -> np.ndarray:
        return np.concatenate([[0], np.cumsum([_NQ[int(t)] for t in self.joint_type])]).astype(np.int64)

    @property
    def v_off(self) -> np.ndarray:
        return np.concatenate([[0], np.cumsum([_NV[int(t)] for t in self.joint_type])]).astype(np.int64)


# ----------------------------------------------------------------------------- random pieces

def _quat_to_R(qx, qy, qz, qw) -> np.ndarray:
    """Rotation matrix of a unit quaternion (x, y, z, w); used to DRAW random fixed offsets."""
    x, y, z, w = qx, qy, qz, qw
    return np.array([
        [1 - 2 * (y * y + z * z), 2 * (x * y - z * w), 2 * (x * z + y * w)],
        [2 * (x * y + z * w), 1 - 2 * (x * x + z * z), 2 * (y * z - x * w)],
        [2 * (x * z - y * w), 2 * (y * z + x * w), 1 - 2 * (x * x + y * y)],
    ])


def _Rt12(R: np.ndarray, t: np.ndarray) -> np.ndarray:
    return np.concatenate([R, t.reshape(3, 1)], axis=1).reshape(12)


_IDENTITY12 = _Rt12(np.eye(3), np.zeros(3))


def _draw_link(rng: np.random.Generator):
    """One body's draws, always in this order: axis index, 4 normals (quaternion),
    t_pre, mass, COM, box sides."""
    axis_idx = int(rng.integers(0, 3))
    quat = rng.normal(size=4)
    quat /= np.linalg.norm(quat)
    t_pre = rng.uniform(-0.2, 0.2, size=3)
    mass = float(np.exp(rng.normal(0.0, 0.5)))
    com = rng.uniform(-0.1, 0.1, size=3)
    a, b, c = rng.uniform(0.05, 0.3, size=3)
    ixx, iyy, izz = mass / 12 * (b * b + c * c), mass / 12 * (a * a + c * c), mass / 12 * (a * a + b * b)
    inertia = np.array([ixx, 0.0, 0.0, iyy, 0.0, izz])
    return axis_idx, quat, t_pre, mass, com, inertia


def build_robot(name: str, parent, joint_type, seed: int, fixed_axes=None, frames=(), gravity=(0.0, 0.0, -9.81),
                random_T_post: bool = False, random_frame_offsets: bool = False, full_inertia: bool = False) -> RobotDesc:
    """Seeded link parameters on a given topology.  ``fixed_axes`` maps body -> 0/1/2 to override the drawn axis."""
    rng = np.random.default_rng(seed)
    nb = len(parent)
    axis = np.zeros((nb, 3))
    T_pre = np.zeros((nb, 12))
    mass = np.zeros(nb)
    com = np.zeros((nb, 3))
    inertia = np.zeros((nb, 6))
    for i in range(nb):
        ai, quat, t_pre, m, c, I = _draw_link(rng)
        if fixed_axes and i in fixed_axes:
            ai = fixed_axes[i]
        if int(joint_type[i]) == FREE:
            T_pre[i] = _IDENTITY12
        else:
            T_pre[i] = _Rt12(_quat_to_R(*quat), t_pre)
            if int(joint_type[i]) in (REVOLUTE, PRISMATIC):
                axis[i, ai] = 1.0
        mass[i], com[i], inertia[i] = m, c, I
    T_post = None
    # extras used only by unit-test robots; drawn AFTER the per-link stream so configs 0-3 are unaffected
    if random_T_post:
        T_post = np.zeros((nb, 12))
        for i in range(nb):
            quat = rng.normal(size=4)
            quat /= np.linalg.norm(quat)
            t = rng.uniform(-0.15, 0.15, size=3)
            T_post[i] = _IDENTITY12 if int(joint_type[i]) == FREE else _Rt12(_quat_to_R(*quat), t)
        for i in range(nb):  # general (non axis-aligned) joint axes as well
            if int(joint_type[i]) in (REVOLUTE, PRISMATIC):
                axis[i] = rng.normal(size=3) * rng.uniform(0.5, 2.0)  # deliberately not unit length
    if full_inertia:
        for i in range(nb):  # rotate the box inertia into a general symmetric positive-definite tensor
            quat = rng.normal(size=4)
            quat /= np.linalg.norm(quat)
            R = _quat_to_R(*quat)
            D = np.diag([inertia[i, 0], inertia[i, 3], inertia[i, 5]])
            F = R @ D @ R.T
            inertia[i] = [F[0, 0], F[0, 1], F[0, 2], F[1, 1], F[1, 2], F[2, 2]]
    frame_body = np.asarray(frames, dtype=np.int32)
    frame_offset = rng.uniform(-0.1, 0.1, size=(len(frame_body), 3)) if random_frame_offsets else None
    return RobotDesc(name=name, parent=np.asarray(parent, np.int32), joint_type=np.asarray(joint_type, np.int32),
                     axis=axis, T_pre=T_pre, T_post=T_post, mass=mass, com=com, inertia=inertia,
                     gravity=np.asarray(gravity, float), frame_body=frame_body, frame_offset=frame_offset)


# ----------------------------------------------------------------------------- BASELINE.json configs

def chain7() -> RobotDesc:
    """config 0: 7-DOF fixed-base serial chain of revolute joints, depth 7; frame = end effector."""
    return build_robot("chain7", [-1, 0, 1, 2, 3, 4, 5], [REVOLUTE] * 7, seed=1000, frames=[6])


def quadruped12() -> RobotDesc:
    """config 1: free base + 4 legs x (hip x, hip y, knee y); frames = 4 feet; nv 18."""
    parent = [-1, 0, 1, 2, 0, 4, 5, 0, 7, 8, 0, 10, 11]
    jt = [FREE] + [REVOLUTE] * 12
    fixed = {}
    for leg in range(4):
        fixed[1 + 3 * leg] = 0
        fixed[2 + 3 * leg] = 1
        fixed[3 + 3 * leg] = 1
    return build_robot("quadruped12", parent, jt, seed=1001, fixed_axes=fixed, frames=[3, 6, 9, 12])


def spined_quadruped11() -> RobotDesc:
    """config 2: free base, 3-revolute spine (bodies 1-3), rear legs on spine link 1, front legs on
    spine link 3, 2 revolute joints per leg; frames = 4 feet; nv 17; max depth 6."""
    parent = [-1, 0, 1, 2, 1, 4, 1, 6, 3, 8, 3, 10]
    jt = [FREE] + [REVOLUTE] * 11
    return build_robot("spined_quadruped11", parent, jt, seed=1002, frames=[5, 7, 9, 11])


def humanoid23() -> RobotDesc:
    """config 3: free base, torso chain 1-3, arms (4 DOF) on torso link 2, legs (6 DOF) on the base;
    frames = hands 7, 11 and feet 17, 23; nv 29; max depth 7."""
    parent = [-1, 0, 1, 2, 2, 4, 5, 6, 2, 8, 9, 10, 0, 12, 13, 14, 15, 16, 0, 18, 19, 20, 21, 22]
    jt = [FREE] + [REVOLUTE] * 23
    return build_robot("humanoid23", parent, jt, seed=1003, frames=[7, 11, 17, 23])


CONFIGS = {0: chain7, 1: quadruped12, 2: spined_quadruped11, 3: humanoid23}
CONFIG_NAMES = {0: "chain7", 1: "quadruped12", 2: "spined_quadruped11", 3: "humanoid23"}


def config_robot(cfg: int) -> RobotDesc:
    return CONFIGS[cfg]()


def random_tree(seed: int, nb: int, joint_types=(REVOLUTE, PRISMATIC, FIXED), free_root: bool = False,
                shape: str = "random", nframes: int = 2, general: bool = True) -> RobotDesc:
    """Unit-test robots: random topology (``random`` / ``chain`` / ``star`` / ``unbalanced``), all joint
    types, non-identity T_post, non-unit general axes, full inertia tensors, frame offsets."""
    rng = np.random.default_rng(seed)
    parent = [-1]
    for i in range(1, nb):
        if shape == "chain":
            parent.append(i - 1)
        elif shape == "star":
            parent.append(0)
        elif shape == "unbalanced":
            parent.append(i - 1 if i % 3 else max(0, i - 3))
        else:
            lo = -1 if (not free_root and rng.random() < 0.1) else 0   # occasionally a second root (forest)
            parent.append(int(rng.integers(lo, i)))
    jt = [int(rng.choice(joint_types)) for _ in range(nb)]
    if free_root:
        jt[0] = FREE
    nf = min(nframes, nb)
    frames = sorted(int(x) for x in rng.choice(nb, size=nf, replace=False))
    return build_robot(f"tree{seed}", parent, jt, seed=seed + 7919, frames=frames, random_T_post=general,
                       random_frame_offsets=general, full_inertia=general)


# ----------------------------------------------------------------------------- states

def sample_states(desc: RobotDesc, B: int, seed: int, dtype=np.float32, zero_qd=False, zero_qdd=False):
    """q ~ U(-pi, pi) for revolute (and prismatic, in metres), base p ~ U(-1,1)^3, base quaternion =
    normalised 4 normals, qd ~ N(0,1), qdd ~ N(0,1); drawn in fp64, rounded once to ``dtype``."""
    rng = np.random.default_rng(seed)
    q = np.zeros((desc.nq, B))
    qo = desc.q_off
    for i, t in enumerate(desc.joint_type):
        t = int(t)
        if t in (REVOLUTE, PRISMATIC):
            q[qo[i]] = rng.uniform(-np.pi, np.pi, size=B)
        elif t == FREE:
            q[qo[i]:qo[i] + 3] = rng.uniform(-1.0, 1.0, size=(3, B))
            quat = rng.normal(size=(4, B))
            quat /= np.linalg.norm(quat, axis=0, keepdims=True)
            q[qo[i] + 3:qo[i] + 7] = quat
    qd = rng.normal(size=(desc.nv, B))
    qdd = rng.normal(size=(desc.nv, B))
    if zero_qd:
        qd[:] = 0
    if zero_qdd:
        qdd[:] = 0
    return (np.ascontiguousarray(q.astype(dtype)), np.ascontiguousarray(qd.astype(dtype)),
            np.ascontiguousarray(qdd.astype(dtype)))


def config_states(cfg: int, B: int, step: int = 0, dtype=np.float32):
    """State seed 2000 + config (+ step), SURVEY 8(d)."""
    return sample_states(config_robot(cfg), B, seed=2000 + cfg + 100 * step, dtype=dtype)
