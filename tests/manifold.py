"""Test helper: the configuration-manifold step q (+) dv written in numpy, independently of the oracle's C code.

Used by the oracle pins as a finite-difference stencil (Jacobians, potential gradient, kinetic-energy rate), as the
second formulation that pins ``bard_oracle_euler_step`` (tests/test_euler.py), and to roll config 2 forward on the
host.  It is test code: neither ``oracle/`` nor ``paper_2605_31481_b200/`` imports it.
"""
from __future__ import annotations

import numpy as np

from paper_2605_31481_b200.workloads import FREE, PRISMATIC, REVOLUTE, RobotDesc, config_robot, sample_states


def _quat_to_R(x, y, z, w) -> np.ndarray:
    return np.array([
        [1 - 2 * (y * y + z * z), 2 * (x * y - z * w), 2 * (x * z + y * w)],
        [2 * (x * y + z * w), 1 - 2 * (x * x + z * z), 2 * (y * z - x * w)],
        [2 * (x * z - y * w), 2 * (y * z + x * w), 1 - 2 * (x * x + y * y)],
    ])


def manifold_step(desc: RobotDesc, q: np.ndarray, dv: np.ndarray) -> np.ndarray:
    """q (+) dv: revolute/prismatic add; free base p += R(quat) v, quat += 1/2 quat (x) (omega, 0), renormalised.
    ``dv`` is a tangent increment (already multiplied by dt), layout [nv, B].  Used to roll config 2 forward
    (explicit Euler) and for finite-difference test stencils."""
    q = np.array(q, dtype=np.float64, copy=True)
    qo, vo = desc.q_off, desc.v_off
    for i, t in enumerate(desc.joint_type):
        t = int(t)
        if t in (REVOLUTE, PRISMATIC):
            q[qo[i]] += dv[vo[i]]
        elif t == FREE:
            x, y, z, w = q[qo[i] + 3:qo[i] + 7]
            n = np.sqrt(x * x + y * y + z * z + w * w)
            x, y, z, w = x / n, y / n, z / n, w / n
            v, om = dv[vo[i]:vo[i] + 3], dv[vo[i] + 3:vo[i] + 6]
            R = _quat_to_R(x, y, z, w)  # [3,3,B]
            q[qo[i]:qo[i] + 3] += np.einsum("ijb,jb->ib", R, v)
            # quaternion product quat (x) (om, 0): body-frame angular increment
            ox, oy, oz = om
            dx = 0.5 * (w * ox + y * oz - z * oy)
            dy = 0.5 * (w * oy + z * ox - x * oz)
            dz = 0.5 * (w * oz + x * oy - y * ox)
            dw = 0.5 * (-x * ox - y * oy - z * oz)
            nq4 = np.stack([x + dx, y + dy, z + dz, w + dw])
            nq4 /= np.linalg.norm(nq4, axis=0, keepdims=True)
            q[qo[i] + 3:qo[i] + 7] = nq4
    return q


def euler_rollout(cfg: int, B: int, steps: int = 24, dt: float = 0.005, dtype=np.float32):
    """config 2 style trajectory: per step fresh seeded qdd, qd += dt qdd, q (+)= dt qd.  Returns a list of
    (q, qd, qdd) per step, each rounded once to ``dtype`` (the state carried forward stays fp64)."""
    desc = config_robot(cfg)
    q, qd, _ = sample_states(desc, B, seed=2000 + cfg, dtype=np.float64)
    out = []
    for s in range(steps):
        rng = np.random.default_rng(2000 + cfg + 100 * (s + 1))
        qdd = rng.normal(size=(desc.nv, B))
        out.append((np.ascontiguousarray(q.astype(dtype)), np.ascontiguousarray(qd.astype(dtype)),
                    np.ascontiguousarray(qdd.astype(dtype))))
        qd = qd + dt * qdd
        q = manifold_step(desc, q, dt * qd)
    return out
