"""Algorithmic bytes and FP32 FLOPs per environment for each operator (counting only; no kernel arithmetic).

The roofline of north_star is "the slower of analytically counted FP32 FLOPs at peak and the bytes of
q, qd, qdd in plus outputs out at HBM bandwidth".  This module re-derives SURVEY.md section 8(d)'s table from
the robot description with the primitive costs of SURVEY.md Appendix A (mul and add 1 FLOP each, FMA 2,
sin/cos/rsqrt 1 each; T_post = I; structural zeros of S = [a; 0] and of world-attached bodies skipped):

  Rodrigues R_pc (eq. (4)) incl. sincos 39 | unit quaternion -> R 36 | pose compose 63 |
  axis to world 15 | Jacobian column 12 (revolute) / 30 (free base, 6 columns) |
  RNEA non-root revolute body 332 = 39 + 48 (v) + 72 (a) + 120 (f) + 5 (tau) + 48 (force to parent)
  RNEA root revolute body 188, free root body 177 |
  CRBA: 39 per revolute + 36 per free + 145 per non-root body (inertia congruence + accumulate)
        + 29 per revolute DOF (F = I^c S, S^T F) + 47 per (DOF, revolute ancestor DOF) pair
        + 42 per (DOF, free-base ancestor) pair.

The roofline fraction always uses these ALGORITHMIC counts, never the executed ones.
"""
from __future__ import annotations

import json
import os

import numpy as np

REVOLUTE, PRISMATIC, FIXED, FREE = 0, 1, 2, 3
SM_COUNT = 148
FP32_LANES_PER_SM = 128
HBM_FALLBACK_GBS = 6650.0      # B200_PROFILING.md fallback
SM_MAX_MHZ_FALLBACK = 1965.0


def measured_peaks(root: str | None = None, fp32_measured: float | None = None) -> dict:
    """HBM GB/s from MEASURED_PEAKS.json (driver-written) or the profiling guide's fallback; the plain-FP32
    peak is derived: 148 SMs x 128 FMA lanes x 2 FLOP x max SM clock.  If the caller measured
    the FFMA throughput on the box (``binding.measure_fp32_peak``: an FFMA-chain kernel) both figures are recorded and
    the "alu" roofline divides by min(measured, nominal) -- what the FMA pipes of THIS box deliver."""
    root = root or os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    p = os.path.join(root, "MEASURED_PEAKS.json")
    hbm, mhz, src = HBM_FALLBACK_GBS, SM_MAX_MHZ_FALLBACK, "fallback"
    if os.path.exists(p):
        try:
            d = json.load(open(p))
            hbm, mhz, src = float(d["hbm_gbs"]), float(d.get("sm_max_mhz", mhz)), "measured"
        except Exception:
            pass
    nominal = SM_COUNT * FP32_LANES_PER_SM * 2 * mhz * 1e6 / 1e12
    fp32 = min(nominal, fp32_measured) if fp32_measured else nominal
    return {"hbm_gbs": hbm, "fp32_tflops": fp32, "fp32_tflops_nominal": nominal, "fp32_tflops_measured": fp32_measured,
            "sm_max_mhz": mhz, "source": src}


def _ancestors(parent, i):
    out = []
    j = int(parent[i])
    while j >= 0:
        out.append(j)
        j = int(parent[j])
    return out


def counts(desc) -> dict:
    """{op: {"in": bytes, "out": bytes, "bytes": total, "flop": FLOPs}} per environment."""
    parent = np.asarray(desc.parent)
    jt = [int(t) for t in desc.joint_type]
    nb = len(jt)
    nq = sum({REVOLUTE: 1, PRISMATIC: 1, FIXED: 0, FREE: 7}[t] for t in jt)
    nv = sum({REVOLUTE: 1, PRISMATIC: 1, FIXED: 0, FREE: 6}[t] for t in jt)
    frames = [int(b) for b in np.asarray(desc.frame_body).reshape(-1)]
    nf = len(frames)

    def xform(t):
        return 36 if t == FREE else (39 if t == REVOLUTE else (12 if t == PRISMATIC else 0))

    fk = sum(xform(jt[i]) + (63 if parent[i] >= 0 else 0) for i in range(nb))

    used = set()
    for b in frames:
        used.add(b)
        used.update(_ancestors(parent, b))
    jac = sum(xform(jt[i]) + (63 if parent[i] >= 0 else 0) for i in used)
    jac += sum(15 for i in used if jt[i] in (REVOLUTE, PRISMATIC))
    for b in frames:
        for i in [b] + _ancestors(parent, b):
            jac += 12 if jt[i] in (REVOLUTE, PRISMATIC) else (30 if jt[i] == FREE else 0)

    rnea = 0
    for i in range(nb):
        root = parent[i] < 0
        if jt[i] == FREE:
            rnea += 177 if root else 177 + 42 + 42 + 30 + 48
        elif jt[i] == FIXED:
            rnea += (15 if root else 84) + 120 + (0 if root else 48)
        else:
            rnea += (188 if root else 332) - (39 - xform(jt[i]))

    crba = sum(xform(jt[i]) + (145 if parent[i] >= 0 else 0) for i in range(nb))
    for i in range(nb):
        nd_i = {REVOLUTE: 1, PRISMATIC: 1, FIXED: 0, FREE: 6}[jt[i]]
        if jt[i] in (REVOLUTE, PRISMATIC):
            crba += 29
        for j in _ancestors(parent, i):
            if jt[j] in (REVOLUTE, PRISMATIC):
                crba += 47 * nd_i
            elif jt[j] == FREE:
                crba += 42 * nd_i

    # ABA, three passes, compact algebra, per body: joint transform; v (48) and c = v x S qd (24);
    # p^A = v x* I v (72); U = I^A S (66), D (5), u (6), I^a = I^A - U U^T / D (48), p^a = p^A + I^a c + U u / D (78);
    # X^T I^a X as rotate (I, M symmetric 75 each, H general 90) + translate (96) = 336, X^T p^a (42), accumulate (27);
    # pass 3: a' = X a_p + c (48), qdd = (u - U^T a') / D (13), a = a' + S qdd (6).  Root bodies skip the parent terms;
    # a free root solves a 6x6 SPD system instead (LDL^T ~ 200).
    aba = 0
    for i in range(nb):
        root = parent[i] < 0
        if jt[i] == FREE:
            aba += 36 + 72 + 200 + 30
        else:
            has_dof = jt[i] != FIXED
            aba += xform(jt[i]) + (0 if root else 48 + 24) + 72 + (66 + 5 + 6 if has_dof else 0)
            aba += (0 if root else (48 if has_dof else 0) + 78 + 336 + 42 + 27) + (48 + (13 + 6 if has_dof else 0))

    # RNEA VJP w.r.t. the inertial parameters, one outward pass, per body: joint transform; X_up on v, a and
    # the pushed cotangent lambda (42 each: R^T w 15, w x t 9, + 3, R^T (.) 15); S qd, S qdd, S dtau and their adds (36);
    # a += v x S qd (36); u = v x lambda (30); the ten bilinear terms (86: m 11, h 45, Io 30); the batch sum (10).
    # Root bodies: v = S qd, a = R^T (-g) + S qdd, lambda = S dtau.  Free joints: the joint vectors are the inputs themselves.
    vjp = 0
    for i in range(nb):
        root = parent[i] < 0
        if jt[i] == FREE:
            vjp += 36 + (18 if root else 126 + 18 + 36) + 30 + 86 + 10
        elif jt[i] == FIXED:
            vjp += (15 if root else 126) + 30 + 86 + 10
        else:
            vjp += xform(jt[i]) + (36 if root else 126 + 36 + 36) + 30 + 86 + 10

    def row(i, o, f):
        return {"in": i, "out": o, "bytes": i + o, "flop": f}

    return {
        "fk": row(4 * nq, 48 * nb, fk),
        "jacobian": row(4 * nq, 24 * nf * nv, jac),
        "rnea": row(4 * (nq + 2 * nv), 4 * nv, rnea),
        "crba": row(4 * nq, 4 * nv * nv, crba),
        "aba": row(4 * (nq + 2 * nv), 4 * nv, aba),
        "rnea_vjp": row(4 * (nq + 3 * nv), 0, vjp),
        # bard_kinematics: q read once; FK is part of CRBA's walk, the Jacobian adds its axis and column work
        "kin": row(4 * nq, 48 * nb + 24 * nf * nv + 4 * nv * nv, crba + jac - sum(xform(jt[i]) + (63 if parent[i] >= 0 else 0) for i in used)),
    }


def roofline(desc, peaks: dict | None = None) -> dict:
    """Per op: which roof binds and the roofline time per environment (seconds)."""
    pk = peaks or measured_peaks()
    out = {}
    for op, c in counts(desc).items():
        t_hbm = c["bytes"] / (pk["hbm_gbs"] * 1e9)
        t_alu = c["flop"] / (pk["fp32_tflops"] * 1e12)
        bound = "hbm" if t_hbm >= t_alu else "alu"
        out[op] = dict(c, bound=bound, t_env=max(t_hbm, t_alu), t_hbm=t_hbm, t_alu=t_alu)
    return out


if __name__ == "__main__":
    from . import workloads as W
    pk = measured_peaks()
    print(pk)
    for cfg in range(4):
        d = W.config_robot(cfg)
        for op, r in roofline(d, pk).items():
            print(f"c{cfg} {d.name:20s} {op:9s} in {r['in']:5d} out {r['out']:5d} total {r['bytes']:5d} B  "
                  f"{r['flop']:5d} FLOP  {r['flop'] / r['bytes']:5.1f} FLOP/B  {r['bound']:3s}  "
                  f"{1e-9 / r['t_env']:6.2f} Genv/s")
