"""fp64 CPU oracle for the batched rigid-body operators -- TEST INFRASTRUCTURE, not product.

Thin ctypes wrapper around ``oracle/bard_oracle.c`` (plain C, dense 6x6 Featherstone recursions,
see the header of ``bard_oracle.h`` for conventions and citations).  Only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may
import this package.  It imports nothing from ``paper_2605_31481_b200`` and shares no code with it.

A robot description is any object with the attributes
``parent, joint_type, axis, T_pre, T_post (or None), mass, com, inertia, gravity,
frame_body, frame_offset (or None)`` (numpy-convertible).  Batched arrays are SoA, batch last:
``q[nq, B]``, ``qd[nv, B]``, ``pose[nb, 12, B]``, ``J[nframes, 6, nv, B]``, ``M[nv, nv, B]``.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "bard_oracle.c")
_HDR = os.path.join(_HERE, "bard_oracle.h")
_SO = os.path.join(_HERE, "libbard_oracle.so")


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (C99, -O2, OpenMP over environments only)."""
    stale = (not os.path.exists(_SO)) or os.path.getmtime(_SO) < max(os.path.getmtime(_SRC), os.path.getmtime(_HDR))
    if force or stale:
        tmp = _SO + f".tmp{os.getpid()}"
        cmd = ["gcc", "-std=c99", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", tmp, _SRC, "-lm"]
        subprocess.run(cmd, check=True, cwd=_HERE)
        os.replace(tmp, _SO)
    return _SO


class _Desc(C.Structure):
    _fields_ = [
        ("nb", C.c_int32),
        ("parent", C.POINTER(C.c_int32)),
        ("joint_type", C.POINTER(C.c_int32)),
        ("axis", C.POINTER(C.c_double)),
        ("T_pre", C.POINTER(C.c_double)),
        ("T_post", C.POINTER(C.c_double)),
        ("mass", C.POINTER(C.c_double)),
        ("com", C.POINTER(C.c_double)),
        ("inertia", C.POINTER(C.c_double)),
        ("gravity", C.c_double * 3),
        ("nframes", C.c_int32),
        ("frame_body", C.POINTER(C.c_int32)),
        ("frame_offset", C.POINTER(C.c_double)),
    ]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        dp = C.POINTER(C.c_double)
        P = C.POINTER(_Desc)
        L.bard_oracle_dims.argtypes = [P, C.POINTER(C.c_int32), C.POINTER(C.c_int32), C.POINTER(C.c_int32)]
        L.bard_oracle_table.argtypes = [P, C.c_int, C.POINTER(C.c_int64), C.c_int64]
        L.bard_oracle_rodrigues.argtypes = [P, dp]
        L.bard_oracle_fk_rodrigues.argtypes = [P, C.c_int64, dp, dp]
        L.bard_oracle_fk.argtypes = [P, C.c_int64, dp, dp]
        L.bard_oracle_jacobian.argtypes = [P, C.c_int64, dp, dp]
        L.bard_oracle_rnea.argtypes = [P, C.c_int64, dp, dp, dp, dp]
        L.bard_oracle_crba.argtypes = [P, C.c_int64, dp, dp]
        L.bard_oracle_body_velocity.argtypes = [P, C.c_int64, dp, dp, dp]
        L.bard_oracle_euler_step.argtypes = [P, C.c_int64, C.c_double, dp, dp, dp]
        L.bard_oracle_spatial_inertia.argtypes = [P, C.c_int32, dp]
        L.bard_oracle_rnea_params.argtypes = [P, C.c_int64, dp, dp, dp, dp, dp]
        L.bard_oracle_inertial_params.argtypes = [P, dp]
        L.bard_oracle_rnea_vjp_params.argtypes = [P, C.c_int64, dp, dp, dp, dp, dp]
        L.bard_oracle_set_threads.argtypes = [C.c_int]
        L.bard_oracle_get_threads.restype = C.c_int
        _lib = L
    return _lib


def set_threads(n: int) -> None:
    lib().bard_oracle_set_threads(int(n))


def get_threads() -> int:
    return int(lib().bard_oracle_get_threads())


TABLES = {
    "LEVEL_PTR": 0, "LEVEL_BODY": 1, "BODY_LEVEL": 2, "PARENT_SLOT": 3,
    "Q_OFF": 4, "V_OFF": 5, "DOF_BODY": 6, "ANC_MASK": 7,
}


def _dptr(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _f64(a, shape=None):
    a = np.ascontiguousarray(np.asarray(a, dtype=np.float64))
    if shape is not None:
        a = a.reshape(shape)
    return a


class Oracle:
    """Holds one robot description and evaluates the four operators in fp64 on the host."""

    def __init__(self, desc):
        self._keep = {}
        nb = int(len(np.asarray(desc.parent)))
        k = self._keep
        k["parent"] = np.ascontiguousarray(np.asarray(desc.parent, dtype=np.int32))
        k["joint_type"] = np.ascontiguousarray(np.asarray(desc.joint_type, dtype=np.int32))
        k["axis"] = _f64(desc.axis, (nb, 3))
        k["T_pre"] = _f64(desc.T_pre, (nb, 12))
        k["T_post"] = None if getattr(desc, "T_post", None) is None else _f64(desc.T_post, (nb, 12))
        k["mass"] = _f64(desc.mass, (nb,))
        k["com"] = _f64(desc.com, (nb, 3))
        k["inertia"] = _f64(desc.inertia, (nb, 6))
        fb = getattr(desc, "frame_body", None)
        k["frame_body"] = np.ascontiguousarray(np.asarray([] if fb is None else fb, dtype=np.int32))
        fo = getattr(desc, "frame_offset", None)
        k["frame_offset"] = None if fo is None else _f64(fo, (len(k["frame_body"]), 3))
        d = _Desc()
        d.nb = nb
        ip = C.POINTER(C.c_int32)
        d.parent = k["parent"].ctypes.data_as(ip)
        d.joint_type = k["joint_type"].ctypes.data_as(ip)
        d.axis = _dptr(k["axis"])
        d.T_pre = _dptr(k["T_pre"])
        d.T_post = _dptr(k["T_post"]) if k["T_post"] is not None else None
        d.mass = _dptr(k["mass"])
        d.com = _dptr(k["com"])
        d.inertia = _dptr(k["inertia"])
        g = _f64(desc.gravity, (3,))
        for i in range(3):
            d.gravity[i] = float(g[i])
        d.nframes = len(k["frame_body"])
        d.frame_body = k["frame_body"].ctypes.data_as(ip) if d.nframes else None
        d.frame_offset = _dptr(k["frame_offset"]) if k["frame_offset"] is not None else None
        self._d = d
        nq, nv, nl = C.c_int32(), C.c_int32(), C.c_int32()
        rc = lib().bard_oracle_dims(C.byref(d), C.byref(nq), C.byref(nv), C.byref(nl))
        if rc:
            raise ValueError(f"oracle rejected the robot description (code {rc})")
        self.nb, self.nq, self.nv, self.nlevels, self.nframes = nb, nq.value, nv.value, nl.value, d.nframes

    # -- tables -------------------------------------------------------------------------
    def table(self, name: str) -> np.ndarray:
        cap = max(self.nb, self.nv, self.nlevels) + 2
        out = np.zeros(cap, dtype=np.int64)
        n = lib().bard_oracle_table(C.byref(self._d), TABLES[name], out.ctypes.data_as(C.POINTER(C.c_int64)), cap)
        if n < 0:
            raise RuntimeError(f"oracle table {name} failed ({n})")
        out = out[:n]
        return out.view(np.uint64) if name == "ANC_MASK" else out

    def rodrigues(self) -> np.ndarray:
        out = np.zeros((self.nb, 36))
        self._chk(lib().bard_oracle_rodrigues(C.byref(self._d), _dptr(out)))
        return out

    # -- operators ----------------------------------------------------------------------
    @staticmethod
    def _chk(rc):
        if rc:
            raise RuntimeError(f"oracle call failed (code {rc})")

    def _in(self, a, n):
        a = _f64(a)
        if a.ndim == 1:
            a = a.reshape(n, 1)
        assert a.shape[0] == n, (a.shape, n)
        return a

    def fk(self, q) -> np.ndarray:
        q = self._in(q, self.nq)
        B = q.shape[1]
        out = np.zeros((self.nb, 12, B))
        self._chk(lib().bard_oracle_fk(C.byref(self._d), B, _dptr(q), _dptr(out)))
        return out

    def fk_rodrigues(self, q) -> np.ndarray:
        q = self._in(q, self.nq)
        B = q.shape[1]
        out = np.zeros((self.nb, 12, B))
        self._chk(lib().bard_oracle_fk_rodrigues(C.byref(self._d), B, _dptr(q), _dptr(out)))
        return out

    def jacobian(self, q) -> np.ndarray:
        q = self._in(q, self.nq)
        B = q.shape[1]
        out = np.zeros((self.nframes, 6, self.nv, B))
        self._chk(lib().bard_oracle_jacobian(C.byref(self._d), B, _dptr(q), _dptr(out)))
        return out

    def rnea(self, q, qd, qdd) -> np.ndarray:
        q = self._in(q, self.nq)
        qd = self._in(qd, self.nv)
        qdd = self._in(qdd, self.nv)
        B = q.shape[1]
        out = np.zeros((self.nv, B))
        self._chk(lib().bard_oracle_rnea(C.byref(self._d), B, _dptr(q), _dptr(qd), _dptr(qdd), _dptr(out)))
        return out

    def crba(self, q) -> np.ndarray:
        q = self._in(q, self.nq)
        B = q.shape[1]
        out = np.zeros((self.nv, self.nv, B))
        self._chk(lib().bard_oracle_crba(C.byref(self._d), B, _dptr(q), _dptr(out)))
        return out

    def euler_step(self, dt, q, qd, qdd):
        """One explicit Euler step of the config-2 rollout: returns the new (q, qd)."""
        q = np.array(self._in(q, self.nq), copy=True)
        qd = np.array(self._in(qd, self.nv), copy=True)
        qdd = self._in(qdd, self.nv)
        self._chk(lib().bard_oracle_euler_step(C.byref(self._d), q.shape[1], float(dt), _dptr(q), _dptr(qd), _dptr(qdd)))
        return q, qd

    def aba(self, q, qd, tau) -> np.ndarray:
        """Forward dynamics by its definition: the qdd that solves M(q) qdd + C(q, qd) = tau, with M from CRBA,
        C = RNEA(q, qd, 0) (gravity included) and a dense fp64 solve per environment (numpy.linalg.solve).  The
        paper's ABA reaches exactly this result by an O(n) recursion."""
        q = self._in(q, self.nq)
        qd = self._in(qd, self.nv)
        tau = self._in(tau, self.nv)
        M = self.crba(q)                                      # [nv, nv, B]
        C0 = self.rnea(q, qd, np.zeros_like(qd))              # [nv, B]
        rhs = (tau - C0).T[:, :, None]                        # [B, nv, 1]
        return np.ascontiguousarray(np.linalg.solve(np.moveaxis(M, 2, 0), rhs)[:, :, 0].T)

    # -- RNEA as a function of the inertial parameters --------------------
    def inertial_params(self) -> np.ndarray:
        """[nb, 10]: m, h = m c, Io (xx,xy,xz,yy,yz,zz about the body origin) of every link of the description."""
        out = np.zeros((self.nb, 10))
        self._chk(lib().bard_oracle_inertial_params(C.byref(self._d), _dptr(out)))
        return out

    def rnea_params(self, q, qd, qdd, params) -> np.ndarray:
        q = self._in(q, self.nq)
        qd = self._in(qd, self.nv)
        qdd = self._in(qdd, self.nv)
        params = _f64(params, (self.nb, 10))
        B = q.shape[1]
        out = np.zeros((self.nv, B))
        self._chk(lib().bard_oracle_rnea_params(C.byref(self._d), B, _dptr(q), _dptr(qd), _dptr(qdd), _dptr(params), _dptr(out)))
        return out

    def rnea_vjp_params(self, q, qd, qdd, dtau) -> np.ndarray:
        """dparams[nb, 10] = sum_b (d tau_b / d params)^T dtau_b, by the definition (linearity in the parameters)."""
        q = self._in(q, self.nq)
        qd = self._in(qd, self.nv)
        qdd = self._in(qdd, self.nv)
        dtau = self._in(dtau, self.nv)
        out = np.zeros((self.nb, 10))
        self._chk(lib().bard_oracle_rnea_vjp_params(C.byref(self._d), q.shape[1], _dptr(q), _dptr(qd), _dptr(qdd), _dptr(dtau), _dptr(out)))
        return out

    def body_velocity(self, q, qd) -> np.ndarray:
        q = self._in(q, self.nq)
        qd = self._in(qd, self.nv)
        B = q.shape[1]
        out = np.zeros((self.nb, 6, B))
        self._chk(lib().bard_oracle_body_velocity(C.byref(self._d), B, _dptr(q), _dptr(qd), _dptr(out)))
        return out

    def spatial_inertia(self, body: int) -> np.ndarray:
        out = np.zeros((6, 6))
        self._chk(lib().bard_oracle_spatial_inertia(C.byref(self._d), int(body), _dptr(out)))
        return out
