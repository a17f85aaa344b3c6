"""Thin ctypes binding of ``libbard.so`` (``include/bard.h``): argument marshalling only.

Every step of the hot path runs in the CUDA kernels of the library.  There is NO CPU fallback: if the
library is missing and cannot be built, importing fails loudly; operator calls on a machine without CUDA
raise ``BardError``.  PyTorch is used by callers only for device memory and streams; tensors are passed
as raw device pointers (``tensor.data_ptr()``) and the current CUDA stream handle.

Layouts are the library's: SoA, batch last -- ``q[nq, B]``, ``qd[nv, B]``, ``qdd[nv, B]``,
``pose[nb, 12, B]``, ``J[nframes, 6, nv, B]``, ``tau[nv, B]``, ``M[nv, nv, B]`` (fp32, contiguous).
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

BARD_OK = 0
STATUS = {0: "BARD_OK", 1: "BARD_ERR_INVALID_ARG", 2: "BARD_ERR_TOPOLOGY", 3: "BARD_ERR_UNSUPPORTED",
          4: "BARD_ERR_ALLOC", 5: "BARD_ERR_CUDA"}
VJP_STATIC_SCRATCH_FLOATS = 262144      # BARD_VJP_STATIC_SCRATCH_FLOATS in include/bard.h
OPS = {"fk": 1, "jacobian": 2, "rnea": 4, "crba": 8, "fused": 16, "aba": 32, "rnea_roles": 64, "crba_roles": 128, "rnea_pack2": 256, "kin": 512, "rnea_vjp": 1024}
DTYPES = {"f32": 0, "f64": 1}
LAYOUTS = {"soa": 0, "aos": 1}
TABLES = {"LEVEL_PTR": (0, np.int32), "LEVEL_BODY": (1, np.int32), "BODY_LEVEL": (2, np.int32),
          "PARENT_SLOT": (3, np.int32), "Q_OFF": (4, np.int32), "V_OFF": (5, np.int32), "DOF_BODY": (6, np.int32),
          "ANC_MASK": (7, np.uint64), "RODRIGUES": (8, np.float32)}
EXPORTS = ["bard_model_create", "bard_model_destroy", "bard_model_dims", "bard_model_get_table",
           "bard_model_set_frames", "bard_model_set_option", "bard_model_get_option", "bard_model_specialize", "bard_model_specialized_source", "bard_fk", "bard_jacobian", "bard_rnea", "bard_crba", "bard_kinematics", "bard_step", "bard_euler_step", "bard_euler_step_to", "bard_aba", "bard_aba_workspace_floats", "bard_rnea_vjp_params", "bard_rnea_vjp_params_static", "bard_rnea_vjp_workspace_floats",
           "bard_model_inertial_params", "bard_model_set_inertial_params", "bard_model_specialize_variant", "bard_model_variant_source",
           "bard_variant_workspace_bytes", "bard_fk_v", "bard_jacobian_v", "bard_rnea_v", "bard_crba_v", "bard_measure_fp32_peak",
           "bard_status_string", "bard_last_error", "bard_launch_count"]


class BardError(RuntimeError):
    def __init__(self, code: int, detail: str):
        super().__init__(f"{STATUS.get(code, code)}: {detail}")
        self.code = code


class _Desc(C.Structure):
    _fields_ = [("nb", C.c_int32), ("parent", C.POINTER(C.c_int32)), ("joint_type", C.POINTER(C.c_int32)),
                ("axis", C.POINTER(C.c_double)), ("T_pre", C.POINTER(C.c_double)), ("T_post", C.POINTER(C.c_double)),
                ("mass", C.POINTER(C.c_double)), ("com", C.POINTER(C.c_double)), ("inertia", C.POINTER(C.c_double)),
                ("gravity", C.c_double * 3)]


_lib = None


def lib():
    """Load (building first if stale) the C-ABI library; raises if it cannot be produced."""
    global _lib
    if _lib is None:
        path = _build.build()
        if not os.path.exists(path):
            raise ImportError("libbard.so is missing and could not be built; there is no CPU fallback")
        L = C.CDLL(path)
        vp, i64, fp = C.c_void_p, C.c_int64, C.c_void_p
        L.bard_model_create.argtypes = [C.POINTER(_Desc), C.c_int, C.POINTER(vp)]
        L.bard_model_destroy.argtypes = [vp]
        L.bard_model_destroy.restype = None
        L.bard_model_dims.argtypes = [vp] + [C.POINTER(C.c_int32)] * 4
        L.bard_model_get_table.argtypes = [vp, C.c_int, vp, C.c_size_t, C.POINTER(C.c_size_t)]
        L.bard_model_set_frames.argtypes = [vp, C.c_int32, C.POINTER(C.c_int32), C.POINTER(C.c_double)]
        L.bard_model_set_option.argtypes = [vp, C.c_char_p, C.c_int64]
        L.bard_model_get_option.argtypes = [vp, C.c_char_p, C.POINTER(C.c_int64)]
        L.bard_model_specialize.argtypes = [vp, C.c_uint32]
        L.bard_model_specialized_source.argtypes = [vp, C.c_uint32, C.c_char_p, C.c_size_t, C.POINTER(C.c_size_t)]
        L.bard_fk.argtypes = [vp, i64, fp, fp, vp]
        L.bard_jacobian.argtypes = [vp, i64, fp, fp, vp]
        L.bard_rnea.argtypes = [vp, i64, fp, fp, fp, fp, vp]
        L.bard_crba.argtypes = [vp, i64, fp, fp, vp]
        L.bard_kinematics.argtypes = [vp, i64, fp, fp, fp, fp, vp]
        L.bard_step.argtypes = [vp, i64, fp, fp, fp, fp, fp, fp, fp, vp]
        L.bard_euler_step.argtypes = [vp, i64, C.c_float, fp, fp, fp, vp]
        L.bard_euler_step_to.argtypes = [vp, i64, C.c_float, fp, fp, fp, fp, fp, vp]
        L.bard_aba.argtypes = [vp, i64, fp, fp, fp, fp, fp, vp]
        L.bard_aba_workspace_floats.argtypes = [vp, i64]
        L.bard_aba_workspace_floats.restype = C.c_size_t
        L.bard_rnea_vjp_workspace_floats.argtypes = [vp, i64]
        L.bard_rnea_vjp_workspace_floats.restype = C.c_size_t
        L.bard_rnea_vjp_params.argtypes = [vp, i64, fp, fp, fp, fp, fp, fp, vp]
        L.bard_rnea_vjp_params_static.argtypes = [vp, i64, fp, fp, fp, fp, fp, vp]
        L.bard_model_inertial_params.argtypes = [vp, C.POINTER(C.c_double)]
        L.bard_model_set_inertial_params.argtypes = [vp, C.POINTER(C.c_double)]
        L.bard_model_specialize_variant.argtypes = [vp, C.c_uint32, C.c_int, C.c_int]
        L.bard_model_variant_source.argtypes = [vp, C.c_uint32, C.c_int, C.c_int, C.c_char_p, C.c_size_t, C.POINTER(C.c_size_t)]
        L.bard_variant_workspace_bytes.argtypes = [vp, C.c_uint32, C.c_int, C.c_int, i64]
        L.bard_variant_workspace_bytes.restype = C.c_size_t
        L.bard_fk_v.argtypes = [vp, C.c_int, C.c_int, i64, fp, fp, fp, vp]
        L.bard_jacobian_v.argtypes = [vp, C.c_int, C.c_int, i64, fp, fp, fp, vp]
        L.bard_rnea_v.argtypes = [vp, C.c_int, C.c_int, i64, fp, fp, fp, fp, fp, vp]
        L.bard_crba_v.argtypes = [vp, C.c_int, C.c_int, i64, fp, fp, fp, vp]
        L.bard_measure_fp32_peak.argtypes = [C.c_int, C.POINTER(C.c_double)]
        L.bard_status_string.argtypes = [C.c_int]
        L.bard_status_string.restype = C.c_char_p
        L.bard_last_error.restype = C.c_char_p
        L.bard_launch_count.restype = C.c_int64
        _lib = L
    return _lib


def _check(code: int):
    if code != BARD_OK:
        raise BardError(code, lib().bard_last_error().decode())


def measure_fp32_peak(device: int = 0) -> float:
    """Measured plain-FP32 FMA throughput of the device in TFLOP/s (``bard_measure_fp32_peak``)."""
    v = C.c_double()
    _check(lib().bard_measure_fp32_peak(int(device), C.byref(v)))
    return float(v.value)


def launch_count() -> int:
    return int(lib().bard_launch_count())


def _f64(a, shape):
    return np.ascontiguousarray(np.asarray(a, dtype=np.float64).reshape(shape))


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _ptr(t):
    """Raw pointer of a torch tensor / anything with data_ptr(); ints pass through."""
    if t is None:
        return None
    if isinstance(t, int):
        return t
    return int(t.data_ptr())


class Model:
    """An immutable robot model on one CUDA device (``device=-1``: host-only, tables can be queried)."""

    def __init__(self, desc, device: int = 0):
        L = lib()
        nb = int(len(np.asarray(desc.parent)))
        keep = {
            "parent": np.ascontiguousarray(np.asarray(desc.parent, dtype=np.int32)),
            "joint_type": np.ascontiguousarray(np.asarray(desc.joint_type, dtype=np.int32)),
            "axis": _f64(desc.axis, (nb, 3)), "T_pre": _f64(desc.T_pre, (nb, 12)),
            "T_post": None if getattr(desc, "T_post", None) is None else _f64(desc.T_post, (nb, 12)),
            "mass": _f64(desc.mass, (nb,)), "com": _f64(desc.com, (nb, 3)), "inertia": _f64(desc.inertia, (nb, 6)),
        }
        d = _Desc()
        ip = C.POINTER(C.c_int32)
        d.nb = nb
        d.parent = keep["parent"].ctypes.data_as(ip)
        d.joint_type = keep["joint_type"].ctypes.data_as(ip)
        d.axis, d.T_pre = _dp(keep["axis"]), _dp(keep["T_pre"])
        d.T_post = _dp(keep["T_post"]) if keep["T_post"] is not None else None
        d.mass, d.com, d.inertia = _dp(keep["mass"]), _dp(keep["com"]), _dp(keep["inertia"])
        g = np.asarray(desc.gravity, dtype=np.float64).reshape(3)
        for k in range(3):
            d.gravity[k] = float(g[k])
        h = C.c_void_p()
        _check(L.bard_model_create(C.byref(d), int(device), C.byref(h)))
        self._h = h
        self.device = int(device)
        v = [C.c_int32() for _ in range(4)]
        _check(L.bard_model_dims(h, *[C.byref(x) for x in v]))
        self.nb, self.nq, self.nv, self.nlevels = (int(x.value) for x in v)
        self.nframes = 0
        fb = getattr(desc, "frame_body", None)
        if fb is not None and len(fb):
            self.set_frames(fb, getattr(desc, "frame_offset", None))

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            lib().bard_model_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_frames(self, body, offset=None):
        body = np.ascontiguousarray(np.asarray(body, dtype=np.int32))
        off = None if offset is None else _f64(offset, (len(body), 3))
        _check(lib().bard_model_set_frames(self._h, len(body), body.ctypes.data_as(C.POINTER(C.c_int32)),
                                           _dp(off) if off is not None else None))
        self.nframes = len(body)

    def set_option(self, key: str, value: int):
        """``bard_model_set_option``: a launch / code-generation knob of THIS model (see ``include/bard.h``)."""
        _check(lib().bard_model_set_option(self._h, key.encode(), int(value)))

    def get_option(self, key: str) -> int:
        v = C.c_int64()
        _check(lib().bard_model_get_option(self._h, key.encode(), C.byref(v)))
        return int(v.value)

    def specialize(self, ops=("rnea",)):
        """JIT-compile model-specialised kernels for the named operators (``bard_model_specialize``)."""
        mask = 0
        for o in ops:
            mask |= OPS[o]
        _check(lib().bard_model_specialize(self._h, mask))

    def specialized_source(self, op: str) -> str:
        need = C.c_size_t()
        lib().bard_model_specialized_source(self._h, OPS[op], None, 0, C.byref(need))
        buf = C.create_string_buffer(max(need.value, 1))
        _check(lib().bard_model_specialized_source(self._h, OPS[op], buf, need.value, C.byref(need)))
        return buf.value.decode()

    def table(self, name: str) -> np.ndarray:
        tid, dt = TABLES[name]
        need = C.c_size_t()
        lib().bard_model_get_table(self._h, tid, None, 0, C.byref(need))
        out = np.zeros(need.value // np.dtype(dt).itemsize, dtype=dt)
        _check(lib().bard_model_get_table(self._h, tid, out.ctypes.data_as(C.c_void_p), out.nbytes, C.byref(need)))
        return out

    # ---- operators: raw device pointers in, one kernel launch each, asynchronous on `stream`
    def fk(self, B, q, pose, stream=0):
        _check(lib().bard_fk(self._h, int(B), _ptr(q), _ptr(pose), stream or None))

    def jacobian(self, B, q, J, stream=0):
        _check(lib().bard_jacobian(self._h, int(B), _ptr(q), _ptr(J), stream or None))

    def rnea(self, B, q, qd, qdd, tau, stream=0):
        _check(lib().bard_rnea(self._h, int(B), _ptr(q), _ptr(qd), _ptr(qdd), _ptr(tau), stream or None))

    def kinematics(self, B, q, pose, J, M, stream=0):
        """Poses, Jacobians and mass matrix of one batch: one kernel where the kinematics-fused kernel exists (``bard_kinematics``)."""
        _check(lib().bard_kinematics(self._h, int(B), _ptr(q), _ptr(pose), _ptr(J), _ptr(M), stream or None))

    def step(self, B, q, qd, qdd, pose, J, tau, M, stream=0):
        """All four operators of one (q, qd, qdd) batch: one fused kernel if specialised with "fused"."""
        _check(lib().bard_step(self._h, int(B), _ptr(q), _ptr(qd), _ptr(qdd), _ptr(pose), _ptr(J), _ptr(tau), _ptr(M),
                               stream or None))

    def euler_step(self, B, dt, q, qd, qdd, stream=0):
        """qd += dt qdd ; q (+)= dt qd in place (``bard_euler_step``)."""
        _check(lib().bard_euler_step(self._h, int(B), float(dt), _ptr(q), _ptr(qd), _ptr(qdd), stream or None))

    def euler_step_to(self, B, dt, q, qd, qdd, q_out, qd_out, stream=0):
        """(q_out, qd_out) = Euler step of (q, qd, qdd), out of place (``bard_euler_step_to``)."""
        _check(lib().bard_euler_step_to(self._h, int(B), float(dt), _ptr(q), _ptr(qd), _ptr(qdd), _ptr(q_out), _ptr(qd_out), stream or None))

    def aba_workspace_floats(self, B) -> int:
        return int(lib().bard_aba_workspace_floats(self._h, int(B)))

    def aba(self, B, q, qd, tau, qdd, workspace, stream=0):
        """Forward dynamics qdd = M^-1 (tau - C) (``bard_aba``); needs ``specialize(("aba",))`` first."""
        _check(lib().bard_aba(self._h, int(B), _ptr(q), _ptr(qd), _ptr(tau), _ptr(qdd), _ptr(workspace), stream or None))

    # ---- dtype / layout variants (``bard_*_v``): dtype "f32" | "f64", layout "soa" | "aos" (batch-first, the paper's)
    def specialize_variant(self, ops, dtype="f32", layout="soa"):
        mask = 0
        for o in ops:
            mask |= OPS[o]
        _check(lib().bard_model_specialize_variant(self._h, mask, DTYPES[dtype], LAYOUTS[layout]))

    def variant_source(self, op: str, dtype="f32", layout="soa") -> str:
        need = C.c_size_t()
        lib().bard_model_variant_source(self._h, OPS[op], DTYPES[dtype], LAYOUTS[layout], None, 0, C.byref(need))
        buf = C.create_string_buffer(max(need.value, 1))
        _check(lib().bard_model_variant_source(self._h, OPS[op], DTYPES[dtype], LAYOUTS[layout], buf, need.value, C.byref(need)))
        return buf.value.decode()

    def variant_workspace_bytes(self, op, dtype, layout, B) -> int:
        return int(lib().bard_variant_workspace_bytes(self._h, OPS[op], DTYPES[dtype], LAYOUTS[layout], int(B)))

    def fk_v(self, dtype, layout, B, q, pose, workspace=None, stream=0):
        _check(lib().bard_fk_v(self._h, DTYPES[dtype], LAYOUTS[layout], int(B), _ptr(q), _ptr(pose), _ptr(workspace), stream or None))

    def jacobian_v(self, dtype, layout, B, q, J, workspace=None, stream=0):
        _check(lib().bard_jacobian_v(self._h, DTYPES[dtype], LAYOUTS[layout], int(B), _ptr(q), _ptr(J), _ptr(workspace), stream or None))

    def rnea_v(self, dtype, layout, B, q, qd, qdd, tau, workspace=None, stream=0):
        _check(lib().bard_rnea_v(self._h, DTYPES[dtype], LAYOUTS[layout], int(B), _ptr(q), _ptr(qd), _ptr(qdd), _ptr(tau),
                                 _ptr(workspace), stream or None))

    def crba_v(self, dtype, layout, B, q, M, workspace=None, stream=0):
        _check(lib().bard_crba_v(self._h, DTYPES[dtype], LAYOUTS[layout], int(B), _ptr(q), _ptr(M), _ptr(workspace), stream or None))

    def rnea_vjp_workspace_floats(self, B) -> int:
        return int(lib().bard_rnea_vjp_workspace_floats(self._h, int(B)))

    def rnea_vjp_params(self, B, q, qd, qdd, dtau, dparams, workspace, stream=0):
        """dparams[nb, 10] = sum_b (d tau_b / d theta)^T dtau_b (``bard_rnea_vjp_params``), theta = (m, m c, Io) per link."""
        _check(lib().bard_rnea_vjp_params(self._h, int(B), _ptr(q), _ptr(qd), _ptr(qdd), _ptr(dtau), _ptr(dparams),
                                          _ptr(workspace), stream or None))

    def rnea_vjp_params_static(self, B, q, qd, qdd, dtau, dparams, stream=0):
        """``bard_rnea_vjp_params_static``: the same with the library's static scratch array (no allocation; calls that
        overlap on the GPU race on it; refused above ``VJP_STATIC_SCRATCH_FLOATS`` floats of scratch)."""
        _check(lib().bard_rnea_vjp_params_static(self._h, int(B), _ptr(q), _ptr(qd), _ptr(qdd), _ptr(dtau), _ptr(dparams), stream or None))

    def inertial_params(self) -> np.ndarray:
        out = np.zeros((self.nb, 10))
        _check(lib().bard_model_inertial_params(self._h, _dp(out)))
        return out

    def set_inertial_params(self, params):
        p = _f64(params, (self.nb, 10))
        _check(lib().bard_model_set_inertial_params(self._h, _dp(p)))

    def crba(self, B, q, M, stream=0):
        _check(lib().bard_crba(self._h, int(B), _ptr(q), _ptr(M), stream or None))
