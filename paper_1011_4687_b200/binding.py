"""Thin ctypes binding of include/qmmm_field.h (argument marshalling only).

Every step of the path runs in the CUDA library; PyTorch is used here only for device
memory and streams (tensor ``data_ptr()`` and ``torch.cuda.current_stream()``).  There is
no CPU fallback: if ``libqmmm_field.so`` is missing the import of this module raises.
Function names mirror the C ABI: ``qmmm_field_create``, ``qmmm_field_eval``,
``qmmm_field_eval_host``, ``qmmm_field_destroy`` (PAPER.md:117 create/eval split).
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Tuple

import numpy as np

QMMM_FP64 = 0
QMMM_FP32_ACC64 = 1
_PREC = {"fp64": QMMM_FP64, "fp32": QMMM_FP32_ACC64, QMMM_FP64: QMMM_FP64,
         QMMM_FP32_ACC64: QMMM_FP32_ACC64}
_STATUS = {0: "QMMM_OK", 1: "QMMM_ERR_INVALID_ARG", 2: "QMMM_ERR_ALLOC", 3: "QMMM_ERR_CUDA",
           4: "QMMM_ERR_UNSUPPORTED_DEVICE"}

# QMMM_FIELD_LIB selects another build of the same library (a tuning variant made with
# build.build(defines=..., out=...)); the default is the in-tree build.
LIB_PATH = os.environ.get("QMMM_FIELD_LIB") or os.path.join(
    os.path.dirname(os.path.abspath(__file__)), "libqmmm_field.so")
EXPORTED_SYMBOLS = ("qmmm_field_create", "qmmm_field_eval", "qmmm_field_eval_host",
                    "qmmm_field_eval_moves_host", "qmmm_field_eval_move_host", "qmmm_field_create_grid", "qmmm_field_eval_energy",
                    "qmmm_field_eval_moves",
                    "qmmm_field_share", "qmmm_field_create_grid3",
                    "qmmm_field_set_layout", "qmmm_field_get_grid_info",
                    "qmmm_field_destroy", "qmmm_field_set_plan", "qmmm_field_get_info",
                    "qmmm_field_set_timing", "qmmm_field_last_timing", "qmmm_field_set_overlap",
                    "qmmm_field_set_local_lattice", "qmmm_field_set_accurate_v", "qmmm_field_eval_noalloc",
                    "qmmm_field_min_distance", "qmmm_sum_rank_partials", "qmmm_probe_peak", "qmmm_last_error")


class QmmmError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"{_STATUS.get(status, status)}: {message}")
        self.status = status


class qmmm_plan(ctypes.Structure):
    _fields_ = [("points_per_thread", ctypes.c_int32), ("point_warps", ctypes.c_int32),
                ("slices", ctypes.c_int32), ("stages", ctypes.c_int32)]


class qmmm_field_info(ctypes.Structure):
    _fields_ = [("M", ctypes.c_int64), ("K", ctypes.c_int64), ("max_points", ctypes.c_int64),
                ("n_chunks", ctypes.c_int64), ("bytes_fp64", ctypes.c_int64),
                ("bytes_fp32", ctypes.c_int64), ("bytes_workspace", ctypes.c_int64),
                ("last_plan", qmmm_plan), ("last_point_blocks", ctypes.c_int32),
                ("last_launches", ctypes.c_int32), ("sm_count", ctypes.c_int32),
                ("last_dz_table", ctypes.c_int32), ("device_errors", ctypes.c_int32),
                ("last_local_lattice", ctypes.c_int32), ("last_accurate_v", ctypes.c_int32),
                ("last_kernel", ctypes.c_char * 192)]


class qmmm_grid_info(ctypes.Structure):
    _fields_ = [("present", ctypes.c_int32), ("has_list", ctypes.c_int32),
                ("layout", ctypes.c_int32), ("last_layout", ctypes.c_int32),
                ("n", ctypes.c_int32 * 3), ("reserved", ctypes.c_int32),
                ("origin", ctypes.c_double * 3), ("spacing", ctypes.c_double),
                ("n_gchunks", ctypes.c_int64), ("bytes_fp32", ctypes.c_int64),
                ("bytes_fp64", ctypes.c_int64), ("spacing3", ctypes.c_double * 3)]


QMMM_LAYOUT_AUTO, QMMM_LAYOUT_LIST, QMMM_LAYOUT_GRID = 0, 1, 2
_LAYOUT = {"auto": 0, "list": 1, "grid": 2, 0: 0, 1: 1, 2: 2}


def _load() -> ctypes.CDLL:
    if not os.path.exists(LIB_PATH):
        raise ImportError(
            f"{LIB_PATH} is missing: build it with `python -m paper_1011_4687_b200.build` "
            "(there is no CPU fallback)")
    lib = ctypes.CDLL(LIB_PATH)
    vp, i64, ci = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int
    lib.qmmm_field_create.restype = ci
    lib.qmmm_field_create.argtypes = [vp, vp, i64, vp, vp, i64, i64, ctypes.POINTER(vp)]
    lib.qmmm_field_eval.restype = ci
    lib.qmmm_field_eval.argtypes = [vp, vp, i64, i64, vp, vp, ci, vp]
    lib.qmmm_field_eval_energy.restype = ci
    lib.qmmm_field_eval_energy.argtypes = [vp, vp, i64, i64, vp, ci, vp]
    lib.qmmm_field_eval_host.restype = ci
    lib.qmmm_field_eval_host.argtypes = [vp, vp, i64, i64, vp, vp, ci, vp]
    lib.qmmm_field_min_distance.restype = ci
    lib.qmmm_field_min_distance.argtypes = [vp, vp, i64, ctypes.POINTER(ctypes.c_double), vp]
    lib.qmmm_field_eval_move_host.restype = ci
    lib.qmmm_field_eval_move_host.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp, vp, ci, vp]
    lib.qmmm_field_eval_moves_host.restype = ci
    lib.qmmm_field_eval_moves_host.argtypes = [vp, vp, i64, i64, vp, vp, ci, vp,
                                               ctypes.POINTER(ctypes.c_double)]
    lib.qmmm_field_eval_moves.restype = ci
    lib.qmmm_field_eval_moves.argtypes = [vp, vp, i64, i64, vp, vp, ci, vp]
    lib.qmmm_field_create_grid.restype = ci
    lib.qmmm_field_create_grid.argtypes = [ctypes.POINTER(ctypes.c_double), ctypes.c_double,
                                           ctypes.POINTER(i64), vp, vp, vp, i64, i64,
                                           ctypes.POINTER(vp)]
    lib.qmmm_field_share.restype = ci
    lib.qmmm_field_share.argtypes = [vp, i64, ctypes.POINTER(vp)]
    lib.qmmm_field_create_grid3.restype = ci
    lib.qmmm_field_create_grid3.argtypes = [ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double),
                                            ctypes.POINTER(i64), vp, vp, vp, i64, i64,
                                            ctypes.POINTER(vp)]
    lib.qmmm_field_set_layout.restype = ci
    lib.qmmm_field_set_layout.argtypes = [vp, ci]
    lib.qmmm_field_get_grid_info.restype = ci
    lib.qmmm_field_get_grid_info.argtypes = [vp, ctypes.POINTER(qmmm_grid_info)]
    lib.qmmm_field_destroy.restype = ci
    lib.qmmm_field_destroy.argtypes = [vp]
    lib.qmmm_field_set_plan.restype = ci
    lib.qmmm_field_set_plan.argtypes = [vp, ctypes.POINTER(qmmm_plan)]
    lib.qmmm_field_get_info.restype = ci
    lib.qmmm_field_get_info.argtypes = [vp, ctypes.POINTER(qmmm_field_info)]
    lib.qmmm_field_set_timing.restype = ci
    lib.qmmm_field_set_timing.argtypes = [vp, ci]
    lib.qmmm_field_set_overlap.restype = ci
    lib.qmmm_field_set_overlap.argtypes = [vp, ci]
    lib.qmmm_field_set_local_lattice.restype = ci
    lib.qmmm_field_set_local_lattice.argtypes = [vp, ci]
    lib.qmmm_field_set_accurate_v.restype = ci
    lib.qmmm_field_set_accurate_v.argtypes = [vp, ci]
    lib.qmmm_field_last_timing.restype = ci
    lib.qmmm_field_last_timing.argtypes = [vp, ctypes.POINTER(ctypes.c_double),
                                           ctypes.POINTER(ctypes.c_double)]
    lib.qmmm_probe_peak.restype = ci
    lib.qmmm_probe_peak.argtypes = [ci, ci, ctypes.POINTER(ctypes.c_double),
                                    ctypes.POINTER(ctypes.c_double), vp]
    lib.qmmm_field_eval_noalloc.restype = ci
    lib.qmmm_field_eval_noalloc.argtypes = [vp, vp, i64, vp, vp, i64, vp, i64, vp, vp, vp]
    lib.qmmm_sum_rank_partials.restype = ci
    lib.qmmm_sum_rank_partials.argtypes = [vp, i64, i64, vp, vp]
    lib.qmmm_last_error.restype = ctypes.c_char_p
    lib.qmmm_last_error.argtypes = []
    return lib


_lib = _load()


def _check(status: int) -> None:
    if status != 0:
        raise QmmmError(status, _lib.qmmm_last_error().decode())


def _ptr(a) -> Optional[int]:
    """Raw address of a numpy array (host) or torch tensor (host or device); None -> NULL."""
    if a is None:
        return None
    if isinstance(a, np.ndarray):
        assert a.dtype == np.float64 and a.flags.c_contiguous
        return a.ctypes.data if a.size else None
    assert a.dtype.is_floating_point and a.element_size() == 8 and a.is_contiguous()
    return a.data_ptr() if a.numel() else None


def _stream(stream) -> Optional[int]:
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream or None
    return getattr(stream, "cuda_stream", stream) or None


def qmmm_field_create(src_xyz, src_q, nuc_xyz, nuc_Z, max_points: int) -> int:
    """Upload + pack one environment; arrays are FP64 numpy arrays or torch tensors (host
    or device).  Returns the opaque handle."""
    M = int(src_q.shape[0]) if src_q is not None else 0
    K = int(nuc_Z.shape[0]) if nuc_Z is not None else 0
    out = ctypes.c_void_p()
    _check(_lib.qmmm_field_create(_ptr(src_xyz), _ptr(src_q), M, _ptr(nuc_xyz), _ptr(nuc_Z), K,
                                  int(max_points), ctypes.byref(out)))
    return out.value


def qmmm_field_create_grid(origin, spacing: float, n, cell_q, nuc_xyz, nuc_Z,
                           max_points: int) -> int:
    """Environment given as a regular grid: node (0,0,0) at ``origin``, edge ``spacing`` (a
    number, or (hx, hy, hz) for orthorhombic cells),
    ``cell_q`` [n0,n1,n2] FP64 cell charges (C order; 0 = no cell), host or device."""
    org = (ctypes.c_double * 3)(*[float(v) for v in origin])
    dims = (ctypes.c_int64 * 3)(*[int(v) for v in n])
    assert cell_q is not None and tuple(cell_q.shape) == tuple(int(v) for v in n)
    K = int(nuc_Z.shape[0]) if nuc_Z is not None else 0
    out = ctypes.c_void_p()
    if np.ndim(spacing) == 0:
        _check(_lib.qmmm_field_create_grid(org, float(spacing), dims, _ptr(cell_q), _ptr(nuc_xyz),
                                           _ptr(nuc_Z), K, int(max_points), ctypes.byref(out)))
    else:                                       # (hx, hy, hz): orthorhombic cells
        sp = (ctypes.c_double * 3)(*[float(v) for v in spacing])
        _check(_lib.qmmm_field_create_grid3(org, sp, dims, _ptr(cell_q), _ptr(nuc_xyz),
                                            _ptr(nuc_Z), K, int(max_points), ctypes.byref(out)))
    return out.value


def qmmm_field_share(parent: int, max_points: int) -> int:
    """A second handle on the same environment (shares the packed sources, own workspace):
    one per stream / host thread for concurrent evaluations."""
    out = ctypes.c_void_p()
    _check(_lib.qmmm_field_share(parent, int(max_points), ctypes.byref(out)))
    return out.value


def qmmm_field_set_layout(handle: int, layout="auto") -> None:
    """"auto" | "list" | "grid": which copy of the sources eval uses."""
    _check(_lib.qmmm_field_set_layout(handle, _LAYOUT[layout]))


def qmmm_field_get_grid_info(handle: int) -> dict:
    info = qmmm_grid_info()
    _check(_lib.qmmm_field_get_grid_info(handle, ctypes.byref(info)))
    names = {0: "auto", 1: "list", 2: "grid"}
    return {"present": bool(info.present), "has_list": bool(info.has_list),
            "layout": names[info.layout], "last_layout": names[info.last_layout],
            "n": tuple(info.n), "origin": tuple(info.origin), "spacing": info.spacing,
            "spacing3": tuple(info.spacing3),
            "n_gchunks": info.n_gchunks, "bytes_fp32": info.bytes_fp32,
            "bytes_fp64": info.bytes_fp64}


def qmmm_field_eval(handle: int, elec_xyz, W: int, N: int, V, E=None, precision="fp64",
                    stream=None) -> None:
    """Asynchronous evaluation on device tensors (elec_xyz [W*N,3], V [W*N], E [W*N,3])."""
    _check(_lib.qmmm_field_eval(handle, _ptr(elec_xyz), int(W), int(N), _ptr(V), _ptr(E),
                                _PREC[precision], _stream(stream)))


def qmmm_field_eval_energy(handle: int, elec_xyz, W: int, N: int, U, precision="fp64",
                           stream=None) -> None:
    """U[w] = -sum_i V(r_{w,i}) per walker (Eq. 4), device tensors, asynchronous."""
    _check(_lib.qmmm_field_eval_energy(handle, _ptr(elec_xyz), int(W), int(N), _ptr(U),
                                       _PREC[precision], _stream(stream)))


def qmmm_field_eval_host(handle: int, elec_xyz, W: int, N: int, V, E=None, precision="fp64",
                         stream=None) -> None:
    """Per-step host loop of PAPER.md:117: host buffers in/out, synchronises the stream."""
    _check(_lib.qmmm_field_eval_host(handle, _ptr(elec_xyz), int(W), int(N), _ptr(V), _ptr(E),
                                     _PREC[precision], _stream(stream)))


def qmmm_field_min_distance(handle: int, elec_xyz, stream=None) -> float:
    """Debug helper: smallest distance (bohr) between the points (device tensor [P,3]) and the
    charged sources of the handle."""
    out = ctypes.c_double()
    _check(_lib.qmmm_field_min_distance(handle, _ptr(elec_xyz), int(elec_xyz.numel() // 3), ctypes.byref(out),
                                        _stream(stream)))
    return out.value


def qmmm_field_eval_move_host(handle: int, r_old, r_new, V_old=None, E_old=None, V_new=None, E_new=None,
                              dV=None, dE=None, precision="fp64", stream=None) -> None:
    """One single-electron move: V, E at r_new and their change from r_old; host
    arrays (numpy float64).  V_old / E_old = the values a previous call returned at r_old, or None:
    then both points are evaluated in one launch.  Argument marshalling only."""
    _check(_lib.qmmm_field_eval_move_host(handle, _ptr(r_old), _ptr(r_new), _ptr(V_old), _ptr(E_old),
                                          _ptr(V_new), _ptr(E_new), _ptr(dV), _ptr(dE),
                                          _PREC[precision], _stream(stream)))


def qmmm_field_eval_moves_host(handle: int, elec_xyz, n: int, N: int, V, E=None, precision="fp64",
                               stream=None) -> float:
    """n sequential single-configuration evaluations through the per-move path (the paper's
    deployed loop); host arrays elec_xyz [n,N,3], V [n,N], E [n,N,3].  Returns
    the host wall-clock seconds of the loop."""
    secs = ctypes.c_double()
    _check(_lib.qmmm_field_eval_moves_host(handle, _ptr(elec_xyz), int(n), int(N), _ptr(V), _ptr(E),
                                           _PREC[precision], _stream(stream), ctypes.byref(secs)))
    return secs.value


def qmmm_field_eval_moves(handle: int, elec_xyz, n: int, N: int, V, E=None, precision="fp64",
                          stream=None) -> None:
    """n independent single-configuration evaluations with all positions known up front
    (device tensors elec_xyz [n,N,3], V [n,N], E [n,N,3]): one overlapped kernel per move,
    issued from C.  Asynchronous on the stream."""
    _check(_lib.qmmm_field_eval_moves(handle, _ptr(elec_xyz), int(n), int(N), _ptr(V), _ptr(E),
                                      _PREC[precision], _stream(stream)))


QMMM_NOALLOC_MAX_POINTS = 4096


def qmmm_field_eval_noalloc(src_xyz, src_q, nuc_xyz, nuc_Z, elec_xyz, V, E=None, stream=None) -> None:
    """V and E without a handle and without any allocation (fixed __device__ scratch array in
    the library; include/qmmm_field.h): all arguments are DEVICE FP64 tensors, src_xyz [M,3],
    src_q [M], nuc_xyz [K,3], nuc_Z [K] (either pair may be None), elec_xyz [P,3] with
    P <= QMMM_NOALLOC_MAX_POINTS, V [P], E [P,3] or None.  Asynchronous on the stream."""
    M = int(src_q.shape[0]) if src_q is not None else 0
    K = int(nuc_Z.shape[0]) if nuc_Z is not None else 0
    P = int(elec_xyz.shape[0])
    _check(_lib.qmmm_field_eval_noalloc(_ptr(src_xyz), _ptr(src_q), M, _ptr(nuc_xyz), _ptr(nuc_Z), K,
                                        _ptr(elec_xyz), P, _ptr(V), _ptr(E), _stream(stream)))


def qmmm_sum_rank_partials(parts, out, stream=None) -> None:
    """out[i] = parts[0][i] + parts[1][i] + ... in rank order (device tensors: parts [R, n]
    contiguous FP64, out [n]); sharding by sources, Eq. 5 across GPUs."""
    R = int(parts.shape[0])
    n = int(parts.numel() // R) if R else 0
    _check(_lib.qmmm_sum_rank_partials(_ptr(parts), R, n, _ptr(out), _stream(stream)))


def qmmm_field_destroy(handle: Optional[int]) -> None:
    _check(_lib.qmmm_field_destroy(handle))


def qmmm_field_set_plan(handle: int, points_per_thread=0, point_warps=0, slices=0, stages=0):
    pl = qmmm_plan(points_per_thread, point_warps, slices, stages)
    _check(_lib.qmmm_field_set_plan(handle, ctypes.byref(pl)))


def qmmm_field_get_info(handle: int) -> dict:
    info = qmmm_field_info()
    _check(_lib.qmmm_field_get_info(handle, ctypes.byref(info)))
    d = {k: getattr(info, k) for k, _ in info._fields_ if k not in ("last_plan", "reserved")}
    d["last_kernel"] = info.last_kernel.decode()
    d["last_plan"] = {k: getattr(info.last_plan, k) for k, _ in qmmm_plan._fields_}
    return d


def qmmm_field_set_timing(handle: int, enable: bool) -> None:
    _check(_lib.qmmm_field_set_timing(handle, int(bool(enable))))


def qmmm_field_set_overlap(handle: int, enable: bool) -> None:
    """Back-to-back evaluations on one stream may overlap (programmatic dependent launch); see
    include/qmmm_field.h for the precondition on elec_xyz."""
    _check(_lib.qmmm_field_set_overlap(handle, int(bool(enable))))


def qmmm_field_set_local_lattice(handle: int, mode: int = -1) -> None:
    """FP32 grid kernels: coordinate lattice per work unit (-1 automatic, 0 never, 1 always)."""
    _check(_lib.qmmm_field_set_local_lattice(handle, int(mode)))


def qmmm_field_set_accurate_v(handle: int, enable: bool = True) -> None:
    """FP32 batched grid V + E kernel: accurate V (default on; off = the 6 % faster kernel)."""
    _check(_lib.qmmm_field_set_accurate_v(handle, int(bool(enable))))


def qmmm_field_last_timing(handle: int) -> Tuple[float, float]:
    """(pair_kernel_ms, 0.0) of the most recent eval (waits for it); the finalize step is
    fused into the pair kernel."""
    a, b = ctypes.c_double(), ctypes.c_double()
    _check(_lib.qmmm_field_last_timing(handle, ctypes.byref(a), ctypes.byref(b)))
    return a.value, b.value


def qmmm_probe_peak(kind: int, iters: int = 0, stream=None) -> Tuple[float, float]:
    """(rate, seconds): kind 0 FFMA, 1 DFMA, 2 MUFU.RSQ lane-ops/s; 3 launch+sync seconds;
    4 / 5 read bandwidth in bytes/s over a 33 MB (L2) / 537 MB (HBM) buffer."""
    rate, secs = ctypes.c_double(), ctypes.c_double()
    _check(_lib.qmmm_probe_peak(kind, iters, ctypes.byref(rate), ctypes.byref(secs),
                                _stream(stream)))
    return rate.value, secs.value


class FieldEvaluator:
    """Convenience owner of a handle (context manager); still argument marshalling only."""

    def __init__(self, src_xyz, src_q, nuc_xyz, nuc_Z, max_points: int):
        self.handle = qmmm_field_create(src_xyz, src_q, nuc_xyz, nuc_Z, max_points)

    def eval(self, elec_xyz, precision="fp64", want_E=True, stream=None):
        """elec_xyz: CUDA FP64 tensor [..., 3]; returns (V [...], E [..., 3] or None)."""
        import torch
        pts = elec_xyz.reshape(-1, 3).contiguous()
        P = pts.shape[0]
        V = torch.empty(P, dtype=torch.float64, device=pts.device)
        E = torch.empty((P, 3), dtype=torch.float64, device=pts.device) if want_E else None
        qmmm_field_eval(self.handle, pts, 1, P, V, E, precision, stream)
        lead = elec_xyz.shape[:-1]
        return V.reshape(lead), (E.reshape(*lead, 3) if want_E else None)

    def close(self):
        if self.handle is not None:
            qmmm_field_destroy(self.handle)
            self.handle = None

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
