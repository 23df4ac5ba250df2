"""ctypes binding of include/fstat.h.  Argument marshalling only -- no arithmetic of the method."""
from __future__ import annotations

import ctypes as C
import os
import threading
from typing import Optional, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libfstat_b200.so")
_lock = threading.Lock()
_lib = None

STATUS = {0: "FSTAT_OK", 1: "FSTAT_EINVAL", 2: "FSTAT_ENOMEM", 3: "FSTAT_ECUDA", 4: "FSTAT_EUNSUPPORTED"}

# every symbol include/fstat.h declares (tests check the library exports exactly these)
EXPORTED_SYMBOLS = (
    "fstat_default_options", "fstat_plan_create", "fstat_plan_set_partitions", "fstat_eval_batch",
    "fstat_eval_batch_noalloc", "fstat_noalloc_scratch_bytes",
    "fstat_eval_batch_host", "fstat_eval_batch_bands", "fstat_eval_batch_bands_host", "fstat_eval_amplitudes_bands", "fstat_eval_batch_channels", "fstat_eval_amplitudes", "fstat_eval_template", "fstat_plan_destroy", "fstat_plan_n_bins",
    "fstat_plan_n_part", "fstat_plan_device", "fstat_plan_n_ctas", "fstat_plan_launch_count", "fstat_plan_table_bytes", "fstat_plan_band_stats",
    "fstat_plan_main_kernel_ms", "fstat_plan_level_bins", "fstat_edges_equal_bins", "fstat_probe_pipe_peak",
    "fstat_status_str", "fstat_last_error", "fstat_extrinsic_from_amplitudes", "fstat_amplitudes_from_extrinsic",
    "fstat_pso_default_options", "fstat_pso_create", "fstat_pso_create_boxes", "fstat_pso_iterate", "fstat_pso_best", "fstat_pso_state",
    "fstat_pso_iterations_done", "fstat_pso_destroy",
)


class FstatError(RuntimeError):
    def __init__(self, status: int, where: str, detail: str = ""):
        self.status = int(status)
        super().__init__("%s: %s%s" % (where, STATUS.get(int(status), str(status)), (" -- " + detail) if detail else ""))


class Options(C.Structure):
    """fstat_options of include/fstat.h."""
    _fields_ = [("f_ref_e0", C.c_double), ("arm_length_m", C.c_double), ("orbit_kappa", C.c_double),
                ("orbit_lambda", C.c_double), ("device", C.c_int32), ("inputs_on_device", C.c_int32),
                ("max_segment_bins", C.c_int32), ("force_level", C.c_int32), ("interp_tol", C.c_double),
                ("tdi_channel", C.c_int32), ("no_channel_fusion", C.c_int32), ("min_stride_level", C.c_int32)]


TDI_CHANNELS = {"X": 0, "Y": 1, "Z": 2, "A": 3, "E": 4, "T": 5}      # fstat_tdi_channel


class PsoOptions(C.Structure):
    """fstat_pso_options of include/fstat.h."""
    _fields_ = [("c1", C.c_double), ("c2", C.c_double), ("v_max", C.c_double), ("w_start", C.c_double),
                ("w_end", C.c_double), ("band_n_seg", C.c_int32), ("band_lattice", C.c_int32)]


def library_path() -> str:
    return _LIB_PATH


def load_library():
    """dlopen the in-tree CUDA library; fails loudly if it has not been built."""
    global _lib
    with _lock:
        if _lib is not None:
            return _lib
        if not os.path.exists(_LIB_PATH):
            raise ImportError("%s is missing: run `python -m paper_2407_10797_b200.build` "
                              "(there is no CPU fallback)" % _LIB_PATH)
        L = C.CDLL(_LIB_PATH)
        vp, dp, i64, i32 = C.c_void_p, C.POINTER(C.c_double), C.c_int64, C.c_int32
        L.fstat_default_options.argtypes = [C.POINTER(Options)]
        L.fstat_default_options.restype = None
        L.fstat_plan_create.argtypes = [C.POINTER(vp), i64, vp, vp, vp, i32, C.POINTER(i64), C.POINTER(Options)]
        L.fstat_plan_create.restype = C.c_int
        L.fstat_plan_set_partitions.argtypes = [vp, i32, C.POINTER(i64)]
        L.fstat_plan_set_partitions.restype = C.c_int
        L.fstat_eval_batch.argtypes = [vp, i64, vp, vp, vp, vp]
        L.fstat_eval_batch.restype = C.c_int
        L.fstat_eval_batch_noalloc.argtypes = [vp, i64, vp, vp, vp, vp]
        L.fstat_eval_batch_noalloc.restype = C.c_int
        L.fstat_noalloc_scratch_bytes.argtypes = []
        L.fstat_noalloc_scratch_bytes.restype = i64
        L.fstat_eval_amplitudes.argtypes = [vp, i64, vp, vp, vp]
        L.fstat_eval_amplitudes.restype = C.c_int
        L.fstat_eval_batch_bands.argtypes = [vp, i64, vp, C.c_int32, C.c_int32, vp, vp, vp, vp]
        L.fstat_eval_batch_bands.restype = C.c_int
        L.fstat_eval_batch_bands_host.argtypes = [vp, i64, vp, C.c_int32, C.c_int32, vp, vp, vp, vp]
        L.fstat_eval_batch_bands_host.restype = C.c_int
        L.fstat_eval_amplitudes_bands.argtypes = [vp, i64, vp, C.c_int32, C.c_int32, vp, vp]
        L.fstat_eval_amplitudes_bands.restype = C.c_int
        L.fstat_eval_batch_channels.argtypes = [C.POINTER(vp), C.c_int32, i64, vp, vp, vp, vp]
        L.fstat_eval_batch_channels.restype = C.c_int
        L.fstat_eval_batch_host.argtypes = [vp, i64, vp, vp, vp, vp]
        L.fstat_eval_batch_host.restype = C.c_int
        L.fstat_eval_template.argtypes = [vp, dp, vp, vp, vp]
        L.fstat_eval_template.restype = C.c_int
        L.fstat_plan_destroy.argtypes = [vp]
        L.fstat_plan_destroy.restype = None
        L.fstat_plan_n_bins.argtypes = [vp]
        L.fstat_plan_n_bins.restype = i64
        L.fstat_plan_n_part.argtypes = [vp]
        L.fstat_plan_n_part.restype = i32
        L.fstat_plan_device.argtypes = [vp]
        L.fstat_plan_device.restype = i32
        L.fstat_plan_n_ctas.argtypes = [vp, i64]
        L.fstat_plan_n_ctas.restype = i64
        L.fstat_plan_launch_count.argtypes = [vp]
        L.fstat_plan_launch_count.restype = i64
        L.fstat_plan_band_stats.argtypes = [vp, C.POINTER(i64)]
        L.fstat_plan_band_stats.restype = C.c_int
        L.fstat_plan_table_bytes.argtypes = [vp]
        L.fstat_plan_table_bytes.restype = i64
        L.fstat_plan_level_bins.argtypes = [vp, C.POINTER(i64), C.POINTER(i64)]
        L.fstat_plan_level_bins.restype = C.c_int
        L.fstat_plan_main_kernel_ms.argtypes = [vp, i32, dp]
        L.fstat_plan_main_kernel_ms.restype = i32
        L.fstat_edges_equal_bins.argtypes = [i64, i32, C.POINTER(i64)]
        L.fstat_edges_equal_bins.restype = C.c_int
        L.fstat_probe_pipe_peak.argtypes = [i32, i32, C.c_double, dp, C.POINTER(i32)]
        L.fstat_probe_pipe_peak.restype = C.c_int
        L.fstat_pso_default_options.argtypes = [C.POINTER(PsoOptions)]
        L.fstat_pso_default_options.restype = None
        L.fstat_pso_create.argtypes = [C.POINTER(vp), vp, i32, i32, i32, dp, dp, C.c_uint64, C.POINTER(PsoOptions), vp]
        L.fstat_pso_create.restype = C.c_int
        L.fstat_pso_create_boxes.argtypes = [C.POINTER(vp), vp, i32, i32, i32, dp, dp, C.c_uint64, C.POINTER(PsoOptions), vp]
        L.fstat_pso_create_boxes.restype = C.c_int
        L.fstat_pso_iterate.argtypes = [vp, i32, vp]
        L.fstat_pso_iterate.restype = C.c_int
        L.fstat_pso_best.argtypes = [vp, dp, dp, vp]
        L.fstat_pso_best.restype = C.c_int
        L.fstat_pso_state.argtypes = [vp, dp, dp, dp, dp, dp, vp]
        L.fstat_pso_state.restype = C.c_int
        L.fstat_pso_iterations_done.argtypes = [vp]
        L.fstat_pso_iterations_done.restype = i32
        L.fstat_pso_destroy.argtypes = [vp]
        L.fstat_pso_destroy.restype = None
        L.fstat_extrinsic_from_amplitudes.argtypes = [dp, C.c_double, dp]
        L.fstat_extrinsic_from_amplitudes.restype = C.c_int
        L.fstat_amplitudes_from_extrinsic.argtypes = [C.c_double] * 4 + [dp]
        L.fstat_amplitudes_from_extrinsic.restype = C.c_int
        L.fstat_status_str.argtypes = [C.c_int]
        L.fstat_status_str.restype = C.c_char_p
        L.fstat_last_error.argtypes = [vp]
        L.fstat_last_error.restype = C.c_char_p
        _lib = L
        return _lib


class Plan:
    """Owner of one ``fstat_plan*``.  Use ``fstat_plan_destroy(plan)`` / ``with`` / garbage collection."""

    def __init__(self, handle: int, n_bins: int, n_part: int):
        self._h = C.c_void_p(handle)
        self.n_bins = int(n_bins)
        self.n_part = int(n_part)

    @property
    def handle(self) -> C.c_void_p:
        if not self._h:
            raise FstatError(1, "Plan", "plan already destroyed")
        return self._h

    def close(self) -> None:
        if getattr(self, "_h", None):
            load_library().fstat_plan_destroy(self._h)
            self._h = C.c_void_p(None)

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def _check(status: int, where: str, plan: Optional[Plan] = None) -> None:
    if status != 0:
        h = plan._h if (plan is not None and plan._h) else None
        detail = load_library().fstat_last_error(h)
        raise FstatError(status, where, detail.decode() if detail else "")


def _is_tensor(x) -> bool:
    return hasattr(x, "data_ptr") and hasattr(x, "is_cuda")


def _dev_ptr(t, name: str, n_elem: int) -> int:
    """Pointer of a contiguous float64 CUDA tensor with at least n_elem elements."""
    import torch
    if not _is_tensor(t) or not t.is_cuda or t.dtype != torch.float64 or not t.is_contiguous():
        raise TypeError("%s must be a contiguous float64 CUDA tensor" % name)
    if t.numel() < n_elem:
        raise ValueError("%s has %d elements, needs %d" % (name, t.numel(), n_elem))
    return t.data_ptr()


def _stream_ptr(stream) -> Optional[int]:
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream if torch.cuda.is_available() else None
    if hasattr(stream, "cuda_stream"):
        return stream.cuda_stream
    return int(stream)


def fstat_default_options(**kw) -> Options:
    o = Options()
    load_library().fstat_default_options(C.byref(o))
    for k, v in kw.items():
        setattr(o, k, v)
    return o


def fstat_edges_equal_bins(n_bins: int, n_part: int) -> np.ndarray:
    e = np.zeros(int(n_part) + 1 if n_part >= 0 else 1, dtype=np.int64)
    st = load_library().fstat_edges_equal_bins(int(n_bins), int(n_part), e.ctypes.data_as(C.POINTER(C.c_int64)))
    if st != 0:
        raise FstatError(st, "fstat_edges_equal_bins")
    return e


def fstat_plan_create(freq_hz, dw, inv_sn, part_edges, opts: Optional[Options] = None) -> Plan:
    """freq_hz [N] f8, dw [N] c16 (or [N][2] f8), inv_sn [N] f8: numpy arrays (host) or CUDA tensors
    (device; sets opts.inputs_on_device).  part_edges [N_p+1] int64 host."""
    L = load_library()
    o = fstat_default_options() if opts is None else opts
    edges = np.ascontiguousarray(part_edges, dtype=np.int64)
    n_part = int(edges.shape[0]) - 1
    keep = []
    if _is_tensor(freq_hz):
        import torch
        n = int(freq_hz.numel())
        dwt = torch.view_as_real(dw) if dw.is_complex() else dw
        dwt = dwt.contiguous()
        keep.append(dwt)
        pf, pd, pi = _dev_ptr(freq_hz, "freq_hz", n), _dev_ptr(dwt, "dw", 2 * n), _dev_ptr(inv_sn, "inv_sn", n)
        o.inputs_on_device = 1
    else:
        f = np.ascontiguousarray(freq_hz, dtype=np.float64)
        n = int(f.shape[0])
        d = np.ascontiguousarray(dw)
        d = d.astype(np.complex128, copy=False).view(np.float64) if np.iscomplexobj(d) else d.astype(np.float64, copy=False)
        d = np.ascontiguousarray(d)
        w = np.ascontiguousarray(inv_sn, dtype=np.float64)
        if d.size != 2 * n or w.size != n:
            raise ValueError("dw / inv_sn sizes do not match freq_hz")
        keep += [f, d, w]
        pf, pd, pi = f.ctypes.data, d.ctypes.data, w.ctypes.data
        o.inputs_on_device = 0
    out = C.c_void_p()
    st = L.fstat_plan_create(C.byref(out), n, pf, pd, pi, n_part, edges.ctypes.data_as(C.POINTER(C.c_int64)), C.byref(o))
    if st != 0:
        raise FstatError(st, "fstat_plan_create", L.fstat_last_error(None).decode())
    return Plan(out.value, n, n_part)


def fstat_plan_set_partitions(plan: Plan, part_edges) -> None:
    edges = np.ascontiguousarray(part_edges, dtype=np.int64)
    n_part = int(edges.shape[0]) - 1
    _check(load_library().fstat_plan_set_partitions(plan.handle, n_part, edges.ctypes.data_as(C.POINTER(C.c_int64))),
           "fstat_plan_set_partitions", plan)
    plan.n_part = n_part


def fstat_eval_batch(plan: Plan, params, F=None, Fk=None, stream=None, want_Fk: bool = True):
    """params [P][6] float64 CUDA tensor -> (F [P], Fk [P][N_p] or None) CUDA tensors.  Asynchronous on
    ``stream`` (default: torch's current stream)."""
    import torch
    P = int(params.shape[0])
    pp = _dev_ptr(params, "params", 6 * P)
    if F is None:
        F = torch.empty(P, dtype=torch.float64, device=params.device)
    if Fk is None and want_Fk:
        Fk = torch.empty((P, plan.n_part), dtype=torch.float64, device=params.device)
    pF = _dev_ptr(F, "F", P)
    pFk = _dev_ptr(Fk, "Fk", P * plan.n_part) if Fk is not None else None
    _check(load_library().fstat_eval_batch(plan.handle, P, pp, pF, pFk, _stream_ptr(stream)), "fstat_eval_batch", plan)
    return F, Fk


def fstat_eval_batch_noalloc(plan: Plan, params, F, Fk=None, stream=None):
    """fstat_eval_batch with the workspace in the library's static 32 MiB device array: no device allocation inside the call
    (the caller passes every buffer: params [P][6], F [P], Fk [P][N_p] or None, float64 CUDA tensors).  Calls that overlap
    on the GPU race on that array; see include/fstat.h for the size limit and the set-up it needs."""
    P = int(params.shape[0])
    pp = _dev_ptr(params, "params", 6 * P)
    pF = _dev_ptr(F, "F", P)
    pFk = _dev_ptr(Fk, "Fk", P * plan.n_part) if Fk is not None else None
    _check(load_library().fstat_eval_batch_noalloc(plan.handle, P, pp, pF, pFk, _stream_ptr(stream)),
           "fstat_eval_batch_noalloc", plan)
    return F, Fk


def fstat_noalloc_scratch_bytes() -> int:
    return int(load_library().fstat_noalloc_scratch_bytes())


def fstat_eval_batch_bands(plan: Plan, params, n_seg: int, edge_lattice: int = 1, stream=None, want_Fk: bool = True,
                           want_band: bool = True):
    """Row f2: params [P][6] float64 CUDA tensor -> (F [P], Fk [P][n_seg] or None,
    band [P][2] int64 or None) CUDA tensors, with every template windowed to its own band and that band
    cut into n_seg partitions.  Asynchronous on ``stream``."""
    import torch
    P = int(params.shape[0])
    pp = _dev_ptr(params, "params", 6 * P)
    F = torch.empty(P, dtype=torch.float64, device=params.device)
    Fk = torch.empty((P, int(n_seg)), dtype=torch.float64, device=params.device) if want_Fk else None
    band = torch.empty((P, 2), dtype=torch.int64, device=params.device) if want_band else None
    _check(load_library().fstat_eval_batch_bands(plan.handle, P, pp, int(n_seg), int(edge_lattice), _dev_ptr(F, "F", P),
                                                 _dev_ptr(Fk, "Fk", P * int(n_seg)) if want_Fk else None,
                                                 band.data_ptr() if want_band else None, _stream_ptr(stream)),
           "fstat_eval_batch_bands", plan)
    return F, Fk, band


def fstat_eval_batch_bands_host(plan: Plan, params, n_seg: int, edge_lattice: int = 1, stream=None):
    """HOST buffers: params [P][6] float64 numpy array or CPU tensor (pinned for async DMA) -> (F [P], Fk [P][n_seg],
    band [P][2] int64) of the same kind, filled when the call returns."""
    if _is_tensor(params):
        import torch
        if params.is_cuda or params.dtype != torch.float64 or not params.is_contiguous():
            raise TypeError("params must be a contiguous float64 CPU tensor or numpy array")
        P = int(params.shape[0])
        pin = params.is_pinned()
        F = torch.empty(P, dtype=torch.float64, pin_memory=pin)
        Fk = torch.empty((P, int(n_seg)), dtype=torch.float64, pin_memory=pin)
        band = torch.empty((P, 2), dtype=torch.int64, pin_memory=pin)
        ptrs = (params.data_ptr(), F.data_ptr(), Fk.data_ptr(), band.data_ptr())
    else:
        params = np.ascontiguousarray(params, dtype=np.float64).reshape(-1, 6)
        P = params.shape[0]
        F, Fk, band = np.empty(P), np.empty((P, int(n_seg))), np.empty((P, 2), dtype=np.int64)
        ptrs = (params.ctypes.data, F.ctypes.data, Fk.ctypes.data, band.ctypes.data)
    _check(load_library().fstat_eval_batch_bands_host(plan.handle, P, ptrs[0], int(n_seg), int(edge_lattice),
                                                      ptrs[1], ptrs[2], ptrs[3], _stream_ptr(stream)),
           "fstat_eval_batch_bands_host", plan)
    return F, Fk, band


def fstat_eval_amplitudes_bands(plan: Plan, params, n_seg: int, edge_lattice: int = 1, stream=None):
    """Rows f2 x f3: params [P][6] float64 CUDA tensor -> amp [P][n_seg][4] CUDA tensor, the amplitudes a = M^-1 N of
    every partition of every template's own band."""
    import torch
    P = int(params.shape[0])
    amp = torch.empty((P, int(n_seg), 4), dtype=torch.float64, device=params.device)
    _check(load_library().fstat_eval_amplitudes_bands(plan.handle, P, _dev_ptr(params, "params", 6 * P), int(n_seg),
                                                      int(edge_lattice), _dev_ptr(amp, "amp", 4 * P * int(n_seg)),
                                                      _stream_ptr(stream)), "fstat_eval_amplitudes_bands", plan)
    return amp


def fstat_eval_batch_channels(plans, params, stream=None, want_Fk: bool = True):
    """Row f4 (Eq. 3): one plan per TDI channel (same grid and partitions) -> (F [P], Fk [P][N_p] or
    None) CUDA tensors of the statistic with the four amplitudes common to all channels.  Asynchronous."""
    import torch
    plans = list(plans)
    P = int(params.shape[0])
    pp = _dev_ptr(params, "params", 6 * P)
    F = torch.empty(P, dtype=torch.float64, device=params.device)
    Fk = torch.empty((P, plans[0].n_part), dtype=torch.float64, device=params.device) if want_Fk else None
    arr = (C.c_void_p * len(plans))(*[pl.handle for pl in plans])
    _check(load_library().fstat_eval_batch_channels(arr, len(plans), P, pp, _dev_ptr(F, "F", P),
                                                    _dev_ptr(Fk, "Fk", P * plans[0].n_part) if want_Fk else None,
                                                    _stream_ptr(stream)), "fstat_eval_batch_channels", plans[0])
    return F, Fk


def fstat_eval_amplitudes(plan: Plan, params, amp=None, stream=None):
    """params [P][6] float64 CUDA tensor -> amp [P][N_p][4] CUDA tensor (a_1..a_4 of PAPER.md Eq. 5 / 10)."""
    import torch
    P = int(params.shape[0])
    pp = _dev_ptr(params, "params", 6 * P)
    if amp is None:
        amp = torch.empty((P, plan.n_part, 4), dtype=torch.float64, device=params.device)
    pa = _dev_ptr(amp, "amp", 4 * P * plan.n_part)
    _check(load_library().fstat_eval_amplitudes(plan.handle, P, pp, pa, _stream_ptr(stream)),
           "fstat_eval_amplitudes", plan)
    return amp


def fstat_eval_batch_host(plan: Plan, params, F=None, Fk=None, stream=None, want_Fk: bool = True):
    """HOST buffers: params [P][6] float64 numpy array or CPU tensor (pinned for async DMA) ->
    (F, Fk) of the same kind, filled when the call returns."""
    tensor_in = _is_tensor(params)
    if tensor_in:
        import torch
        if params.is_cuda or params.dtype != torch.float64 or not params.is_contiguous():
            raise TypeError("params must be a contiguous float64 CPU tensor or numpy array")
        P = int(params.shape[0])
        if F is None:
            F = torch.empty(P, dtype=torch.float64, pin_memory=params.is_pinned())
        if Fk is None and want_Fk:
            Fk = torch.empty((P, plan.n_part), dtype=torch.float64, pin_memory=params.is_pinned())
        pp, pF, pFk = params.data_ptr(), F.data_ptr(), (Fk.data_ptr() if Fk is not None else None)
    else:
        params = np.ascontiguousarray(params, dtype=np.float64)
        P = int(params.shape[0])
        if F is None:
            F = np.empty(P)
        if Fk is None and want_Fk:
            Fk = np.empty((P, plan.n_part))
        pp, pF, pFk = params.ctypes.data, F.ctypes.data, (Fk.ctypes.data if Fk is not None else None)
    _check(load_library().fstat_eval_batch_host(plan.handle, P, pp, pF, pFk, _stream_ptr(stream)),
           "fstat_eval_batch_host", plan)
    return F, Fk


def fstat_eval_template(plan: Plan, params6, stream=None) -> Tuple["object", "object"]:
    """(u_plus, u_cross) complex128 CUDA tensors [N] for one parameter vector (host, 6 doubles)."""
    import torch
    q = np.ascontiguousarray(params6, dtype=np.float64).reshape(6)
    dev = torch.device("cuda", fstat_plan_device(plan))
    up = torch.empty((plan.n_bins, 2), dtype=torch.float64, device=dev)
    uc = torch.empty((plan.n_bins, 2), dtype=torch.float64, device=dev)
    _check(load_library().fstat_eval_template(plan.handle, q.ctypes.data_as(C.POINTER(C.c_double)), up.data_ptr(),
                                              uc.data_ptr(), _stream_ptr(stream)), "fstat_eval_template", plan)
    return torch.view_as_complex(up), torch.view_as_complex(uc)


def fstat_plan_destroy(plan: Optional[Plan]) -> None:
    if plan is not None:
        plan.close()


def fstat_plan_n_bins(plan: Plan) -> int:
    return int(load_library().fstat_plan_n_bins(plan.handle))


def fstat_plan_n_part(plan: Plan) -> int:
    return int(load_library().fstat_plan_n_part(plan.handle))


def fstat_plan_device(plan: Plan) -> int:
    return int(load_library().fstat_plan_device(plan.handle))


def fstat_plan_n_ctas(plan: Plan, P: int) -> int:
    return int(load_library().fstat_plan_n_ctas(plan.handle, int(P)))


def fstat_plan_launch_count(plan: Plan) -> int:
    return int(load_library().fstat_plan_launch_count(plan.handle))


def fstat_plan_band_stats(plan: Plan) -> np.ndarray:
    """[5] int64: warp-level bins, node intervals, intervals with a cut, runs of the last band call; invariant flag."""
    out = np.zeros(5, dtype=np.int64)
    _check(load_library().fstat_plan_band_stats(plan.handle, out.ctypes.data_as(C.POINTER(C.c_int64))),
           "fstat_plan_band_stats", plan)
    return out


def fstat_plan_table_bytes(plan: Plan) -> int:
    return int(load_library().fstat_plan_table_bytes(plan.handle))


def fstat_plan_level_bins(plan: Plan) -> Tuple[np.ndarray, np.ndarray]:
    """(bins[8], subblocks[8]) of the most recent evaluation: index 0 = direct kernel, 1..7 = stride 8..512."""
    b, s = np.zeros(8, dtype=np.int64), np.zeros(8, dtype=np.int64)
    _check(load_library().fstat_plan_level_bins(plan.handle, b.ctypes.data_as(C.POINTER(C.c_int64)),
                                                s.ctypes.data_as(C.POINTER(C.c_int64))), "fstat_plan_level_bins", plan)
    return b, s


def fstat_plan_main_kernel_ms(plan: Plan, n_last: int = 1) -> np.ndarray:
    """Device milliseconds of the main kernel in the last ``n_last`` evaluations (oldest first)."""
    out = np.zeros(max(int(n_last), 1))
    n = load_library().fstat_plan_main_kernel_ms(plan.handle, int(n_last), out.ctypes.data_as(C.POINTER(C.c_double)))
    return out[:n]


def fstat_probe_pipe_peak(which: int, millis: float = 50.0, device: int = -1) -> Tuple[float, int]:
    """(thread-level instructions per second, SM count) of pipe 0 = FP64 FMA, 1 = FP32 FMA, 2 = MUFU."""
    r, n = C.c_double(), C.c_int32()
    st = load_library().fstat_probe_pipe_peak(int(device), int(which), float(millis), C.byref(r), C.byref(n))
    if st != 0:
        raise FstatError(st, "fstat_probe_pipe_peak")
    return r.value, n.value


def fstat_status_str(status: int) -> str:
    return load_library().fstat_status_str(int(status)).decode()


def fstat_last_error(plan: Optional[Plan] = None) -> str:
    h = plan._h if (plan is not None and plan._h) else None
    return load_library().fstat_last_error(h).decode()


# ------------------------------------------------------------------------------------------ device PSO
class Pso:
    """Owner of one ``fstat_pso*`` (device-resident swarms bound to a Plan)."""

    def __init__(self, handle: int, plan: Plan, n_swarms: int, n_particles: int):
        self._h = C.c_void_p(handle)
        self.plan, self.n_swarms, self.n_particles = plan, int(n_swarms), int(n_particles)

    def close(self) -> None:
        if getattr(self, "_h", None):
            load_library().fstat_pso_destroy(self._h)
            self._h = C.c_void_p(None)

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def fstat_pso_default_options(**kw) -> PsoOptions:
    o = PsoOptions()
    load_library().fstat_pso_default_options(C.byref(o))
    for k, v in kw.items():
        setattr(o, k, v)
    return o


def fstat_pso_create(plan: Plan, n_swarms: int, n_particles: int, n_iter_total: int, lo, hi, seed: int = 0,
                     opts: Optional[PsoOptions] = None, stream=None) -> Pso:
    """lo, hi: [6] (one box for every swarm -> fstat_pso_create) or [n_swarms][6] (one box per swarm ->
    fstat_pso_create_boxes)."""
    lo = np.ascontiguousarray(lo, dtype=np.float64)
    hi = np.ascontiguousarray(hi, dtype=np.float64)
    per_swarm = lo.ndim == 2
    lo = lo.reshape(int(n_swarms), 6) if per_swarm else lo.reshape(6)
    hi = hi.reshape(int(n_swarms), 6) if per_swarm else hi.reshape(6)
    out = C.c_void_p()
    dp = C.POINTER(C.c_double)
    L = load_library()
    fn = L.fstat_pso_create_boxes if per_swarm else L.fstat_pso_create
    st = fn(C.byref(out), plan.handle, int(n_swarms), int(n_particles), int(n_iter_total),
            lo.ctypes.data_as(dp), hi.ctypes.data_as(dp), C.c_uint64(int(seed)),
            C.byref(opts) if opts is not None else None, _stream_ptr(stream))
    if st != 0:
        raise FstatError(st, "fstat_pso_create", fstat_last_error(plan))
    return Pso(out.value, plan, n_swarms, n_particles)


def fstat_pso_iterate(pso: Pso, n_iter: int, stream=None) -> None:
    st = load_library().fstat_pso_iterate(pso._h, int(n_iter), _stream_ptr(stream))
    if st != 0:
        raise FstatError(st, "fstat_pso_iterate", fstat_last_error(pso.plan))


def fstat_pso_best(pso: Pso, stream=None) -> Tuple[np.ndarray, np.ndarray]:
    bp, bf = np.empty((pso.n_swarms, 6)), np.empty(pso.n_swarms)
    dp = C.POINTER(C.c_double)
    st = load_library().fstat_pso_best(pso._h, bp.ctypes.data_as(dp), bf.ctypes.data_as(dp), _stream_ptr(stream))
    if st != 0:
        raise FstatError(st, "fstat_pso_best")
    return bp, bf


def fstat_pso_state(pso: Pso, stream=None):
    """(x, v, pbest [N][6], pbest_f, f_last [N]) host copies."""
    n = pso.n_swarms * pso.n_particles
    x, v, pb = np.empty((n, 6)), np.empty((n, 6)), np.empty((n, 6))
    pf, fl = np.empty(n), np.empty(n)
    dp = C.POINTER(C.c_double)
    st = load_library().fstat_pso_state(pso._h, x.ctypes.data_as(dp), v.ctypes.data_as(dp), pb.ctypes.data_as(dp),
                                        pf.ctypes.data_as(dp), fl.ctypes.data_as(dp), _stream_ptr(stream))
    if st != 0:
        raise FstatError(st, "fstat_pso_state")
    return x, v, pb, pf, fl


def fstat_pso_iterations_done(pso: Pso) -> int:
    return int(load_library().fstat_pso_iterations_done(pso._h))


def fstat_pso_destroy(pso: Optional[Pso]) -> None:
    if pso is not None:
        pso.close()
