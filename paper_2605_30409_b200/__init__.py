"""B200-native Gated DeltaNet chunk forward -- thin Python binding over the C ABI of include/gdn.h.

Argument marshalling only: every step of the path runs in the CUDA kernels of
``libgdn_b200.so`` (built in-tree by ``paper_2605_30409_b200.build``).  PyTorch is used for device
memory and streams, nothing else.  There is no CPU fallback: if the library is missing this module
raises on first use, and on a non-sm_100 device every compute call returns ``GDN_ERR_ARCH``.

The functions ``gdn_plan`` / ``gdn_forward_chunk`` / ``gdn_forward_chunk_norm`` /
``gdn_forward_chunk_host`` / ``gdn_destroy`` mirror the C entry points one to one.
"""
from __future__ import annotations

import ctypes
from pathlib import Path
from typing import Optional

__all__ = [
    "GdnError", "GdnConfig", "GdnPlanInfo", "lib", "gdn_plan", "gdn_forward_chunk", "gdn_forward_chunk_norm",
    "gdn_forward_chunk_host", "gdn_destroy", "gdn_plan_get_info", "gdn_plan_set_profiling", "gdn_plan_kernel_times",
    "gdn_status_string", "gdn_last_error", "gdn_version", "GdnPlan", "GDN_BF16", "GDN_FP32", "GDN_FLAG_NORMALIZER", "GDN_FLAG_BIDIR",
    "GDN_FLAG_LOG_ALPHA", "GDN_FLAG_FORCE_SIMT", "GDN_FLAG_UNFUSED", "PATH_NAMES", "EXPORTED_SYMBOLS",
]

_PKG = Path(__file__).resolve().parent
LIB_PATH = _PKG / "libgdn_b200.so"

GDN_OK = 0
GDN_ERR_INVALID_ARG, GDN_ERR_UNSUPPORTED, GDN_ERR_ALIGNMENT, GDN_ERR_NOMEM, GDN_ERR_ARCH, GDN_ERR_CUDA = 1, 2, 3, 4, 5, 6
GDN_BF16, GDN_FP32 = 0, 1
GDN_FLAG_NORMALIZER, GDN_FLAG_BIDIR, GDN_FLAG_LOG_ALPHA, GDN_FLAG_FORCE_SIMT, GDN_FLAG_UNFUSED = 1, 2, 4, 8, 16
PATH_NAMES = {0: "simt_fp32", 1: "tc_token", 2: "tc_frame"}
EXPORTED_SYMBOLS = [
    "gdn_plan", "gdn_forward_chunk", "gdn_forward_chunk_norm", "gdn_forward_chunk_host", "gdn_destroy",
    "gdn_feature_map", "gdn_compute_gates", "gdn_compute_gates_static", "gdn_forward_chunk_full",
    "gdn_plan_get_info", "gdn_plan_set_profiling", "gdn_plan_kernel_times", "gdn_status_string", "gdn_last_error",
    "gdn_version",
]


class GdnConfig(ctypes.Structure):
    """Mirror of gdn_config_t (include/gdn.h)."""
    _fields_ = [
        ("struct_size", ctypes.c_uint32),
        ("B", ctypes.c_int32), ("H", ctypes.c_int32), ("T", ctypes.c_int32),
        ("d_k", ctypes.c_int32), ("d_v", ctypes.c_int32),
        ("group", ctypes.c_int32), ("chunk", ctypes.c_int32), ("io_dtype", ctypes.c_int32),
        ("scale", ctypes.c_float), ("eps", ctypes.c_float), ("flags", ctypes.c_uint32),
        ("q_token_stride", ctypes.c_int64), ("k_token_stride", ctypes.c_int64),
        ("v_token_stride", ctypes.c_int64), ("o_token_stride", ctypes.c_int64),
    ]


class GdnPlanInfo(ctypes.Structure):
    """Mirror of gdn_plan_info_t."""
    _fields_ = [("path", ctypes.c_int32), ("chunk", ctypes.c_int32), ("launches_per_call", ctypes.c_int32),
                ("sm_count", ctypes.c_int32), ("workspace_bytes", ctypes.c_uint64)]


class GdnFeatmapArgs(ctypes.Structure):
    """Mirror of gdn_featmap_args_t."""
    _fields_ = [("q", ctypes.c_void_p), ("k", ctypes.c_void_p), ("rms_wq", ctypes.c_void_p), ("rms_wk", ctypes.c_void_p),
                ("rope_cos", ctypes.c_void_p), ("rope_sin", ctypes.c_void_p), ("rms_eps", ctypes.c_float)]


class GdnGateArgs(ctypes.Structure):
    """Mirror of gdn_gate_args_t."""
    _fields_ = [("x", ctypes.c_void_p), ("x_token_stride", ctypes.c_int64), ("w_alpha", ctypes.c_void_p),
                ("b_alpha", ctypes.c_void_p), ("a_log", ctypes.c_void_p), ("w_beta", ctypes.c_void_p), ("b_beta", ctypes.c_void_p)]


class GdnError(RuntimeError):
    def __init__(self, status: int, detail: str = ""):
        self.status = int(status)
        name = gdn_status_string(status) if _lib is not None else str(status)
        super().__init__(f"{name}: {detail}" if detail else name)


_lib = None


def lib() -> ctypes.CDLL:
    """Load libgdn_b200.so (fails loudly if it was not built: there is no fallback path)."""
    global _lib
    if _lib is None:
        if not LIB_PATH.exists():
            raise FileNotFoundError(
                f"{LIB_PATH} is missing: build it with `python -m paper_2605_30409_b200.build` "
                "(or __graft_entry__.build()). There is no CPU or PyTorch fallback.")
        L = ctypes.CDLL(str(LIB_PATH))
        vp, fp, cp = ctypes.c_void_p, ctypes.c_void_p, ctypes.c_char_p
        L.gdn_plan.restype = ctypes.c_int
        L.gdn_plan.argtypes = [ctypes.POINTER(GdnConfig), ctypes.POINTER(vp)]
        L.gdn_forward_chunk.restype = ctypes.c_int
        L.gdn_forward_chunk.argtypes = [vp, vp, vp, vp, fp, fp, fp, vp, fp, vp]
        L.gdn_forward_chunk_norm.restype = ctypes.c_int
        L.gdn_forward_chunk_norm.argtypes = [vp] + [vp] * 5 + [fp] * 4 + [vp, fp, fp, vp]
        L.gdn_forward_chunk_host.restype = ctypes.c_int
        L.gdn_forward_chunk_host.argtypes = [vp, vp, vp, vp, fp, fp, fp, vp, fp, vp]
        L.gdn_feature_map.restype = ctypes.c_int
        L.gdn_feature_map.argtypes = [vp, ctypes.POINTER(GdnFeatmapArgs), vp, vp, vp, vp, vp]
        L.gdn_compute_gates.restype = ctypes.c_int
        L.gdn_compute_gates.argtypes = [vp, ctypes.POINTER(GdnGateArgs), fp, fp, vp]
        L.gdn_compute_gates_static.restype = ctypes.c_int
        L.gdn_compute_gates_static.argtypes = [ctypes.POINTER(GdnGateArgs)] + [ctypes.c_int] * 6 + [fp, fp, vp]
        L.gdn_forward_chunk_full.restype = ctypes.c_int
        L.gdn_forward_chunk_full.argtypes = [vp, ctypes.POINTER(GdnFeatmapArgs), vp, ctypes.POINTER(GdnGateArgs), fp, fp, vp,
                                             fp, fp, vp, fp, fp, vp]
        L.gdn_destroy.restype = ctypes.c_int
        L.gdn_destroy.argtypes = [vp]
        L.gdn_plan_get_info.restype = ctypes.c_int
        L.gdn_plan_get_info.argtypes = [vp, ctypes.POINTER(GdnPlanInfo)]
        L.gdn_plan_set_profiling.restype = ctypes.c_int
        L.gdn_plan_set_profiling.argtypes = [vp, ctypes.c_int]
        L.gdn_plan_kernel_times.restype = ctypes.c_int
        L.gdn_plan_kernel_times.argtypes = [vp, ctypes.c_int, ctypes.POINTER(cp), ctypes.POINTER(ctypes.c_float),
                                            ctypes.POINTER(ctypes.c_int)]
        L.gdn_status_string.restype = cp
        L.gdn_status_string.argtypes = [ctypes.c_int]
        L.gdn_last_error.restype = cp
        L.gdn_last_error.argtypes = [vp]
        L.gdn_version.restype = cp
        L.gdn_version.argtypes = []
        _lib = L
    return _lib


def _ptr(x) -> Optional[int]:
    """Raw address of a torch tensor / int / None."""
    if x is None:
        return None
    if isinstance(x, int):
        return x
    return int(x.data_ptr())


def _stream_handle(stream) -> Optional[int]:
    if stream is None:
        import torch
        return int(torch.cuda.current_stream().cuda_stream)
    if isinstance(stream, int):
        return stream or None
    return int(stream.cuda_stream)


def gdn_status_string(status: int) -> str:
    return lib().gdn_status_string(int(status)).decode()


def gdn_last_error(plan: Optional[int]) -> str:
    return lib().gdn_last_error(plan).decode()


def gdn_version() -> str:
    return lib().gdn_version().decode()


def make_config(B, H, T, d_k, d_v, *, group=1, chunk=0, io_dtype=GDN_BF16, scale=1.0, eps=1e-6, flags=0,
                q_token_stride=0, k_token_stride=0, v_token_stride=0, o_token_stride=0) -> GdnConfig:
    return GdnConfig(ctypes.sizeof(GdnConfig), B, H, T, d_k, d_v, group, chunk, io_dtype, scale, eps, flags,
                     q_token_stride, k_token_stride, v_token_stride, o_token_stride)


def gdn_plan(cfg: GdnConfig) -> int:
    """-> opaque plan handle (int). Raises GdnError on failure."""
    handle = ctypes.c_void_p()
    st = lib().gdn_plan(ctypes.byref(cfg), ctypes.byref(handle))
    if st != GDN_OK:
        raise GdnError(st, gdn_last_error(None))
    return handle.value


def _check(plan, st):
    if st != GDN_OK:
        raise GdnError(st, gdn_last_error(plan))


def gdn_forward_chunk(plan, q, k, v, alpha, beta, state_in, out, state_out, stream=None) -> None:
    _check(plan, lib().gdn_forward_chunk(plan, _ptr(q), _ptr(k), _ptr(v), _ptr(alpha), _ptr(beta), _ptr(state_in),
                                         _ptr(out), _ptr(state_out), _stream_handle(stream)))


def gdn_forward_chunk_norm(plan, q_rot, k_rot, v, q_raw, k_raw, alpha, beta, S_in, z_in, out, S_out, z_out,
                           stream=None) -> None:
    _check(plan, lib().gdn_forward_chunk_norm(plan, _ptr(q_rot), _ptr(k_rot), _ptr(v), _ptr(q_raw), _ptr(k_raw),
                                              _ptr(alpha), _ptr(beta), _ptr(S_in), _ptr(z_in), _ptr(out), _ptr(S_out),
                                              _ptr(z_out), _stream_handle(stream)))


def gdn_forward_chunk_host(plan, q, k, v, alpha, beta, state_in, out, state_out, stream=None) -> None:
    """Host (CPU, ideally pinned) tensors in and out; the caller synchronises the stream afterwards."""
    _check(plan, lib().gdn_forward_chunk_host(plan, _ptr(q), _ptr(k), _ptr(v), _ptr(alpha), _ptr(beta),
                                              _ptr(state_in), _ptr(out), _ptr(state_out), _stream_handle(stream)))


def make_featmap_args(q, k, rms_wq, rms_wk, rope_cos, rope_sin, rms_eps=1e-6) -> GdnFeatmapArgs:
    return GdnFeatmapArgs(_ptr(q), _ptr(k), _ptr(rms_wq), _ptr(rms_wk), _ptr(rope_cos), _ptr(rope_sin), rms_eps)


def make_gate_args(x, w_alpha, b_alpha, a_log, w_beta, b_beta, x_token_stride=0) -> GdnGateArgs:
    return GdnGateArgs(_ptr(x), x_token_stride, _ptr(w_alpha), _ptr(b_alpha), _ptr(a_log), _ptr(w_beta), _ptr(b_beta))


def gdn_feature_map(plan, fm: GdnFeatmapArgs, q_rot, k_rot, q_raw, k_raw, stream=None) -> None:
    _check(plan, lib().gdn_feature_map(plan, ctypes.byref(fm), _ptr(q_rot), _ptr(k_rot), _ptr(q_raw), _ptr(k_raw),
                                       _stream_handle(stream)))


def gdn_compute_gates(plan, ga: GdnGateArgs, alpha_out, beta_out, stream=None) -> None:
    _check(plan, lib().gdn_compute_gates(plan, ctypes.byref(ga), _ptr(alpha_out), _ptr(beta_out), _stream_handle(stream)))


def gdn_compute_gates_static(ga: GdnGateArgs, B: int, T: int, H: int, D: int, group: int, log_alpha: bool, alpha_out, beta_out,
                             stream=None) -> None:
    """The gates without a plan and without any allocation (static device scratch; see include/gdn.h for the limit)."""
    _check(None, lib().gdn_compute_gates_static(ctypes.byref(ga), B, T, H, D, group, int(bool(log_alpha)), _ptr(alpha_out),
                                                _ptr(beta_out), _stream_handle(stream)))


def gdn_forward_chunk_full(plan, fm: GdnFeatmapArgs, v, gates: Optional[GdnGateArgs], alpha, beta, out_gate, S_in, z_in,
                           out, S_out, z_out, stream=None) -> None:
    _check(plan, lib().gdn_forward_chunk_full(plan, ctypes.byref(fm), _ptr(v), ctypes.byref(gates) if gates is not None else None,
                                              _ptr(alpha), _ptr(beta), _ptr(out_gate), _ptr(S_in), _ptr(z_in), _ptr(out),
                                              _ptr(S_out), _ptr(z_out), _stream_handle(stream)))


def gdn_destroy(plan) -> None:
    if plan:
        lib().gdn_destroy(plan)


def gdn_plan_get_info(plan) -> GdnPlanInfo:
    info = GdnPlanInfo()
    st = lib().gdn_plan_get_info(plan, ctypes.byref(info))
    if st != GDN_OK:
        raise GdnError(st)
    return info


def gdn_plan_set_profiling(plan, enable: int) -> None:
    _check(plan, lib().gdn_plan_set_profiling(plan, int(enable)))


def gdn_plan_kernel_times(plan, max_n: int = 16):
    """-> (names, avg_ms) of each kernel of a call since profiling was enabled."""
    names = (ctypes.c_char_p * max_n)()
    ms = (ctypes.c_float * max_n)()
    n = ctypes.c_int(0)
    _check(plan, lib().gdn_plan_kernel_times(plan, max_n, names, ms, ctypes.byref(n)))
    return [names[i].decode() for i in range(n.value)], [float(ms[i]) for i in range(n.value)]


class GdnPlan:
    """RAII wrapper: ``with GdnPlan(B=..., ...) as p: p.forward(q, k, v, alpha, beta, state_in, out, state_out)``."""

    def __init__(self, **kw):
        self.cfg = make_config(**kw)
        self.handle = gdn_plan(self.cfg)

    @property
    def info(self) -> GdnPlanInfo:
        return gdn_plan_get_info(self.handle)

    def forward(self, q, k, v, alpha, beta, state_in, out, state_out, stream=None):
        gdn_forward_chunk(self.handle, q, k, v, alpha, beta, state_in, out, state_out, stream)

    def forward_norm(self, *a, stream=None):
        gdn_forward_chunk_norm(self.handle, *a, stream=stream)

    def feature_map(self, fm, q_rot, k_rot, q_raw, k_raw, stream=None):
        gdn_feature_map(self.handle, fm, q_rot, k_rot, q_raw, k_raw, stream)

    def compute_gates(self, ga, alpha_out, beta_out, stream=None):
        gdn_compute_gates(self.handle, ga, alpha_out, beta_out, stream)

    def forward_full(self, fm, v, gates, alpha, beta, out_gate, S_in, z_in, out, S_out, z_out, stream=None):
        gdn_forward_chunk_full(self.handle, fm, v, gates, alpha, beta, out_gate, S_in, z_in, out, S_out, z_out, stream)

    def forward_host(self, q, k, v, alpha, beta, state_in, out, state_out, stream=None):
        gdn_forward_chunk_host(self.handle, q, k, v, alpha, beta, state_in, out, state_out, stream)

    def close(self):
        if self.handle:
            gdn_destroy(self.handle)
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
