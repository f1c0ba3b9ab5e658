"""CPU oracle for the Gated DeltaNet forward -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference``
legs may import this package.  It shares no code with ``paper_2605_30409_b200`` (the CUDA path) and
neither imports the other.  The arithmetic lives in ``gdn_oracle.c`` (plain C, fp64, the paper's
predict-then-correct recurrence, Eq. 17-22); this file only compiles it with gcc
and marshals numpy arrays through ctypes.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "gdn_oracle.c"
_LIB = _HERE / "libgdn_oracle.so"
_lib = None


class _Strides(ctypes.Structure):
    _fields_ = [("batch", ctypes.c_int64), ("token", ctypes.c_int64), ("head", ctypes.c_int64)]


def build(force: bool = False) -> Path:
    """Compile gdn_oracle.c -> libgdn_oracle.so (gcc -O2 -fopenmp). Building is not using."""
    if force or (not _LIB.exists()) or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        tmp = _LIB.with_suffix(f".so.tmp{os.getpid()}")
        cmd = ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c11", "-o", str(tmp), str(_SRC)]
        subprocess.run(cmd, check=True, capture_output=True)
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(str(_LIB))
        fp = ctypes.POINTER(ctypes.c_float)
        dp = ctypes.POINTER(ctypes.c_double)
        sp = ctypes.POINTER(_Strides)
        lib.gdn_oracle_forward.restype = ctypes.c_int
        lib.gdn_oracle_forward.argtypes = [ctypes.c_int] * 6 + [fp, sp] * 5 + [fp, fp, dp, dp,
                                          ctypes.c_double, ctypes.c_double, ctypes.c_int,
                                          dp, dp, dp, ctypes.c_int]
        lib.gdn_oracle_forward_bidir.restype = ctypes.c_int
        lib.gdn_oracle_forward_bidir.argtypes = lib.gdn_oracle_forward.argtypes
        lib.gdn_oracle_max_threads.restype = ctypes.c_int
        _lib = lib
    return _lib


def max_threads() -> int:
    return int(_load().gdn_oracle_max_threads())


def _as_f32(x):
    """torch tensor (any float dtype, e.g. bf16) or ndarray -> fp32 ndarray (exact for bf16/fp32)."""
    if x is None:
        return None
    if hasattr(x, "detach"):
        x = x.detach().cpu().float().numpy()
    a = np.asarray(x, dtype=np.float32)
    if a.strides[-1] != a.itemsize:
        a = np.ascontiguousarray(a)
    return a


def _as_f64(x):
    if x is None:
        return None
    if hasattr(x, "detach"):
        x = x.detach().cpu().double().numpy()
    return np.ascontiguousarray(np.asarray(x, dtype=np.float64))


def _ptr_strides(a):
    it = a.itemsize
    assert a.ndim == 4 and a.strides[3] == it
    st = _Strides(a.strides[0] // it, a.strides[1] // it, a.strides[2] // it)
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_float)), ctypes.byref(st), st


def gdn_forward(q, k, v, alpha, beta, S_in=None, *, group: int = 1, scale: float = 1.0,
                q_raw=None, k_raw=None, z_in=None, eps: float = 1e-6, normalizer: bool = False,
                bidir: bool = False, nthreads: int = 0):
    """Run the oracle.  ``bidir``: the bidirectional in-chunk scan of PAPER.md Alg. 1 lines 8-22 (forward scan from
    the cache plus a reverse scan over the frames of this call, one readout on the summed histories); S_out / z_out
    stay the forward terminal states.

    q,k: [B,T,H,d_k]; v: [B,T,H,d_v]; alpha: [B,H,T/group]; beta: [B,H,T]; S_in: [B,H,d_k,d_v] or None.
    Returns (out [B,T,H,d_v] fp64, S_out [B,H,d_k,d_v] fp64) and, with ``normalizer``, also z_out.
    """
    lib = _load()
    q, k, v = _as_f32(q), _as_f32(k), _as_f32(v)
    B, T, H, dk = q.shape
    dv = v.shape[3]
    assert k.shape == (B, T, H, dk) and v.shape == (B, T, H, dv)
    assert group >= 1 and T % group == 0
    alpha = np.ascontiguousarray(_as_f32(alpha)).reshape(B, H, T // group)
    beta = np.ascontiguousarray(_as_f32(beta)).reshape(B, H, T)
    S_in = _as_f64(S_in)
    z_in = _as_f64(z_in)
    if S_in is not None:
        assert S_in.shape == (B, H, dk, dv)
    out = np.empty((B, T, H, dv), dtype=np.float64)
    S_out = np.empty((B, H, dk, dv), dtype=np.float64)
    z_out = np.zeros((B, H, dk), dtype=np.float64)
    dp = ctypes.POINTER(ctypes.c_double)
    fpt = ctypes.POINTER(ctypes.c_float)
    keep = []

    def ps(a):
        if a is None:
            return ctypes.cast(None, fpt), ctypes.cast(None, ctypes.POINTER(_Strides))
        p, ref, st = _ptr_strides(a)
        keep.append(st)
        return p, ref

    if normalizer:
        q_raw, k_raw = _as_f32(q_raw), _as_f32(k_raw)
        assert q_raw.shape == q.shape and k_raw.shape == k.shape
    else:
        q_raw = k_raw = None
    args = [B, H, T, dk, dv, group]
    for a in (q, k, v, q_raw, k_raw):
        args.extend(ps(a))
    args += [alpha.ctypes.data_as(fpt), beta.ctypes.data_as(fpt),
             S_in.ctypes.data_as(dp) if S_in is not None else ctypes.cast(None, dp),
             z_in.ctypes.data_as(dp) if z_in is not None else ctypes.cast(None, dp),
             float(scale), float(eps), int(bool(normalizer)),
             out.ctypes.data_as(dp), S_out.ctypes.data_as(dp), z_out.ctypes.data_as(dp), int(nthreads)]
    rc = (lib.gdn_oracle_forward_bidir if bidir else lib.gdn_oracle_forward)(*args)
    if rc != 0:
        raise RuntimeError(f"gdn_oracle_forward failed with code {rc}")
    if normalizer:
        return out, S_out, z_out
    return out, S_out
