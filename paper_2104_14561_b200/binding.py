"""ctypes binding of the C ABI in include/fk.h (libfk_b200.so): argument marshalling only.

Same names as the C entry points (`fk_create`, `fk_set_coeffs`, `fk_set_coeffs_range`,
`fk_evolve`, `fk_reset`, `fk_read`, `fk_reduce`, `fk_reduce_static`, `fk_check`, `fk_profile`, `fk_profile_read`,
`fk_profile_updates`, `fk_work`, `fk_paths`, `fk_peak_fp64`, `fk_launch_count`, `fk_destroy`,
`fk_last_error`, `fk_gauss_hermite`).  Arrays may be numpy arrays (host
pointers) or torch CUDA tensors (device pointers); every step of the path runs in the CUDA
kernels behind the ABI.  There is no CPU fallback: a missing library raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

FK_OK, FK_EINVAL, FK_ENOMEM, FK_ECUDA, FK_ESTATE = 0, 1, 2, 3, 4
FK_FACE_ABSORB, FK_FACE_CLAMP, FK_FACE_PERIODIC = 0, 1, 2
FK_MEM_HOST, FK_MEM_DEVICE, FK_MEM_HOST_PINNED = 0, 1, 2
FK_ALL_STEPS = -1
FK_MAX_Q = 32
FK_REDUCE_STATIC_MAX_CHUNKS = 64
FK_FLAG_VALIDATE = 1
FK_FLAG_WEIGHTED_SLOPES = 2
FK_FLAG_MULTISTEP = 4
FK_FLAG_COUNT_PATHS = 8
PATHS = ("3d_same", "3d_merged", "3d_wide", "3d_wide_merged", "3d_rowwise", "2d_banded", "2d_scattered")
FK_PATH_COUNT = 8
FK_K_ASSEMBLE, FK_K_SLOPES, FK_K_APPLY, FK_K_FUSED, FK_K_ROWBLOCK, FK_K_FAR2D, FK_K_LINE1D, FK_K_COUNT = 0, 1, 2, 3, 4, 5, 6, 7
KERNEL_CLASSES = ("assemble", "slopes", "apply", "fused", "rowblock", "far2d", "line1d")

LIB_PATH = os.path.join(os.path.dirname(os.path.abspath(__file__)), "libfk_b200.so")

EXPORTS = ("fk_create", "fk_set_coeffs", "fk_set_coeffs_range", "fk_evolve", "fk_reset",
           "fk_read", "fk_reduce", "fk_reduce_static", "fk_check", "fk_profile", "fk_profile_read",
           "fk_profile_updates", "fk_work", "fk_paths", "fk_peak_fp64", "fk_launch_count", "fk_destroy",
           "fk_last_error", "fk_gauss_hermite")


class FkError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"fk error {code}: {msg}")
        self.code = code


class fk_params(C.Structure):
    _fields_ = [("d", C.c_int), ("n", C.c_int * 3), ("x", C.POINTER(C.c_double) * 3),
                ("dt", C.c_double), ("N", C.c_int), ("Q", C.c_int * 3),
                ("face_kind", (C.c_int * 2) * 3), ("face_value", (C.c_double * 2) * 3),
                ("coeff_slots", C.c_int), ("device", C.c_int), ("stream", C.c_void_p),
                ("flags", C.c_uint), ("shard_index", C.c_int), ("shard_count", C.c_int)]


_lib = None


def lib():
    """Load libfk_b200.so (built in-tree by paper_2104_14561_b200.build); raise if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(
                f"{LIB_PATH} is missing: build it with `python -m paper_2104_14561_b200.build` "
                "(the Feynman-Kac path runs only in its CUDA kernels; there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        dp, vp = C.POINTER(C.c_double), C.c_void_p
        L.fk_create.argtypes = [C.POINTER(fk_params), C.POINTER(vp)]
        L.fk_set_coeffs.argtypes = [vp, C.c_int, vp, vp, C.c_int]
        L.fk_set_coeffs_range.argtypes = [vp, C.c_int, C.c_int, vp, vp, C.c_int]
        L.fk_evolve.argtypes = [vp, C.c_int, C.c_int]
        L.fk_reset.argtypes = [vp]
        L.fk_read.argtypes = [vp, C.c_int, C.c_int, vp, C.c_int]
        L.fk_reduce.argtypes = [vp, vp, C.c_int, C.c_int, vp, C.c_int]
        L.fk_reduce_static.argtypes = [vp, vp, C.c_int, C.c_int, vp]
        L.fk_check.argtypes = [vp]
        L.fk_profile.argtypes = [vp, C.c_int]
        L.fk_profile_read.argtypes = [vp, dp, C.POINTER(C.c_longlong)]
        L.fk_profile_updates.argtypes = [vp, dp]
        L.fk_work.argtypes = [vp, dp]
        L.fk_paths.argtypes = [vp, C.POINTER(C.c_longlong)]
        L.fk_peak_fp64.argtypes = [C.c_int, vp, C.c_int, dp, dp]
        L.fk_launch_count.argtypes = [vp]
        L.fk_launch_count.restype = C.c_longlong
        L.fk_destroy.argtypes = [vp]
        L.fk_destroy.restype = None
        L.fk_last_error.argtypes = [vp]
        L.fk_last_error.restype = C.c_char_p
        L.fk_gauss_hermite.argtypes = [C.c_int, dp, dp]
        _lib = L
    return _lib


def _check(ctx, code):
    if code != FK_OK:
        raise FkError(code, lib().fk_last_error(ctx).decode())


def _buffer(a, elems=None):
    """(pointer, mem kind, keep-alive) of a float64 C-contiguous numpy array or CUDA tensor."""
    if hasattr(a, "data_ptr"):                      # torch tensor
        import torch
        if a.dtype != torch.float64 or not a.is_contiguous():
            raise TypeError("tensor must be contiguous float64")
        if elems is not None and a.numel() != elems:
            raise ValueError(f"expected {elems} elements, got {a.numel()}")
        return C.c_void_p(a.data_ptr()), (FK_MEM_DEVICE if a.is_cuda else FK_MEM_HOST), a
    if not isinstance(a, np.ndarray) or a.dtype != np.float64 or not a.flags.c_contiguous:
        a = np.ascontiguousarray(a, dtype=np.float64)
    if elems is not None and a.size != elems:
        raise ValueError(f"expected {elems} elements, got {a.size}")
    return C.c_void_p(a.ctypes.data), FK_MEM_HOST, a


def fk_gauss_hermite(Q):
    a, w = np.empty(Q), np.empty(Q)
    dp = C.POINTER(C.c_double)
    rc = lib().fk_gauss_hermite(int(Q), a.ctypes.data_as(dp), w.ctypes.data_as(dp))
    if rc != FK_OK:
        raise FkError(rc, "Q must be 1..32")
    return a, w


def fk_create(x, dt, N, Q, face_kind, face_value, coeff_slots=0, device=0, stream=0, flags=0,
              shard_index=0, shard_count=1):
    """-> opaque context handle.  x: list of d node arrays; Q, face_kind[d][2], face_value[d][2]."""
    p = fk_params()
    d = len(x)
    p.d = d
    keep = []
    for k in range(min(d, 3)):
        xa = np.ascontiguousarray(x[k], dtype=np.float64)
        keep.append(xa)
        p.n[k] = xa.size
        p.x[k] = xa.ctypes.data_as(C.POINTER(C.c_double))
        p.Q[k] = int(Q[k])
        for s in range(2):
            p.face_kind[k][s] = int(face_kind[k][s])
            p.face_value[k][s] = float(face_value[k][s])
    p.dt = float(dt)
    p.N = int(N)
    p.coeff_slots = int(coeff_slots)
    p.device = int(device)
    p.stream = C.c_void_p(int(stream) or None)
    p.flags = int(flags)
    p.shard_index = int(shard_index)
    p.shard_count = int(shard_count)
    ctx = C.c_void_p()
    rc = lib().fk_create(C.byref(p), C.byref(ctx))
    if rc != FK_OK:
        raise FkError(rc, lib().fk_last_error(None).decode())
    return ctx


def fk_set_coeffs(ctx, step, b, sigma):
    pb, mb, kb = _buffer(b)
    ps, ms, ks = _buffer(sigma)
    if mb != ms:
        raise ValueError("b and sigma must both be host or both be device arrays")
    _check(ctx, lib().fk_set_coeffs(ctx, int(step), pb, ps, mb))


def fk_set_coeffs_range(ctx, step0, count, b, sigma, pinned_async=False):
    """pinned_async: b and sigma are page-locked torch CPU tensors that the caller keeps alive and
    unchanged until the context's stream has passed the copies (FK_MEM_HOST_PINNED: no sync)."""
    pb, mb, kb = _buffer(b)
    ps, ms, ks = _buffer(sigma)
    if mb != ms:
        raise ValueError("b and sigma must both be host or both be device arrays")
    if pinned_async:
        if mb != FK_MEM_HOST or not (hasattr(b, "is_pinned") and b.is_pinned() and sigma.is_pinned()):
            raise ValueError("pinned_async needs page-locked torch CPU tensors")
        mb = FK_MEM_HOST_PINNED
    _check(ctx, lib().fk_set_coeffs_range(ctx, int(step0), int(count), pb, ps, mb))


def fk_evolve(ctx, n_from, n_to):
    _check(ctx, lib().fk_evolve(ctx, int(n_from), int(n_to)))


def fk_reset(ctx):
    _check(ctx, lib().fk_reset(ctx))


def fk_read(ctx, m0, m1, out):
    """Columns m0..m1-1 into `out` ([m1-m0][J] float64; numpy array or CUDA tensor)."""
    po, mo, ko = _buffer(out)
    if ko is not out:
        raise TypeError("out must be a C-contiguous float64 numpy array or torch tensor")
    _check(ctx, lib().fk_read(ctx, int(m0), int(m1), po, mo))
    return out


def fk_reduce(ctx, weights, m0, m1, out):
    """out[m - m0] = sum_j weights[j] P(t_m, x_j); weights [J] and out [m1-m0] both numpy arrays or
    both CUDA tensors."""
    pw, mw, kw = _buffer(weights)
    po, mo, ko = _buffer(out, m1 - m0)
    if ko is not out:
        raise TypeError("out must be a C-contiguous float64 numpy array or torch tensor")
    if mw != mo:
        raise ValueError("weights and out must both be host or both be device arrays")
    _check(ctx, lib().fk_reduce(ctx, pw, int(m0), int(m1), po, mo))
    return out


def fk_reduce_static(ctx, weights, m0, m1, out):
    """fk_reduce for callers that cannot allocate device memory: weights [J] and out [m1-m0] must be
    CUDA tensors, the range may touch at most FK_REDUCE_STATIC_MAX_CHUNKS 32-column chunks, and the
    partial sums go to a fixed array inside the library that all calls on a device share (do not let
    two calls overlap on the GPU).  Asynchronous on the context's stream; see include/fk.h."""
    pw, mw, kw = _buffer(weights)
    po, mo, ko = _buffer(out, m1 - m0)
    if ko is not out:
        raise TypeError("out must be a contiguous float64 CUDA tensor")
    _check(ctx, lib().fk_reduce_static(ctx, pw, int(m0), int(m1), po))
    return out


def fk_check(ctx):
    """Synchronise the stream; raise FkError(FK_EINVAL) if the device found a bad coefficient."""
    _check(ctx, lib().fk_check(ctx))


def fk_profile(ctx, on):
    _check(ctx, lib().fk_profile(ctx, int(bool(on))))


def fk_profile_read(ctx):
    """-> {class: (ms, launches)} for the kernel classes assemble / slopes / apply / fused."""
    ms = (C.c_double * FK_K_COUNT)()
    ln = (C.c_longlong * FK_K_COUNT)()
    _check(ctx, lib().fk_profile_read(ctx, ms, ln))
    return {KERNEL_CLASSES[k]: (float(ms[k]), int(ln[k])) for k in range(FK_K_COUNT)}


def fk_profile_updates(ctx):
    """-> {class: node-step updates processed since the last fk_reset}."""
    upd = (C.c_double * FK_K_COUNT)()
    _check(ctx, lib().fk_profile_updates(ctx, upd))
    return {KERNEL_CLASSES[k]: float(upd[k]) for k in range(FK_K_COUNT)}


def fk_work(ctx):
    """-> dict(updates_near, fma_near, updates_other, fma_other): algorithmic work counted on the device."""
    w = (C.c_double * 4)()
    _check(ctx, lib().fk_work(ctx, w))
    return {"updates_near": w[0], "fma_near": w[1], "updates_other": w[2], "fma_other": w[3]}


def fk_paths(ctx):
    """-> {path: (group of four rows, step) pairs it served}; needs FK_FLAG_COUNT_PATHS at fk_create."""
    n = (C.c_longlong * FK_PATH_COUNT)()
    _check(ctx, lib().fk_paths(ctx, n))
    return {PATHS[k]: int(n[k]) for k in range(len(PATHS))}


def fk_peak_fp64(device=0, stream=0, iters=1 << 15):
    """-> (TFLOP/s, ms) of the DFMA microkernel (measurement only)."""
    tf, ms = C.c_double(), C.c_double()
    rc = lib().fk_peak_fp64(int(device), C.c_void_p(int(stream) or None), int(iters), C.byref(tf), C.byref(ms))
    if rc != FK_OK:
        raise FkError(rc, "fk_peak_fp64 failed")
    return tf.value, ms.value


def fk_launch_count(ctx):
    return int(lib().fk_launch_count(ctx))


def fk_destroy(ctx):
    if ctx:
        lib().fk_destroy(ctx)


def fk_last_error(ctx):
    return lib().fk_last_error(ctx).decode()
