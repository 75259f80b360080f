"""Thin ctypes binding of include/demons.h -- argument marshalling only.

Every function has the name and the argument order of its C entry point; tensors are passed as
raw device (or host) pointers, streams as `torch.cuda.Stream.cuda_stream`.  Nothing is computed
here: every step of the path runs in the CUDA kernels of libdemons.so.  PyTorch is used by
callers for device allocations and streams only.  There is no fallback: if libdemons.so is
missing or does not load, importing this module's `lib()` raises.
"""
from __future__ import annotations

import ctypes
import os

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libdemons.so")

PASSIVE, EVOLVED_PASSIVE, ACTIVE, DOUBLE, ADJUSTED_DOUBLE, INVERSE_CONSISTENT = range(6)
VARIANT_NAMES = ["passive", "evolved_passive", "active", "double", "adjusted_double", "inverse_consistent"]
OK, E_ARG, E_CUDA, E_WORKSPACE, E_UNSUPPORTED = 0, -1, -2, -3, -4

# name -> (restype, argtypes); mirrors include/demons.h one to one
_c_int3 = ctypes.POINTER(ctypes.c_int)
_c_float3 = ctypes.POINTER(ctypes.c_float)
_vp = ctypes.c_void_p
SIGNATURES = {
    "demons_create": (ctypes.c_int, [ctypes.POINTER(_vp), _c_int3, _c_float3, ctypes.c_int, ctypes.c_float,
                                     ctypes.c_float]),
    "demons_destroy": (None, [_vp]),
    "demons_workspace_bytes": (ctypes.c_size_t, [_vp, ctypes.c_int]),
    "demons_workspace_bytes_batch": (ctypes.c_size_t, [_vp, ctypes.c_int, ctypes.c_int]),
    "demons_set_workspace": (ctypes.c_int, [_vp, _vp, ctypes.c_size_t]),
    "demons_level_dims": (ctypes.c_int, [_vp, ctypes.c_int, _c_int3]),
    "demons_launch_count": (ctypes.c_longlong, [_vp]),
    "demons_get_profile": (ctypes.c_int, [_vp, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_longlong)]),
    "demons_set_option": (ctypes.c_int, [_vp, ctypes.c_char_p, ctypes.c_int]),
    "demons_register": (ctypes.c_int, [_vp, _vp, _vp, _vp, _vp, ctypes.c_int, _c_int3, ctypes.c_double, _vp, _vp,
                                       _vp]),
    "demons_register_batch": (ctypes.c_int, [_vp, ctypes.c_int, _vp, _vp, _vp, _vp, ctypes.c_int, _c_int3, ctypes.c_double,
                                             _vp, _vp, _vp]),
    "demons_register_host": (ctypes.c_int, [_vp, _vp, _vp, _vp, _vp, ctypes.c_int, _c_int3, ctypes.c_double, _vp,
                                            _vp, _vp]),
    "demons_workspace_bytes_queue": (ctypes.c_size_t, [_vp, ctypes.c_int]),
    "demons_register_host_queue": (ctypes.c_int, [_vp, ctypes.c_int, _vp, _vp, _vp, _vp, ctypes.c_int, _c_int3,
                                                  ctypes.c_double, _vp, _vp, _vp]),
    "demons_warp_force": (ctypes.c_int, [_vp, _c_int3, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp]),
    "demons_warp_force_slab": (ctypes.c_int, [_vp, _c_int3, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int, _vp, _vp,
                                              _vp, _vp, _vp, _vp, _vp, _vp]),
    "demons_smooth": (ctypes.c_int, [_vp, _c_int3, _vp, _vp, ctypes.c_int, ctypes.c_float, _vp]),
    "demons_restrict": (ctypes.c_int, [_vp, _c_int3, _vp, _vp, _vp]),
    "demons_prolong": (ctypes.c_int, [_vp, _c_int3, _vp, _c_int3, _vp, _vp]),
    "demons_ssd": (ctypes.c_int, [_vp, _c_int3, _vp, _vp, _vp, _vp, _vp, _vp]),
    "demons_ic_error": (ctypes.c_int, [_vp, _c_int3, _vp, _vp, _vp, _vp]),
    "demons_cc": (ctypes.c_int, [_vp, _c_int3, _vp, _vp, _vp, _vp, _vp, _vp]),
    "demons_point_error": (ctypes.c_int, [_vp, _c_int3, _vp, ctypes.c_int, _vp, _vp, _vp, _vp]),
    "demons_ssd_static": (ctypes.c_int, [_c_int3, _vp, _vp, _vp, _vp, _vp, _vp]),
    "demons_last_error": (ctypes.c_char_p, []),
}

_lib = None


class DemonsError(RuntimeError):
    def __init__(self, code, message):
        super().__init__(f"demons error {code}: {message}")
        self.code = code


def lib():
    """Loads libdemons.so (built in-tree by paper_0909_0928_b200.build).  Raises if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} not found: build it with `python -m paper_0909_0928_b200.build` "
                              "(there is no CPU fallback)")
        L = ctypes.CDLL(LIB_PATH)
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(L, name)
            fn.restype = res
            fn.argtypes = args
        _lib = L
    return _lib


def _check(rc):
    if rc != OK:
        raise DemonsError(rc, lib().demons_last_error().decode())


def _int3(v):
    return (ctypes.c_int * 3)(int(v[0]), int(v[1]), int(v[2]))


def _ptr(t):
    """Raw pointer of a torch tensor / numpy array / int / None."""
    if t is None:
        return None
    if isinstance(t, int):
        return t
    if hasattr(t, "data_ptr"):
        assert t.is_contiguous(), "tensors must be contiguous"
        return t.data_ptr()
    return t.ctypes.data


def _stream(stream):
    if stream is None:
        return None
    return stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream)


def dims_of(t):
    """(nx, ny, nz) of a (.., nz, ny, nx) tensor."""
    nz, ny, nx = t.shape[-3:]
    return (int(nx), int(ny), int(nz))


# ---- the C entry points, same names ------------------------------------------------------------

def demons_create(dims, spacing, variant, alpha, sigma):
    ctx = _vp()
    sp = (ctypes.c_float * 3)(*[float(s) for s in spacing])
    _check(lib().demons_create(ctypes.byref(ctx), _int3(dims), sp, int(variant), float(alpha), float(sigma)))
    return ctx


def demons_destroy(ctx):
    lib().demons_destroy(ctx)


def demons_workspace_bytes(ctx, levels):
    return int(lib().demons_workspace_bytes(ctx, int(levels)))


def demons_workspace_bytes_batch(ctx, levels, nbatch):
    return int(lib().demons_workspace_bytes_batch(ctx, int(levels), int(nbatch)))


def demons_set_workspace(ctx, d_ws, nbytes):
    _check(lib().demons_set_workspace(ctx, _ptr(d_ws), int(nbytes)))


def demons_level_dims(ctx, level):
    out = (ctypes.c_int * 3)()
    _check(lib().demons_level_dims(ctx, int(level), out))
    return tuple(out)


def demons_launch_count(ctx):
    return int(lib().demons_launch_count(ctx))


def demons_get_profile(ctx):
    ms = (ctypes.c_double * 4)()
    n = (ctypes.c_longlong * 4)()
    _check(lib().demons_get_profile(ctx, ms, n))
    names = ("force", "warp", "smooth", "pyramid")
    return {k: {"ms": ms[i], "groups": int(n[i])} for i, k in enumerate(names)}


def demons_set_option(ctx, name, value):
    _check(lib().demons_set_option(ctx, name.encode(), int(value)))


def demons_register(ctx, d_static, d_moving, d_u, d_u_back, iters_per_level, eps=0.0, h_stats=None,
                    h_iters_done=None, stream=None):
    levels = len(iters_per_level)
    it = (ctypes.c_int * levels)(*[int(i) for i in iters_per_level])
    _check(lib().demons_register(ctx, _ptr(d_static), _ptr(d_moving), _ptr(d_u), _ptr(d_u_back), levels, it,
                                 float(eps), _ptr(h_stats), _ptr(h_iters_done), _stream(stream)))


def demons_register_batch(ctx, nbatch, d_static, d_moving, d_u, d_u_back, iters_per_level, eps=0.0, h_stats=None,
                          h_iters_done=None, stream=None):
    levels = len(iters_per_level)
    it = (ctypes.c_int * levels)(*[int(i) for i in iters_per_level])
    _check(lib().demons_register_batch(ctx, int(nbatch), _ptr(d_static), _ptr(d_moving), _ptr(d_u), _ptr(d_u_back),
                                       levels, it, float(eps), _ptr(h_stats), _ptr(h_iters_done), _stream(stream)))


def demons_register_host(ctx, h_static, h_moving, h_u, h_u_back, iters_per_level, eps=0.0, h_stats=None,
                         h_iters_done=None, stream=None):
    levels = len(iters_per_level)
    it = (ctypes.c_int * levels)(*[int(i) for i in iters_per_level])
    _check(lib().demons_register_host(ctx, _ptr(h_static), _ptr(h_moving), _ptr(h_u), _ptr(h_u_back), levels, it,
                                      float(eps), _ptr(h_stats), _ptr(h_iters_done), _stream(stream)))


def demons_workspace_bytes_queue(ctx, levels):
    return int(lib().demons_workspace_bytes_queue(ctx, int(levels)))


def demons_register_host_queue(ctx, h_static, h_moving, h_u, h_u_back, iters_per_level, eps=0.0, h_stats=None,
                               h_iters_done=None, stream=None):
    """h_static, h_moving, h_u (h_u_back): sequences of n host buffers (pinned torch tensors or numpy arrays)."""
    n = len(h_static)
    levels = len(iters_per_level)
    it = (ctypes.c_int * levels)(*[int(i) for i in iters_per_level])

    def ptrs(seq):
        return None if seq is None else (ctypes.c_void_p * n)(*[_ptr(t) for t in seq])
    pS, pM, pU, pUb = ptrs(h_static), ptrs(h_moving), ptrs(h_u), ptrs(h_u_back)
    _check(lib().demons_register_host_queue(ctx, n, pS, pM, pU, pUb, levels, it, float(eps), _ptr(h_stats),
                                            _ptr(h_iters_done), _stream(stream)))


def demons_warp_force(ctx, dims, d_static, d_moving, d_u_in, d_u_out, d_ub_in=None, d_ub_out=None, d_metrics=None,
                      stream=None):
    _check(lib().demons_warp_force(ctx, _int3(dims), _ptr(d_static), _ptr(d_moving), _ptr(d_u_in), _ptr(d_u_out),
                                   _ptr(d_ub_in), _ptr(d_ub_out), _ptr(d_metrics), _stream(stream)))


def demons_warp_force_slab(ctx, dims, z_begin, z_count, own_begin, own_count, d_static, d_moving, d_u_in, d_u_out,
                           d_ub_in=None, d_ub_out=None, d_metrics=None, stream=None):
    _check(lib().demons_warp_force_slab(ctx, _int3(dims), int(z_begin), int(z_count), int(own_begin), int(own_count),
                                        _ptr(d_static), _ptr(d_moving), _ptr(d_u_in), _ptr(d_u_out), _ptr(d_ub_in),
                                        _ptr(d_ub_out), _ptr(d_metrics), _stream(stream)))


def demons_smooth(ctx, dims, d_in, d_out, ncomp, sigma, stream=None):
    _check(lib().demons_smooth(ctx, _int3(dims), _ptr(d_in), _ptr(d_out), int(ncomp), float(sigma), _stream(stream)))


def demons_restrict(ctx, fine_dims, d_fine, d_coarse, stream=None):
    _check(lib().demons_restrict(ctx, _int3(fine_dims), _ptr(d_fine), _ptr(d_coarse), _stream(stream)))


def demons_prolong(ctx, coarse_dims, d_uc, fine_dims, d_uf, stream=None):
    _check(lib().demons_prolong(ctx, _int3(coarse_dims), _ptr(d_uc), _int3(fine_dims), _ptr(d_uf), _stream(stream)))


def demons_ssd(ctx, dims, d_static, d_moving, d_u, d_ub, d_out, stream=None):
    _check(lib().demons_ssd(ctx, _int3(dims), _ptr(d_static), _ptr(d_moving), _ptr(d_u), _ptr(d_ub), _ptr(d_out),
                            _stream(stream)))


def demons_ic_error(ctx, dims, d_uf, d_ub, d_out, stream=None):
    _check(lib().demons_ic_error(ctx, _int3(dims), _ptr(d_uf), _ptr(d_ub), _ptr(d_out), _stream(stream)))


def demons_cc(ctx, dims, d_static, d_moving, d_u, d_ub, d_out, stream=None):
    _check(lib().demons_cc(ctx, _int3(dims), _ptr(d_static), _ptr(d_moving), _ptr(d_u), _ptr(d_ub), _ptr(d_out),
                           _stream(stream)))


def demons_point_error(ctx, dims, d_u, n_points, d_points, d_expect, d_err, stream=None):
    _check(lib().demons_point_error(ctx, _int3(dims), _ptr(d_u), int(n_points), _ptr(d_points), _ptr(d_expect),
                                    _ptr(d_err), _stream(stream)))


SSD_STATIC_MAX_VOXELS = 1 << 26


def demons_ssd_static(dims, d_static, d_moving, d_u, d_ub, d_out, stream=None):
    """SSD without a context or a workspace (scratch is a fixed array inside libdemons.so); see include/demons.h."""
    _check(lib().demons_ssd_static(_int3(dims), _ptr(d_static), _ptr(d_moving), _ptr(d_u), _ptr(d_ub), _ptr(d_out),
                                   _stream(stream)))


def demons_last_error():
    return lib().demons_last_error().decode()


# ---- convenience: a context plus its torch-allocated workspace ------------------------------------

class Demons:
    """Owns a demons_ctx and the torch tensor backing its workspace (allocation only)."""

    def __init__(self, dims, spacing=(1.0, 1.0, 1.0), variant=PASSIVE, alpha=1.0, sigma=1.0, levels=1,
                 device="cuda:0", nbatch=1, queue=False):
        import torch
        self.dims = tuple(int(d) for d in dims)
        self.variant = int(variant)
        self.levels = int(levels)
        self.sigma = float(sigma)
        self.ctx = demons_create(self.dims, spacing, variant, alpha, sigma)
        self.nbatch = int(nbatch)
        nbytes = demons_workspace_bytes_batch(self.ctx, levels, nbatch)
        if queue:  # second staging slot of demons_register_host_queue
            nbytes = max(nbytes, demons_workspace_bytes_queue(self.ctx, levels))
        self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=device)
        off = (-self.workspace.data_ptr()) % 256
        self._ws_ptr = self.workspace.data_ptr() + off
        demons_set_workspace(self.ctx, self._ws_ptr, nbytes)

    def close(self):
        if self.ctx is not None:
            demons_destroy(self.ctx)
            self.ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
