"""Thin Python binding of the C-ABI library `libbem_b200.so` (include/bem.h).

Argument marshalling only: every step of the boundary-element matrix-vector
product y = S[q] - D[phi] (arXiv 1905.01341) runs in
the CUDA kernels of paper_1905_01341_b200/csrc.  Names follow the C functions:
bem_create, bem_set_option, bem_setup, bem_apply, bem_solve, ...

There is NO CPU fallback: importing works anywhere (so that the exported
symbols can be checked), but every compute call needs a CUDA device and raises
`BemError` otherwise.  The library is built in-tree by
`python -m paper_1905_01341_b200.build` (see __graft_entry__.build()).
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libbem_b200.so")

BEM_OK, BEM_ERR_INVALID_ARG, BEM_ERR_BAD_MESH, BEM_ERR_NOT_SETUP, BEM_ERR_CUDA, BEM_ERR_OOM, BEM_ERR_NOT_CONVERGED = range(7)
STATUS_NAMES = ["BEM_OK", "BEM_ERR_INVALID_ARG", "BEM_ERR_BAD_MESH", "BEM_ERR_NOT_SETUP", "BEM_ERR_CUDA",
                "BEM_ERR_OOM", "BEM_ERR_NOT_CONVERGED"]
TIMING_NAMES = ["lift", "p2m", "m2m", "m2l", "l2l_reduce", "l2p", "p2p", "spmv", "total"]
STAT_NAMES = ["n_targets", "n_sources", "lmax", "n_src_leaves", "n_tgt_leaves", "p2p_pairs", "m2l_pairs", "csr_nnz",
              "near_triangles", "setup_ms", "n_src_boxes", "n_tgt_boxes", "device_bytes", "exp_stride",
              "kernel_launches_per_apply", "m2l_flop", "m2l_row_bytes", "p_dipole", "p2p_pairs_executed", "p2p_pairs_wx", "m2m_pairs", "m2m_parents"]

# every symbol include/bem.h declares
EXPORTS = ["bem_create", "bem_create_points", "bem_create_evaluator", "bem_set_option", "bem_set_stream", "bem_setup", "bem_apply", "bem_solve", "bem_get_timings",
           "bem_get_stats", "bem_get_free_term", "bem_fp64_peak", "bem_fp64_tensor_peak", "bem_last_error", "bem_destroy",
           "bem_surface_velocity", "bem_surface_curvature", "bem_bubble_volume", "bem_filter_create", "bem_filter_apply", "bem_filter_last_error", "bem_filter_destroy",
           "bem_direct_sum_static", "bem_direct_sum_static_last_error"]
DIRECT_STATIC_MAX_TARGETS = 65536      # BEM_DIRECT_STATIC_MAX_TARGETS of include/bem.h


class BemError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"{STATUS_NAMES[status] if 0 <= status < len(STATUS_NAMES) else status}: {message}")
        self.status = status


_lib = None


def load_library() -> ctypes.CDLL:
    """dlopen the in-tree C-ABI library; fails loudly when it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_1905_01341_b200.build` "
                          "(there is no CPU fallback)")
    lib = ctypes.CDLL(LIB_PATH)
    vp, i64, i32, dbl = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int, ctypes.c_double
    lib.bem_create.argtypes = [vp, i64, vp, i64, vp, ctypes.POINTER(vp)]
    lib.bem_create_points.argtypes = [vp, i64, vp, i64, ctypes.POINTER(vp)]
    lib.bem_create_evaluator.argtypes = [vp, vp, i64, ctypes.POINTER(vp)]
    lib.bem_set_option.argtypes = [vp, ctypes.c_char_p, dbl]
    lib.bem_set_stream.argtypes = [vp, vp]
    lib.bem_setup.argtypes = [vp, i32, i32, dbl]
    lib.bem_apply.argtypes = [vp, vp, vp, vp]
    lib.bem_solve.argtypes = [vp, vp, vp, i32, dbl, i32, ctypes.POINTER(i32), ctypes.POINTER(dbl)]
    lib.bem_get_timings.argtypes = [vp, vp, i32]
    lib.bem_get_stats.argtypes = [vp, vp, i32]
    lib.bem_get_free_term.argtypes = [vp, vp]
    lib.bem_fp64_peak.argtypes = [vp, ctypes.POINTER(dbl)]
    lib.bem_fp64_tensor_peak.argtypes = [vp, ctypes.POINTER(dbl)]
    lib.bem_last_error.argtypes = [vp]
    lib.bem_last_error.restype = ctypes.c_char_p
    lib.bem_destroy.argtypes = [vp]
    lib.bem_destroy.restype = None
    lib.bem_surface_velocity.argtypes = [vp, vp, vp, vp, vp, vp]
    lib.bem_surface_curvature.argtypes = [vp, vp]
    lib.bem_bubble_volume.argtypes = [vp, vp, i64]
    lib.bem_filter_create.argtypes = [vp, vp, i64, i32, ctypes.POINTER(vp)]
    lib.bem_filter_apply.argtypes = [vp, vp, i64, vp, vp]
    lib.bem_filter_last_error.argtypes = [vp]
    lib.bem_filter_last_error.restype = ctypes.c_char_p
    lib.bem_filter_destroy.argtypes = [vp]
    lib.bem_filter_destroy.restype = None
    lib.bem_direct_sum_static.argtypes = [vp, i64, vp, vp, vp, i64, vp, vp]
    lib.bem_direct_sum_static_last_error.argtypes = []
    lib.bem_direct_sum_static_last_error.restype = ctypes.c_char_p
    for name in EXPORTS:
        if name not in ("bem_last_error", "bem_destroy", "bem_filter_last_error", "bem_filter_destroy",
                        "bem_direct_sum_static_last_error"):
            getattr(lib, name).restype = ctypes.c_int
    _lib = lib
    return lib


def _ptr(a):
    """Raw address of a numpy array (host) or a torch tensor (host or device), or NULL."""
    if a is None:
        return ctypes.c_void_p(0)
    if isinstance(a, np.ndarray):
        if a.dtype != np.float64 or not a.flags.c_contiguous:
            raise TypeError("numpy arguments must be C-contiguous float64")
        return ctypes.c_void_p(a.ctypes.data)
    if hasattr(a, "data_ptr"):
        import torch
        if a.dtype != torch.float64 or not a.is_contiguous():
            raise TypeError("tensor arguments must be contiguous float64")
        return ctypes.c_void_p(a.data_ptr())
    raise TypeError(f"unsupported array type {type(a)}")


class Bem:
    """One mesh + its setup: the object the C calls operate on (an owned `bem_ctx *`)."""

    def __init__(self, vertices, triangles, bubble_id=None, _points=None, _evaluator=None):
        self._lib = load_library()
        self._ctx = ctypes.c_void_p(0)
        if _evaluator is not None:                   # bem_create_evaluator(mesh_ctx, targets)
            mesh, T = _evaluator[0], np.ascontiguousarray(_evaluator[1], dtype=np.float64)
            if T.ndim != 2 or T.shape[1] != 3:
                raise ValueError("targets must be [n,3]")
            self._mesh = mesh                        # keeps the mesh context alive
            self.n_vertices, self.n_triangles, self.n_sources = T.shape[0], 0, 3 * mesh.n_triangles
            st = self._lib.bem_create_evaluator(mesh._ctx, T.ctypes.data, T.shape[0], ctypes.byref(self._ctx))
            if st != BEM_OK:
                self._ctx = ctypes.c_void_p(0)
                raise BemError(st, self._lib.bem_last_error(None).decode())
            return
        if _points is not None:                      # bem_create_points(sources, targets)
            S = np.ascontiguousarray(_points[0], dtype=np.float64)
            T = np.ascontiguousarray(_points[1], dtype=np.float64)
            if S.ndim != 2 or S.shape[1] != 3 or T.ndim != 2 or T.shape[1] != 3:
                raise ValueError("sources and targets must be [n,3]")
            self.n_vertices, self.n_triangles, self.n_sources = T.shape[0], 0, S.shape[0]
            st = self._lib.bem_create_points(S.ctypes.data, S.shape[0], T.ctypes.data, T.shape[0], ctypes.byref(self._ctx))
            if st != BEM_OK:
                self._ctx = ctypes.c_void_p(0)
                raise BemError(st, "bem_create_points failed (a CUDA device is required): " + self._lib.bem_last_error(None).decode())
            return
        V = np.ascontiguousarray(vertices, dtype=np.float64)
        F = np.ascontiguousarray(triangles, dtype=np.int32)
        if V.ndim != 2 or V.shape[1] != 3 or F.ndim != 2 or F.shape[1] != 3:
            raise ValueError("vertices must be [N,3], triangles [T,3]")
        B = None if bubble_id is None else np.ascontiguousarray(bubble_id, dtype=np.int32)
        self.n_vertices, self.n_triangles = V.shape[0], F.shape[0]
        st = self._lib.bem_create(V.ctypes.data, V.shape[0], F.ctypes.data, F.shape[0],
                                  None if B is None else B.ctypes.data, ctypes.byref(self._ctx))
        if st != BEM_OK:
            self._ctx = ctypes.c_void_p(0)
            raise BemError(st, "bem_create failed (mesh must be a closed, outward-oriented manifold; a CUDA device is required): "
                           + self._lib.bem_last_error(None).decode())

    # -- the C calls, same names --------------------------------------------------
    def _check(self, st, allow=()):
        if st != BEM_OK and st not in allow:
            raise BemError(st, self._lib.bem_last_error(self._ctx).decode())
        return st

    def bem_set_option(self, key: str, value: float):
        self._check(self._lib.bem_set_option(self._ctx, key.encode(), float(value)))

    def bem_set_stream(self, stream_handle: int):
        self._check(self._lib.bem_set_stream(self._ctx, ctypes.c_void_p(stream_handle)))

    def bem_setup(self, p: int, leaf_size: int, near_radius: float):
        self._check(self._lib.bem_setup(self._ctx, int(p), int(leaf_size), float(near_radius)))

    def bem_apply(self, q, phi, y):
        """y = S q - D phi.  q, phi: arrays/tensors of n_vertices float64 or None; y: output (same kinds)."""
        self._check(self._lib.bem_apply(self._ctx, _ptr(q), _ptr(phi), _ptr(y)))
        return y

    def bem_solve(self, phi, q, use_q_as_x0=False, tol=1e-6, max_iter=100):
        """Solve S q = -c phi + D phi.  Returns (status, iterations, relative residual); q is filled."""
        it = ctypes.c_int(0)
        rr = ctypes.c_double(0.0)
        st = self._lib.bem_solve(self._ctx, _ptr(phi), _ptr(q), int(bool(use_q_as_x0)), float(tol), int(max_iter),
                                 ctypes.byref(it), ctypes.byref(rr))
        self._check(st, allow=(BEM_ERR_NOT_CONVERGED,))
        return st, it.value, rr.value

    def bem_get_timings(self):
        t = np.zeros(len(TIMING_NAMES))
        self._check(self._lib.bem_get_timings(self._ctx, t.ctypes.data, t.size))
        return dict(zip(TIMING_NAMES, t.tolist()))

    def bem_get_stats(self):
        s = np.zeros(len(STAT_NAMES))
        self._check(self._lib.bem_get_stats(self._ctx, s.ctypes.data, s.size))
        return dict(zip(STAT_NAMES, s.tolist()))

    def bem_get_free_term(self):
        c = np.zeros(self.n_vertices)
        self._check(self._lib.bem_get_free_term(self._ctx, c.ctypes.data))
        return c

    def bem_fp64_peak(self) -> float:
        g = ctypes.c_double(0.0)
        self._check(self._lib.bem_fp64_peak(self._ctx, ctypes.byref(g)))
        return g.value

    def bem_fp64_tensor_peak(self) -> float:
        g = ctypes.c_double(0.0)
        self._check(self._lib.bem_fp64_tensor_peak(self._ctx, ctypes.byref(g)))
        return g.value

    def bem_surface_velocity(self, phi, q, v=None, normals_out=None, areas_out=None):
        """v = n q + v_t (Eqs. 22-27), vertex normals and areas (Eq. 17); outputs may be None (at least one given)."""
        self._check(self._lib.bem_surface_velocity(self._ctx, _ptr(phi), _ptr(q), _ptr(v), _ptr(normals_out), _ptr(areas_out)))
        return v

    def bem_surface_curvature(self, H):
        """Mean curvature by the fitted paraboloid (Eqs. 28-29); H: [n_vertices] output."""
        self._check(self._lib.bem_surface_curvature(self._ctx, _ptr(H)))
        return H

    def bem_bubble_volume(self, vol_out):
        """vol_out [n_bubbles] <- V_m of every bubble; host or device float64."""
        n = vol_out.numel() if hasattr(vol_out, "numel") else vol_out.size
        self._check(self._lib.bem_bubble_volume(self._ctx, _ptr(vol_out), int(n)))
        return vol_out

    def bem_destroy(self):
        if self._ctx:
            self._lib.bem_destroy(self._ctx)
            self._ctx = ctypes.c_void_p(0)

    def __del__(self):
        try:
            self.bem_destroy()
        except Exception:
            pass


def bem_create(vertices, triangles, bubble_id=None) -> Bem:
    return Bem(vertices, triangles, bubble_id)


def bem_create_points(sources, targets) -> Bem:
    """Point-cloud mode (include/bem.h): bem_apply(q[n_sources], d[n_sources, 3] or None, y[n_targets])."""
    return Bem(None, None, None, _points=(sources, targets))


def bem_create_evaluator(mesh_ctx: Bem, targets) -> Bem:
    """Off-surface evaluation of S[q] - D[phi] of a mesh context (include/bem.h): after bem_setup,
    bem_apply(q[n_vertices of the mesh], phi[...], u[n_targets])."""
    return Bem(None, None, None, _evaluator=(mesh_ctx, targets))


class BemFilter:
    """Shape filter of bandwidth p_f (an owned `bem_filter *`): bem_filter_create / bem_filter_apply / bem_filter_destroy."""

    def __init__(self, theta, phi, p_f: int):
        self._lib = load_library()
        self._f = ctypes.c_void_p(0)
        th = np.ascontiguousarray(theta, dtype=np.float64)
        ph = np.ascontiguousarray(phi, dtype=np.float64)
        if th.ndim != 1 or th.shape != ph.shape:
            raise ValueError("theta and phi must be [n_d]")
        self.n_d, self.p_f = th.shape[0], int(p_f)
        st = self._lib.bem_filter_create(th.ctypes.data, ph.ctypes.data, th.shape[0], int(p_f), ctypes.byref(self._f))
        if st != BEM_OK:
            self._f = ctypes.c_void_p(0)
            raise BemError(st, "bem_filter_create failed (need 1 <= p_f <= 16, p_f^2 < n_d, angles that resolve the band, a CUDA device)")

    def bem_filter_apply(self, x, n_cols: int, xhat, stream_handle: int = 0):
        st = self._lib.bem_filter_apply(self._f, _ptr(x), int(n_cols), _ptr(xhat), ctypes.c_void_p(stream_handle))
        if st != BEM_OK:
            raise BemError(st, self._lib.bem_filter_last_error(self._f).decode())
        return xhat

    def bem_filter_destroy(self):
        if self._f:
            self._lib.bem_filter_destroy(self._f)
            self._f = ctypes.c_void_p(0)

    def __del__(self):
        try:
            self.bem_filter_destroy()
        except Exception:
            pass


def bem_filter_create(theta, phi, p_f: int) -> BemFilter:
    return BemFilter(theta, phi, p_f)


def bem_direct_sum_static(sources, q, d, targets, y, stream_handle: int = 0):
    """y_i = sum_j [ q_j / (4 pi r) - d_j . (x_i - y_j) / (4 pi r^3) ] over a point cloud (Eq. 13) through
    the one entry of the library that allocates no device memory -- for a caller whose GPU is already full of its own
    arenas, who runs under a fixed memory budget, or who cannot take the device-wide stall of a cudaMalloc in its loop.
    Its scratch is an 8 MiB array compiled into the library, shared by every call on a device: at most
    DIRECT_STATIC_MAX_TARGETS targets per call, and calls that overlap on the GPU race (one stream, or events).

    sources [ns x 3], q [ns] or None, d [ns x 3] or None, targets [nt x 3], y [nt]: contiguous float64 CUDA tensors of
    the current device (host arrays are refused by the library: copying them would need a buffer).  Enqueued on
    `stream_handle` (0 = default stream), never synchronised.  The first call on a device looks up the scratch
    address; make it at start-up, outside any stream capture."""
    lib = load_library()
    for name, a in (("sources", sources), ("targets", targets)):
        if a.dim() != 2 or a.shape[1] != 3:
            raise ValueError(f"{name} must be [n, 3]")
    ns, nt = sources.shape[0], targets.shape[0]
    if q is not None and q.numel() != ns:
        raise ValueError("q must be [n_sources]")
    if d is not None and tuple(d.shape) != (ns, 3):
        raise ValueError("d must be [n_sources, 3]")
    if y.numel() != nt:
        raise ValueError("y must be [n_targets]")
    st = lib.bem_direct_sum_static(_ptr(sources), ns, _ptr(q), _ptr(d), _ptr(targets), nt, _ptr(y), ctypes.c_void_p(stream_handle))
    if st != BEM_OK:
        raise BemError(st, lib.bem_direct_sum_static_last_error().decode())
    return y
