"""Thin Python binding of the C ABI in include/celes.h: argument marshalling only.

Every step of the hot path runs in the CUDA kernels of libceles.so; PyTorch is used for device memory and
streams.  There is no CPU fallback: a missing library raises ImportError-like RuntimeError at first use, and
a missing GPU makes celes_setup raise CelesError(CELES_ECUDA).

Function names and semantics are those of include/celes.h (which cites the paper passage for each).
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libceles.so")

CELES_OK, CELES_EINVAL, CELES_ENOMEM, CELES_ECUDA, CELES_ENOCONV, CELES_ELIMIT = 0, -1, -2, -3, -4, -5
CELES_FAR_FIELD_NOALLOC_MAX_DIR = 2048
CELES_GMRES, CELES_BICGSTAB = 0, 1
CELES_PRECOND_NONE, CELES_PRECOND_BLOCKDIAG = 0, 1
CELES_TRANSLATION_ROTATED, CELES_TRANSLATION_DIRECT = 0, 1
TRANSLATIONS = {"rotated": CELES_TRANSLATION_ROTATED, "direct": CELES_TRANSLATION_DIRECT}
CELES_MAX_HISTORY = 4096
EXPORTS = ["celes_setup", "celes_coupling_matvec", "celes_system_matvec", "celes_coupling_matvec_host",
           "celes_system_matvec_host", "celes_solve", "celes_destroy", "celes_strerror", "celes_nmax",
           "celes_launch_config", "celes_translation_table", "celes_fp32_peak_probe", "celes_precond_setup",
           "celes_precond_apply", "celes_partition", "celes_far_field", "celes_gaussian_beam", "celes_plane_wave",
           "celes_scattered_field", "celes_coupling_matvec_rows", "celes_system_matvec_rows", "celes_work_partition",
           "celes_plan_work", "celes_range_info", "celes_far_field_noalloc"]


class CelesError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        super().__init__(f"{where}: {strerror(code)} ({code})")


class celes_options(ctypes.Structure):
    _fields_ = [("emitter_tile", ctypes.c_int), ("emitter_splits", ctypes.c_int), ("skip_overlap_check", ctypes.c_int),
                ("translation", ctypes.c_int), ("hankel", ctypes.c_int), ("hankel_dr", ctypes.c_double),
                ("range", ctypes.c_int), ("levels", ctypes.c_int)]


class celes_solve_opts(ctypes.Structure):
    _fields_ = [("method", ctypes.c_int), ("restart", ctypes.c_int), ("rtol", ctypes.c_double),
                ("max_iters", ctypes.c_int), ("precond", ctypes.c_int)]


class celes_beam(ctypes.Structure):
    _fields_ = [("waist", ctypes.c_double), ("center", ctypes.c_double * 3), ("alpha_G", ctypes.c_double),
                ("E0_re", ctypes.c_double), ("E0_im", ctypes.c_double), ("n_beta", ctypes.c_int)]


class celes_precond_info(ctypes.Structure):
    _fields_ = [("n_groups", ctypes.c_int), ("max_group_spheres", ctypes.c_int), ("block_bytes", ctypes.c_longlong),
                ("seconds", ctypes.c_double)]


class celes_solve_info(ctypes.Structure):
    _fields_ = [("iterations", ctypes.c_int), ("matvecs", ctypes.c_int), ("converged", ctypes.c_int),
                ("rel_residual", ctypes.c_double), ("seconds", ctypes.c_double), ("n_history", ctypes.c_int),
                ("history", ctypes.c_double * CELES_MAX_HISTORY)]


_LIB = None


def lib() -> ctypes.CDLL:
    """The loaded libceles.so (fails loudly if it has not been built: run `python -m paper_1706_02145_b200.build`)."""
    global _LIB
    if _LIB is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_1706_02145_b200.build` "
                               "(there is no CPU fallback)")
        L = ctypes.CDLL(LIB_PATH)
        i, d, p = ctypes.c_int, ctypes.c_double, ctypes.c_void_p
        L.celes_setup.restype = i
        L.celes_setup.argtypes = [ctypes.POINTER(p), i, i, p, p, p, d, ctypes.POINTER(celes_options), p]
        for name in ("celes_coupling_matvec", "celes_system_matvec", "celes_coupling_matvec_host",
                     "celes_system_matvec_host"):
            getattr(L, name).restype = i
            getattr(L, name).argtypes = [p, p, p, p]
        L.celes_solve.restype = i
        L.celes_solve.argtypes = [p, p, p, ctypes.POINTER(celes_solve_opts), ctypes.POINTER(celes_solve_info), p]
        L.celes_destroy.restype = None
        L.celes_destroy.argtypes = [p]
        L.celes_strerror.restype = ctypes.c_char_p
        L.celes_strerror.argtypes = [i]
        L.celes_nmax.restype = i
        L.celes_nmax.argtypes = [i]
        L.celes_launch_config.restype = i
        L.celes_launch_config.argtypes = [p] + [ctypes.POINTER(i)] * 4
        L.celes_plan_work.restype = i
        L.celes_plan_work.argtypes = [i, i, i, i, i, ctypes.POINTER(i), ctypes.POINTER(i), ctypes.POINTER(i), p, i]
        L.celes_range_info.restype = i
        L.celes_range_info.argtypes = [p, ctypes.POINTER(d), ctypes.POINTER(i)]
        L.celes_work_partition.restype = i
        L.celes_work_partition.argtypes = [p] + [ctypes.POINTER(i)] * 3
        for f in (L.celes_coupling_matvec_rows, L.celes_system_matvec_rows):
            f.restype = i
            f.argtypes = [p, i, i, p, p, p]
        L.celes_translation_table.restype = i
        L.celes_translation_table.argtypes = [i, p, p]
        L.celes_precond_setup.restype = i
        L.celes_precond_setup.argtypes = [p, p, ctypes.POINTER(celes_precond_info), p]
        L.celes_precond_apply.restype = i
        L.celes_precond_apply.argtypes = [p, p, p, p]
        L.celes_partition.restype = i
        L.celes_partition.argtypes = [i, p, p, p, ctypes.POINTER(i)]
        L.celes_scattered_field.restype = i
        L.celes_scattered_field.argtypes = [p, p, i, p, p, p]
        L.celes_plane_wave.restype = i
        L.celes_plane_wave.argtypes = [p, d, d, i, d, d, p, p]
        L.celes_gaussian_beam.restype = i
        L.celes_gaussian_beam.argtypes = [p, ctypes.POINTER(celes_beam), p, p]
        L.celes_far_field.restype = i
        L.celes_far_field.argtypes = [p, p, i, p, p, p, p]
        L.celes_far_field_noalloc.restype = i
        L.celes_far_field_noalloc.argtypes = [p, p, i, p, p, p, p]
        L.celes_fp32_peak_probe.restype = i
        L.celes_fp32_peak_probe.argtypes = [i, i, ctypes.POINTER(d), ctypes.POINTER(d), p]
        _LIB = L
    return _LIB


def strerror(code: int) -> str:
    return lib().celes_strerror(code).decode()


def celes_nmax(lmax: int) -> int:
    n = lib().celes_nmax(lmax)
    if n < 0:
        raise CelesError(n, "celes_nmax")
    return n


def _stream(stream) -> int:
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    return int(getattr(stream, "cuda_stream", stream))


def _check_vec(t, ctx, name):
    import torch
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.complex64 and t.is_contiguous()
            and t.numel() == ctx.N * ctx.nmax):
        raise ValueError(f"{name}: need a contiguous CUDA complex64 tensor with {ctx.N * ctx.nmax} elements")


class Context:
    """Owner of a celes_ctx*; destroyed with the object (or explicitly with celes_destroy)."""

    def __init__(self, handle: int, N: int, lmax: int):
        self.handle, self.N, self.lmax, self.nmax = handle, N, lmax, celes_nmax(lmax)

    def __del__(self):
        celes_destroy(self)


def celes_setup(pos_xyz, radii, mie_q, k: float, lmax: int, *, emitter_tile: int = 0, emitter_splits: int = 0,
                skip_overlap_check: bool = False, translation: str = "rotated", hankel: str = "registers",
                hankel_dr: float = 0.0, range: str = "auto", levels: int = 0, stream=None) -> Context:
    """celes_setup of include/celes.h.  pos_xyz [N,3] float64, radii [N] float64, mie_q [N,2,lmax] complex128 (host)."""
    pos = np.ascontiguousarray(pos_xyz, dtype=np.float64)
    rad = np.ascontiguousarray(radii, dtype=np.float64)
    q = np.ascontiguousarray(mie_q, dtype=np.complex128)
    N = pos.shape[0] if pos.ndim == 2 else 0
    if pos.ndim != 2 or pos.shape[1] != 3 or rad.shape != (N,) or q.shape != (N, 2, lmax):
        raise ValueError("celes_setup: pos_xyz [N,3], radii [N], mie_q [N,2,lmax] expected")
    if translation not in TRANSLATIONS:
        raise ValueError("translation: one of " + ", ".join(TRANSLATIONS))
    opt = celes_options(int(emitter_tile), int(emitter_splits), int(bool(skip_overlap_check)),
                        TRANSLATIONS[translation], {"registers": 0, "table": 1}[hankel], float(hankel_dr),
                        {"auto": 0, "standard": 1, "extended": 2}[range], int(levels))
    h = ctypes.c_void_p()
    import torch
    s = _stream(stream) if torch.cuda.is_available() else 0
    rc = lib().celes_setup(ctypes.byref(h), N, int(lmax), pos.ctypes.data, rad.ctypes.data, q.ctypes.data,
                           float(k), ctypes.byref(opt), s)
    if rc != CELES_OK:
        raise CelesError(rc, "celes_setup")
    return Context(h.value, N, int(lmax))


def celes_destroy(ctx: Context) -> None:
    if getattr(ctx, "handle", None):
        lib().celes_destroy(ctx.handle)
        ctx.handle = None


def celes_coupling_matvec(ctx: Context, b, y=None, stream=None):
    """y = W b (device tensors, complex64 [N,nmax]); asynchronous on the stream."""
    import torch
    _check_vec(b, ctx, "b")
    if y is None:
        y = torch.empty_like(b)
    _check_vec(y, ctx, "y")
    rc = lib().celes_coupling_matvec(ctx.handle, b.data_ptr(), y.data_ptr(), _stream(stream))
    if rc != CELES_OK:
        raise CelesError(rc, "celes_coupling_matvec")
    return y


def celes_system_matvec(ctx: Context, b, out=None, stream=None):
    """out = b - T (W b) (device tensors); asynchronous on the stream."""
    import torch
    _check_vec(b, ctx, "b")
    if out is None:
        out = torch.empty_like(b)
    _check_vec(out, ctx, "out")
    rc = lib().celes_system_matvec(ctx.handle, b.data_ptr(), out.data_ptr(), _stream(stream))
    if rc != CELES_OK:
        raise CelesError(rc, "celes_system_matvec")
    return out


def _matvec_rows(fn, name, ctx, row_begin, row_end, b, out, stream):
    import torch
    _check_vec(b, ctx, "b")
    rows = int(row_end) - int(row_begin)
    if out is None:
        out = torch.empty(max(rows, 0), ctx.nmax, dtype=torch.complex64, device=b.device)
    if not (out.is_cuda and out.dtype == torch.complex64 and out.is_contiguous() and out.numel() == max(rows, 0) * ctx.nmax):
        raise ValueError(f"{name}: out must be a contiguous CUDA complex64 tensor with (row_end - row_begin) * nmax elements")
    rc = fn(ctx.handle, int(row_begin), int(row_end), b.data_ptr(), out.data_ptr(), _stream(stream))
    if rc != CELES_OK:
        raise CelesError(rc, name)
    return out


def celes_coupling_matvec_rows(ctx: Context, row_begin: int, row_end: int, b, y_rows=None, stream=None):
    """rows [row_begin, row_end) of y = W b from the full device vector b; asynchronous on the stream."""
    return _matvec_rows(lib().celes_coupling_matvec_rows, "celes_coupling_matvec_rows", ctx, row_begin, row_end, b, y_rows, stream)


def celes_system_matvec_rows(ctx: Context, row_begin: int, row_end: int, b, out_rows=None, stream=None):
    """rows [row_begin, row_end) of b - T (W b) from the full device vector b; asynchronous on the stream."""
    return _matvec_rows(lib().celes_system_matvec_rows, "celes_system_matvec_rows", ctx, row_begin, row_end, b, out_rows, stream)


def _host_vec(a, ctx, name):
    if not (isinstance(a, np.ndarray) and a.dtype == np.complex64 and a.flags.c_contiguous and a.size == ctx.N * ctx.nmax):
        raise ValueError(f"{name}: need a C-contiguous complex64 ndarray with {ctx.N * ctx.nmax} elements")


def celes_coupling_matvec_host(ctx: Context, b_host: np.ndarray, y_host: np.ndarray | None = None, stream=None):
    """y = W b with HOST buffers (numpy complex64, ideally backed by pinned memory); synchronous."""
    _host_vec(b_host, ctx, "b_host")
    if y_host is None:
        y_host = np.empty_like(b_host)
    _host_vec(y_host, ctx, "y_host")
    rc = lib().celes_coupling_matvec_host(ctx.handle, b_host.ctypes.data, y_host.ctypes.data, _stream(stream))
    if rc != CELES_OK:
        raise CelesError(rc, "celes_coupling_matvec_host")
    return y_host


def celes_system_matvec_host(ctx: Context, b_host: np.ndarray, out_host: np.ndarray | None = None, stream=None):
    _host_vec(b_host, ctx, "b_host")
    if out_host is None:
        out_host = np.empty_like(b_host)
    _host_vec(out_host, ctx, "out_host")
    rc = lib().celes_system_matvec_host(ctx.handle, b_host.ctypes.data, out_host.ctypes.data, _stream(stream))
    if rc != CELES_OK:
        raise CelesError(rc, "celes_system_matvec_host")
    return out_host


def celes_precond_setup(ctx: Context, edge_xyz, stream=None) -> dict:
    """celes_precond_setup of include/celes.h: block-diagonal preconditioner on cuboids of edge lengths edge_xyz
    (a scalar means a cube).  Returns the celes_precond_info fields."""
    e = np.ascontiguousarray(np.broadcast_to(np.asarray(edge_xyz, dtype=np.float64), (3,)))
    info = celes_precond_info()
    rc = lib().celes_precond_setup(ctx.handle, e.ctypes.data, ctypes.byref(info), _stream(stream))
    if rc != CELES_OK:
        raise CelesError(rc, "celes_precond_setup")
    return {"n_groups": info.n_groups, "max_group_spheres": info.max_group_spheres, "block_bytes": info.block_bytes,
            "seconds": info.seconds}


def celes_precond_apply(ctx: Context, v, z=None, stream=None):
    """z = blockdiag(M_j^{-1}) v on device tensors."""
    import torch
    _check_vec(v, ctx, "v")
    if z is None:
        z = torch.empty_like(v)
    _check_vec(z, ctx, "z")
    rc = lib().celes_precond_apply(ctx.handle, v.data_ptr(), z.data_ptr(), _stream(stream))
    if rc != CELES_OK:
        raise CelesError(rc, "celes_precond_apply")
    return z


def celes_plane_wave(ctx: Context, alpha: float = 0.0, beta: float = 0.0, polarisation: int = 2, E0: complex = 1.0,
                     a_in=None, stream=None):
    """a_in [N, nmax] complex64 (device) of the plane wave E0 Phi_j(alpha, beta); celes_plane_wave of include/celes.h."""
    import torch
    if a_in is None:
        a_in = torch.empty(ctx.N, ctx.nmax, dtype=torch.complex64, device="cuda")
    _check_vec(a_in, ctx, "a_in")
    rc = lib().celes_plane_wave(ctx.handle, float(alpha), float(beta), int(polarisation), float(complex(E0).real),
                                float(complex(E0).imag), a_in.data_ptr(), _stream(stream))
    if rc != CELES_OK:
        raise CelesError(rc, "celes_plane_wave")
    return a_in


def celes_gaussian_beam(ctx: Context, waist: float, center, alpha_G: float = 0.0, E0: complex = 1.0, n_beta: int = 0,
                        a_in=None, stream=None):
    """a_in [N, nmax] complex64 (device) of the Gaussian beam of Appendix C; celes_gaussian_beam of include/celes.h."""
    import torch
    if a_in is None:
        a_in = torch.empty(ctx.N, ctx.nmax, dtype=torch.complex64, device="cuda")
    _check_vec(a_in, ctx, "a_in")
    c = np.asarray(center, dtype=np.float64).reshape(3)
    beam = celes_beam(float(waist), (ctypes.c_double * 3)(*c), float(alpha_G), float(complex(E0).real),
                      float(complex(E0).imag), int(n_beta))
    rc = lib().celes_gaussian_beam(ctx.handle, ctypes.byref(beam), a_in.data_ptr(), _stream(stream))
    if rc != CELES_OK:
        raise CelesError(rc, "celes_gaussian_beam")
    return a_in


def celes_scattered_field(ctx: Context, b, points, stream=None):
    """E_scat [n_pts, 3] complex64 (device) at the host points [n_pts, 3]; celes_scattered_field of include/celes.h."""
    import torch
    _check_vec(b, ctx, "b")
    pts = np.ascontiguousarray(points, dtype=np.float64)
    if pts.ndim != 2 or pts.shape[1] != 3 or pts.shape[0] < 1:
        raise ValueError("points: [n_pts, 3]")
    E = torch.empty(pts.shape[0], 3, dtype=torch.complex64, device=b.device)
    rc = lib().celes_scattered_field(ctx.handle, b.data_ptr(), int(pts.shape[0]), pts.ctypes.data, E.data_ptr(),
                                     _stream(stream))
    if rc != CELES_OK:
        raise CelesError(rc, "celes_scattered_field")
    return E


def celes_far_field(ctx: Context, b, alpha, beta, g=None, stream=None):
    """g [n_dir, 2] complex64 (device): far-field amplitudes g_1, g_2 of the scattered field with coefficients b in the
    directions (alpha, beta) (host arrays, radians); celes_far_field of include/celes.h."""
    import torch
    _check_vec(b, ctx, "b")
    al = np.ascontiguousarray(alpha, dtype=np.float64).reshape(-1)
    be = np.ascontiguousarray(beta, dtype=np.float64).reshape(-1)
    if al.shape != be.shape or al.size < 1:
        raise ValueError("alpha and beta: same non-zero length")
    if g is None:
        g = torch.empty(al.size, 2, dtype=torch.complex64, device=b.device)
    if not (g.is_cuda and g.dtype == torch.complex64 and g.is_contiguous() and g.numel() == 2 * al.size):
        raise ValueError("g: contiguous CUDA complex64 tensor with 2 * n_dir elements")
    rc = lib().celes_far_field(ctx.handle, b.data_ptr(), int(al.size), al.ctypes.data, be.ctypes.data, g.data_ptr(),
                               _stream(stream))
    if rc != CELES_OK:
        raise CelesError(rc, "celes_far_field")
    return g


def celes_far_field_noalloc(ctx: Context, b, alpha, beta, g, stream=None):
    """celes_far_field_noalloc of include/celes.h: the far field from the library's static scratch array, no allocation in
    the call (at most CELES_FAR_FIELD_NOALLOC_MAX_DIR directions; g [n_dir, 2] complex64 is the CALLER's tensor).
    alpha, beta: contiguous float64 host arrays of equal length (no conversion or copy is made here)."""
    _check_vec(b, ctx, "b")
    for a in (alpha, beta):
        if not (isinstance(a, np.ndarray) and a.dtype == np.float64 and a.flags.c_contiguous and a.ndim == 1):
            raise ValueError("alpha and beta: contiguous 1-d float64 ndarrays")
    if alpha.shape != beta.shape or alpha.size < 1:
        raise ValueError("alpha and beta: same non-zero length")
    if not (g.is_cuda and g.is_contiguous() and g.numel() == 2 * alpha.size and g.element_size() == 8):
        raise ValueError("g: contiguous CUDA complex64 tensor with 2 * n_dir elements")
    rc = lib().celes_far_field_noalloc(ctx.handle, b.data_ptr(), int(alpha.size), alpha.ctypes.data, beta.ctypes.data,
                                       g.data_ptr(), _stream(stream))
    if rc != CELES_OK:
        raise CelesError(rc, "celes_far_field_noalloc")
    return g


def celes_partition(pos_xyz, edge_xyz):
    """(group_of [N] int32, n_groups): the cuboid partition of celes_precond_setup (host only, needs no GPU)."""
    pos = np.ascontiguousarray(pos_xyz, dtype=np.float64)
    e = np.ascontiguousarray(np.broadcast_to(np.asarray(edge_xyz, dtype=np.float64), (3,)))
    g = np.empty(pos.shape[0], dtype=np.int32)
    n = ctypes.c_int()
    rc = lib().celes_partition(pos.shape[0], pos.ctypes.data, e.ctypes.data, g.ctypes.data, ctypes.byref(n))
    if rc != CELES_OK:
        raise CelesError(rc, "celes_partition")
    return g, n.value


def celes_solve(ctx: Context, a_in, x, *, restart: int = 30, rtol: float = 1e-4, max_iters: int = 1000,
                precond: bool = False, method: str = "gmres", stream=None):
    """Solve eq. (8) in place in x (in: x0, out: b).  precond=True uses the block-diagonal preconditioner built by
    celes_precond_setup.  Returns a dict with the celes_solve_info fields; raises CelesError on failure other than
    CELES_ENOCONV (reported as converged = 0)."""
    _check_vec(a_in, ctx, "a_in")
    _check_vec(x, ctx, "x")
    if method not in ("gmres", "bicgstab"):
        raise ValueError("method: 'gmres' or 'bicgstab'")
    o = celes_solve_opts(CELES_BICGSTAB if method == "bicgstab" else CELES_GMRES, int(restart), float(rtol), int(max_iters),
                         CELES_PRECOND_BLOCKDIAG if precond else CELES_PRECOND_NONE)
    info = celes_solve_info()
    rc = lib().celes_solve(ctx.handle, a_in.data_ptr(), x.data_ptr(), ctypes.byref(o), ctypes.byref(info), _stream(stream))
    if rc not in (CELES_OK, CELES_ENOCONV):
        raise CelesError(rc, "celes_solve")
    return {"iterations": info.iterations, "matvecs": info.matvecs, "converged": bool(info.converged),
            "rel_residual": info.rel_residual, "seconds": info.seconds,
            "history": [info.history[i] for i in range(info.n_history)], "code": rc}


def celes_launch_config(ctx: Context) -> dict:
    v = [ctypes.c_int() for _ in range(4)]
    rc = lib().celes_launch_config(ctx.handle, *[ctypes.byref(x) for x in v])
    if rc != CELES_OK:
        raise CelesError(rc, "celes_launch_config")
    return dict(zip(("receiver_blocks", "emitter_splits", "block_threads", "emitter_tile"), (x.value for x in v)))


def celes_range_info(ctx: Context) -> dict:
    kd, ext = ctypes.c_double(), ctypes.c_int()
    rc = lib().celes_range_info(ctx.handle, ctypes.byref(kd), ctypes.byref(ext))
    if rc != CELES_OK:
        raise CelesError(rc, "celes_range_info")
    return {"kd_max": kd.value, "extended": bool(ext.value)}


def celes_work_partition(ctx: Context) -> dict:
    v = [ctypes.c_int() for _ in range(3)]
    rc = lib().celes_work_partition(ctx.handle, *[ctypes.byref(x) for x in v])
    if rc != CELES_OK:
        raise CelesError(rc, "celes_work_partition")
    return dict(zip(("ctas", "segments", "receivers_per_block"), (x.value for x in v)))


def celes_plan_work(N: int, emitter_tile: int = 32, resident_ctas: int = 296, levels: int = 0, emitter_splits: int = 0) -> dict:
    """Host-only: the work partition celes_setup would build; 'segments' is an int array [n][5] of
    (cta, receiver block, e_begin, e_end, slot)."""
    v = [ctypes.c_int() for _ in range(3)]
    rc = lib().celes_plan_work(int(N), int(emitter_tile), int(resident_ctas), int(levels), int(emitter_splits),
                               *[ctypes.byref(x) for x in v], None, 0)
    if rc != CELES_OK:
        raise CelesError(rc, "celes_plan_work")
    seg = np.zeros((v[1].value, 5), dtype=np.int32)
    rc = lib().celes_plan_work(int(N), int(emitter_tile), int(resident_ctas), int(levels), int(emitter_splits), None, None, None,
                               seg.ctypes.data, seg.shape[0])
    if rc != CELES_OK:
        raise CelesError(rc, "celes_plan_work")
    return {"ctas": v[0].value, "receivers_per_block": v[2].value, "segments": seg}


def celes_translation_table(lmax: int):
    """(a5_re, b5_im) [H,H,P] float64 as the library evaluates them on the host (needs no GPU)."""
    H, P = lmax * (lmax + 2), 2 * lmax + 1
    a = np.zeros((H, H, P)); b = np.zeros((H, H, P))
    rc = lib().celes_translation_table(int(lmax), a.ctypes.data, b.ctypes.data)
    if rc != CELES_OK:
        raise CelesError(rc, "celes_translation_table")
    return a, b


def celes_fp32_peak_probe(variant: int = 0, iters: int = 4096, stream=None) -> dict:
    f, ms = ctypes.c_double(), ctypes.c_double()
    rc = lib().celes_fp32_peak_probe(int(variant), int(iters), ctypes.byref(f), ctypes.byref(ms), _stream(stream))
    if rc != CELES_OK:
        raise CelesError(rc, "celes_fp32_peak_probe")
    return {"flops_per_s": f.value, "ms": ms.value}
