"""Thin ctypes binding of libchfsi.so (include/chfsi.h).  Argument marshalling only: every step of
the hot path runs in the library's CUDA kernels.  There is no CPU fallback: if the shared library
is missing or fails to load, importing `lib()` raises.

PyTorch appears here only as the owner of device memory and streams (tensors are passed by
`data_ptr()`, the current stream by its `cuda_stream` handle).
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libchfsi.so")

OK, EINVAL, ENOMEM, ECUDA, ESTATE, EUNSUPPORTED = range(6)
FP64, FP32, TF32, TF32X3, FP32_STORED = range(5)
RECUR_STANDARD, RECUR_RESIDUAL = 0, 1
PREC = {"fp64": FP64, "fp32": FP32, "tf32": TF32, "tf32x3": TF32X3, "fp32s": FP32_STORED}

EXPORTS = [
    "chfsi_mesh_create", "chfsi_mesh_destroy", "chfsi_mesh_set_cell_kernel", "chfsi_mesh_num_nodes", "chfsi_mesh_node_coords",
    "chfsi_mesh_mass", "chfsi_ham_set", "chfsi_workspace_bytes", "chfsi_apply_H", "chfsi_cheb_filter",
    "chfsi_profile_enable", "chfsi_profile_read",
    "chfsi_bfp_stream_bytes", "chfsi_bfp_encode", "chfsi_bfp_decode", "chfsi_bfp_gather_encode",
    "chfsi_bfp_decode_scatter_add",
    "chfsi_rr_project", "chfsi_rr_rotate_workspace_bytes", "chfsi_rr_rotate", "chfsi_rr_rotate_static", "chfsi_measure_pipe_peaks",
    "chfsi_poisson_set_quadrature", "chfsi_poisson_kdiag", "chfsi_poisson_apply_K", "chfsi_poisson_workspace_bytes", "chfsi_poisson_pcg",
    "chfsi_last_launch_count", "chfsi_last_error", "chfsi_version",
]

_lib = None


class ChfsiError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"chfsi status {status}: {msg}")
        self.status = status


def lib() -> C.CDLL:
    """Load libchfsi.so (fails loudly if it has not been built: run `python -m paper_2605_30128_b200.build`)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} not found: build it with `python -m paper_2605_30128_b200.build` "
                          "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    dp, ip, llp, vp = C.POINTER(C.c_double), C.POINTER(C.c_int), C.POINTER(C.c_longlong), C.c_void_p
    L.chfsi_mesh_create.argtypes = [C.c_int] * 3 + [C.c_double] * 3 + [C.c_int, dp, C.c_int, C.POINTER(vp)]
    L.chfsi_mesh_destroy.argtypes = [vp]
    L.chfsi_mesh_set_cell_kernel.argtypes = [vp, C.c_int, C.c_int]
    L.chfsi_mesh_num_nodes.argtypes = [vp, llp]
    L.chfsi_mesh_node_coords.argtypes = [vp, dp]
    L.chfsi_mesh_mass.argtypes = [vp, dp]
    L.chfsi_ham_set.argtypes = [vp, dp, dp, dp, dp, C.c_int, llp, llp, ip, dp, dp, dp]
    L.chfsi_workspace_bytes.argtypes = [vp, C.c_int, C.c_int, C.c_int, C.POINTER(C.c_size_t)]
    L.chfsi_apply_H.argtypes = [vp, C.c_int, C.c_int, vp, C.c_longlong, vp, C.c_longlong, vp, C.c_size_t, vp]
    L.chfsi_cheb_filter.argtypes = [vp, C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double,
                                    C.c_int, C.c_int, vp, C.c_longlong, dp, vp, C.c_longlong, vp,
                                    C.c_size_t, vp]
    L.chfsi_profile_enable.argtypes = [vp, C.c_int]
    L.chfsi_profile_read.argtypes = [vp, dp, llp, dp]
    L.chfsi_bfp_stream_bytes.argtypes = [C.c_int, C.c_longlong, C.POINTER(C.c_size_t)]
    L.chfsi_bfp_encode.argtypes = [C.c_int, vp, C.c_longlong, vp, vp]
    L.chfsi_bfp_decode.argtypes = [C.c_int, vp, C.c_longlong, vp, vp]
    L.chfsi_bfp_gather_encode.argtypes = [C.c_int, vp, C.c_int, C.c_longlong, C.c_int, vp, C.c_longlong, vp, vp]
    L.chfsi_bfp_decode_scatter_add.argtypes = [C.c_int, vp, vp, C.c_longlong, C.c_int, vp, C.c_int, C.c_longlong, vp]
    L.chfsi_rr_project.argtypes = [vp, C.c_longlong, C.c_int, vp, C.c_longlong, vp, C.c_longlong, C.c_int, C.c_int, vp, vp]
    L.chfsi_rr_rotate_workspace_bytes.argtypes = [C.c_int, C.POINTER(C.c_size_t)]
    L.chfsi_rr_rotate.argtypes = [C.c_int, C.c_longlong, C.c_int, vp, C.c_longlong, vp, vp, C.c_longlong, vp, C.c_size_t, vp]
    L.chfsi_rr_rotate_static.argtypes = [C.c_int, C.c_longlong, C.c_int, vp, C.c_longlong, vp, vp, C.c_longlong, vp]
    L.chfsi_measure_pipe_peaks.argtypes = [C.c_int, dp]
    L.chfsi_poisson_set_quadrature.argtypes = [vp, C.c_int]
    L.chfsi_poisson_kdiag.argtypes = [vp, dp]
    L.chfsi_poisson_apply_K.argtypes = [vp, C.c_int, vp, C.c_longlong, vp, C.c_longlong, vp]
    L.chfsi_poisson_workspace_bytes.argtypes = [vp, C.c_int, C.POINTER(C.c_size_t)]
    L.chfsi_poisson_pcg.argtypes = [vp, C.c_int, vp, C.c_longlong, vp, C.c_longlong, C.c_int, C.c_double, C.c_double, C.c_double,
                                    C.c_int, C.c_int, vp, C.c_size_t, ip, dp, vp]
    for name in EXPORTS:
        if name not in ("chfsi_last_launch_count", "chfsi_last_error", "chfsi_version"):
            getattr(L, name).restype = C.c_int
    L.chfsi_last_launch_count.restype = C.c_longlong
    L.chfsi_last_error.restype = C.c_char_p
    L.chfsi_version.restype = C.c_char_p
    _lib = L
    return L


def _check(st):
    if st != OK:
        raise ChfsiError(st, lib().chfsi_last_error().decode())


def _dptr(a):
    return None if a is None else a.ctypes.data_as(C.POINTER(C.c_double))


def _f64(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float64)


# ---- the C-ABI calls, same names ---------------------------------------------------------------
def chfsi_mesh_create(ncell, L, p, kfrac=None, device=0):
    nc = (ncell,) * 3 if np.ndim(ncell) == 0 else tuple(ncell)
    Ls = (L,) * 3 if np.ndim(L) == 0 else tuple(L)
    k = None if kfrac is None else _f64(kfrac)
    h = C.c_void_p()
    _check(lib().chfsi_mesh_create(int(nc[0]), int(nc[1]), int(nc[2]), float(Ls[0]), float(Ls[1]), float(Ls[2]),
                                   int(p), _dptr(k), int(device), C.byref(h)))
    return h


def chfsi_mesh_destroy(mesh):
    _check(lib().chfsi_mesh_destroy(mesh))


CELL_DEFAULT, CELL_XYZ, CELL_MARCH, CELL_MMA = range(4)


def chfsi_mesh_set_cell_kernel(mesh, prec, kernel):
    _check(lib().chfsi_mesh_set_cell_kernel(mesh, int(prec), int(kernel)))


def chfsi_mesh_num_nodes(mesh) -> int:
    n = C.c_longlong()
    _check(lib().chfsi_mesh_num_nodes(mesh, C.byref(n)))
    return n.value


def chfsi_mesh_node_coords(mesh) -> np.ndarray:
    xyz = np.empty((chfsi_mesh_num_nodes(mesh), 3), dtype=np.float64)
    _check(lib().chfsi_mesh_node_coords(mesh, _dptr(xyz)))
    return xyz


def chfsi_mesh_mass(mesh) -> np.ndarray:
    m = np.empty(chfsi_mesh_num_nodes(mesh), dtype=np.float64)
    _check(lib().chfsi_mesh_mass(mesh, _dptr(m)))
    return m


def chfsi_ham_set(mesh, V, Bx, By, Bz, supp_off=None, supp_node=None, nproj=None, P=None, D=None):
    """P: complex128 concatenated per-atom [n_supp_a, nproj_a] blocks; D: complex128 per-atom matrices."""
    V, Bx, By, Bz = _f64(V), _f64(Bx), _f64(By), _f64(Bz)
    natoms = 0 if supp_off is None else len(supp_off) - 1
    if natoms > 0:
        so = np.ascontiguousarray(supp_off, dtype=np.int64)
        sn = np.ascontiguousarray(supp_node, dtype=np.int64)
        npj = np.ascontiguousarray(nproj, dtype=np.int32)
        Pc = np.ascontiguousarray(P, dtype=np.complex128).reshape(-1)
        Pre, Pim = np.ascontiguousarray(Pc.real), np.ascontiguousarray(Pc.imag)
        Dc = np.ascontiguousarray(np.concatenate([np.asarray(d, np.complex128).reshape(-1) for d in D]))
        Dv = Dc.view(np.float64)
        llp = C.POINTER(C.c_longlong)
        st = lib().chfsi_ham_set(mesh, _dptr(V), _dptr(Bx), _dptr(By), _dptr(Bz), natoms,
                                 so.ctypes.data_as(llp), sn.ctypes.data_as(llp),
                                 npj.ctypes.data_as(C.POINTER(C.c_int)), _dptr(Pre), _dptr(Pim), _dptr(Dv))
    else:
        st = lib().chfsi_ham_set(mesh, _dptr(V), _dptr(Bx), _dptr(By), _dptr(Bz), 0, None, None, None, None,
                                 None, None)
    _check(st)


def chfsi_workspace_bytes(mesh, prec, recur, chunk) -> int:
    n = C.c_size_t()
    _check(lib().chfsi_workspace_bytes(mesh, int(prec), int(recur), int(chunk), C.byref(n)))
    return n.value


def _ptr(t):
    return C.c_void_p(t.data_ptr())


def _stream(stream):
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


def chfsi_apply_H(mesh, prec, X, Y, work, stream=None, nvec=None, ldx=None, ldy=None):
    """X, Y: torch complex128 CUDA tensors [M, 2, ld]; work: torch uint8 CUDA tensor."""
    nvec = X.shape[-1] if nvec is None else nvec
    ldx = X.stride(-2) if ldx is None else ldx
    ldy = Y.stride(-2) if ldy is None else ldy
    _check(lib().chfsi_apply_H(mesh, int(prec), int(nvec), _ptr(X), int(ldx), _ptr(Y), int(ldy), _ptr(work),
                               work.numel(), _stream(stream)))


def chfsi_cheb_filter(mesh, prec, recur, degree, a, b, a0, X, lam, Y, work, chunk=0, stream=None,
                      nvec=None, ldx=None, ldy=None):
    nvec = X.shape[-1] if nvec is None else nvec
    ldx = X.stride(-2) if ldx is None else ldx
    ldy = Y.stride(-2) if ldy is None else ldy
    lam_h = None if lam is None else np.ascontiguousarray(lam, dtype=np.float64)
    _check(lib().chfsi_cheb_filter(mesh, int(prec), int(recur), int(degree), float(a), float(b), float(a0),
                                   int(nvec), int(chunk), _ptr(X), int(ldx), _dptr(lam_h), _ptr(Y), int(ldy),
                                   _ptr(work), work.numel(), _stream(stream)))


def chfsi_profile_enable(mesh, on: bool):
    _check(lib().chfsi_profile_enable(mesh, int(bool(on))))


def chfsi_profile_read(mesh):
    """(cell-kernel ms summed, launches, algorithmic bytes summed) since the last read; synchronises."""
    ms, n, by = C.c_double(), C.c_longlong(), C.c_double()
    _check(lib().chfsi_profile_read(mesh, C.byref(ms), C.byref(n), C.byref(by)))
    return ms.value, n.value, by.value


def chfsi_last_launch_count() -> int:
    return int(lib().chfsi_last_launch_count())


def chfsi_version() -> str:
    return lib().chfsi_version().decode()


# ---- BFP codec ----------------------------------------------------------------
def chfsi_bfp_stream_bytes(nbits, n) -> int:
    b = C.c_size_t()
    _check(lib().chfsi_bfp_stream_bytes(int(nbits), int(n), C.byref(b)))
    return b.value


def chfsi_bfp_encode(nbits, src, dst, stream=None):
    """src: torch float32 CUDA tensor (numel % 4 == 0); dst: torch uint8 CUDA tensor of chfsi_bfp_stream_bytes."""
    _check(lib().chfsi_bfp_encode(int(nbits), _ptr(src), src.numel(), _ptr(dst), _stream(stream)))


def chfsi_bfp_decode(nbits, src, dst, stream=None):
    _check(lib().chfsi_bfp_decode(int(nbits), _ptr(src), dst.numel(), _ptr(dst), _stream(stream)))


def chfsi_bfp_gather_encode(nbits, X, rows, dst, stream=None):
    """X: torch complex128 / complex64 CUDA tensor [nrows_total, ld]; rows: torch int64 CUDA tensor."""
    _check(lib().chfsi_bfp_gather_encode(int(nbits), _ptr(X), X.element_size(), X.stride(0), X.shape[1], _ptr(rows),
                                         rows.numel(), _ptr(dst), _stream(stream)))


def chfsi_bfp_decode_scatter_add(nbits, src, rows, Y, stream=None):
    _check(lib().chfsi_bfp_decode_scatter_add(int(nbits), _ptr(src), _ptr(rows), rows.numel(), Y.shape[1], _ptr(Y),
                                              Y.element_size(), Y.stride(0), _stream(stream)))


# ---- Rayleigh-Ritz pieces --------------------------------------------------------
def chfsi_rr_project(mesh, A, B, S, use_mass=True, hermitian=True, stream=None):
    """A, B: torch complex128 CUDA tensors [..., ld] viewed as [nrows, ld]; S: torch complex128 [nvec, nvec]."""
    nvec = S.shape[0]
    nrows = A.numel() // A.shape[-1]
    _check(lib().chfsi_rr_project(mesh, nrows, nvec, _ptr(A), A.stride(-2), _ptr(B), B.stride(-2), int(bool(use_mass)),
                                  int(bool(hermitian)), _ptr(S), _stream(stream)))


def chfsi_rr_rotate_workspace_bytes(nvec) -> int:
    b = C.c_size_t()
    _check(lib().chfsi_rr_rotate_workspace_bytes(int(nvec), C.byref(b)))
    return b.value


def chfsi_rr_rotate(prec, Y, Q, Yout, work, stream=None):
    nvec = Q.shape[0]
    nrows = Y.numel() // Y.shape[-1]
    _check(lib().chfsi_rr_rotate(int(prec), nrows, nvec, _ptr(Y), Y.stride(-2), _ptr(Q), _ptr(Yout), Yout.stride(-2), _ptr(work),
                                 work.numel(), _stream(stream)))


RR_STATIC_MAX_NVEC = 512


def chfsi_rr_rotate_static(prec, Y, Q, Yout, stream=None):
    """chfsi_rr_rotate on the library's static device scratch (no workspace, no allocation; nvec <= RR_STATIC_MAX_NVEC)."""
    nvec = Q.shape[0]
    nrows = Y.numel() // Y.shape[-1]
    _check(lib().chfsi_rr_rotate_static(int(prec), nrows, nvec, _ptr(Y), Y.stride(-2), _ptr(Q), _ptr(Yout), Yout.stride(-2),
                                        _stream(stream)))


def chfsi_measure_pipe_peaks(device=0) -> dict:
    """TFLOP/s of the FP64 FMA, FP32 FMA, mma.m8n8k4.f64 and mma.m16n8k8.tf32 pipes, measured now on `device`."""
    out = (C.c_double * 4)()
    _check(lib().chfsi_measure_pipe_peaks(int(device), out))
    return {"fp64_fma": out[0], "fp32_fma": out[1], "fp64_mma": out[2], "tf32_mma": out[3]}


# ---- Poisson solve ----------------------------------------------------------------
def chfsi_poisson_set_quadrature(mesh, rule):
    """rule 0: GLL collocation (default); 1: Gauss-Legendre, the paper's Kx."""
    _check(lib().chfsi_poisson_set_quadrature(mesh, int(rule)))


def chfsi_poisson_kdiag(mesh) -> np.ndarray:
    kd = np.empty(chfsi_mesh_num_nodes(mesh), dtype=np.float64)
    _check(lib().chfsi_poisson_kdiag(mesh, _dptr(kd)))
    return kd


def chfsi_poisson_apply_K(mesh, U, W, stream=None):
    """U, W: torch complex128 CUDA tensors [M, 2, ld] (4 nvec independent real columns)."""
    _check(lib().chfsi_poisson_apply_K(mesh, U.shape[-1], _ptr(U), U.stride(-2), _ptr(W), W.stride(-2), _stream(stream)))


def chfsi_poisson_workspace_bytes(mesh, nvec) -> int:
    b = C.c_size_t()
    _check(lib().chfsi_poisson_workspace_bytes(mesh, int(nvec), C.byref(b)))
    return b.value


def chfsi_poisson_pcg(mesh, F, X, cheb_degree, lmin, lmax, tol, maxit, work, check_every=10, stream=None, want_stats=True):
    """Returns (iterations, residual norms) per real column [2, nvec, 2] = (spin, vector, re/im) when want_stats."""
    nvec = F.shape[-1]
    it = np.zeros(4 * nvec, dtype=np.int32) if want_stats else None
    rn = np.zeros(4 * nvec, dtype=np.float64) if want_stats else None
    _check(lib().chfsi_poisson_pcg(mesh, nvec, _ptr(F), F.stride(-2), _ptr(X), X.stride(-2), int(cheb_degree), float(lmin),
                                   float(lmax), float(tol), int(maxit), int(check_every), _ptr(work), work.numel(),
                                   None if it is None else it.ctypes.data_as(C.POINTER(C.c_int)), _dptr(rn), _stream(stream)))
    if not want_stats:
        return None, None
    return it.reshape(2, nvec, 2), rn.reshape(2, nvec, 2)
