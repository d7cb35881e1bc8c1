"""Thin ctypes binding over libpwham.so (C ABI in include/pwham.h) -- argument marshalling only.

Every step of the path runs in the library's CUDA kernels; PyTorch is used here for device memory and streams
and nothing else.  There is no CPU fallback: importing works without a GPU (so that the symbol table can be
checked), but every compute entry point needs CUDA tensors, and loading fails loudly if the library has not
been built (`python paper_2604_11139_b200/build.py` or `__graft_entry__.build()`).

Array conventions (see synth.py): a block is a complex128 tensor of shape (nband, npw) whose rows are bands, i.e. the
paper's N x M matrix Psi column-major with leading dimension `stride(0)`.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libpwham.so")

EXPORTS = ["pwh_ham_setup", "pwh_ham_destroy", "pwh_workspace_bytes", "pwh_apply_h", "pwh_cheb_filter",
           "pwh_gram_workspace_bytes", "pwh_gram", "pwh_gram_herm", "pwh_ham_kernels", "pwh_apply_h_host", "pwh_cheb_filter_host", "pwh_sweep_host",
           "pwh_launch_count", "pwh_ham_info", "pwh_last_error", "pwh_profile_begin", "pwh_profile_end",
           "pwh_probe_fp64_tensor_peak",
           "pwh_rayleigh_quotients", "pwh_residual_norms", "pwh_rotate", "pwh_dense_workspace_bytes", "pwh_potrf",
           "pwh_heev", "pwh_hegv", "pwh_rr_workspace_bytes", "pwh_chol_ortho", "pwh_rayleigh_ritz",
           "pwh_chebfi_workspace_bytes", "pwh_chebfi_iteration",
           "pwh_ham_set_paw", "pwh_apply_hs", "pwh_apply_sinv", "pwh_cheb_filter_gen",
           "pwh_lobpcg_workspace_bytes", "pwh_lobpcg",
           "pwh_density_workspace_bytes", "pwh_density_accumulate",
           "pwh_chol_ortho_gen", "pwh_lobpcg_gen_workspace_bytes", "pwh_lobpcg_gen", "pwh_gram_static"]

STAGES = ["scatter_zinv", "plane", "zfwd_gather", "zgemm_cn", "splitk_reduce", "zgemm_nn", "colstats", "dense_small",
          "jacobi", "axpy", "reserved10", "reserved11"]

_lib = None


class PwhamError(RuntimeError):
    pass


def load_library() -> ctypes.CDLL:
    """dlopen libpwham.so and declare the prototypes of include/pwham.h.  Raises if the library is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise PwhamError(f"{LIB_PATH} is missing: build the CUDA library first (python paper_2604_11139_b200/build.py "
                         "or __graft_entry__.build()); there is no CPU fallback")
    L = ctypes.CDLL(LIB_PATH)
    vp, i64, i32, dbl, sz = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int, ctypes.c_double, ctypes.c_size_t
    L.pwh_ham_setup.argtypes = [ctypes.POINTER(vp), vp, vp, vp, i64, vp, vp, i64, vp, i64, vp, vp]
    L.pwh_ham_setup.restype = i32
    L.pwh_ham_destroy.argtypes = [vp]
    L.pwh_ham_destroy.restype = i32
    L.pwh_workspace_bytes.argtypes = [vp, i64]
    L.pwh_workspace_bytes.restype = sz
    L.pwh_apply_h.argtypes = [vp, i64, vp, i64, vp, i64, vp, sz, vp]
    L.pwh_apply_h.restype = i32
    L.pwh_cheb_filter.argtypes = [vp, i64, vp, i64, i32, dbl, dbl, dbl, vp, sz, vp]
    L.pwh_cheb_filter.restype = i32
    L.pwh_gram_workspace_bytes.argtypes = [i64, i64, i64]
    L.pwh_gram_workspace_bytes.restype = sz
    L.pwh_gram.argtypes = [i64, i64, vp, i64, i64, vp, i64, vp, i64, vp, sz, vp]
    L.pwh_gram.restype = i32
    L.pwh_gram_herm.argtypes = [i64, i64, vp, i64, vp, i64, vp, i64, vp, sz, vp]
    L.pwh_gram_static.argtypes = [i64, i64, vp, i64, i64, vp, i64, vp, i64, vp]
    L.pwh_gram_static.restype = i32
    L.pwh_gram_herm.restype = i32
    L.pwh_ham_kernels.argtypes = [vp, ctypes.c_char_p, sz]
    L.pwh_ham_kernels.restype = i32
    L.pwh_apply_h_host.argtypes = [vp, i64, vp, i64, vp, i64, vp]
    L.pwh_apply_h_host.restype = i32
    L.pwh_cheb_filter_host.argtypes = [vp, i64, i64, vp, i64, i32, dbl, dbl, dbl, vp]
    L.pwh_cheb_filter_host.restype = i32
    L.pwh_sweep_host.argtypes = [vp, i64, i64, vp, i64, i32, dbl, dbl, dbl, vp, i64, vp, i64, vp]
    L.pwh_sweep_host.restype = i32
    L.pwh_launch_count.argtypes = []
    L.pwh_launch_count.restype = i64
    L.pwh_ham_info.argtypes = [vp, vp]
    L.pwh_ham_info.restype = i32
    L.pwh_profile_begin.argtypes = []
    L.pwh_profile_begin.restype = i32
    L.pwh_profile_end.argtypes = [vp, vp]
    L.pwh_profile_end.restype = i32
    L.pwh_probe_fp64_tensor_peak.argtypes = [i32, vp, vp]
    L.pwh_probe_fp64_tensor_peak.restype = i32
    L.pwh_last_error.argtypes = []
    L.pwh_last_error.restype = ctypes.c_char_p
    L.pwh_rayleigh_quotients.argtypes = [i64, i64, vp, i64, vp, i64, vp, i64, vp, vp, vp]
    L.pwh_rayleigh_quotients.restype = i32
    L.pwh_residual_norms.argtypes = [i64, i64, vp, i64, vp, i64, vp, i64, vp, vp, i64, vp, vp]
    L.pwh_residual_norms.restype = i32
    L.pwh_rotate.argtypes = [i64, i64, vp, i64, i64, vp, i64, vp, i64, vp]
    L.pwh_rotate.restype = i32
    L.pwh_dense_workspace_bytes.argtypes = [i64]
    L.pwh_dense_workspace_bytes.restype = sz
    L.pwh_potrf.argtypes = [i64, vp, i64, vp, vp]
    L.pwh_potrf.restype = i32
    L.pwh_heev.argtypes = [i64, vp, i64, vp, vp, i64, vp, vp, sz, vp]
    L.pwh_heev.restype = i32
    L.pwh_hegv.argtypes = [i64, vp, i64, vp, i64, vp, vp, i64, vp, vp, sz, vp]
    L.pwh_hegv.restype = i32
    L.pwh_rr_workspace_bytes.argtypes = [i64, i64]
    L.pwh_rr_workspace_bytes.restype = sz
    L.pwh_chol_ortho.argtypes = [i64, i64, vp, i64, vp, i64, vp, i64, vp, vp, sz, vp]
    L.pwh_chol_ortho.restype = i32
    L.pwh_rayleigh_ritz.argtypes = [i64, i64, vp, i64, vp, i64, vp, i64, vp, vp, vp, sz, vp]
    L.pwh_rayleigh_ritz.restype = i32
    L.pwh_chebfi_workspace_bytes.argtypes = [vp, i64, i64]
    L.pwh_chebfi_workspace_bytes.restype = sz
    L.pwh_chebfi_iteration.argtypes = [vp, i64, i64, vp, i64, vp, i64, vp, i64, i32, dbl, dbl, vp, vp, vp, vp, vp, sz, vp]
    L.pwh_chebfi_iteration.restype = i32
    L.pwh_ham_set_paw.argtypes = [vp, i64, vp, vp, vp, vp, vp]
    L.pwh_ham_set_paw.restype = i32
    L.pwh_apply_hs.argtypes = [vp, i64, vp, i64, vp, i64, vp, i64, vp, sz, vp]
    L.pwh_apply_hs.restype = i32
    L.pwh_apply_sinv.argtypes = [vp, i64, vp, i64, vp, sz, vp]
    L.pwh_apply_sinv.restype = i32
    L.pwh_cheb_filter_gen.argtypes = [vp, i64, vp, i64, i32, dbl, dbl, dbl, vp, sz, vp]
    L.pwh_cheb_filter_gen.restype = i32
    L.pwh_chol_ortho_gen.argtypes = [i64, i64, vp, i64, vp, i64, vp, i64, vp, i64, vp, vp, sz, vp]
    L.pwh_chol_ortho_gen.restype = i32
    L.pwh_lobpcg_gen_workspace_bytes.argtypes = [vp, i64, i64]
    L.pwh_lobpcg_gen_workspace_bytes.restype = sz
    L.pwh_lobpcg_gen.argtypes = [vp, i64, i64, i32, dbl, vp, i64, vp, i64, vp, i64, vp, vp, vp, vp, vp, sz, vp]
    L.pwh_lobpcg_gen.restype = i32
    L.pwh_density_workspace_bytes.argtypes = [vp, i64]
    L.pwh_density_workspace_bytes.restype = sz
    L.pwh_density_accumulate.argtypes = [vp, i64, vp, i64, vp, dbl, vp, vp, sz, vp]
    L.pwh_density_accumulate.restype = i32
    L.pwh_lobpcg_workspace_bytes.argtypes = [vp, i64, i64]
    L.pwh_lobpcg_workspace_bytes.restype = sz
    L.pwh_lobpcg.argtypes = [vp, i64, i64, i32, dbl, vp, i64, vp, i64, vp, vp, vp, vp, vp, sz, vp]
    L.pwh_lobpcg.restype = i32
    _lib = L
    return L


def _check(rc: int, what: str) -> None:
    if rc != 0:
        msg = load_library().pwh_last_error().decode("utf-8", "replace")
        raise PwhamError(f"{what} failed with code {rc}: {msg}")


def _stream_ptr(device) -> int:
    return int(torch.cuda.current_stream(device).cuda_stream)


def _dev_tensor(x, dtype, device) -> torch.Tensor:
    if isinstance(x, np.ndarray):
        x = torch.from_numpy(np.ascontiguousarray(x))
    return x.to(device=device, dtype=dtype).contiguous()


def _block_args(t: torch.Tensor, npw: int, name: str):
    if not (t.is_cuda and t.dtype == torch.complex128 and t.dim() == 2):
        raise PwhamError(f"{name} must be a 2-D CUDA complex128 tensor of shape (nband, npw)")
    if t.shape[1] != npw or t.stride(1) != 1 or (t.shape[0] > 1 and t.stride(0) < npw):
        raise PwhamError(f"{name}: expected shape (nband, {npw}) with unit stride along plane waves")
    ld = t.stride(0) if t.shape[0] > 1 else max(npw, t.stride(0))
    return t.data_ptr(), int(ld)


class Ham:
    """Owner of one pwh_ham handle plus the device tensors it borrows (projectors) and its cached workspace."""

    def __init__(self, handle: int, device, npw: int, nproj: int, keep):
        self.handle = ctypes.c_void_p(handle)
        self.device = device
        self.npw = npw
        self.nproj = nproj
        self._keep = keep
        self._ws: Optional[torch.Tensor] = None

    def workspace(self, nband: int) -> torch.Tensor:
        need = int(load_library().pwh_workspace_bytes(self.handle, nband))
        if self._ws is None or self._ws.numel() < need:
            self._ws = None
            self._ws = torch.empty(need, dtype=torch.uint8, device=self.device)
        return self._ws

    def info(self) -> dict:
        arr = (ctypes.c_int64 * 8)()
        _check(load_library().pwh_ham_info(self.handle, arr), "pwh_ham_info")
        keys = ["npw", "nproj", "n1", "n2", "n3", "n_zcolumns", "n_xlines", "band_group"]
        return dict(zip(keys, [int(v) for v in arr]))

    def kernels(self) -> list:
        """pwh_ham_kernels: the kernel families this handle launches."""
        buf = ctypes.create_string_buffer(256)
        _check(load_library().pwh_ham_kernels(self.handle, buf, 256), "pwh_ham_kernels")
        return buf.value.decode().split()

    def destroy(self) -> None:
        if self.handle:
            load_library().pwh_ham_destroy(self.handle)
            self.handle = ctypes.c_void_p(None)
            self._keep = None
            self._ws = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def ham_setup(lattice, kpt, fft_dims, gvec, vloc, proj, dij, device="cuda:0") -> Ham:
    """pwh_ham_setup: build the handle.  gvec (npw,3) int32, vloc (n3,n2,n1) float64, proj (nproj,npw) complex128
    (row i = <G|p_i>, i.e. column-major npw x nproj), dij (nproj,) float64; numpy arrays or torch tensors."""
    L = load_library()
    if not torch.cuda.is_available():
        raise PwhamError("CUDA is not available: libpwham has no CPU fallback")
    device = torch.device(device)
    lattice = np.ascontiguousarray(np.asarray(lattice, dtype=np.float64).reshape(9))
    kpt = np.ascontiguousarray(np.asarray(kpt, dtype=np.float64).reshape(3))
    dims = np.ascontiguousarray(np.asarray(fft_dims, dtype=np.int32).reshape(3))
    g = _dev_tensor(gvec, torch.int32, device)
    npw = int(g.shape[0])
    v = _dev_tensor(vloc, torch.float64, device)
    if tuple(v.shape) != (int(dims[2]), int(dims[1]), int(dims[0])):
        raise PwhamError("vloc must have shape (n3, n2, n1)")
    if proj is None or len(proj) == 0:
        nproj, p, d, p_ptr, d_ptr, ldp = 0, None, None, None, None, npw
    else:
        if isinstance(proj, torch.Tensor) and proj.is_cuda and proj.dtype == torch.complex128 and proj.dim() == 2 \
                and proj.stride(1) == 1 and (proj.shape[0] == 1 or proj.stride(0) >= proj.shape[1]):
            p = proj                                  # borrowed as is: rows may be padded (ldp = stride(0) > npw)
        else:
            p = _dev_tensor(proj, torch.complex128, device)
        d = _dev_tensor(dij, torch.float64, device)
        nproj = int(p.shape[0])
        if p.shape[1] != npw or d.shape[0] != nproj:
            raise PwhamError("proj must be (nproj, npw) and dij (nproj,)")
        p_ptr, d_ptr, ldp = p.data_ptr(), d.data_ptr(), (int(p.stride(0)) if nproj > 1 else max(npw, int(p.stride(0))))
    handle = ctypes.c_void_p()
    with torch.cuda.device(device):
        rc = L.pwh_ham_setup(ctypes.byref(handle), lattice.ctypes.data, kpt.ctypes.data, dims.ctypes.data, npw,
                             g.data_ptr(), v.data_ptr(), nproj, p_ptr, ldp, d_ptr, _stream_ptr(device))
    _check(rc, "pwh_ham_setup")
    return Ham(handle.value, device, npw, nproj, keep=(p,))


def ham_destroy(ham: Ham) -> None:
    ham.destroy()


def apply_h(ham: Ham, psi: torch.Tensor, out: Optional[torch.Tensor] = None) -> torch.Tensor:
    """pwh_apply_h: out = H psi for a block psi (nband, npw)."""
    L = load_library()
    p_ptr, ldp = _block_args(psi, ham.npw, "psi")
    if out is None:
        out = torch.empty((psi.shape[0], ham.npw), dtype=torch.complex128, device=psi.device)
    o_ptr, ldo = _block_args(out, ham.npw, "out")
    nband = int(psi.shape[0])
    ws = ham.workspace(nband)
    with torch.cuda.device(ham.device):
        rc = L.pwh_apply_h(ham.handle, nband, p_ptr, ldp, o_ptr, ldo, ws.data_ptr(), ws.numel(), _stream_ptr(ham.device))
    _check(rc, "pwh_apply_h")
    return out


def cheb_filter(ham: Ham, psi: torch.Tensor, degree: int, a: float, b: float, a0: float) -> torch.Tensor:
    """pwh_cheb_filter: in place psi <- T_m((H-c)/e)/T_m((a0-c)/e) psi; returns psi."""
    L = load_library()
    p_ptr, ld = _block_args(psi, ham.npw, "psi")
    nband = int(psi.shape[0])
    ws = ham.workspace(nband)
    with torch.cuda.device(ham.device):
        rc = L.pwh_cheb_filter(ham.handle, nband, p_ptr, ld, int(degree), float(a), float(b), float(a0), ws.data_ptr(),
                               ws.numel(), _stream_ptr(ham.device))
    _check(rc, "pwh_cheb_filter")
    return psi


def density_accumulate(ham: Ham, psi: torch.Tensor, occ, rho: torch.Tensor, weight: float = 1.0) -> torch.Tensor:
    """pwh_density_accumulate: rho (n3, n2, n1) float64 += weight * sum_i occ[i] |u_i(r)|^2 for the block psi; returns rho."""
    L = load_library()
    p_ptr, ld = _block_args(psi, ham.npw, "psi")
    nband = int(psi.shape[0])
    f = _dev_tensor(occ if isinstance(occ, torch.Tensor) else np.asarray(occ, dtype=np.float64), torch.float64, ham.device)
    info = ham.info()
    if f.dim() != 1 or f.shape[0] != nband:
        raise PwhamError("occ must have shape (nband,)")
    if not (rho.is_cuda and rho.dtype == torch.float64 and rho.is_contiguous()
            and tuple(rho.shape) == (info["n3"], info["n2"], info["n1"])):
        raise PwhamError("rho must be a contiguous CUDA float64 tensor of shape (n3, n2, n1)")
    need = int(L.pwh_density_workspace_bytes(ham.handle, nband))
    ws = torch.empty(need, dtype=torch.uint8, device=ham.device)
    with torch.cuda.device(ham.device):
        rc = L.pwh_density_accumulate(ham.handle, nband, p_ptr, ld, f.data_ptr(), float(weight), rho.data_ptr(),
                                      ws.data_ptr(), ws.numel(), _stream_ptr(ham.device))
    _check(rc, "pwh_density_accumulate")
    return rho


_gram_ws = {}


def gram(x: torch.Tensor, y: torch.Tensor, hermitian: bool = False) -> torch.Tensor:
    """pwh_gram (pwh_gram_herm when `hermitian`): returns G of shape (nx, ny) with G[i, j] = <x_i, y_j> =
    sum_g conj(x[i, g]) y[j, g]."""
    L = load_library()
    npw = int(x.shape[1])
    x_ptr, ldx = _block_args(x, npw, "x")
    y_ptr, ldy = _block_args(y, npw, "y")
    nx, ny = int(x.shape[0]), int(y.shape[0])
    g_cm = torch.empty((ny, nx), dtype=torch.complex128, device=x.device)   # column-major nx x ny
    need = int(L.pwh_gram_workspace_bytes(npw, nx, ny))
    key = (x.device.index, )
    ws = _gram_ws.get(key)
    if ws is None or ws.numel() < need:
        _gram_ws[key] = None
        ws = _gram_ws[key] = torch.empty(need, dtype=torch.uint8, device=x.device)
    with torch.cuda.device(x.device):
        if hermitian:
            if nx != ny:
                raise PwhamError("hermitian gram needs nx == ny")
            rc = L.pwh_gram_herm(npw, nx, x_ptr, ldx, y_ptr, ldy, g_cm.data_ptr(), nx, ws.data_ptr(), ws.numel(),
                                 _stream_ptr(x.device))
        else:
            rc = L.pwh_gram(npw, nx, x_ptr, ldx, ny, y_ptr, ldy, g_cm.data_ptr(), nx, ws.data_ptr(), ws.numel(),
                            _stream_ptr(x.device))
    _check(rc, "pwh_gram_herm" if hermitian else "pwh_gram")
    return g_cm.T


GRAM_STATIC_MAX_ENTRIES = 1048576      # PWH_GRAM_STATIC_MAX_ENTRIES of include/pwham.h


def gram_static(x: torch.Tensor, y: torch.Tensor, out: Optional[torch.Tensor] = None) -> torch.Tensor:
    """pwh_gram_static: G = X^H Y with the split-K scratch in the library's static device array (no workspace, no allocation
    inside the call; nx * ny <= GRAM_STATIC_MAX_ENTRIES).  `out`: optional (ny, nx) complex128 CUDA tensor that receives the
    column-major result, so that the binding allocates nothing either; returns G of shape (nx, ny)."""
    L = load_library()
    npw = int(x.shape[1])
    x_ptr, ldx = _block_args(x, npw, "x")
    y_ptr, ldy = _block_args(y, npw, "y")
    nx, ny = int(x.shape[0]), int(y.shape[0])
    if out is None:
        out = torch.empty((ny, nx), dtype=torch.complex128, device=x.device)
    elif not (out.is_cuda and out.dtype == torch.complex128 and tuple(out.shape) == (ny, nx) and out.is_contiguous()):
        raise PwhamError("out must be a contiguous CUDA complex128 tensor of shape (ny, nx)")
    with torch.cuda.device(x.device):
        rc = L.pwh_gram_static(npw, nx, x_ptr, ldx, ny, y_ptr, ldy, out.data_ptr(), nx, _stream_ptr(x.device))
    _check(rc, "pwh_gram_static")
    return out.T


def _host_block(a, npw: int, name: str):
    if isinstance(a, torch.Tensor):
        if a.is_cuda or a.dtype != torch.complex128 or a.dim() != 2 or a.shape[1] != npw or not a.is_contiguous():
            raise PwhamError(f"{name} must be a contiguous host complex128 tensor (nband, npw)")
        return a.data_ptr(), int(a.shape[0])
    if not (isinstance(a, np.ndarray) and a.dtype == np.complex128 and a.ndim == 2 and a.shape[1] == npw
            and a.flags.c_contiguous):
        raise PwhamError(f"{name} must be a C-contiguous host complex128 array (nband, npw)")
    return a.ctypes.data, int(a.shape[0])


def apply_h_host(ham: Ham, psi_host, hpsi_host) -> None:
    """pwh_apply_h_host: host buffers in, host buffers out (copies inside the call)."""
    L = load_library()
    p, nband = _host_block(psi_host, ham.npw, "psi_host")
    o, nb2 = _host_block(hpsi_host, ham.npw, "hpsi_host")
    if nb2 != nband:
        raise PwhamError("psi_host / hpsi_host band counts differ")
    with torch.cuda.device(ham.device):
        rc = L.pwh_apply_h_host(ham.handle, nband, p, ham.npw, o, ham.npw, _stream_ptr(ham.device))
    _check(rc, "pwh_apply_h_host")


def cheb_filter_host(ham: Ham, psi_host, degree: int, a: float, b: float, a0: float, block: int = 0) -> None:
    """pwh_cheb_filter_host: in place on a host block, bands filtered in column blocks of `block`."""
    L = load_library()
    p, nband = _host_block(psi_host, ham.npw, "psi_host")
    with torch.cuda.device(ham.device):
        rc = L.pwh_cheb_filter_host(ham.handle, nband, int(block), p, ham.npw, int(degree), float(a), float(b),
                                    float(a0), _stream_ptr(ham.device))
    _check(rc, "pwh_cheb_filter_host")


def sweep_host(ham: Ham, psi_host, degree: int, a: float, b: float, a0: float, g_host, block: int = 0,
               hpsi_host=None) -> None:
    """pwh_sweep_host: psi_host <- p_m(H) psi_host, then g_host (nband, nband; g_host[j, i] = <psi_i, H psi_j>,
    i.e. the column-major Gram matrix) -- degree+1 H applications per band and one Gram product, host to host."""
    L = load_library()
    p, nband = _host_block(psi_host, ham.npw, "psi_host")
    if isinstance(g_host, torch.Tensor):
        g_ptr, ok = g_host.data_ptr(), (g_host.dtype == torch.complex128 and tuple(g_host.shape) == (nband, nband)
                                        and g_host.is_contiguous() and not g_host.is_cuda)
    else:
        g_ptr, ok = g_host.ctypes.data, (g_host.dtype == np.complex128 and g_host.shape == (nband, nband)
                                         and g_host.flags.c_contiguous)
    if not ok:
        raise PwhamError("g_host must be a contiguous host complex128 (nband, nband) array")
    h_ptr = None
    if hpsi_host is not None:
        h_ptr, nb2 = _host_block(hpsi_host, ham.npw, "hpsi_host")
        if nb2 != nband:
            raise PwhamError("hpsi_host band count differs")
    with torch.cuda.device(ham.device):
        rc = L.pwh_sweep_host(ham.handle, nband, int(block), p, ham.npw, int(degree), float(a), float(b), float(a0),
                              h_ptr, ham.npw, g_ptr, nband, _stream_ptr(ham.device))
    _check(rc, "pwh_sweep_host")


# ----------------------------------------------------------------------------------------------------------------
# Rayleigh-Ritz companion steps (include/pwham.h, second half).  Small matrices cross this binding as torch tensors of
# shape (n, n) indexed [row, column]; the library's column-major layout is their transpose's memory.
# ----------------------------------------------------------------------------------------------------------------
_scratch = {}


def _ws(device, need: int, tag: str = "rr") -> torch.Tensor:
    key = (torch.device(device).index, tag)
    t = _scratch.get(key)
    if t is None or t.numel() < need:
        _scratch[key] = None
        t = _scratch[key] = torch.empty(max(need, 256), dtype=torch.uint8, device=device)
    return t


def _cm(a: torch.Tensor) -> torch.Tensor:
    """A fresh contiguous tensor holding a^T, i.e. the matrix `a` in column-major order (the solvers work in place)."""
    return a.to(torch.complex128).T.contiguous().clone()


def _opt_block(t: Optional[torch.Tensor], npw: int, name: str):
    return (None, npw) if t is None else _block_args(t, npw, name)


def rayleigh_quotients(psi: torch.Tensor, hpsi: torch.Tensor, spsi: Optional[torch.Tensor] = None):
    """pwh_rayleigh_quotients: (lambda (nband,), minmax (2,)) as device tensors; spsi = S psi (None: S = I)."""
    L = load_library()
    npw = int(psi.shape[1])
    p, ld = _block_args(psi, npw, "psi")
    h, ldh = _block_args(hpsi, npw, "hpsi")
    s_, lds = _opt_block(spsi, npw, "spsi")
    nb = int(psi.shape[0])
    lam = torch.empty(nb, dtype=torch.float64, device=psi.device)
    mm = torch.empty(2, dtype=torch.float64, device=psi.device)
    with torch.cuda.device(psi.device):
        _check(L.pwh_rayleigh_quotients(npw, nb, p, ld, h, ldh, s_, lds, lam.data_ptr(), mm.data_ptr(),
                                        _stream_ptr(psi.device)), "pwh_rayleigh_quotients")
    return lam, mm


def residual_norms(psi: torch.Tensor, hpsi: torch.Tensor, lam: torch.Tensor, want_w: bool = False,
                   spsi: Optional[torch.Tensor] = None):
    """pwh_residual_norms: norms (nband,) and, when want_w, W = hpsi - lam spsi (spsi None: psi)."""
    L = load_library()
    npw = int(psi.shape[1])
    p, ld = _block_args(psi, npw, "psi")
    h, ldh = _block_args(hpsi, npw, "hpsi")
    s_, lds = _opt_block(spsi, npw, "spsi")
    nb = int(psi.shape[0])
    lam = lam.to(device=psi.device, dtype=torch.float64).contiguous()
    norms = torch.empty(nb, dtype=torch.float64, device=psi.device)
    w = torch.empty_like(psi) if want_w else None
    with torch.cuda.device(psi.device):
        _check(L.pwh_residual_norms(npw, nb, p, ld, h, ldh, s_, lds, lam.data_ptr(), w.data_ptr() if want_w else None, npw,
                                    norms.data_ptr(), _stream_ptr(psi.device)), "pwh_residual_norms")
    return (norms, w) if want_w else norms


def rotate(x: torch.Tensor, q: torch.Tensor) -> torch.Tensor:
    """pwh_rotate: Y = X Q for a block x (m, npw) and q (m, n) indexed [i, j]; returns (n, npw)."""
    L = load_library()
    npw = int(x.shape[1])
    xp, ldx = _block_args(x, npw, "x")
    m, n = int(q.shape[0]), int(q.shape[1])
    q_cm = _cm(q)                                      # (n, m) memory = column-major m x n
    y = torch.empty((n, npw), dtype=torch.complex128, device=x.device)
    with torch.cuda.device(x.device):
        _check(L.pwh_rotate(npw, m, xp, ldx, n, q_cm.data_ptr(), m, y.data_ptr(), npw, _stream_ptr(x.device)), "pwh_rotate")
    return y


def potrf(s: torch.Tensor):
    """pwh_potrf: returns (U [row, column] upper triangular with S = U^H U, info)."""
    L = load_library()
    a = _cm(s)
    n = int(a.shape[0])
    info = torch.zeros(1, dtype=torch.int32, device=a.device)
    with torch.cuda.device(a.device):
        _check(L.pwh_potrf(n, a.data_ptr(), n, info.data_ptr(), _stream_ptr(a.device)), "pwh_potrf")
    return a.T, int(info.item())


def heev(a: torch.Tensor):
    """pwh_heev: (w ascending (n,), X [row, column] with eigenvectors in its columns, sweeps)."""
    L = load_library()
    a_cm = _cm(a)
    n = int(a_cm.shape[0])
    w = torch.empty(n, dtype=torch.float64, device=a.device)
    x = torch.empty((n, n), dtype=torch.complex128, device=a.device)
    info = torch.zeros(1, dtype=torch.int32, device=a.device)
    ws = _ws(a.device, int(L.pwh_dense_workspace_bytes(n)))
    with torch.cuda.device(a.device):
        _check(L.pwh_heev(n, a_cm.data_ptr(), n, w.data_ptr(), x.data_ptr(), n, info.data_ptr(), ws.data_ptr(), ws.numel(),
                          _stream_ptr(a.device)), "pwh_heev")
    return w, x.T, int(info.item())


def hegv(a: torch.Tensor, b: torch.Tensor):
    """pwh_hegv: A X = B X diag(w), X^H B X = I; returns (w, X [row, column], info)."""
    L = load_library()
    a_cm, b_cm = _cm(a), _cm(b)
    n = int(a_cm.shape[0])
    w = torch.empty(n, dtype=torch.float64, device=a.device)
    x = torch.empty((n, n), dtype=torch.complex128, device=a.device)
    info = torch.zeros(1, dtype=torch.int32, device=a.device)
    ws = _ws(a.device, int(L.pwh_dense_workspace_bytes(n)))
    with torch.cuda.device(a.device):
        _check(L.pwh_hegv(n, a_cm.data_ptr(), n, b_cm.data_ptr(), n, w.data_ptr(), x.data_ptr(), n, info.data_ptr(),
                          ws.data_ptr(), ws.numel(), _stream_ptr(a.device)), "pwh_hegv")
    return w, x.T, int(info.item())


def chol_ortho(psi: torch.Tensor, hpsi: Optional[torch.Tensor] = None):
    """pwh_chol_ortho, in place on psi (and hpsi): returns (U [row, column], info)."""
    L = load_library()
    npw = int(psi.shape[1])
    p, ld = _block_args(psi, npw, "psi")
    nb = int(psi.shape[0])
    h, ldh = (None, npw) if hpsi is None else _block_args(hpsi, npw, "hpsi")
    u = torch.empty((nb, nb), dtype=torch.complex128, device=psi.device)
    info = torch.zeros(1, dtype=torch.int32, device=psi.device)
    ws = _ws(psi.device, int(L.pwh_rr_workspace_bytes(npw, nb)))
    with torch.cuda.device(psi.device):
        _check(L.pwh_chol_ortho(npw, nb, p, ld, h, ldh, u.data_ptr(), nb, info.data_ptr(), ws.data_ptr(), ws.numel(),
                                _stream_ptr(psi.device)), "pwh_chol_ortho")
    return u.T, int(info.item())


def chol_ortho_gen(psi: torch.Tensor, hpsi: Optional[torch.Tensor], spsi: torch.Tensor):
    """pwh_chol_ortho_gen, in place on psi, spsi (and hpsi): returns (U [row, column], info)."""
    L = load_library()
    npw = int(psi.shape[1])
    p, ld = _block_args(psi, npw, "psi")
    sp, lds = _block_args(spsi, npw, "spsi")
    nb = int(psi.shape[0])
    h, ldh = (None, npw) if hpsi is None else _block_args(hpsi, npw, "hpsi")
    u = torch.empty((nb, nb), dtype=torch.complex128, device=psi.device)
    info = torch.zeros(1, dtype=torch.int32, device=psi.device)
    ws = _ws(psi.device, int(L.pwh_rr_workspace_bytes(npw, nb)))
    with torch.cuda.device(psi.device):
        _check(L.pwh_chol_ortho_gen(npw, nb, p, ld, h, ldh, sp, lds, u.data_ptr(), nb, info.data_ptr(), ws.data_ptr(),
                                    ws.numel(), _stream_ptr(psi.device)), "pwh_chol_ortho_gen")
    return u.T, int(info.item())


def rayleigh_ritz(psi: torch.Tensor, hpsi: torch.Tensor, spsi: Optional[torch.Tensor] = None):
    """pwh_rayleigh_ritz, in place on psi, hpsi (and spsi): returns (lambda (nband,), info)."""
    L = load_library()
    npw = int(psi.shape[1])
    p, ld = _block_args(psi, npw, "psi")
    h, ldh = _block_args(hpsi, npw, "hpsi")
    s_, lds = _opt_block(spsi, npw, "spsi")
    nb = int(psi.shape[0])
    lam = torch.empty(nb, dtype=torch.float64, device=psi.device)
    info = torch.zeros(1, dtype=torch.int32, device=psi.device)
    ws = _ws(psi.device, int(L.pwh_rr_workspace_bytes(npw, nb)))
    with torch.cuda.device(psi.device):
        _check(L.pwh_rayleigh_ritz(npw, nb, p, ld, h, ldh, s_, lds, lam.data_ptr(), info.data_ptr(), ws.data_ptr(), ws.numel(),
                                   _stream_ptr(psi.device)), "pwh_rayleigh_ritz")
    return lam, int(info.item())


def chebfi_iteration(ham: Ham, psi: torch.Tensor, hpsi: torch.Tensor, degree: int, b: float, a0_margin: float = 0.0,
                     block: int = 0, spsi: Optional[torch.Tensor] = None):
    """pwh_chebfi_iteration, in place on psi / hpsi (/ spsi: generalised problem, needs set_paw): returns
    dict(lam, resid (device tensors), a0, a, info)."""
    L = load_library()
    p, ld = _block_args(psi, ham.npw, "psi")
    h, ldh = _block_args(hpsi, ham.npw, "hpsi")
    s_, lds = _opt_block(spsi, ham.npw, "spsi")
    nb = int(psi.shape[0])
    lam = torch.empty(nb, dtype=torch.float64, device=psi.device)
    res = torch.empty(nb, dtype=torch.float64, device=psi.device)
    info = torch.zeros(1, dtype=torch.int32, device=psi.device)
    bounds = (ctypes.c_double * 2)()
    ws = _ws(psi.device, int(L.pwh_chebfi_workspace_bytes(ham.handle, nb, int(block))), tag="chebfi")
    with torch.cuda.device(ham.device):
        _check(L.pwh_chebfi_iteration(ham.handle, nb, int(block), p, ld, h, ldh, s_, lds, int(degree), float(b), float(a0_margin),
                                      lam.data_ptr(), res.data_ptr(), bounds, info.data_ptr(), ws.data_ptr(), ws.numel(),
                                      _stream_ptr(ham.device)), "pwh_chebfi_iteration")
    return {"lam": lam, "resid": res, "a0": float(bounds[0]), "a": float(bounds[1]), "info": int(info.item())}


def lobpcg(ham: Ham, psi: torch.Tensor, hpsi: torch.Tensor, nblocks: int, nline: int, tol: float = 0.0):
    """pwh_lobpcg (Algorithm 11, S = I), in place on psi / hpsi: returns dict(lam, resid, history (nblocks, nline, m) device
    tensors -- history entries of passes skipped by the early exit are NaN --, info)."""
    L = load_library()
    p, ld = _block_args(psi, ham.npw, "psi")
    h, ldh = _block_args(hpsi, ham.npw, "hpsi")
    nb = int(psi.shape[0])
    need = int(L.pwh_lobpcg_workspace_bytes(ham.handle, nb, int(nblocks)))
    if need == 0:
        raise PwhamError("pwh_lobpcg_workspace_bytes: nband must be a positive multiple of nblocks")
    lam = torch.empty(nb, dtype=torch.float64, device=psi.device)
    res = torch.empty(nb, dtype=torch.float64, device=psi.device)
    hist = torch.full((int(nblocks), max(int(nline), 0), nb // int(nblocks)), float("nan"), dtype=torch.float64, device=psi.device)
    info = torch.zeros(1, dtype=torch.int32, device=psi.device)
    ws = _ws(psi.device, need, tag="lobpcg")
    with torch.cuda.device(ham.device):
        _check(L.pwh_lobpcg(ham.handle, nb, int(nblocks), int(nline), float(tol), p, ld, h, ldh, lam.data_ptr(), res.data_ptr(),
                            hist.data_ptr() if hist.numel() else None, info.data_ptr(), ws.data_ptr(), ws.numel(),
                            _stream_ptr(ham.device)), "pwh_lobpcg")
    return {"lam": lam, "resid": res, "history": hist, "info": int(info.item())}


def lobpcg_gen(ham: Ham, psi: torch.Tensor, hpsi: torch.Tensor, spsi: torch.Tensor, nblocks: int, nline: int, tol: float = 0.0):
    """pwh_lobpcg_gen (Algorithm 11 with the PAW overlap S of the handle), in place on psi / hpsi / spsi: returns the same dict
    as `lobpcg`."""
    L = load_library()
    p, ld = _block_args(psi, ham.npw, "psi")
    h, ldh = _block_args(hpsi, ham.npw, "hpsi")
    sp, lds = _block_args(spsi, ham.npw, "spsi")
    nb = int(psi.shape[0])
    need = int(L.pwh_lobpcg_gen_workspace_bytes(ham.handle, nb, int(nblocks)))
    if need == 0:
        raise PwhamError("pwh_lobpcg_gen_workspace_bytes: nband must be a positive multiple of nblocks")
    lam = torch.empty(nb, dtype=torch.float64, device=psi.device)
    res = torch.empty(nb, dtype=torch.float64, device=psi.device)
    hist = torch.full((int(nblocks), max(int(nline), 0), nb // int(nblocks)), float("nan"), dtype=torch.float64, device=psi.device)
    info = torch.zeros(1, dtype=torch.int32, device=psi.device)
    ws = _ws(psi.device, need, tag="lobpcg")
    with torch.cuda.device(ham.device):
        _check(L.pwh_lobpcg_gen(ham.handle, nb, int(nblocks), int(nline), float(tol), p, ld, h, ldh, sp, lds, lam.data_ptr(),
                                res.data_ptr(), hist.data_ptr() if hist.numel() else None, info.data_ptr(), ws.data_ptr(),
                                ws.numel(), _stream_ptr(ham.device)), "pwh_lobpcg_gen")
    return {"lam": lam, "resid": res, "history": hist, "info": int(info.item())}


# ----------------------------------------------------------------------------------------------------------------
# PAW-style generalised problem
# ----------------------------------------------------------------------------------------------------------------
def ham_set_paw(ham: Ham, offsets, dblocks, qblocks) -> int:
    """pwh_ham_set_paw: per-atom dense blocks D^R, Q^R (lists of (n_R, n_R) arrays indexed [i, j]); returns info."""
    L = load_library()
    offsets = np.ascontiguousarray(np.asarray(offsets, dtype=np.int32))

    def pack(blocks):
        flat = np.concatenate([np.asarray(b, dtype=np.complex128).T.reshape(-1) for b in blocks])   # column-major
        return torch.from_numpy(np.ascontiguousarray(flat)).to(ham.device)

    d, q = pack(dblocks), pack(qblocks)
    info = torch.zeros(1, dtype=torch.int32, device=ham.device)
    with torch.cuda.device(ham.device):
        _check(L.pwh_ham_set_paw(ham.handle, len(offsets) - 1, offsets.ctypes.data, d.data_ptr(), q.data_ptr(),
                                 info.data_ptr(), _stream_ptr(ham.device)), "pwh_ham_set_paw")
    ham._ws = None                     # the workspace layout grows with the PAW blocks
    return int(info.item())


def apply_hs(ham: Ham, psi: torch.Tensor):
    """pwh_apply_hs: returns (H psi, S psi)."""
    L = load_library()
    p, ldp = _block_args(psi, ham.npw, "psi")
    nband = int(psi.shape[0])
    hpsi, spsi = torch.empty_like(psi), torch.empty_like(psi)
    ws = ham.workspace(nband)
    with torch.cuda.device(ham.device):
        _check(L.pwh_apply_hs(ham.handle, nband, p, ldp, hpsi.data_ptr(), ham.npw, spsi.data_ptr(), ham.npw, ws.data_ptr(),
                              ws.numel(), _stream_ptr(ham.device)), "pwh_apply_hs")
    return hpsi, spsi


def apply_sinv(ham: Ham, x: torch.Tensor) -> torch.Tensor:
    """pwh_apply_sinv: x <- S^-1 x in place; returns x."""
    L = load_library()
    p, ld = _block_args(x, ham.npw, "x")
    nband = int(x.shape[0])
    ws = ham.workspace(nband)
    with torch.cuda.device(ham.device):
        _check(L.pwh_apply_sinv(ham.handle, nband, p, ld, ws.data_ptr(), ws.numel(), _stream_ptr(ham.device)), "pwh_apply_sinv")
    return x


def cheb_filter_gen(ham: Ham, psi: torch.Tensor, degree: int, a: float, b: float, a0: float) -> torch.Tensor:
    """pwh_cheb_filter_gen: in place psi <- p_m(S^-1 H) psi; returns psi."""
    L = load_library()
    p, ld = _block_args(psi, ham.npw, "psi")
    nband = int(psi.shape[0])
    ws = ham.workspace(nband)
    with torch.cuda.device(ham.device):
        _check(L.pwh_cheb_filter_gen(ham.handle, nband, p, ld, int(degree), float(a), float(b), float(a0), ws.data_ptr(),
                                     ws.numel(), _stream_ptr(ham.device)), "pwh_cheb_filter_gen")
    return psi


def launch_count() -> int:
    return int(load_library().pwh_launch_count())


def profile_begin() -> None:
    _check(load_library().pwh_profile_begin(), "pwh_profile_begin")


def profile_end() -> dict:
    """Returns {stage: (milliseconds, launches)} summed over the launches since profile_begin()."""
    ms = (ctypes.c_double * len(STAGES))()
    n = (ctypes.c_int64 * len(STAGES))()
    _check(load_library().pwh_profile_end(ms, n), "pwh_profile_end")
    return {STAGES[i]: (float(ms[i]), int(n[i])) for i in range(len(STAGES)) if n[i]}


def probe_fp64_tensor_peak(iters: int = 20000, device="cuda:0") -> float:
    """TFLOP/s of a register-resident DMMA loop on this GPU at its current clocks (roofline denominator)."""
    out = ctypes.c_double(0.0)
    with torch.cuda.device(device):
        _check(load_library().pwh_probe_fp64_tensor_peak(int(iters), ctypes.byref(out), _stream_ptr(torch.device(device))),
               "pwh_probe_fp64_tensor_peak")
    return float(out.value)
