"""ctypes binding of libqe_hpsi.so (include/qe_hpsi.h; the measurement / test helpers of include/qe_hpsi_test.h are
bound too and marked as such). Argument marshalling only: every step of H|psi> runs in the library's CUDA kernels.
PyTorch supplies device memory and streams. There is NO fallback: if the shared library is missing or cannot be
loaded, importing callers get a RuntimeError.

Function names mirror the C ABI (qe_hpsi_gsphere, qe_hpsi_create, qe_hpsi_apply, ...); `Hpsi` is a small RAII
convenience around a handle.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np
import torch

_PKG = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_PKG, "libqe_hpsi.so")

QE_HPSI_OK, QE_HPSI_EINVAL, QE_HPSI_EGRID, QE_HPSI_ENOMEM, QE_HPSI_ECUDA, QE_HPSI_ESTATE = 0, -1, -2, -3, -4, -5
QE_HPSI_BORROW_BETA = 1
QE_HPSI_GENERIC_FFT = 2
QE_HPSI_FP64_DMMA = 4      # the default accuracy class (FP64 tensor pipe); the flag only names it
QE_HPSI_PROJ_INT8 = 8      # opt-in: a6 / a8 as exact int8 digit products (block fixed point, 8S-1 bits under a row exponent)
QE_HPSI_PROJ_CERTIFY = 16  # with PROJ_INT8: a-posteriori check of every chunk + FP64 re-computation of failing bands
QE_HPSI_PROJ_3M_OFF, QE_HPSI_PROJ_3M_A6, QE_HPSI_PROJ_3M_ALL = 1 << 12, 2 << 12, 3 << 12
QE_HPSI_NO_GAMMA_SYM = 32   # keep the general complex contraction at k = 0 (see include/qe_hpsi.h)
QE_HPSI_NPROBE = 8
QE_HPSI_MAX_N = 720


def QE_HPSI_PROJ_DIGITS(s: int) -> int:
    """Digit-count field of the create flags (4..7; 0 = 7)."""
    return (int(s) & 15) << 8


_c = ctypes
_vp, _i64, _i32, _dbl = _c.c_void_p, _c.c_int64, _c.c_int, _c.c_double
_pd, _pi32, _pi64 = _c.POINTER(_c.c_double), _c.POINTER(_c.c_int32), _c.POINTER(_c.c_int64)

# name -> (restype, argtypes); the single source the loader and the symbol test use
SIGNATURES = {
    "qe_hpsi_gsphere": (_i32, [_pd, _pd, _dbl, _pi32, _pi64, _pi32]),
    "qe_hpsi_create": (_i32, [_c.POINTER(_vp), _pd, _dbl, _pd, _pi32, _vp, _i32, _vp, _i64, _i32, _pi32, _pd, _i32,
                              _c.c_uint, _vp]),
    "qe_hpsi_apply": (_i32, [_vp, _vp, _i64, _vp, _i64, _i32, _vp]),
    "qe_hpsi_apply_host": (_i32, [_vp, _vp, _i64, _vp, _i64, _i32]),
    "qe_hpsi_destroy": (_i32, [_vp]),
    "qe_hpsi_npw": (_i64, [_vp]),
    "qe_hpsi_nsticks": (_i64, [_vp]),
    "qe_hpsi_nplanes": (_i64, [_vp]),
    "qe_hpsi_get_maps": (_i32, [_vp, _vp, _vp, _vp, _vp]),
    "qe_hpsi_get_becp": (_i32, [_vp, _vp, _vp, _vp]),
    "qe_hpsi_launch_count": (_i64, [_vp, _i32]),
    "qe_hpsi_info": (_i32, [_vp, _pi64]),
    "qe_hpsi_strerror": (_c.c_char_p, [_i32]),
    "qe_hpsi_last_error": (_i32, [_vp]),
    "qe_hpsi_set_proj_tolerance": (_i32, [_vp, _dbl]),
    "qe_hpsi_get_proj_check": (_i32, [_vp, _vp, _vp, _vp]),
    "qe_hpsi_residual": (_i32, [_vp, _vp, _i64, _vp, _i64, _vp, _vp, _i64, _i32, _vp, _vp]),
    "qe_hpsi_scale": (_i32, [_vp, _vp, _i64, _i32, _vp, _vp]),
    # ---- include/qe_hpsi_test.h: measurement and test helpers, not the product boundary ----
    "qe_hpsi_test_set_int8_kmax": (_i32, [_i64]),
    "qe_hpsi_test_set_sym_min": (_i32, [_i64]),
    "qe_hpsi_test_check_guards": (_i64, [_vp]),
    "qe_hpsi_probe_fp64": (_i32, [_dbl, _pd, _pd]),
    "qe_hpsi_profile": (_i32, [_vp, _i32]),
    "qe_hpsi_profile_read": (_i32, [_vp, _pd, _pi64]),
    "qe_hpsi_fft_local": (_i32, [_vp, _vp, _i64, _vp, _i64, _i32, _vp]),
    "qe_hpsi_nonlocal": (_i32, [_vp, _vp, _i64, _vp, _i64, _i32, _vp]),
    "qe_hpsi_set_s": (_i32, [_vp, _pd]),
    "qe_hpsi_apply_hs": (_i32, [_vp, _vp, _i64, _vp, _i64, _vp, _i64, _i32, _vp]),
    "qe_hpsi_overlap": (_i32, [_vp, _vp, _i64, _i32, _vp, _i64, _i32, _vp, _i64, _vp]),
    "qe_hpsi_overlap_static_init": (_i32, []),
    "qe_hpsi_overlap_static": (_i32, [_vp, _i64, _i32, _vp, _i64, _i32, _i64, _vp, _i64, _vp]),
    "qe_hpsi_density": (_i32, [_vp, _vp, _i64, _i32, _vp, _dbl, _vp, _vp]),
    "qe_hpsi_hdiag": (_i32, [_vp, _dbl, _vp, _vp, _vp]),
    "qe_hpsi_precond": (_i32, [_vp, _vp, _i64, _i32, _vp, _vp, _vp, _vp]),
    "qe_hpsi_rotate": (_i32, [_vp, _vp, _i64, _i32, _vp, _i64, _vp, _i64, _i32, _i32, _vp]),
    "qe_hpsi_gamma_gsphere": (_i32, [_pd, _dbl, _pi32, _pi64, _pi32]),
    "qe_hpsi_gamma_create": (_i32, [_c.POINTER(_vp), _pd, _dbl, _pi32, _vp, _i32, _vp, _i64, _i32, _pi32, _pd, _i32,
                                    _c.c_uint, _vp]),
    "qe_hpsi_gamma_apply": (_i32, [_vp, _vp, _i64, _vp, _i64, _i32, _vp]),
    "qe_hpsi_gamma_ngw": (_i64, [_vp]),
    "qe_hpsi_gamma_destroy": (_i32, [_vp]),
}

_lib = None


def load_library():
    """dlopen libqe_hpsi.so (built by paper_2104_10502_b200.build). Fails loudly; never falls back."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_2104_10502_b200.build` (nvcc, sm_100a). "
                           "There is no CPU fallback.")
    lib = ctypes.CDLL(LIB_PATH)
    for name, (res, args) in SIGNATURES.items():
        fn = getattr(lib, name)  # AttributeError if the symbol is not exported
        fn.restype = res
        fn.argtypes = args
    _lib = lib
    return lib


class QeHpsiError(RuntimeError):
    def __init__(self, status, cuda=0):
        msg = load_library().qe_hpsi_strerror(int(status)).decode()
        super().__init__(f"qe_hpsi status {status}: {msg}" + (f" (cudaError {cuda})" if cuda else ""))
        self.status = int(status)
        self.cuda = int(cuda)


def _check(rc, handle=None):
    if rc != 0:
        raise QeHpsiError(rc, load_library().qe_hpsi_last_error(handle))


def _darr(x, n):
    a = np.ascontiguousarray(np.asarray(x, dtype=np.float64).reshape(-1))
    assert a.size == n
    return a, a.ctypes.data_as(_pd)


def _iarr(x, n):
    a = np.ascontiguousarray(np.asarray(x, dtype=np.int32).reshape(-1))
    assert a.size == n
    return a, a.ctypes.data_as(_pi32)


def _stream_ptr(stream):
    if stream is None:
        stream = torch.cuda.current_stream()
    return _vp(stream.cuda_stream)


def qe_hpsi_gsphere(at, xk, ecutwfc, nr) -> np.ndarray:
    """Canonical sphere: int32 Miller triples [npw, 3] (host), ascending FFT linear index."""
    lib = load_library()
    _a, pa = _darr(at, 9)
    _k, pk = _darr(xk, 3)
    _n, pn = _iarr(nr, 3)
    npw = _c.c_int64(0)
    _check(lib.qe_hpsi_gsphere(pa, pk, float(ecutwfc), pn, _c.byref(npw), None))
    mil = np.zeros((max(npw.value, 0), 3), dtype=np.int32)
    if npw.value > 0:
        _check(lib.qe_hpsi_gsphere(pa, pk, float(ecutwfc), pn, _c.byref(npw), mil.ctypes.data_as(_pi32)))
    return mil


def qe_hpsi_test_set_int8_kmax(kmax: int):
    """(qe_hpsi_test.h) K range per CTA of the int8 GEMMs for handles created from now on; 0 = natural."""
    _check(load_library().qe_hpsi_test_set_int8_kmax(int(kmax)))


def qe_hpsi_test_set_sym_min(entries: int):
    """(qe_hpsi_test.h) smallest nproj * npw that takes the Gamma-symmetric projector mode; negative = default (2^20), 0 = always."""
    _check(load_library().qe_hpsi_test_set_sym_min(int(entries)))


QE_HPSI_OVERLAP_STATIC_MAX = 128


def qe_hpsi_overlap_static_init():
    """Once-per-device set-up of qe_hpsi_overlap_static for the current device (allocates nothing)."""
    _check(load_library().qe_hpsi_overlap_static_init())


def qe_hpsi_overlap_static(a, b, npw, out, stream=None):
    """qe_hpsi_overlap_static: out[i][j] = <a_i|b_j> over the leading npw entries, without a handle and without any
    allocation (split-K partials in the library's static device array; na, nb <= QE_HPSI_OVERLAP_STATIC_MAX; calls
    that overlap on the GPU race).  The caller passes `out` ([na, >= nb] complex128 on the device)."""
    for t in (a, b, out):
        assert t.is_cuda and t.dtype == torch.complex128 and t.dim() == 2 and t.stride(1) == 1
    na, nb = int(a.shape[0]), int(b.shape[0])
    lda = int(a.stride(0)) if na > 1 else int(a.shape[1])
    ldb = int(b.stride(0)) if nb > 1 else int(b.shape[1])
    ldo = int(out.stride(0)) if na > 1 else int(out.shape[1])
    _check(load_library().qe_hpsi_overlap_static(_vp(a.data_ptr()), lda, na, _vp(b.data_ptr()), ldb, nb, int(npw),
                                                 _vp(out.data_ptr()), ldo, _stream_ptr(stream)))
    return out


def qe_hpsi_probe_fp64(millis=200.0):
    """(qe_hpsi_test.h) (DMMA TFLOP/s, DFMA TFLOP/s) measured on the current device."""
    lib = load_library()
    a, b = _c.c_double(0), _c.c_double(0)
    _check(lib.qe_hpsi_probe_fp64(float(millis), _c.byref(a), _c.byref(b)))
    return a.value, b.value


class Hpsi:
    """One handle = one (cell, k, cutoff, grid, V(r), projectors, D). See include/qe_hpsi.h for the contract."""

    def __init__(self, at, ecutwfc, xk, nr, vr: torch.Tensor, beta: torch.Tensor | None = None, blk_off=None,
                 dblocks=None, max_batch: int = 128, flags: int = 0, stream=None):
        lib = load_library()
        self._lib = lib
        self._h = _vp(None)
        assert vr.is_cuda and vr.dtype == torch.float64 and vr.is_contiguous()
        assert tuple(vr.shape) == tuple(int(x) for x in nr)
        _a, pa = _darr(at, 9)
        _k, pk = _darr(xk, 3)
        _n, pn = _iarr(nr, 3)
        nproj = 0 if beta is None else int(beta.shape[0])
        if nproj:
            assert beta.is_cuda and beta.dtype == torch.complex128 and beta.stride(1) == 1
            ldbeta = int(beta.stride(0)) if beta.shape[0] > 1 else int(beta.shape[1])
            blk = np.ascontiguousarray(np.asarray(blk_off, dtype=np.int32))
            dpk = np.ascontiguousarray(np.concatenate([np.asarray(d, dtype=np.float64).reshape(-1) for d in dblocks]))
            pb, nblocks = blk.ctypes.data_as(_pi32), blk.size - 1
            pdk = dpk.ctypes.data_as(_pd)
            bptr = _vp(beta.data_ptr())
        else:
            ldbeta, pb, nblocks, pdk, bptr = 0, None, 0, None, _vp(None)
        self._keep = (vr, beta) if (flags & QE_HPSI_BORROW_BETA) else None
        rc = lib.qe_hpsi_create(_c.byref(self._h), pa, float(ecutwfc), pk, pn, _vp(vr.data_ptr()), nproj, bptr,
                                ldbeta, nblocks, pb, pdk, int(max_batch), int(flags), _stream_ptr(stream))
        _check(rc)
        self.npw = int(lib.qe_hpsi_npw(self._h))
        self.nproj = nproj
        self.max_batch = int(max_batch)

    # -- hot path ----------------------------------------------------------------------------------------
    def _call(self, fn, psi, hpsi, stream):
        assert psi.is_cuda and psi.dtype == torch.complex128 and psi.dim() == 2 and psi.stride(1) == 1
        nb = int(psi.shape[0])
        if hpsi is None:
            hpsi = torch.zeros_like(psi)
        assert hpsi.is_cuda and hpsi.dtype == torch.complex128 and hpsi.shape[0] == nb and hpsi.stride(1) == 1
        ldp = int(psi.stride(0)) if nb > 1 else int(psi.shape[1])
        ldh = int(hpsi.stride(0)) if nb > 1 else int(hpsi.shape[1])
        _check(fn(self._h, _vp(psi.data_ptr()), ldp, _vp(hpsi.data_ptr()), ldh, nb, _stream_ptr(stream)), self._h)
        return hpsi

    def apply(self, psi, hpsi=None, stream=None):
        """qe_hpsi_apply: hpsi[b][:npw] = H psi[b] (asynchronous on `stream`)."""
        return self._call(self._lib.qe_hpsi_apply, psi, hpsi, stream)

    def fft_local(self, psi, hpsi=None, stream=None):
        return self._call(self._lib.qe_hpsi_fft_local, psi, hpsi, stream)

    def nonlocal_add(self, psi, hpsi, stream=None):
        return self._call(self._lib.qe_hpsi_nonlocal, psi, hpsi, stream)

    def apply_host(self, psi_host: torch.Tensor, hpsi_host: torch.Tensor):
        """qe_hpsi_apply_host: host (pinned) buffers, copies inside the call, synchronous."""
        assert (not psi_host.is_cuda) and (not hpsi_host.is_cuda)
        assert psi_host.dtype == torch.complex128 and hpsi_host.dtype == torch.complex128
        nb = int(psi_host.shape[0])
        ldp = int(psi_host.stride(0)) if nb > 1 else int(psi_host.shape[1])
        ldh = int(hpsi_host.stride(0)) if nb > 1 else int(hpsi_host.shape[1])
        _check(self._lib.qe_hpsi_apply_host(self._h, _vp(psi_host.data_ptr()), ldp, _vp(hpsi_host.data_ptr()), ldh, nb),
               self._h)
        return hpsi_host

    # -- rows marked "next" in SURVEY.md 8(f) ------------------------------------------------------------
    def set_s(self, qblocks):
        """qe_hpsi_set_s: per-atom real symmetric q blocks of the overlap operator (same packing as D)."""
        qpk = np.ascontiguousarray(np.concatenate([np.asarray(q, dtype=np.float64).reshape(-1) for q in qblocks])) \
            if self.nproj else np.zeros(1)
        self._nq = qpk.size
        _check(self._lib.qe_hpsi_set_s(self._h, qpk.ctypes.data_as(_pd)), self._h)

    def apply_hs(self, psi, hpsi=None, spsi=None, stream=None, want_h=True):
        """qe_hpsi_apply_hs: (H psi, S psi) with becp shared; want_h=False computes S psi only (returns (None, spsi))."""
        assert psi.is_cuda and psi.dtype == torch.complex128 and psi.dim() == 2 and psi.stride(1) == 1
        nb = int(psi.shape[0])
        if spsi is None:
            spsi = torch.zeros_like(psi)
        if want_h and hpsi is None:
            hpsi = torch.zeros_like(psi)
        ld = lambda t: int(t.stride(0)) if nb > 1 else int(t.shape[1])
        hp = _vp(hpsi.data_ptr()) if want_h else _vp(None)
        _check(self._lib.qe_hpsi_apply_hs(self._h, _vp(psi.data_ptr()), ld(psi), hp, ld(hpsi) if want_h else 0,
                                          _vp(spsi.data_ptr()), ld(spsi), nb, _stream_ptr(stream)), self._h)
        return (hpsi if want_h else None), spsi

    def overlap(self, a, b, out=None, stream=None):
        """qe_hpsi_overlap: out[i][j] = <a_i|b_j> over the npw sphere entries; a [na, ld], b [nb, ld] complex128."""
        for t in (a, b):
            assert t.is_cuda and t.dtype == torch.complex128 and t.dim() == 2 and t.stride(1) == 1
        na, nb = int(a.shape[0]), int(b.shape[0])
        if out is None:
            out = torch.zeros((na, nb), dtype=torch.complex128, device=a.device)
        assert out.is_cuda and out.dtype == torch.complex128 and out.stride(1) == 1
        lda = int(a.stride(0)) if na > 1 else int(a.shape[1])
        ldb = int(b.stride(0)) if nb > 1 else int(b.shape[1])
        ldo = int(out.stride(0)) if na > 1 else int(out.shape[1])
        _check(self._lib.qe_hpsi_overlap(self._h, _vp(a.data_ptr()), lda, na, _vp(b.data_ptr()), ldb, nb,
                                         _vp(out.data_ptr()), ldo, _stream_ptr(stream)), self._h)
        return out

    def hdiag(self, vbar, want_s=False, stream=None):
        """qe_hpsi_hdiag: (hdiag, sdiag or None) as CUDA float64 [npw] tensors."""
        dev = torch.device("cuda", torch.cuda.current_device())
        hd = torch.empty(self.npw, dtype=torch.float64, device=dev)
        sd = torch.empty(self.npw, dtype=torch.float64, device=dev) if want_s else None
        _check(self._lib.qe_hpsi_hdiag(self._h, float(vbar), _vp(hd.data_ptr()), _vp(sd.data_ptr()) if want_s else _vp(None),
                                       _stream_ptr(stream)), self._h)
        return hd, sd

    def precond(self, r, e, hdiag, sdiag=None, stream=None):
        """qe_hpsi_precond: in place on r [nb, ld]; e CUDA float64 [nb]."""
        assert r.is_cuda and r.dtype == torch.complex128 and r.stride(1) == 1 and e.is_cuda and e.dtype == torch.float64
        nb = int(r.shape[0])
        ldr = int(r.stride(0)) if nb > 1 else int(r.shape[1])
        _check(self._lib.qe_hpsi_precond(self._h, _vp(r.data_ptr()), ldr, nb, _vp(e.data_ptr()), _vp(hdiag.data_ptr()),
                                         _vp(sdiag.data_ptr()) if sdiag is not None else _vp(None), _stream_ptr(stream)),
               self._h)
        return r

    def rotate(self, x, coef, y=None, accumulate=False, stream=None):
        """qe_hpsi_rotate: y[k] (+)= sum_j coef[k][j] x[j]; x [nx, ld], coef [ny, nx] complex128 (CUDA)."""
        assert x.is_cuda and x.dtype == torch.complex128 and x.stride(1) == 1
        assert coef.is_cuda and coef.dtype == torch.complex128 and coef.stride(1) == 1 and coef.shape[1] == x.shape[0]
        nx, ny = int(x.shape[0]), int(coef.shape[0])
        if y is None:
            y = torch.zeros((ny, x.shape[1]), dtype=torch.complex128, device=x.device)
        ldx = int(x.stride(0)) if nx > 1 else int(x.shape[1])
        ldc = int(coef.stride(0)) if ny > 1 else int(coef.shape[1])
        ldy = int(y.stride(0)) if ny > 1 else int(y.shape[1])
        _check(self._lib.qe_hpsi_rotate(self._h, _vp(x.data_ptr()), ldx, nx, _vp(coef.data_ptr()), ldc, _vp(y.data_ptr()),
                                        ldy, ny, 1 if accumulate else 0, _stream_ptr(stream)), self._h)
        return y

    def residual(self, hx, sx, e, r=None, want_norm=True, stream=None):
        """qe_hpsi_residual: r = hx - e[b] sx over the sphere entries and rnorm2[b] = |r_b|^2 (CUDA float64 [nb])."""
        nb = int(hx.shape[0])
        for t in (hx, sx):
            assert t.is_cuda and t.dtype == torch.complex128 and t.stride(1) == 1 and t.shape[0] == nb
        assert e.is_cuda and e.dtype == torch.float64 and e.numel() == nb
        if r is None:
            r = torch.zeros_like(hx)
        n2 = torch.empty(nb, dtype=torch.float64, device=hx.device) if want_norm else None
        ld = lambda t: int(t.stride(0)) if nb > 1 else int(t.shape[1])
        _check(self._lib.qe_hpsi_residual(self._h, _vp(hx.data_ptr()), ld(hx), _vp(sx.data_ptr()), ld(sx), _vp(e.data_ptr()),
                                          _vp(r.data_ptr()), ld(r), nb, _vp(n2.data_ptr()) if want_norm else _vp(None),
                                          _stream_ptr(stream)), self._h)
        return r, n2

    def scale(self, x, fac, stream=None):
        """qe_hpsi_scale: x[b] *= fac[b] in place (fac CUDA float64 [nb])."""
        nb = int(x.shape[0])
        assert x.is_cuda and x.dtype == torch.complex128 and x.stride(1) == 1
        assert fac.is_cuda and fac.dtype == torch.float64 and fac.numel() == nb
        ldx = int(x.stride(0)) if nb > 1 else int(x.shape[1])
        _check(self._lib.qe_hpsi_scale(self._h, _vp(x.data_ptr()), ldx, nb, _vp(fac.data_ptr()), _stream_ptr(stream)), self._h)
        return x

    def set_proj_tolerance(self, tol: float):
        """qe_hpsi_set_proj_tolerance (handles created with QE_HPSI_PROJ_INT8 | QE_HPSI_PROJ_CERTIFY)."""
        _check(self._lib.qe_hpsi_set_proj_tolerance(self._h, float(tol)), self._h)

    def proj_check(self, nb):
        """qe_hpsi_get_proj_check: (est_b / |v_b| float64 [nb], redo int32 [nb]) of the last chunk applied (CUDA tensors)."""
        dev = torch.device("cuda", torch.cuda.current_device())
        rel = torch.empty(nb, dtype=torch.float64, device=dev)
        redo = torch.empty(nb, dtype=torch.int32, device=dev)
        _check(self._lib.qe_hpsi_get_proj_check(self._h, _vp(rel.data_ptr()), _vp(redo.data_ptr()), _stream_ptr(None)), self._h)
        return rel, redo

    def density(self, psi, occ, scale, rho, stream=None):
        """qe_hpsi_density: rho[N1,N2,N3] += scale * sum_b occ[b] |psi_b(r)|^2 (rho, occ: CUDA float64 tensors)."""
        assert psi.is_cuda and psi.dtype == torch.complex128 and psi.dim() == 2 and psi.stride(1) == 1
        nb = int(psi.shape[0])
        assert occ.is_cuda and occ.dtype == torch.float64 and occ.numel() == nb and occ.is_contiguous()
        assert rho.is_cuda and rho.dtype == torch.float64 and rho.is_contiguous()
        ldp = int(psi.stride(0)) if nb > 1 else int(psi.shape[1])
        _check(self._lib.qe_hpsi_density(self._h, _vp(psi.data_ptr()), ldp, nb, _vp(occ.data_ptr()), float(scale),
                                         _vp(rho.data_ptr()), _stream_ptr(stream)), self._h)
        return rho

    # -- accessors ---------------------------------------------------------------------------------------
    def maps(self):
        """(miller [npw,3] int32, fft_index [npw] int32, g2kin [npw] float64) as CUDA tensors."""
        dev = torch.device("cuda", torch.cuda.current_device())
        mil = torch.empty((self.npw, 3), dtype=torch.int32, device=dev)
        idx = torch.empty((self.npw,), dtype=torch.int32, device=dev)
        g2 = torch.empty((self.npw,), dtype=torch.float64, device=dev)
        _check(self._lib.qe_hpsi_get_maps(self._h, _vp(mil.data_ptr()), _vp(idx.data_ptr()), _vp(g2.data_ptr()),
                                          _stream_ptr(None)), self._h)
        return mil, idx, g2

    def becp(self, nb):
        """(becp, dbecp) [nproj, nb] complex128 of the last chunk applied (nb must be that chunk's band count)."""
        dev = torch.device("cuda", torch.cuda.current_device())
        a = torch.empty((self.nproj, nb), dtype=torch.complex128, device=dev)
        b = torch.empty((self.nproj, nb), dtype=torch.complex128, device=dev)
        _check(self._lib.qe_hpsi_get_becp(self._h, _vp(a.data_ptr()), _vp(b.data_ptr()), _stream_ptr(None)), self._h)
        return a, b

    def info(self) -> dict:
        buf = (_c.c_int64 * 16)()
        _check(self._lib.qe_hpsi_info(self._h, buf), self._h)
        keys = ["npw", "S", "P", "fft_nb", "nsplit", "workspace_bytes", "npass1", "npass2", "npass3", "kchunk",
                "x_split", "num_sms", "fft2p", "ozaki_slices", "ozaki_nsplit", "ozaki_3m"]
        d = {k: int(buf[i]) for i, k in enumerate(keys)}
        d["gamma_sym"] = (d["fft2p"] >> 1) & 1
        d["x_half"] = (d["fft2p"] >> 2) & 1
        d["fft2p"] &= 1
        d["certify"] = d["ozaki_3m"] >> 2
        d["ozaki_3m"] &= 3
        return d

    PROFILE_SLOTS = ["a6_becp", "a7_reduce_dmul", "a1_a5_fft_chain", "a8_vnl_add", "a1_scatter_zinv", "a2_yinv",
                     "a3_x_vmul", "a4_yfwd", "a5_zfwd_gather", "a6_a8_int8_digits", "certify_check_redo"]

    def profile(self, mode: int):
        """qe_hpsi_profile: 0 off, 1 stage events, 2 per-FFT-kernel events. Resets the accumulators."""
        _check(self._lib.qe_hpsi_profile(self._h, int(mode)), self._h)

    def profile_read(self) -> dict:
        """{slot name: (total ms, spans)} accumulated since the last profile() call (synchronises)."""
        ms = (_c.c_double * 16)()
        cnt = (_c.c_int64 * 16)()
        _check(self._lib.qe_hpsi_profile_read(self._h, ms, cnt), self._h)
        return {n: (float(ms[i]), int(cnt[i])) for i, n in enumerate(self.PROFILE_SLOTS)}

    def check_guards(self) -> int:
        """(qe_hpsi_test.h) number of handle-owned device buffers whose guard band was overwritten (synchronises)."""
        n = int(self._lib.qe_hpsi_test_check_guards(self._h))
        if n < 0:
            _check(n, self._h)
        return n

    def launch_count(self, nbands) -> int:
        return int(self._lib.qe_hpsi_launch_count(self._h, int(nbands)))

    def destroy(self):
        if getattr(self, "_h", None) is not None and self._h.value is not None:
            self._lib.qe_hpsi_destroy(self._h)
            self._h = _vp(None)
        self._keep = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def qe_hpsi_gamma_gsphere(at, ecutwfc, nr) -> np.ndarray:
    """Half sphere of the k = 0 sphere (NEXT-1): int32 [ngw, 3] Miller triples in canonical order, G = 0 first."""
    lib = load_library()
    _a, pa = _darr(at, 9)
    _n, pn = _iarr(nr, 3)
    n = _c.c_int64(0)
    _check(lib.qe_hpsi_gamma_gsphere(pa, float(ecutwfc), pn, _c.byref(n), None))
    mil = np.zeros((max(n.value, 1), 3), dtype=np.int32)
    _check(lib.qe_hpsi_gamma_gsphere(pa, float(ecutwfc), pn, _c.byref(n), mil.ctypes.data_as(_pi32)))
    return mil[:n.value]


class HpsiGamma:
    """Gamma-only handle (k = 0, real wavefunctions on the half sphere). See include/qe_hpsi.h, NEXT-1."""

    def __init__(self, at, ecutwfc, nr, vr: torch.Tensor, beta: torch.Tensor | None = None, blk_off=None, dblocks=None,
                 max_batch: int = 128, flags: int = 0, stream=None):
        lib = load_library()
        self._lib = lib
        self._h = _vp(None)
        assert vr.is_cuda and vr.dtype == torch.float64 and vr.is_contiguous()
        _a, pa = _darr(at, 9)
        _n, pn = _iarr(nr, 3)
        nproj = 0 if beta is None else int(beta.shape[0])
        if nproj:
            assert beta.is_cuda and beta.dtype == torch.complex128 and beta.stride(1) == 1
            ldbeta = int(beta.stride(0)) if beta.shape[0] > 1 else int(beta.shape[1])
            blk = np.ascontiguousarray(np.asarray(blk_off, dtype=np.int32))
            dpk = np.ascontiguousarray(np.concatenate([np.asarray(d, dtype=np.float64).reshape(-1) for d in dblocks]))
            pb, nblocks, pdk, bptr = blk.ctypes.data_as(_pi32), blk.size - 1, dpk.ctypes.data_as(_pd), _vp(beta.data_ptr())
        else:
            ldbeta, pb, nblocks, pdk, bptr = 0, None, 0, None, _vp(None)
        self._keep = (vr, beta) if (flags & QE_HPSI_BORROW_BETA) else None
        _check(lib.qe_hpsi_gamma_create(_c.byref(self._h), pa, float(ecutwfc), pn, _vp(vr.data_ptr()), nproj, bptr, ldbeta,
                                        nblocks, pb, pdk, int(max_batch), int(flags), _stream_ptr(stream)))
        self.ngw = int(lib.qe_hpsi_gamma_ngw(self._h))
        self.nproj = nproj

    def apply(self, psi, hpsi=None, stream=None):
        assert psi.is_cuda and psi.dtype == torch.complex128 and psi.dim() == 2 and psi.stride(1) == 1
        nb = int(psi.shape[0])
        if hpsi is None:
            hpsi = torch.zeros_like(psi)
        ldp = int(psi.stride(0)) if nb > 1 else int(psi.shape[1])
        ldh = int(hpsi.stride(0)) if nb > 1 else int(hpsi.shape[1])
        _check(self._lib.qe_hpsi_gamma_apply(self._h, _vp(psi.data_ptr()), ldp, _vp(hpsi.data_ptr()), ldh, nb,
                                             _stream_ptr(stream)))
        return hpsi

    def destroy(self):
        if getattr(self, "_h", None) is not None and self._h.value is not None:
            self._lib.qe_hpsi_gamma_destroy(self._h)
            self._h = _vp(None)
        self._keep = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass
