"""Thin Python binding of libkspw.so (include/kspw.h): argument marshalling only -- every step of the
hot path runs in the CUDA kernels of csrc/.  torch is used for device buffers and streams.

There is no CPU fallback: importing this module raises if libkspw.so has not been built
(`python -m paper_2501_08697_b200.build` or `__graft_entry__.build()`); ks_create fails without a GPU.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libkspw.so")
if not os.path.exists(LIB_PATH):
    raise ImportError("libkspw.so is missing (%s): build it with `python -m paper_2501_08697_b200.build`; "
                      "there is no CPU fallback" % LIB_PATH)
_lib = C.CDLL(LIB_PATH)

_vp, _i, _d, _l = C.c_void_p, C.c_int, C.c_double, C.c_long
_lib.ks_pw_count.argtypes = [_vp, _vp, _d, _vp]
_lib.ks_pw_list.argtypes = [_vp, _vp, _d, _vp, _vp]
_lib.ks_create.argtypes = [C.POINTER(_vp), _vp, _vp, _d, _vp, _vp, _i, _vp, _i, _vp, _vp]
_lib.ks_destroy.argtypes = [_vp]
_lib.ks_destroy.restype = None
_lib.ks_npw.argtypes = [_vp]
_lib.ks_set_stream.argtypes = [_vp, _vp]
_lib.ks_set_fft_batch.argtypes = [_vp, _i]
_lib.ks_last_error.argtypes = [_vp]
_lib.ks_last_error.restype = C.c_char_p
_lib.ks_supported_sizes.argtypes = [_vp, _i]
_lib.ks_hpsi.argtypes = [_vp, _vp, _vp, _i]
_lib.ks_hpsi_host.argtypes = [_vp, _vp, _vp, _i]
_lib.ks_hpsi_batch.argtypes = [_vp, _i, _vp, _vp, _vp]
_lib.ks_davidson_batch.argtypes = [_vp, _i, _vp, _vp, _vp, _d, _i, _vp, _vp, _vp, _vp]
_lib.ks_density.argtypes = [_vp, _vp, _vp, _i, _vp]
_lib.ks_density_host.argtypes = [_vp, _vp, _vp, _i, _vp]
_lib.ks_set_overlap.argtypes = [_vp, _vp]
_lib.ks_spsi.argtypes = [_vp, _vp, _vp, _i]
_lib.ks_cg.argtypes = [_vp, _vp, _vp, _i, _d, _i, _vp, _vp, _vp]
_lib.ks_chebyshev.argtypes = [_vp, _vp, _vp, _i, _i, _vp, _d, _d]
_lib.ks_davidson.argtypes = [_vp, _vp, _vp, _i, _d, _i, _vp, _vp, _vp]
_lib.ks_davidson_host.argtypes = [_vp, _vp, _vp, _i, _d, _i, _vp, _vp, _vp]
_lib.ks_davidson_profile.argtypes = [_vp, _vp]
_lib.ks_profile_begin.argtypes = [_vp]
_lib.ks_profile_end.argtypes = [_vp, _vp, _vp]
_lib.ks_zgemm_hn.argtypes = [_vp, _i, _i, _i, _vp, _l, _vp, _l, _vp, _l]
_lib.ks_zgemm_hn_static.argtypes = [_vp, _i, _i, _i, _vp, _l, _vp, _l, _vp, _l]
_lib.ks_zgemm_nn.argtypes = [_vp, _i, _i, _i, _vp, _l, _vp, _l, _vp, _l, _i]
_lib.ks_eigh.argtypes = [_vp, _i, _vp, _l, _vp, _vp, _l, _vp]
_lib.ks_dmma_peak.argtypes = [_vp, _vp]
_lib.ks_dmma_latency.argtypes = [_vp, _d]
_lib.ks_fp64_mix_peak.argtypes = [_vp]

KS_OK, KS_NOTCONV = 0, 1
EXPORTS = ("ks_pw_count", "ks_pw_list", "ks_create", "ks_destroy", "ks_npw", "ks_set_stream", "ks_set_fft_batch",
           "ks_last_error", "ks_supported_sizes", "ks_hpsi", "ks_hpsi_host", "ks_hpsi_batch", "ks_davidson_batch", "ks_density", "ks_density_host", "ks_chebyshev", "ks_cg", "ks_set_overlap", "ks_spsi", "ks_davidson", "ks_davidson_host",
           "ks_davidson_profile", "ks_profile_begin", "ks_profile_end", "ks_zgemm_hn", "ks_zgemm_hn_static", "ks_zgemm_nn", "ks_eigh", "ks_dmma_peak", "ks_dmma_latency", "ks_fp64_mix_peak")


class KsError(RuntimeError):
    def __init__(self, rc, msg):
        super().__init__("kspw error %d: %s" % (rc, msg))
        self.rc = rc


def _np(a, dt):
    return np.ascontiguousarray(a, dtype=dt)


def _hp(a):
    return a.ctypes.data_as(_vp) if a is not None else None


def _glob_err():
    return (_lib.ks_last_error(None) or b"").decode()


def ks_pw_count(cell, k_frac, ecutwfc) -> int:
    cell, k = _np(cell, np.float64), _np(k_frac, np.float64)
    n = _i(0)
    rc = _lib.ks_pw_count(_hp(cell), _hp(k), float(ecutwfc), C.byref(n))
    if rc:
        raise KsError(rc, "ks_pw_count")
    return n.value


def ks_pw_list(cell, k_frac, ecutwfc):
    cell, k = _np(cell, np.float64), _np(k_frac, np.float64)
    n = ks_pw_count(cell, k, ecutwfc)
    mil = np.zeros((n, 3), dtype=np.int32)
    g2 = np.zeros(n, dtype=np.float64)
    rc = _lib.ks_pw_list(_hp(cell), _hp(k), float(ecutwfc), _hp(mil), _hp(g2))
    if rc:
        raise KsError(rc, "ks_pw_list")
    return mil, g2


def ks_supported_sizes():
    buf = np.zeros(64, dtype=np.int32)
    n = _lib.ks_supported_sizes(_hp(buf), 64)
    return [int(x) for x in buf[:n]]


def _dev(t, dtype=None):
    import torch
    assert t.is_cuda and t.is_contiguous(), "device buffers must be contiguous CUDA tensors"
    if dtype is not None:
        assert t.dtype == dtype
    return _vp(t.data_ptr())


class Context:
    """ks_ctx*: one k-point.  Methods are the C calls with the same names minus the `ks_` prefix."""

    def __init__(self, cell, k_frac, ecutwfc, grid, vloc_g, beta=None, proj_offset=None, D=None):
        self._h = _vp()
        cell, k = _np(cell, np.float64), _np(k_frac, np.float64)
        grid = _np(grid, np.int32)
        v = _np(vloc_g, np.complex128)
        assert v.shape == tuple(int(x) for x in grid)
        nproj = 0 if beta is None else int(beta.shape[0])
        if nproj:
            beta, off, D = _np(beta, np.complex128), _np(proj_offset, np.int32), _np(D, np.float64)
            natom = off.shape[0] - 1
        else:
            beta = off = D = None
            natom = 0
        rc = _lib.ks_create(C.byref(self._h), _hp(cell), _hp(k), float(ecutwfc), _hp(grid), _hp(v), nproj,
                            _hp(beta), natom, _hp(off), _hp(D))
        if rc:
            raise KsError(rc, _glob_err())
        self.npw = int(_lib.ks_npw(self._h))
        self.nproj = nproj
        self.grid = tuple(int(x) for x in grid)

    @classmethod
    def from_problem(cls, p):
        return cls(p.cell, p.k_frac, p.ecutwfc, p.grid, p.vloc_g,
                   p.beta if p.nproj else None, p.proj_offset, p.D)

    def _check(self, rc):
        if rc < 0:
            raise KsError(rc, (_lib.ks_last_error(self._h) or b"").decode())
        return rc

    def close(self):
        if self._h:
            _lib.ks_destroy(self._h)
            self._h = _vp()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_stream(self, stream=None):
        """stream: torch.cuda.Stream or None (legacy default stream)."""
        self._check(_lib.ks_set_stream(self._h, _vp(stream.cuda_stream) if stream is not None else None))

    def set_fft_batch(self, n: int):
        self._check(_lib.ks_set_fft_batch(self._h, int(n)))

    def hpsi(self, psi, out=None):
        """psi: torch complex128 CUDA tensor [nbands][npw]; returns H psi (same shape)."""
        import torch
        assert psi.dtype == torch.complex128 and psi.dim() == 2 and psi.shape[1] == self.npw
        if out is None:
            out = torch.empty_like(psi)
        self._check(_lib.ks_hpsi(self._h, _dev(psi), _dev(out), int(psi.shape[0])))
        return out

    def density(self, psi, occ, out=None):
        """psi: torch complex128 CUDA [nbands][npw], occ: torch float64 CUDA [nbands]; returns rho [n1][n2][n3]."""
        import torch
        assert psi.dtype == torch.complex128 and psi.dim() == 2 and psi.shape[1] == self.npw
        assert occ.dtype == torch.float64 and occ.shape == (psi.shape[0],)
        if out is None:
            out = torch.empty(tuple(self.grid), dtype=torch.float64, device=psi.device)
        self._check(_lib.ks_density(self._h, _dev(psi), _dev(occ), int(psi.shape[0]), _dev(out)))
        return out

    def chebyshev(self, chi, coef, ebar: float, de: float, out=None):
        """sum_n coef[n] T_n((H - ebar)/de) chi; chi: torch complex128 CUDA [nbands][npw], coef: host floats."""
        import torch
        assert chi.dtype == torch.complex128 and chi.dim() == 2 and chi.shape[1] == self.npw
        coef = _np(coef, np.float64)
        if out is None:
            out = torch.empty_like(chi)
        self._check(_lib.ks_chebyshev(self._h, _dev(chi), _dev(out), int(chi.shape[0]), int(coef.size), _hp(coef),
                                      float(ebar), float(de)))
        return out

    def density_host(self, psi: np.ndarray, occ: np.ndarray) -> np.ndarray:
        psi = _np(psi, np.complex128)
        occ = _np(occ, np.float64)
        assert psi.ndim == 2 and psi.shape[1] == self.npw and occ.shape == (psi.shape[0],)
        out = np.empty(tuple(self.grid), dtype=np.float64)
        self._check(_lib.ks_density_host(self._h, _hp(psi), _hp(occ), int(psi.shape[0]), _hp(out)))
        return out

    def hpsi_host(self, psi: np.ndarray, out: np.ndarray = None) -> np.ndarray:
        psi = _np(psi, np.complex128)
        assert psi.ndim == 2 and psi.shape[1] == self.npw
        if out is None:
            out = np.empty_like(psi)
        self._check(_lib.ks_hpsi_host(self._h, _hp(psi), _hp(out), int(psi.shape[0])))
        return out

    def davidson(self, psi, tol=1e-8, max_iter=400):
        """psi: torch complex128 CUDA [nbands][npw], overwritten with the eigenvectors.
        Returns dict(eig, resid (device tensors), iters, band_applications, converged)."""
        import torch
        assert psi.dtype == torch.complex128 and psi.dim() == 2 and psi.shape[1] == self.npw
        nb = int(psi.shape[0])
        eig = torch.empty(nb, dtype=torch.float64, device=psi.device)
        res = torch.empty(nb, dtype=torch.float64, device=psi.device)
        it, nh = _i(0), C.c_longlong(0)
        rc = self._check(_lib.ks_davidson(self._h, _dev(psi), _dev(eig), nb, float(tol), int(max_iter), _dev(res),
                                          C.byref(it), C.byref(nh)))
        return dict(psi=psi, eig=eig, resid=res, iters=it.value, band_applications=nh.value, converged=(rc == 0))

    def set_overlap(self, Q):
        """S = 1 + sum_a beta_a q^a beta_a^H (Q: concatenated per-atom real symmetric blocks, layout of D); None: S = I."""
        Q = None if Q is None else _np(Q, np.float64)
        self._check(_lib.ks_set_overlap(self._h, _hp(Q)))

    def spsi(self, psi, out=None):
        import torch
        assert psi.dtype == torch.complex128 and psi.dim() == 2 and psi.shape[1] == self.npw
        if out is None:
            out = torch.empty_like(psi)
        self._check(_lib.ks_spsi(self._h, _dev(psi), _dev(out), int(psi.shape[0])))
        return out

    def cg(self, psi, tol=1e-8, kmaxiter=200):
        """Band-by-band preconditioned CG (Fig. 10).  psi: torch complex128 CUDA [nbands][npw], overwritten.
        Returns dict(eig, resid (device tensors), steps, band_applications, converged)."""
        import torch
        assert psi.dtype == torch.complex128 and psi.dim() == 2 and psi.shape[1] == self.npw
        nb = int(psi.shape[0])
        eig = torch.empty(nb, dtype=torch.float64, device=psi.device)
        res = torch.empty(nb, dtype=torch.float64, device=psi.device)
        it, nh = _i(0), C.c_longlong(0)
        rc = self._check(_lib.ks_cg(self._h, _dev(psi), _dev(eig), nb, float(tol), int(kmaxiter), _dev(res),
                                    C.byref(it), C.byref(nh)))
        return dict(psi=psi, eig=eig, resid=res, steps=it.value, band_applications=nh.value, converged=(rc == 0))

    def davidson_host(self, psi0: np.ndarray, tol=1e-8, max_iter=400):
        psi = np.array(psi0, dtype=np.complex128, order="C")
        nb = psi.shape[0]
        eig, res = np.zeros(nb), np.zeros(nb)
        it, nh = _i(0), C.c_longlong(0)
        rc = self._check(_lib.ks_davidson_host(self._h, _hp(psi), _hp(eig), nb, float(tol), int(max_iter), _hp(res),
                                               C.byref(it), C.byref(nh)))
        return dict(psi=psi, eig=eig, resid=res, iters=it.value, band_applications=nh.value, converged=(rc == 0))

    KERNELS = ("k_inv_yz", "k_x", "k_fwd_yz", "k_gemm_hn+reduce", "k_apply_D", "k_gemm_nn", "k_inv_yz+k_rho")

    def profile_begin(self):
        self._check(_lib.ks_profile_begin(self._h))

    def profile_end(self):
        """Returns {kernel: (ms, launches)} accumulated since profile_begin (synchronises)."""
        ms = np.zeros(8)
        n = np.zeros(8, dtype=np.int64)
        self._check(_lib.ks_profile_end(self._h, _hp(ms), _hp(n)))
        return {k: (float(ms[i]), int(n[i])) for i, k in enumerate(self.KERNELS)}

    def davidson_profile(self):
        ms = np.zeros(8)
        self._check(_lib.ks_davidson_profile(self._h, _hp(ms)))
        keys = ("hpsi", "proj_gemm", "eigh", "rot_gemm", "resid_precond", "orth_gemm", "total")
        return {k: float(ms[i]) for i, k in enumerate(keys)}


def _ptr_array(tensors):
    return (_vp * len(tensors))(*[t.data_ptr() if t is not None and t.numel() else None for t in tensors])


def hpsi_batch(ctxs, psis, outs=None):
    """ks_hpsi_batch: ctxs[i].hpsi(psis[i]) for every k-point in one call (work goes to ctxs[0]'s stream)."""
    import torch
    nk = len(ctxs)
    assert len(psis) == nk
    if outs is None:
        outs = [torch.empty_like(t) for t in psis]
    for c, t, o in zip(ctxs, psis, outs):
        assert t.is_cuda and t.is_contiguous() and t.dtype == torch.complex128 and t.shape[1] == c.npw
        assert o.is_cuda and o.is_contiguous() and o.dtype == torch.complex128 and o.shape == t.shape
    if nk == 0:
        return outs
    h = (_vp * nk)(*[c._h for c in ctxs])
    nb = np.array([t.shape[0] for t in psis], dtype=np.int32)
    rc = _lib.ks_hpsi_batch(h, nk, _ptr_array(psis), _ptr_array(outs), _hp(nb))
    if rc < 0:
        raise KsError(rc, (_lib.ks_last_error(ctxs[0]._h) or b"").decode())
    return outs


def davidson_batch(ctxs, psis, tol=1e-8, max_iter=400):
    """ks_davidson_batch: psis[i] is overwritten with the eigenvectors of k-point i.  Returns a list of dicts as
    Context.davidson does."""
    import torch
    nk = len(ctxs)
    assert len(psis) == nk and nk > 0
    eig = [torch.empty(t.shape[0], dtype=torch.float64, device=t.device) for t in psis]
    res = [torch.empty(t.shape[0], dtype=torch.float64, device=t.device) for t in psis]
    for c, t in zip(ctxs, psis):
        assert t.is_cuda and t.is_contiguous() and t.dtype == torch.complex128 and t.shape[1] == c.npw
    h = (_vp * nk)(*[c._h for c in ctxs])
    nb = np.array([t.shape[0] for t in psis], dtype=np.int32)
    its = np.zeros(nk, dtype=np.int32)
    nh = np.zeros(nk, dtype=np.int64)
    st = np.zeros(nk, dtype=np.int32)
    rc = _lib.ks_davidson_batch(h, nk, _ptr_array(psis), _ptr_array(eig), _hp(nb), float(tol), int(max_iter), _ptr_array(res),
                                _hp(its), _hp(nh), _hp(st))
    if rc < 0:
        raise KsError(rc, (_lib.ks_last_error(ctxs[0]._h) or b"").decode())
    return [dict(psi=psis[i], eig=eig[i], resid=res[i], iters=int(its[i]), band_applications=int(nh[i]),
                 converged=(st[i] == KS_OK)) for i in range(nk)]


def _stream_ptr(stream):
    return _vp(stream.cuda_stream) if stream is not None else None


def ks_zgemm_hn(A, B, stream=None):
    """C = A^H B.  A: torch complex128 CUDA [M][K] (row i = column i of the K x M column-major operand),
    B: [N][K].  Returns C as [N][M] (row n = column n of the column-major M x N result)."""
    import torch
    M, K = A.shape
    N = B.shape[0]
    Cm = torch.empty((N, M), dtype=torch.complex128, device=A.device)
    rc = _lib.ks_zgemm_hn(_stream_ptr(stream), M, N, K, _dev(A), K, _dev(B), K, _dev(Cm), M)
    if rc:
        raise KsError(rc, _glob_err())
    return Cm


def ks_zgemm_hn_static(A, B, out, stream=None):
    """ks_zgemm_hn with the split-K partials in the library's static 8 MiB device array: the call allocates nothing, so the
    caller passes the result buffer too.  A: [M][K], B: [N][K], out: [N][M] (complex128 CUDA, contiguous).  M * N <= 524 288."""
    M, K = A.shape
    N = B.shape[0]
    assert out.shape == (N, M) and out.is_contiguous()
    rc = _lib.ks_zgemm_hn_static(_stream_ptr(stream), M, N, K, _dev(A), K, _dev(B), K, _dev(out), M)
    if rc:
        raise KsError(rc, _glob_err())
    return out


def ks_zgemm_nn(A, B, Cm=None, accumulate=False, stream=None):
    """C (+)= A B in column-major terms.  A: [K][M] (row k = column k of the M x K operand), B: [N][K],
    C: [N][M]."""
    import torch
    K, M = A.shape
    N = B.shape[0]
    if Cm is None:
        assert not accumulate
        Cm = torch.empty((N, M), dtype=torch.complex128, device=A.device)
    rc = _lib.ks_zgemm_nn(_stream_ptr(stream), M, N, K, _dev(A), M, _dev(B), K, _dev(Cm), M, 1 if accumulate else 0)
    if rc:
        raise KsError(rc, _glob_err())
    return Cm


def ks_eigh(A, stream=None):
    """A: torch complex128 CUDA [n][n] Hermitian.  Returns (theta[n] ascending, Cm[n][n] with ROW i the
    eigenvector of theta[i] in column-major terms, i.e. Cm[i, :] = v_i), sweeps."""
    import torch
    n = A.shape[0]
    work = A.clone().contiguous()
    th = torch.empty(n, dtype=torch.float64, device=A.device)
    Cm = torch.empty((n, n), dtype=torch.complex128, device=A.device)
    sw = _i(0)
    rc = _lib.ks_eigh(_stream_ptr(stream), n, _dev(work), n, _dev(th), _dev(Cm), n, C.byref(sw))
    if rc:
        raise KsError(rc, _glob_err())
    return th, Cm, sw.value


def ks_dmma_latency(sm_ghz=1.965):
    """clocks per DMMA of one warp per sub-partition with 1, 2, 3, 4, 6, 8 independent accumulators"""
    out = np.zeros(6)
    rc = _lib.ks_dmma_latency(_hp(out), float(sm_ghz))
    if rc:
        raise KsError(rc, _glob_err())
    return dict(zip((1, 2, 3, 4, 6, 8), (float(x) for x in out)))


def ks_fp64_mix_peak():
    """summed TFLOP/s of register-resident loops: DMMA only, DFMA only, one warp of each per sub-partition, both interleaved"""
    out = np.zeros(4)
    rc = _lib.ks_fp64_mix_peak(_hp(out))
    if rc:
        raise KsError(rc, _glob_err())
    return dict(zip(("dmma", "dfma", "split_warps", "interleaved"), (float(x) for x in out)))


def ks_dmma_peak():
    a, b = _d(0), _d(0)
    rc = _lib.ks_dmma_peak(C.byref(a), C.byref(b))
    if rc:
        raise KsError(rc, _glob_err())
    return a.value, b.value
