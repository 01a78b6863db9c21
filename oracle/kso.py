"""ctypes loader for the CPU oracle (oracle/kso.cpp).  TEST INFRASTRUCTURE, NOT THE PRODUCT:
only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs import it.
It imports nothing from paper_2501_08697_b200 (the CUDA path) and vice versa."""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "kso.cpp")
_LIB = os.path.join(_HERE, "libkso.so")


def build(force: bool = False) -> str:
    """g++ -O2 -fopenmp -shared; rebuilt when the source is newer than the library."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp%d" % os.getpid()
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-fopenmp", "-fPIC", "-shared", "-o", tmp, _SRC])
        os.replace(tmp, _LIB)
    return _LIB


_lib = None
_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int)
_vp = C.c_void_p


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.kso_create.argtypes = [C.POINTER(_vp), _vp, _vp, C.c_double, _vp, _vp, C.c_int, _vp, C.c_int, _vp, _vp]
        _lib.kso_destroy.argtypes = [_vp]
        _lib.kso_destroy.restype = None
        _lib.kso_npw.argtypes = [_vp]
        _lib.kso_get_vr.argtypes = [_vp, _vp]
        _lib.kso_hpsi.argtypes = [_vp, _vp, _vp, C.c_int]
        _lib.kso_explicit_h.argtypes = [_vp, _vp]
        _lib.kso_density.argtypes = [_vp, _vp, _vp, C.c_int, _vp]
        _lib.kso_cg.argtypes = [_vp, _vp, _vp, C.c_int, C.c_double, C.c_int, _vp, _vp, _vp]
        _lib.kso_set_overlap.argtypes = [_vp, _vp]
        _lib.kso_spsi.argtypes = [_vp, _vp, _vp, C.c_int]
        _lib.kso_explicit_s.argtypes = [_vp, _vp]
        _lib.kso_davidson_s.argtypes = [_vp, _vp, _vp, C.c_int, C.c_double, C.c_int, _vp, _vp, _vp]
        _lib.kso_chebyshev.argtypes = [_vp, _vp, C.c_int, C.c_int, _vp, C.c_double, C.c_double, _vp]
        _lib.kso_jacobi.argtypes = [C.c_int, _vp, _vp, _vp]
        _lib.kso_fft3d.argtypes = [C.c_int, C.c_int, C.c_int, _vp, C.c_int]
        _lib.kso_pw_count.argtypes = [_vp, _vp, C.c_double, _vp]
        _lib.kso_pw_list.argtypes = [_vp, _vp, C.c_double, _vp, _vp]
        _lib.kso_davidson.argtypes = [_vp, _vp, _vp, C.c_int, C.c_double, C.c_int, _vp, _vp, _vp, _vp, C.c_int]
    return _lib


def _p(a):
    return a.ctypes.data_as(_vp) if a is not None else None


def num_threads() -> int:
    return int(lib().kso_num_threads())


def fft3d(a: np.ndarray, sign: int) -> np.ndarray:
    a = np.array(a, dtype=np.complex128, order="C")
    assert a.ndim == 3
    rc = lib().kso_fft3d(a.shape[0], a.shape[1], a.shape[2], _p(a), sign)
    assert rc == 0
    return a


def pw_list(cell, k_frac, ecutwfc):
    cell = np.ascontiguousarray(cell, dtype=np.float64)
    k = np.ascontiguousarray(k_frac, dtype=np.float64)
    n = C.c_int(0)
    lib().kso_pw_count(_p(cell), _p(k), float(ecutwfc), C.byref(n))
    mil = np.zeros((n.value, 3), dtype=np.int32)
    g2 = np.zeros(n.value, dtype=np.float64)
    lib().kso_pw_list(_p(cell), _p(k), float(ecutwfc), _p(mil), _p(g2))
    return mil, g2


def jacobi(A: np.ndarray):
    A = np.array(A, dtype=np.complex128, order="C")
    n = A.shape[0]
    th = np.zeros(n)
    Cm = np.zeros((n, n), dtype=np.complex128)
    sweeps = lib().kso_jacobi(n, _p(A), _p(th), _p(Cm))
    return th, Cm, sweeps


class Oracle:
    """One k-point (same shapes as the product's ks_* calls, host pointers)."""

    def __init__(self, cell, k_frac, ecutwfc, grid, vloc_g, beta=None, proj_offset=None, D=None):
        self._h = _vp()
        cell = np.ascontiguousarray(cell, dtype=np.float64)
        k = np.ascontiguousarray(k_frac, dtype=np.float64)
        grid = np.ascontiguousarray(grid, dtype=np.int32)
        v = np.ascontiguousarray(vloc_g, dtype=np.complex128)
        assert v.shape == tuple(int(x) for x in grid)
        nproj = 0 if beta is None else int(beta.shape[0])
        if nproj:
            beta = np.ascontiguousarray(beta, dtype=np.complex128)
            off = np.ascontiguousarray(proj_offset, dtype=np.int32)
            D = np.ascontiguousarray(D, dtype=np.float64)
            natom = off.shape[0] - 1
        else:
            beta = off = D = None
            natom = 0
        rc = lib().kso_create(C.byref(self._h), _p(cell), _p(k), float(ecutwfc), _p(grid), _p(v), nproj,
                              _p(beta), natom, _p(off), _p(D))
        if rc != 0:
            raise RuntimeError("kso_create failed rc=%d" % rc)
        self.npw = int(lib().kso_npw(self._h))
        self.grid = tuple(int(x) for x in grid)
        if nproj:
            assert beta.shape[1] == self.npw

    @classmethod
    def from_problem(cls, p):
        return cls(p.cell, p.k_frac, p.ecutwfc, p.grid, p.vloc_g,
                   p.beta if p.nproj else None, p.proj_offset, p.D)

    def close(self):
        if self._h:
            lib().kso_destroy(self._h)
            self._h = _vp()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def vr(self) -> np.ndarray:
        out = np.zeros(self.grid, dtype=np.float64)
        lib().kso_get_vr(self._h, _p(out))
        return out

    def hpsi(self, psi: np.ndarray) -> np.ndarray:
        psi = np.ascontiguousarray(psi, dtype=np.complex128)
        assert psi.ndim == 2 and psi.shape[1] == self.npw
        out = np.empty_like(psi)
        rc = lib().kso_hpsi(self._h, _p(psi), _p(out), psi.shape[0])
        assert rc == 0
        return out

    def density(self, psi: np.ndarray, occ: np.ndarray) -> np.ndarray:
        """rho[n1][n2][n3] = sum_b occ_b |psi_b(r)|^2 (unnormalised inverse transform, Eq. 31)."""
        psi = np.ascontiguousarray(psi, dtype=np.complex128)
        occ = np.ascontiguousarray(occ, dtype=np.float64)
        assert psi.ndim == 2 and psi.shape[1] == self.npw and occ.shape == (psi.shape[0],)
        out = np.empty(self.grid, dtype=np.float64)
        rc = lib().kso_density(self._h, _p(psi), _p(occ), psi.shape[0], _p(out))
        assert rc == 0
        return out

    def chebyshev(self, chi: np.ndarray, coef: np.ndarray, ebar: float, de: float) -> np.ndarray:
        """sum_n coef[n] T_n((H - ebar)/de) chi for a block chi[nb][npw] (three-term recurrence)."""
        chi = np.ascontiguousarray(chi, dtype=np.complex128)
        coef = np.ascontiguousarray(coef, dtype=np.float64)
        assert chi.ndim == 2 and chi.shape[1] == self.npw and de > 0
        out = np.empty_like(chi)
        rc = lib().kso_chebyshev(self._h, _p(chi), chi.shape[0], coef.size, _p(coef), float(ebar), float(de), _p(out))
        assert rc == 0
        return out

    def cg(self, psi0, tol=1e-8, kmaxiter=200):
        """Band-by-band preconditioned CG (Fig. 10).  Returns dict(eig, psi, resid, steps, band_applications, converged)."""
        psi = np.array(psi0, dtype=np.complex128, order="C")
        nb = psi.shape[0]
        eig = np.zeros(nb); res = np.zeros(nb)
        steps = C.c_int(0); nh = C.c_longlong(0)
        rc = lib().kso_cg(self._h, _p(psi), _p(eig), nb, float(tol), int(kmaxiter), _p(res), C.byref(steps), C.byref(nh))
        assert rc >= 0, rc
        return dict(eig=eig, psi=psi, resid=res, steps=steps.value, band_applications=nh.value, converged=(rc == 0))

    def set_overlap(self, Q: np.ndarray):
        """S = 1 + sum_a beta_a q^a beta_a^H; Q: concatenated per-atom real symmetric blocks (layout of D)."""
        Q = np.ascontiguousarray(Q, dtype=np.float64)
        assert lib().kso_set_overlap(self._h, _p(Q)) == 0

    def spsi(self, psi: np.ndarray) -> np.ndarray:
        psi = np.ascontiguousarray(psi, dtype=np.complex128)
        out = np.empty_like(psi)
        assert lib().kso_spsi(self._h, _p(psi), _p(out), psi.shape[0]) == 0
        return out

    def explicit_s(self) -> np.ndarray:
        S = np.empty((self.npw, self.npw), dtype=np.complex128)
        lib().kso_explicit_s(self._h, _p(S))
        return S

    def davidson_s(self, psi0, tol=1e-8, max_iter=400):
        psi = np.array(psi0, dtype=np.complex128, order="C")
        nb = psi.shape[0]
        eig = np.zeros(nb); res = np.zeros(nb)
        it = C.c_int(0); nh = C.c_longlong(0)
        rc = lib().kso_davidson_s(self._h, _p(psi), _p(eig), nb, float(tol), int(max_iter), _p(res), C.byref(it), C.byref(nh))
        assert rc >= 0, rc
        return dict(eig=eig, psi=psi, resid=res, iters=it.value, band_applications=nh.value, converged=(rc == 0))

    def explicit_h(self) -> np.ndarray:
        H = np.empty((self.npw, self.npw), dtype=np.complex128)
        lib().kso_explicit_h(self._h, _p(H))
        return H

    def davidson(self, psi0, tol=1e-8, max_iter=400, max_sub_factor=2, history=False):
        psi = np.array(psi0, dtype=np.complex128, order="C")
        nb = psi.shape[0]
        eig = np.zeros(nb)
        res = np.zeros(nb)
        it = C.c_int(0)
        nh = C.c_longlong(0)
        hist = np.full((max_iter + 1, nb), np.nan) if history else None
        rc = lib().kso_davidson(self._h, _p(psi), _p(eig), nb, float(tol), int(max_iter), _p(res),
                                C.byref(it), C.byref(nh), _p(hist), int(max_sub_factor))
        if rc < 0:
            raise RuntimeError("kso_davidson failed rc=%d" % rc)
        out = dict(psi=psi, eig=eig, resid=res, iters=it.value, nhpsi=nh.value, converged=(rc == 0))
        if history:
            out["ritz_hist"] = hist[: it.value + 1]
        return out
