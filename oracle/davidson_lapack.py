"""Block Davidson of DESIGN.md §3 with LIBRARY PRIMITIVES as its steps.  TEST INFRASTRUCTURE, NOT THE PRODUCT.

Why a second statement of the same listing: the plain-loop `kso_davidson` of oracle/kso.cpp (serial MGS, serial cyclic
Jacobi, full Hc and full rotation recomputed every iteration) needs ~a day of CPU time for the largest config (cfg 3:
520 bands, npw 124 289, subspace 1040).  SURVEY.md §8(d)(4) allows the ONE-OFF full-size reference solve to take a
cheaper route, because converged eigenpairs do not depend on the route (reading C10): a larger subspace, guard bands,
LAPACK instead of Jacobi.  Its iteration and band-application counts are therefore NOT comparable with the GPU's and
are stored only as a record.

What is a library call here (each "may serve as a step"): `numpy.linalg.qr` (orthonormalise), `@` (zgemm: projections
V^H T, V^H W, rotations C^T V), `numpy.linalg.eigh` (subspace problem).  H psi is the oracle's own `kso_hpsi`
(Eq. 32, Eq. 4) -- nothing under paper_2501_08697_b200/ is imported or called.

Listing (numbers = DESIGN.md §3 steps; PAPER.md names the method at L326, L547, L578 and prints no listing):
  0  X <- qr(psi0)                                              nb = nconv + guard vectors
  1  W <- H X ; Hc <- X^H W ; (Theta, C) <- eigh(Hc) ; X <- X C ; HX <- W C ; V <- X ; W <- HX
  2  R_i <- HX_i - eps_i X_i ; rho_i <- ||R_i|| ; stop when rho_i <= tol for every i < nconv
     U <- {i < nb : rho_i > tol}   (guard bands are corrected too, they are only not waited for)
  3  T_i <- K_i R_i, K = Teter-Payne-Allan polynomial (reading C11), x = g2 / max(Ekin_i, 1e-3)
  4  restart V <- X, W <- HX when m + |U| > max_sub_factor * nb
  5  T <- (I - V V^H) T ; T <- qr(T), dropping a column whose |R_jj| < 1e-10 of its norm before ; both twice
  6  V <- [V, T] ; W <- [W, H T]
  7  Hc <- V^H W (only the new columns are computed; the rest is the previous Hc) ; eigh ; rotate

Pins (tests/test_oracle_pins.py): eigenvalues equal numpy.linalg.eigvalsh of the explicit H on cfg 0 and the shrunk
variants, with and without guard bands, and equal `kso_davidson`'s.
"""
from __future__ import annotations

import time

import numpy as np


def _tpa(g2: np.ndarray, ekin: np.ndarray) -> np.ndarray:
    """K_i(G) of step 3, [nu][npw]."""
    x = g2[None, :] / np.maximum(ekin, 1e-3)[:, None]
    n = 27.0 + 18.0 * x + 12.0 * x * x + 8.0 * x * x * x
    return n / (n + 16.0 * x * x * x * x)


def _orth_against(V: np.ndarray, Vc: np.ndarray, T: np.ndarray) -> np.ndarray:
    """T <- T - V (V^H T) for row-stored vectors: rows of V are the basis, Vc = conj(V)."""
    if V.shape[0] == 0:
        return T
    return T - (Vc @ T.T).T @ V


def _qr_rows(T: np.ndarray, ref: np.ndarray, rel: float):
    """Orthonormalise the rows of T (Householder QR of T^T); drop row j if |R_jj| < rel * ref_j.  Returns (Q rows, kept)."""
    keep = np.arange(T.shape[0])
    while True:
        q, r = np.linalg.qr(T[keep].T)
        ok = np.abs(np.diag(r)) >= rel * ref[keep]
        if ok.all():
            return np.ascontiguousarray(q.T), keep
        keep = keep[ok]
        if keep.size == 0:
            return np.zeros((0, T.shape[1]), dtype=T.dtype), keep


def davidson_lapack(o, g2, psi0, nconv=None, tol=1e-8, max_iter=400, max_sub_factor=2, log=None):
    """o: oracle.kso.Oracle (its hpsi is used); g2[npw] = |k+G|^2 (Ry); psi0[nb][npw] start block.
    Converges the lowest `nconv` (default nb) pairs to residual 2-norm <= tol; the other nb - nconv are guard bands."""
    psi0 = np.asarray(psi0, dtype=np.complex128)
    nb, npw = psi0.shape
    nconv = nb if nconv is None else int(nconv)
    assert 1 <= nconv <= nb <= npw and max_sub_factor >= 2
    mmax = max_sub_factor * nb
    t00 = time.time()
    # step 0
    X, kept = _qr_rows(psi0, np.linalg.norm(psi0, axis=1), 1e-10)
    if kept.size != nb:
        raise ValueError("start block is rank deficient")
    # step 1
    V = np.empty((mmax, npw), dtype=np.complex128)
    W = np.empty((mmax, npw), dtype=np.complex128)
    HXw = o.hpsi(X)
    nh = nb
    Hc = X.conj() @ HXw.T
    Hc = 0.5 * (Hc + Hc.conj().T)
    th, Cm = np.linalg.eigh(Hc)
    V[:nb] = Cm.T @ X
    W[:nb] = Cm.T @ HXw
    X = V[:nb].copy()
    HX = W[:nb].copy()
    eps = th.copy()
    m = nb
    Hc = np.diag(eps).astype(np.complex128)
    it = 0
    status = 1
    while True:
        # step 2
        R = HX - eps[:, None] * X
        rho = np.linalg.norm(R, axis=1)
        if log:
            log("it %d m %d nh %d unconverged(all/target) %d/%d max rho target %.3e  t %.0f s" % (
                it, m, nh, int((rho > tol).sum()), int((rho[:nconv] > tol).sum()), rho[:nconv].max(), time.time() - t00))
        if not (rho[:nconv] > tol).any():
            status = 0
            break
        if it >= max_iter:
            break
        U = np.nonzero(rho > tol)[0]
        # step 3
        ekin = (g2[None, :] * (X[U].real ** 2 + X[U].imag ** 2)).sum(axis=1)
        T = _tpa(g2, ekin) * R[U]
        tn0 = np.linalg.norm(T, axis=1)
        del R
        # step 4
        if m + U.size > mmax:
            V[:nb] = X
            W[:nb] = HX
            m = nb
            Hc = np.diag(eps).astype(np.complex128)
        # step 5
        Vm = V[:m]
        Vc = Vm.conj()
        for _ in range(2):
            T = _orth_against(Vm, Vc, T)
            T, kept = _qr_rows(T, tn0, 1e-10)
            tn0 = np.ones(T.shape[0])
            if T.shape[0] == 0:
                break
        nu = T.shape[0]
        if nu == 0:
            break
        # step 6
        HT = o.hpsi(T)
        nh += nu
        V[m:m + nu] = T
        W[m:m + nu] = HT
        # step 7: new columns of Hc = V^H W
        Hn = np.zeros((m + nu, m + nu), dtype=np.complex128)
        Hn[:m, :m] = Hc
        Hn[:m, m:] = Vc @ HT.T
        Hn[m:, m:] = T.conj() @ HT.T
        Hn[m:, :m] = Hn[:m, m:].conj().T
        m += nu
        Hc = 0.5 * (Hn + Hn.conj().T)
        del Vc
        th, Cm = np.linalg.eigh(Hc)
        Cn = np.ascontiguousarray(Cm[:, :nb].T)
        X = Cn @ V[:m]
        HX = Cn @ W[:m]
        eps = th[:nb].copy()
        it += 1
    return dict(psi=X[:nconv], eig=eps[:nconv], resid=rho[:nconv], iters=it, nhpsi=nh, converged=(status == 0),
                eig_guard=eps[nconv:], resid_guard=rho[nconv:])
