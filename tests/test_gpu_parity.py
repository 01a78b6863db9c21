"""GPU parity tests (run on the B200 box): the CUDA path through the C ABI (libkspw.so via the thin
binding) against the CPU oracle on the same seeded inputs.  Tolerances are north_star's:
H psi relative Frobenius error <= 1e-11, |d eps| <= 1e-8 Ry, Davidson residual norms <= 1e-8."""
import numpy as np
import pytest

from paper_2501_08697_b200 import inputs as I

pytestmark = pytest.mark.gpu

HPSI_TOL = 1e-11


@pytest.fixture(scope="module")
def ks():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2501_08697_b200 import kspw
    return kspw


def _t(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _rel(a, b):
    return np.linalg.norm(a - b) / np.linalg.norm(b)


# ------------------------------------------------------------------ building blocks (T1)
@pytest.mark.parametrize("M,N,K", [(8, 8, 515), (160, 37, 1503), (70, 130, 4099), (1, 1, 1), (64, 64, 16), (5, 3, 0),
                                   (512, 1, 37073), (23, 2, 4099), (64, 3, 1503), (7, 4, 8459),
                                   (70, 200, 4099), (33, 520, 2050), (9, 163, 1503),    # N > 160: whole 160-wide tiles + a remainder launch
                                   (1728, 40, 4099), (100, 13, 4099), (64, 24, 2050), (27, 100, 1503), (70, 182, 2050), (9, 41, 515),
                                   (65, 8, 300), (130, 33, 1000)])                      # N <= 40: 8*NJ-wide tiles; ragged tails of 1..24 columns
def test_zgemm_hn(ks, M, N, K):
    rng = np.random.default_rng(M * 1000 + N)
    A = rng.standard_normal((M, K)) + 1j * rng.standard_normal((M, K))
    B = rng.standard_normal((N, K)) + 1j * rng.standard_normal((N, K))
    Cm = ks.ks_zgemm_hn(_t(A), _t(B)).cpu().numpy()            # [N][M]
    ref = (A.conj() @ B.T).T                                     # C[m][n] = sum_k conj(A[m][k]) B[n][k]
    assert np.abs(Cm - ref).max() <= 1e-13 * max(1, K) ** 0.5 * (np.abs(ref).max() + 1)


@pytest.mark.parametrize("M,N,K,acc", [(515, 8, 8, True), (1503, 23, 512, True), (4099, 70, 130, False), (1, 1, 1, False), (130, 65, 17, True),
                                       (37073, 1, 512, True), (4099, 2, 64, False), (1503, 3, 1728, True), (8459, 4, 1, True),
                                       (4099, 40, 130, False), (1503, 13, 512, True), (2050, 520, 64, True), (515, 100, 33, False),
                                       (130, 72, 40, True), (700, 5, 1040, False), (257, 41, 17, True)])   # narrow (8*NJ) tiles and ragged tails
def test_zgemm_nn(ks, M, N, K, acc):
    rng = np.random.default_rng(M + N + K)
    A = rng.standard_normal((K, M)) + 1j * rng.standard_normal((K, M))
    B = rng.standard_normal((N, K)) + 1j * rng.standard_normal((N, K))
    C0 = rng.standard_normal((N, M)) + 1j * rng.standard_normal((N, M))
    Ct = _t(C0)
    ks.ks_zgemm_nn(_t(A), _t(B), Ct, accumulate=acc)
    ref = B @ A + (C0 if acc else 0)
    assert np.abs(Ct.cpu().numpy() - ref).max() <= 1e-13 * max(1, K) ** 0.5 * (np.abs(ref).max() + 1)


@pytest.mark.parametrize("n", [1, 2, 7, 16, 33, 64, 65, 100, 320, 497, 513, 700, 1040])
def test_eigh_vs_oracle_jacobi(ks, oracle_mod, n):
    rng = np.random.default_rng(n)
    A = rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n))
    A = A + A.conj().T
    if n == 7:
        A[:, 3] = A[:, 2]; A[3, :] = A[2, :]; A[3, 3] = A[2, 2]
    th, Cm, sweeps = ks.ks_eigh(_t(A.T.copy()))                 # column-major view of A
    th = th.cpu().numpy()
    V = Cm.cpu().numpy().T                                       # columns = eigenvectors
    if n <= 100:
        tho, _, _ = oracle_mod.jacobi(A)
    else:      # the oracle's cyclic Jacobi is O(n^3) per sweep on one core; above n = 100 LAPACK is the reference
        tho = np.linalg.eigvalsh(A)   # (n >= 512 takes the one-launch-per-round path, 497 pads to 512)
    scale = np.abs(A).max() * n
    assert np.abs(th - tho).max() < 1e-13 * scale
    assert np.abs(A @ V - V * th).max() < 1e-12 * scale
    assert np.abs(V.conj().T @ V - np.eye(n)).max() < 1e-12
    assert (np.diff(th) >= 0).all()


def test_eigh_near_diagonal_and_clusters(ks):
    rng = np.random.default_rng(3)
    n = 200
    d = np.sort(rng.standard_normal(n))
    d[50:60] = d[50]                                             # a 10-fold cluster
    Q, _ = np.linalg.qr(rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n)))
    A = (Q * d) @ Q.conj().T
    A = 0.5 * (A + A.conj().T)
    th, Cm, _ = ks.ks_eigh(_t(A.T.copy()))
    V = Cm.cpu().numpy().T
    # block Jacobi updates every diagonal entry ~n times per sweep: error ~ n * sweeps * eps * |a|
    assert np.abs(th.cpu().numpy() - d).max() < 1e-11
    assert np.abs(V.conj().T @ V - np.eye(n)).max() < 1e-12
    assert np.abs(A @ V - V * th.cpu().numpy()).max() < 1e-11


def test_pw_list_matches_oracle(ks, oracle_mod):
    for c, ik in ((0, 0), (2, 21), (4, 0)):
        cfg = I.config(c)
        m1, g1 = ks.ks_pw_list(cfg.cell, cfg.kpts[ik], cfg.ecutwfc)
        m2, g2 = oracle_mod.pw_list(cfg.cell, cfg.kpts[ik], cfg.ecutwfc)
        assert np.array_equal(m1, m2) and np.array_equal(g1, g2)


# ------------------------------------------------------------------ H psi (T2)
def _hpsi_pair(ks, oracle_mod, p, psi):
    ctx = ks.Context.from_problem(p)
    o = oracle_mod.Oracle.from_problem(p)
    got = ctx.hpsi(_t(psi)).cpu().numpy()
    ref = o.hpsi(psi)
    return got, ref, ctx, o


@pytest.mark.parametrize("name", ["cfg0", "s1", "s2", "s3", "s4", "tiny16", "tiny18"])
def test_hpsi_small(ks, oracle_mod, name):
    if name == "cfg0":
        p = I.make_problem(0)
    elif name == "tiny16":
        p = I.make_problem(0, ecutwfc=4.0, grid=(16, 16, 16), nbands=5)
    elif name == "tiny18":
        p = I.make_problem(0, ecutwfc=5.0, grid=(18, 18, 18), nbands=3)
    else:
        p = I.make_shrunk(name)
    got, ref, ctx, o = _hpsi_pair(ks, oracle_mod, p, p.psi0)
    assert _rel(got, ref) <= HPSI_TOL and _elementwise_ok(got, ref)
    # local + kinetic only and kinetic only (degenerate cases)
    p2 = I.make_problem(p.cfg.index, p.k_index, ecutwfc=p.ecutwfc, grid=tuple(p.grid), nbands=2, with_beta=False)
    got, ref, _, _ = _hpsi_pair(ks, oracle_mod, p2, p2.psi0)
    assert _rel(got, ref) <= HPSI_TOL and _elementwise_ok(got, ref)
    # host-buffer entry point against the device one: the host call cuts the block into chunks (the first one half as long as
    # the others), i.e. another split of the projector sums over K: equal to rounding (bit for bit only where one chunk holds
    # the whole block), as in test_hpsi_host_chunked_pipeline
    h = ctx.hpsi_host(p.psi0)
    dev = ctx.hpsi(_t(p.psi0)).cpu().numpy()
    assert _rel(h, dev) <= 1e-13 and _elementwise_ok(h, dev)


def test_hpsi_edge_cases(ks, oracle_mod):
    import torch
    p = I.make_problem(0)
    ctx = ks.Context.from_problem(p)
    # empty block
    e = torch.empty((0, p.npw), dtype=torch.complex128, device="cuda")
    assert ctx.hpsi(e).shape == (0, p.npw)
    # batch boundaries: nbands not a multiple of the FFT batch, and batch of one
    o = oracle_mod.Oracle.from_problem(p)
    rng = np.random.default_rng(0)
    psi = rng.standard_normal((11, p.npw)) + 1j * rng.standard_normal((11, p.npw))
    ref = o.hpsi(psi)
    for nbatch in (1, 4, 0):
        ctx.set_fft_batch(nbatch)
        assert _rel(ctx.hpsi(_t(psi)).cpu().numpy(), ref) <= HPSI_TOL
    # aliasing is refused
    t = _t(psi)
    with pytest.raises(ks.KsError):
        ctx.hpsi(t, out=t)
    # unsupported / alias-violating grids are refused at create
    with pytest.raises(ks.KsError) as ei:
        ks.Context(p.cell, p.k_frac, p.ecutwfc, (16, 16, 16), np.zeros((16, 16, 16), complex))
    assert ei.value.rc == -2
    with pytest.raises(ks.KsError) as ei:
        v = np.zeros((24, 24, 24), complex); v[1, 0, 0] = 1.0      # V(r) not real
        ks.Context(p.cell, p.k_frac, p.ecutwfc, (24, 24, 24), v)
    assert ei.value.rc == -5
    # a non-default stream
    s = torch.cuda.Stream()
    ctx.set_stream(s)
    with torch.cuda.stream(s):
        out = ctx.hpsi(_t(psi))
    s.synchronize()
    assert _rel(out.cpu().numpy(), ref) <= HPSI_TOL


def _elementwise_ok(got, ref):
    """next to every norm-wise comparison: no single element off by more than 1e-12 of the largest one (measured ~1e-15)"""
    return np.abs(got - ref).max() <= 1e-12 * np.abs(ref).max()


def _boundary_bands(nb, batch, bg=8):
    """bands at both ends of every FFT batch (`batch` bands per launch of the three FFT kernels) and at both ends of a
    k_x band group (bg bands walked by one CTA), plus the middle of the block"""
    s = {0, nb - 1, nb // 2, bg - 1, bg}
    for b0 in range(batch, nb, batch):
        s |= {b0 - 1, b0, b0 + bg - 1, b0 + bg}
    return np.array(sorted(i for i in s if 0 <= i < nb))


# bands per launch of the three FFT kernels: by default the whole block (up to 9 GB of live planes); 125 / 110 were round 1's
# defaults for cfg 3 / cfg 4 and are kept as an explicit second run so that batch boundaries stay covered
@pytest.mark.parametrize("c,k_index,batch", [(2, 0, 32), (2, 21, 32), (2, 63, 32), (1, 0, 160), (3, 0, 125), (4, 0, 110)])
def test_hpsi_full_size(ks, oracle_mod, c, k_index, batch):
    """Full-size configs in the launch configuration bench.py times (whole block in one call); the oracle recomputes
    bands one by one (bands are independent in H psi): every band of cfg 2, and for cfg 1 / 3 / 4 the bands on both sides
    of every FFT-batch boundary and at both ends of a k_x band group."""
    p = I.make_problem(c, k_index)
    ctx = ks.Context.from_problem(p)
    got = ctx.hpsi(_t(p.psi0)).cpu().numpy()
    if batch < p.nbands:
        ctx.set_fft_batch(batch)
        got_b = ctx.hpsi(_t(p.psi0)).cpu().numpy()
        # the FFT batches never change a bit of the local part; the projector products see the same block either way
        assert np.array_equal(got, got_b)
    o = oracle_mod.Oracle.from_problem(p)
    sel = np.arange(p.nbands) if c == 2 else _boundary_bands(p.nbands, batch)
    ref = o.hpsi(p.psi0[sel])
    assert _rel(got[sel], ref) <= HPSI_TOL
    assert _elementwise_ok(got[sel], ref)
    for i, b in enumerate(sel):                     # band by band too: a wrong band cannot hide in the block norm
        assert _rel(got[b], ref[i]) <= HPSI_TOL
    # property at any size: Hermiticity <phi|H psi> = conj <psi|H phi> over the whole block
    G = p.psi0.conj() @ got.T
    assert np.abs(G - G.conj().T).max() <= 1e-11 * np.abs(G).max()


@pytest.mark.parametrize("c,ecut,n,beta", [(0, 4.0, 20, True), (0, 25.0, 40, True), (0, 60.0, 60, True),
                                           (1, 25.0, 80, False), (1, 40.0, 100, False), (3, 30.0, 120, False)])
def test_hpsi_radix5_grids(ks, oracle_mod, c, ecut, n, beta):
    """Grids with a factor 5 (20, 40, 60, 80, 100, 120): radix-5 codelets in all three kernels, plus the density."""
    p = I.make_problem(c, ecutwfc=ecut, grid=(n, n, n), nbands=3, with_beta=beta)
    ctx = ks.Context.from_problem(p)
    o = oracle_mod.Oracle.from_problem(p)
    got, ref = ctx.hpsi(_t(p.psi0)).cpu().numpy(), o.hpsi(p.psi0)
    assert _rel(got, ref) <= HPSI_TOL and _elementwise_ok(got, ref)
    occ = np.array([2.0, 1.0, 0.5])
    ref = o.density(p.psi0, occ)
    assert np.abs(ctx.density(_t(p.psi0), _t(occ)).cpu().numpy() - ref).max() <= 1e-12 * ref.max()


@pytest.mark.parametrize("c,ecut,grid", [(4, 3.0, (96, 96, 288)), (4, 12.0, (96, 96, 288)), (3, 2.5, (128, 128, 128))])
def test_hpsi_large_planes_small_sphere(ks, oracle_mod, c, ecut, grid):
    """The 96 x 288 planes are split over three CTAs per (band, plane) (forward kernel: a cluster exchanging stick tiles
    through distributed shared memory), the 128 x 128 ones use 512-thread CTAs: small spheres on the full grids leave
    planes with a handful of sticks (fewer work items than threads, ranks of the cluster with little to do) and let the
    oracle check every element of every band."""
    p = I.make_problem(c, ecutwfc=ecut, grid=grid, nbands=3, with_beta=False)
    ctx = ks.Context.from_problem(p)
    o = oracle_mod.Oracle.from_problem(p)
    got, ref = ctx.hpsi(_t(p.psi0)).cpu().numpy(), o.hpsi(p.psi0)
    assert _rel(got, ref) <= HPSI_TOL and _elementwise_ok(got, ref)
    occ = np.array([2.0, 1.0, 0.5])
    ref = o.density(p.psi0, occ)
    assert np.abs(ctx.density(_t(p.psi0), _t(occ)).cpu().numpy() - ref).max() <= 1e-12 * ref.max()


def test_hpsi_full_symmetric_D_blocks(ks, oracle_mod):
    """Per-atom D blocks that are full symmetric matrices of uneven sizes (Eq. 4 L221 allows D_ll' coupling)."""
    p = I.make_problem(0)
    rng = np.random.default_rng(21)
    off = np.array([0, 5, 8], dtype=np.int32)
    D = np.concatenate([(0.5 * (a + a.T)).ravel() for a in (rng.standard_normal((5, 5)), rng.standard_normal((3, 3)))])
    ctx = ks.Context(p.cell, p.k_frac, p.ecutwfc, p.grid, p.vloc_g, p.beta, off, D)
    o = oracle_mod.Oracle(p.cell, p.k_frac, p.ecutwfc, p.grid, p.vloc_g, p.beta, off, D)
    assert _rel(ctx.hpsi(_t(p.psi0)).cpu().numpy(), o.hpsi(p.psi0)) <= HPSI_TOL
    w = np.linalg.eigvalsh(o.explicit_h())
    r = ctx.davidson(_t(p.psi0), tol=1e-8)
    assert r["converged"] and np.abs(r["eig"].cpu().numpy() - w[:p.nbands]).max() <= 1e-8


def test_hpsi_ragged_band_group(ks, oracle_mod):
    """cfg 1 geometry with 31 bands: the x kernel walks over band groups of 2, so the last group is ragged;
    a 7-band FFT batch adds a ragged last batch on top."""
    p = I.make_problem(1)
    ctx = ks.Context.from_problem(p)
    o = oracle_mod.Oracle.from_problem(p)
    psi = np.ascontiguousarray(p.psi0[:31])
    sel = np.array([0, 1, 14, 29, 30])
    ref = o.hpsi(psi[sel])
    got = ctx.hpsi(_t(psi)).cpu().numpy()
    assert _rel(got[sel], ref) <= HPSI_TOL and _elementwise_ok(got[sel], ref)
    ctx.set_fft_batch(7)
    got2 = ctx.hpsi(_t(psi)).cpu().numpy()
    assert np.array_equal(got, got2)          # batching never changes a bit: bands are independent


def test_hpsi_host_chunked_pipeline(ks, oracle_mod):
    """ks_hpsi_host on 300 bands of the cfg 1 geometry: ten chunks of 32 bands with a ragged last one (12 bands) run through
    the copy-in / compute / copy-out pipeline, more chunks than the eight event pairs; against the device-resident call on
    the whole block (another split of the projector products, so equal to rounding, not bit for bit) and the oracle."""
    p = I.make_problem(1)
    ctx = ks.Context.from_problem(p)
    psi = np.ascontiguousarray(np.concatenate([p.psi0, 0.5j * p.psi0[::-1][:140]]))
    assert psi.shape[0] == 300
    dev = ctx.hpsi(_t(psi)).cpu().numpy()
    host = ctx.hpsi_host(psi)
    assert _rel(host, dev) <= 1e-13
    sel = np.array([0, 31, 32, 159, 160, 287, 288, 299])
    ref = oracle_mod.Oracle.from_problem(p).hpsi(psi[sel])
    assert _rel(host[sel], ref) <= HPSI_TOL and _elementwise_ok(host[sel], ref)


# ------------------------------------------------------------------ Davidson (T3)
def _check_davidson(ks, oracle_mod, p, tol=1e-8, exact=None, oracle_run=True):
    ctx = ks.Context.from_problem(p)
    o = oracle_mod.Oracle.from_problem(p)
    r = ctx.davidson(_t(p.psi0), tol=tol)
    assert r["converged"], "GPU Davidson did not converge in %d iterations" % r["iters"]
    eig = r["eig"].cpu().numpy()
    X = r["psi"].cpu().numpy()
    nb = p.nbands
    # residuals re-evaluated with the ORACLE's H psi on the GPU's vectors (reading C14)
    hx = o.hpsi(X)
    res = np.linalg.norm(hx - eig[:, None] * X, axis=1)
    assert res.max() <= 1.05 * tol
    assert np.abs(res - r["resid"].cpu().numpy()).max() <= 1e-10
    assert np.abs(X.conj() @ X.T - np.eye(nb)).max() <= 1e-10
    assert (np.diff(eig) >= -1e-12).all()
    if oracle_run:
        ro = o.davidson(p.psi0, tol=tol)
        assert ro["converged"]
        assert np.abs(eig - ro["eig"]).max() <= 1e-8
    if exact is not None:
        assert np.abs(eig - exact[:nb]).max() <= 1e-8
    return r


def test_davidson_cfg0(ks, oracle_mod):
    p = I.make_problem(0)
    o = oracle_mod.Oracle.from_problem(p)
    w = np.linalg.eigvalsh(o.explicit_h())
    r = _check_davidson(ks, oracle_mod, p, exact=w)
    assert 8 * 2 <= r["band_applications"] <= 400
    # host-buffer entry point
    ctx = ks.Context.from_problem(p)
    rh = ctx.davidson_host(p.psi0)
    assert rh["converged"] and np.abs(rh["eig"] - w[:8]).max() <= 1e-8 and rh["resid"].max() <= 1e-8


def test_davidson_free_electron_and_shift(ks, oracle_mod):
    p = I.make_problem(0, with_beta=False, with_vloc=False)
    ctx = ks.Context.from_problem(p)
    r = ctx.davidson(_t(p.psi0), tol=1e-9)
    eig = r["eig"].cpu().numpy()
    assert r["converged"] and np.abs(eig - np.sort(p.g2)[:8]).max() <= 1e-10      # degenerate shells
    v = np.zeros(p.vloc_g.shape, dtype=np.complex128)
    v[0, 0, 0] = -0.321
    ctx2 = ks.Context(p.cell, p.k_frac, p.ecutwfc, p.grid, v)
    r2 = ctx2.davidson(_t(p.psi0), tol=1e-9)
    assert np.abs(r2["eig"].cpu().numpy() - (eig - 0.321)).max() <= 1e-10


@pytest.mark.parametrize("name", ["s1", "s2", "s3", "s4"])
def test_davidson_shrunk(ks, oracle_mod, name):
    p = I.make_shrunk(name)
    o = oracle_mod.Oracle.from_problem(p)
    w = np.linalg.eigvalsh(o.explicit_h())
    _check_davidson(ks, oracle_mod, p, exact=w, oracle_run=(name in ("s2", "s4")))


def test_davidson_not_converged_status(ks):
    p = I.make_problem(0)
    ctx = ks.Context.from_problem(p)
    r = ctx.davidson(_t(p.psi0), tol=1e-8, max_iter=2)
    assert not r["converged"] and r["iters"] == 2 and r["resid"].cpu().numpy().max() > 1e-8


def test_davidson_cfg2_kpoint(ks, oracle_mod):
    """One k-point of config 2 at full size, against the oracle's own Davidson (about 1 min of CPU)."""
    p = I.make_problem(2, 0)
    r = _check_davidson(ks, oracle_mod, p, oracle_run=True)
    eig = r["eig"].cpu().numpy()
    assert abs(eig[15] - eig[16]) < 1e-8            # degenerate pair; compare values only


# ------------------------------------------------------------------ Davidson edge paths (drop rule, rank deficiency)
def _drop_problem():
    # cfg 0 cell at ecutwfc 1.5 Ry: npw = 27 on the 16^3 grid; 16 bands -> 2 nbands = 32 > npw, so the corrections of the
    # first expansion MUST become linearly dependent (at most 27 - 16 = 11 new directions exist)
    return I.make_problem(0, ecutwfc=1.5, grid=(16, 16, 16), nbands=16)


def test_davidson_drop_rule_forced(ks, oracle_mod):
    """D7's drop rule (DESIGN.md §2 'Drop rule'): with 2 nbands > npw the projected corrections are dependent and both
    sides must drop columns; eigenvalues against LAPACK on the explicit 27 x 27 H and against the oracle's own solve."""
    p = _drop_problem()
    assert p.npw == 27
    o = oracle_mod.Oracle.from_problem(p)
    w = np.linalg.eigvalsh(o.explicit_h())
    ro = o.davidson(p.psi0, tol=1e-8)
    assert ro["converged"] and np.abs(ro["eig"] - w[:16]).max() <= 1e-8
    r = ks.Context.from_problem(p).davidson(_t(p.psi0), tol=1e-8)
    assert r["converged"]
    assert np.abs(r["eig"].cpu().numpy() - w[:16]).max() <= 1e-8
    # a drop happened on both sides: fewer band applications than nbands * (iterations + 1) and never more than npw directions
    assert r["band_applications"] < 16 * (r["iters"] + 1) and ro["nhpsi"] < 16 * (ro["iters"] + 1)
    X = r["psi"].cpu().numpy()
    assert np.abs(X.conj() @ X.T - np.eye(16)).max() <= 1e-10
    res = np.linalg.norm(o.hpsi(X) - r["eig"].cpu().numpy()[:, None] * X, axis=1)
    assert res.max() <= 1.05e-8


def test_davidson_whole_space(ks, oracle_mod):
    """nbands = npw (degenerate): the start block spans the whole space, the initial Rayleigh-Ritz step is exact and no
    correction is ever built: nbands band applications, zero iterations -- as in the oracle."""
    p = I.make_problem(0, ecutwfc=1.5, grid=(16, 16, 16), nbands=27)
    o = oracle_mod.Oracle.from_problem(p)
    w = np.linalg.eigvalsh(o.explicit_h())
    r = ks.Context.from_problem(p).davidson(_t(p.psi0), tol=1e-8)
    assert r["converged"] and r["band_applications"] == 27 and r["iters"] == 0
    assert np.abs(r["eig"].cpu().numpy() - w).max() <= 1e-8


def test_davidson_rank_deficient_start_block(ks):
    p = I.make_problem(0)
    psi = p.psi0.copy()
    psi[5] = 2.0 * psi[1] - 0.5j * psi[3]            # a dependent start vector
    ctx = ks.Context.from_problem(p)
    with pytest.raises(ks.KsError) as ei:
        ctx.davidson(_t(psi), tol=1e-8)
    assert ei.value.rc == -1 and "rank deficient" in str(ei.value)
    # the context is still usable
    r = ctx.davidson(_t(p.psi0), tol=1e-8)
    assert r["converged"]


def test_davidson_single_cta_cholesky_path_in_subprocess():
    """KSPW_CHOL_BLOCKED=0 selects the one-CTA Cholesky (k_chol_drop); the switch is read once per process, so the forced-drop
    problem and the rank-deficient start block run in a child process with it set."""
    import os, subprocess, sys
    code = (
        "import numpy as np, torch\n"
        "from paper_2501_08697_b200 import inputs as I, kspw\n"
        "p = I.make_problem(0, ecutwfc=1.5, grid=(16, 16, 16), nbands=16)\n"
        "r = kspw.Context.from_problem(p).davidson(torch.from_numpy(p.psi0).cuda(), tol=1e-8)\n"
        "assert r['converged'] and r['band_applications'] < 16 * (r['iters'] + 1)\n"
        "np.save(__import__('sys').argv[1], r['eig'].cpu().numpy())\n"
        "p = I.make_problem(0); psi = p.psi0.copy(); psi[5] = psi[1]\n"
        "try:\n"
        "    kspw.Context.from_problem(p).davidson(torch.from_numpy(psi).cuda(), tol=1e-8)\n"
        "    raise SystemExit('no error for a rank-deficient start block')\n"
        "except kspw.KsError as e:\n"
        "    assert e.rc == -1\n")
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    out = os.path.join("/tmp", "kspw_chol_single_%d.npy" % os.getpid())
    env = dict(os.environ, KSPW_CHOL_BLOCKED="0", PYTHONPATH=root)
    subprocess.run([sys.executable, "-c", code, out], check=True, env=env, cwd=root, timeout=600)
    eig = np.load(out)
    os.remove(out)
    p = _drop_problem()
    from oracle import kso
    w = np.linalg.eigvalsh(kso.Oracle.from_problem(p).explicit_h())
    assert np.abs(eig - w[:16]).max() <= 1e-8


def test_two_contexts_same_plane_size_different_spheres(ks, oracle_mod):
    """The yz kernels' dynamic shared memory depends on the context's sticks per plane, the opt-in attribute belongs to the
    kernel: a small-sphere context created AFTER a large-sphere one on the same 96 x 96 planes must not break the first."""
    big = I.make_problem(1, nbands=3)
    ctx_big = ks.Context.from_problem(big)
    small = I.make_problem(1, ecutwfc=6.0, grid=(96, 96, 96), nbands=3)
    ctx_small = ks.Context.from_problem(small)
    for p, ctx in ((big, ctx_big), (small, ctx_small), (big, ctx_big)):
        got = ctx.hpsi(_t(p.psi0)).cpu().numpy()
        ref = oracle_mod.Oracle.from_problem(p).hpsi(p.psi0)
        assert _rel(got, ref) <= HPSI_TOL and _elementwise_ok(got, ref)


# ------------------------------------------------------------------ density build
@pytest.mark.parametrize("name", ["cfg0", "s1", "s2", "s4", "tiny18"])
def test_density_small(ks, oracle_mod, name):
    import torch
    if name == "cfg0":
        p = I.make_problem(0)
    elif name == "tiny18":
        p = I.make_problem(0, ecutwfc=5.0, grid=(18, 18, 18), nbands=3)
    else:
        p = I.make_shrunk(name)
    ctx = ks.Context.from_problem(p)
    o = oracle_mod.Oracle.from_problem(p)
    occ = np.linspace(2.0, 0.25, p.nbands)
    ref = o.density(p.psi0, occ)
    got = ctx.density(_t(p.psi0), _t(occ)).cpu().numpy()
    assert np.abs(got - ref).max() <= 1e-12 * np.abs(ref).max()
    # ragged batches give the same bits (fixed summation order per band group is batch dependent, so compare to 1e-13)
    ctx.set_fft_batch(3)
    got2 = ctx.density(_t(p.psi0), _t(occ)).cpu().numpy()
    assert np.abs(got2 - ref).max() <= 1e-12 * np.abs(ref).max()
    # run to run reproducible bit for bit (no atomics)
    assert np.array_equal(got2, ctx.density(_t(p.psi0), _t(occ)).cpu().numpy())
    # host entry point, empty block
    assert np.abs(ctx.density_host(p.psi0, occ) - ref).max() <= 1e-12 * np.abs(ref).max()
    e = torch.empty((0, p.npw), dtype=torch.complex128, device="cuda")
    z = ctx.density(e, torch.empty(0, dtype=torch.float64, device="cuda")).cpu().numpy()
    assert z.shape == tuple(p.grid) and not z.any()


@pytest.mark.parametrize("c,k_index", [(1, 0), (2, 21), (3, 0), (4, 0)])
def test_density_full_size(ks, oracle_mod, c, k_index):
    """Full-size configs: the oracle sums a few bands; Parseval holds for the whole block at any size."""
    p = I.make_problem(c, k_index)
    ctx = ks.Context.from_problem(p)
    o = oracle_mod.Oracle.from_problem(p)
    sel = np.unique(np.linspace(0, p.nbands - 1, 3).astype(int))
    occ = np.zeros(p.nbands)
    occ[sel] = [2.0, 1.0, 0.5][:len(sel)]
    ref = o.density(p.psi0[sel], occ[sel])
    got = ctx.density(_t(p.psi0), _t(occ)).cpu().numpy()          # whole block, zero weight on the other bands
    assert np.abs(got - ref).max() <= 1e-12 * np.abs(ref).max()
    occ = np.linspace(2.0, 0.0, p.nbands)
    got = ctx.density(_t(p.psi0), _t(occ)).cpu().numpy()
    N = got.size
    want = N * (occ * (np.abs(p.psi0) ** 2).sum(axis=1)).sum()
    assert got.min() >= 0.0 and abs(got.sum() - want) <= 1e-11 * want


# ------------------------------------------------------------------ Chebyshev expansion
def _stochastic(p, nchi, seed):
    rng = np.random.default_rng(seed)
    return np.exp(2j * np.pi * rng.uniform(size=(nchi, p.npw))) / np.sqrt(nchi)      # PAPER.md Eq. 52


@pytest.mark.parametrize("name", ["cfg0", "s2", "s4"])
def test_chebyshev_small(ks, oracle_mod, name):
    import torch
    p = I.make_problem(0) if name == "cfg0" else I.make_shrunk(name)
    ctx = ks.Context.from_problem(p)
    o = oracle_mod.Oracle.from_problem(p)
    w = np.linalg.eigvalsh(o.explicit_h())
    ebar, de = 0.5 * (w[-1] + w[0]), 0.51 * (w[-1] - w[0])
    chi = _stochastic(p, 5, 3)
    mu, kT = 0.3, 1.0
    coef = np.polynomial.chebyshev.chebinterpolate(lambda x: 1.0 / np.sqrt(1.0 + np.exp((x * de + ebar - mu) / kT)), 40)
    ref = o.chebyshev(chi, coef, ebar, de)
    got = ctx.chebyshev(_t(chi), coef, ebar, de).cpu().numpy()
    assert _rel(got, ref) <= 1e-11
    # degenerate orders and argument checks
    for nco in (0, 1, 2):
        assert np.abs(ctx.chebyshev(_t(chi), coef[:nco], ebar, de).cpu().numpy() - o.chebyshev(chi, coef[:nco], ebar, de)).max() <= 1e-13
    t = _t(chi)
    with pytest.raises(ks.KsError):
        ctx.chebyshev(t, coef, ebar, de, out=t)
    with pytest.raises(ks.KsError):
        ctx.chebyshev(t, coef, ebar, 0.0)
    e = torch.empty((0, p.npw), dtype=torch.complex128, device="cuda")
    assert ctx.chebyshev(e, coef, ebar, de).shape == (0, p.npw)


def test_chebyshev_full_size_cfg1(ks, oracle_mod):
    """cfg 1 geometry, 96 stochastic orbitals, order 12: the oracle follows 2 of them; a zero-order
    identity and linearity hold for the whole block."""
    p = I.make_problem(1)
    ctx = ks.Context.from_problem(p)
    o = oracle_mod.Oracle.from_problem(p)
    chi = _stochastic(p, 96, 7)
    ebar, de = 0.5 * (p.ecutwfc + 4.0 - 3.0), 0.5 * (p.ecutwfc + 4.0 + 3.0)      # generous bounds: [-3, ecut + 4] Ry
    coef = 1.0 / (1.0 + np.arange(12.0)) ** 2
    got = ctx.chebyshev(_t(chi), coef, ebar, de).cpu().numpy()
    sel = np.array([0, 95])
    ref = o.chebyshev(chi[sel], coef, ebar, de)
    assert _rel(got[sel], ref) <= 1e-11
    half = ctx.chebyshev(_t(0.5 * chi), coef, ebar, de).cpu().numpy()
    assert _rel(2.0 * half, got) <= 1e-14


# ------------------------------------------------------------------ band-by-band CG (Fig. 10)
def _check_cg(ks, oracle_mod, p, exact, kmaxiter=200, need_conv=True):
    ctx = ks.Context.from_problem(p)
    o = oracle_mod.Oracle.from_problem(p)
    r = ctx.cg(_t(p.psi0), tol=1e-8, kmaxiter=kmaxiter)
    nb = p.nbands
    eig = r["eig"].cpu().numpy()
    X = r["psi"].cpu().numpy()
    if need_conv:
        assert r["converged"]
    assert np.abs(eig - exact[:nb]).max() <= 1e-8
    assert np.abs(X.conj() @ X.T - np.eye(nb)).max() <= 1e-10
    res = np.linalg.norm(o.hpsi(X) - eig[:, None] * X, axis=1)       # re-evaluated with the oracle's H psi
    assert np.abs(res - r["resid"].cpu().numpy()).max() <= 1e-10
    if need_conv:
        assert res.max() <= 1.05e-8
    assert (np.diff(eig) >= -1e-12).all()
    assert r["band_applications"] == r["steps"] + nb
    return r, o


def test_cg_cfg0_vs_oracle_and_bruteforce(ks, oracle_mod):
    p = I.make_problem(0)
    o = oracle_mod.Oracle.from_problem(p)
    w = np.linalg.eigvalsh(o.explicit_h())
    r, _ = _check_cg(ks, oracle_mod, p, w)
    ro = o.cg(p.psi0, tol=1e-8)
    assert np.abs(r["eig"].cpu().numpy() - ro["eig"]).max() <= 1e-8
    assert abs(r["steps"] - ro["steps"]) <= 0.1 * ro["steps"]          # same listing: step counts agree to rounding effects
    # Davidson reaches the same pairs
    d = ks.Context.from_problem(p).davidson(_t(p.psi0), tol=1e-8)
    assert np.abs(d["eig"].cpu().numpy() - r["eig"].cpu().numpy()).max() <= 1e-8


@pytest.mark.parametrize("name", ["s2", "s1", "s4"])
def test_cg_shrunk(ks, oracle_mod, name):
    """k != 0 (s2), a clustered 64-atom spectrum (s1: the oracle needs up to ~1000 steps for one band too) and the
    non-cubic slab grid (s4), against LAPACK on the explicit H."""
    p = I.make_shrunk(name)
    o = oracle_mod.Oracle.from_problem(p)
    w = np.linalg.eigvalsh(o.explicit_h())
    _check_cg(ks, oracle_mod, p, w, kmaxiter=1500)


def test_cg_free_electron_and_not_converged(ks):
    p = I.make_problem(0, with_beta=False, with_vloc=False)
    ctx = ks.Context.from_problem(p)
    r = ctx.cg(_t(p.psi0), tol=1e-9)
    assert r["converged"] and np.abs(r["eig"].cpu().numpy() - np.sort(p.g2)[:8]).max() <= 1e-10
    p = I.make_problem(0)
    ctx = ks.Context.from_problem(p)
    r = ctx.cg(_t(p.psi0), tol=1e-8, kmaxiter=2)
    assert not r["converged"] and r["steps"] == 2 * p.nbands


# ------------------------------------------------------------------ generalised problem
def _overlap_q(p, seed=3):
    rng = np.random.default_rng(seed)
    out = []
    for a in range(len(p.proj_offset) - 1):
        n = int(p.proj_offset[a + 1] - p.proj_offset[a])
        m = rng.standard_normal((n, n))
        out.append((0.3 * np.eye(n) + 0.05 * (m + m.T)).ravel())
    return np.concatenate(out)


@pytest.mark.parametrize("name", ["cfg0", "s2", "s4"])
def test_generalised_davidson(ks, oracle_mod, name):
    """H x = eps S x with S = 1 + sum_a beta_a q^a beta_a^H: S psi against the oracle, eigenvalues against
    scipy.linalg.eigh(H, S) of the explicit matrices, X^H S X = I, residuals ||H x - eps S x|| re-evaluated with the
    oracle's operators; the block ends at a gap of the generalised spectrum."""
    import scipy.linalg
    p = I.make_problem(0) if name == "cfg0" else I.make_shrunk(name)
    Q = _overlap_q(p)
    o = oracle_mod.Oracle.from_problem(p)
    o.set_overlap(Q)
    ctx = ks.Context.from_problem(p)
    ctx.set_overlap(Q)
    assert _rel(ctx.spsi(_t(p.psi0)).cpu().numpy(), o.spsi(p.psi0)) <= 1e-13
    S = o.explicit_s()
    w = scipy.linalg.eigh(o.explicit_h(), S, eigvals_only=True)
    nb = 4 + int(np.argmax(np.diff(w[3:p.nbands + 1])))
    r = ctx.davidson(_t(p.psi0[:nb].copy()), tol=1e-8)
    assert r["converged"]
    eig = r["eig"].cpu().numpy()
    X = r["psi"].cpu().numpy()
    assert np.abs(eig - w[:nb]).max() <= 1e-8
    assert np.abs(X.conj() @ S @ X.T - np.eye(nb)).max() <= 1e-10
    res = np.linalg.norm(o.hpsi(X) - eig[:, None] * o.spsi(X), axis=1)
    assert res.max() <= 1.05e-8 and np.abs(res - r["resid"].cpu().numpy()).max() <= 1e-10
    # S = I again: the standard problem, untouched
    ctx.set_overlap(None)
    o2 = oracle_mod.Oracle.from_problem(p)
    w2 = np.linalg.eigvalsh(o2.explicit_h())
    r2 = ctx.davidson(_t(p.psi0), tol=1e-8)
    assert r2["converged"] and np.abs(r2["eig"].cpu().numpy() - w2[:p.nbands]).max() <= 1e-8


# ------------------------------------------------------------------ full-size Davidson against the survey's worked numbers
def _gold():
    import json, os
    return json.load(open(os.path.join(os.path.dirname(__file__), "golden", "survey_c5.json")))


def test_davidson_cfg1_full_size_vs_survey_values(ks, oracle_mod):
    """cfg 1 at full size (npw 37 073, 160 bands) in the configuration bench.py times.  External pin: the eigenvalues the
    survey's independent numpy prototype printed (SURVEY.md §8(c.5), 8 digits); then what holds at any size: residuals
    re-evaluated with the ORACLE's H psi on all 160 vectors, orthonormality, ascending order."""
    p = I.make_problem(1)
    ctx = ks.Context.from_problem(p)
    r = ctx.davidson(_t(p.psi0), tol=1e-8)
    assert r["converged"]
    eig = r["eig"].cpu().numpy()
    g = _gold()["cfg1"]
    assert np.abs(eig[:4] - np.array(g["eps0_3"])).max() <= 1e-8
    assert np.abs(eig[157:160] - np.array(g["eps157_159"])).max() <= 1e-8
    X = r["psi"].cpu().numpy()
    o = oracle_mod.Oracle.from_problem(p)
    res = np.linalg.norm(o.hpsi(X) - eig[:, None] * X, axis=1)
    assert res.max() <= 1.05e-8 and np.abs(res - r["resid"].cpu().numpy()).max() <= 1e-10
    assert np.abs(X.conj() @ X.T - np.eye(p.nbands)).max() <= 1e-10
    assert (np.diff(eig) >= -1e-12).all()


@pytest.mark.parametrize("key", ["k_m38", "k_m18"])
def test_davidson_cfg2_kpoints_vs_survey_values(ks, key):
    g = _gold()["cfg2"][key]
    p = I.make_problem(2, g["k_index"])
    assert p.npw == g["npw"]
    r = ks.Context.from_problem(p).davidson(_t(p.psi0), tol=1e-8)
    eig = r["eig"].cpu().numpy()
    assert r["converged"]
    for i, name in ((0, "eps0"), (15, "eps15"), (16, "eps16"), (31, "eps31")):
        assert abs(eig[i] - g[name]) <= 1e-8


def _golden(name):
    import json, os
    path = os.path.join(os.path.dirname(__file__), "golden", name)
    return json.load(open(path)) if os.path.exists(path) else None


@pytest.mark.parametrize("c", [4, 3])
def test_davidson_large_configs_all_residuals(ks, oracle_mod, c):
    """cfg 4 (slab, 96x96x288) and cfg 3 (216 atoms, 520 bands, subspace up to 1040: the one-launch-per-round Jacobi
    path) at full size: the solve converges, EVERY eigenpair has residual <= tol under the ORACLE's H psi (one oracle
    block apply of all nbands vectors), the block is orthonormal.  The eigenvalues themselves are compared with the
    oracle's stored solves in test_davidson_vs_stored_oracle_solve / test_davidson_cfg3_lowest_bands_vs_stored_oracle_solve."""
    import torch
    p = I.make_problem(c)
    ctx = ks.Context.from_problem(p)
    r = ctx.davidson(_t(p.psi0), tol=1e-8)
    assert r["converged"]
    eig = r["eig"].cpu().numpy()
    X = r["psi"]
    G = X.conj() @ X.T
    assert float((G - torch.eye(p.nbands, dtype=G.dtype, device=G.device)).abs().max()) <= 1e-10
    assert (np.diff(eig) >= -1e-12).all()
    Xh = X.cpu().numpy()
    o = oracle_mod.Oracle.from_problem(p)
    res = np.linalg.norm(o.hpsi(Xh) - eig[:, None] * Xh, axis=1)
    assert res.max() <= 1.05e-8
    assert np.abs(res - r["resid"].cpu().numpy()).max() <= 1e-10
    if c == 3:
        # the lowest levels of THIS 520-band solve against the oracle's stored solves of the same full-size problem for
        # fewer bands (a converged eigenvalue does not depend on how many bands are solved with it): 27 by kso_davidson,
        # 93 and 123 (shell closures further up) by the library-routed listing with guard bands, whichever files exist
        for name in ("oracle_davidson_cfg3_nb27.json", "oracle_davidson_cfg3_nb93.json", "oracle_davidson_cfg3_nb123.json"):
            g = _golden(name)
            if g is not None:
                assert g["converged"] and g["npw"] == p.npw
                assert np.abs(eig[:g["nbands"]] - np.array(g["eig"])).max() <= 1e-8, name


CFG3_LOW_NB = 27     # the lowest four shells of the 216-atom cell's spectrum (1 + 6 + 12 + 8 levels), gap 0.027 Ry above


def test_davidson_cfg3_lowest_bands_vs_stored_oracle_solve(ks):
    """The FULL-SIZE cfg 3 problem (npw 124 289, 128^3 grid, 1728 projectors) solved for its lowest 27 bands: the
    oracle's own kso_davidson (the listing, subspace <= 2 nbands) stored by tests/golden/make_oracle_davidson.py 3 0 27.
    Same listing and same start block on both sides: all 27 eigenvalues to 1e-8 Ry, counts to 10 %.
    (27 = a shell closure.  The 64 lowest bands VERDICT r1 suggested end inside a 24-fold shell of levels ~1e-4 Ry apart:
    with no gap above the block the listing does not converge -- the device stops at max_iter = 400 with 37 bands open,
    and the oracle, the same listing, cannot do better: BASELINE.md section 6.)"""
    g = _golden("oracle_davidson_cfg3_nb%d.json" % CFG3_LOW_NB)
    if g is None:
        pytest.skip("tests/golden/oracle_davidson_cfg3_nb%d.json has not been generated" % CFG3_LOW_NB)
    p = I.make_problem(3, nbands=CFG3_LOW_NB)
    assert p.npw == g["npw"] and g["nbands"] == CFG3_LOW_NB and g["converged"]
    r = ks.Context.from_problem(p).davidson(_t(p.psi0), tol=1e-8)
    assert r["converged"]
    assert np.abs(r["eig"].cpu().numpy() - np.array(g["eig"])).max() <= 1e-8
    assert abs(r["iters"] - g["iterations"]) <= 0.1 * g["iterations"]
    assert abs(r["band_applications"] - g["band_applications"]) <= 0.1 * g["band_applications"]


def test_davidson_cfg3_block_ending_inside_a_shell_does_not_converge(ks):
    """nbands = 64 on the full-size cfg 3 problem cuts the 24-fold shell of levels 58..81: KS_NOTCONV at max_iter with the
    closed shells below converged and orthonormal vectors -- the documented behaviour of the listing without guard bands."""
    p = I.make_problem(3, nbands=64)
    r = ks.Context.from_problem(p).davidson(_t(p.psi0), tol=1e-8, max_iter=400)
    assert not r["converged"] and r["iters"] == 400
    res = r["resid"].cpu().numpy()
    assert (res[:CFG3_LOW_NB] <= 1e-8).all()          # the closed shells below are done (measured: exactly these 27)
    assert (res[57:] > 1e-6).all()                    # the open shell (levels 58..81) is nowhere near (measured: > 1e-3)
    X = r["psi"]
    import torch
    G = X.conj() @ X.T
    assert float((G - torch.eye(64, dtype=G.dtype, device=G.device)).abs().max()) <= 1e-10
    # and the 27 converged values are the same as those of the 27-band solve's golden file, when it exists
    g = _golden("oracle_davidson_cfg3_nb%d.json" % CFG3_LOW_NB)
    if g is not None:
        assert np.abs(r["eig"].cpu().numpy()[:CFG3_LOW_NB] - np.array(g["eig"])).max() <= 1e-8


@pytest.mark.parametrize("c", [1, 4, 3])
def test_davidson_vs_stored_oracle_solve(ks, c):
    """Full-size configs against the ORACLE's own Davidson solve of the same problem, stored once by
    tests/golden/make_oracle_davidson.py (minutes to hours of CPU time): every eigenvalue within north_star's 1e-8 Ry.
    cfg 1 and cfg 4 were solved by kso_davidson (the listing as it stands: counts comparable); cfg 3's 520 bands by the
    library-routed statement of the same listing (oracle/davidson_lapack.py, guard bands, larger subspace: SURVEY.md
    8(d)(4)) -- converged eigenvalues do not depend on the route, its counts are not compared."""
    g = _golden("oracle_davidson_cfg%d.json" % c)
    if g is None:
        pytest.skip("tests/golden/oracle_davidson_cfg%d.json has not been generated" % c)
    p = I.make_problem(c)
    assert p.npw == g["npw"] and p.nbands == g["nbands"] and g["converged"]
    r = ks.Context.from_problem(p).davidson(_t(p.psi0), tol=1e-8)
    assert r["converged"]
    assert np.abs(r["eig"].cpu().numpy() - np.array(g["eig"])).max() <= 1e-8
    if g.get("route", "listing") == "listing":
        # same listing on both sides: iteration and band-application counts agree to a few per cent
        assert abs(r["iters"] - g["iterations"]) <= 0.1 * g["iterations"]
        assert abs(r["band_applications"] - g["band_applications"]) <= 0.1 * g["band_applications"]


# ------------------------------------------------------------------ cfg 2: all 64 k-points
CFG2_STORED_K = (0, 1, 5, 21, 26, 37, 42, 63)      # two k-points from each of the four |k| shells of the 4x4x4 mesh


def test_davidson_cfg2_all_kpoints_time_reversal_and_stored_oracle_solves(ks):
    """Every k-point of the Monkhorst-Pack mesh: the mesh is inversion symmetric, k_{63-i} = -k_i, and
    H(-k) = conj(H(k)) for a real local potential and the real-harmonic projectors, so eps(k_i) = eps(k_{63-i}) band by
    band (time reversal) -- a pin that needs no oracle run.  Eight k-points (two per |k| shell) are
    compared with the oracle's stored kso_davidson solves (tests/golden/oracle_davidson_cfg2_k<i>.json)."""
    eig = []
    for k in range(64):
        p = I.make_problem(2, k)
        ctx = ks.Context.from_problem(p)
        r = ctx.davidson(_t(p.psi0), tol=1e-8)
        assert r["converged"], "k-point %d" % k
        eig.append(r["eig"].cpu().numpy())
        del ctx
    eig = np.array(eig)
    kp = np.array(I.config(2).kpts)
    for i in range(32):
        assert np.allclose(kp[i], -kp[63 - i])
        assert np.abs(eig[i] - eig[63 - i]).max() <= 1e-8, "time reversal broken at k-point %d" % i
    seen = 0
    for k in CFG2_STORED_K:
        g = _golden("oracle_davidson_cfg2_k%d.json" % k)
        if g is None:
            continue
        seen += 1
        assert g["converged"] and g["k_index"] == k
        assert np.abs(eig[k] - np.array(g["eig"])).max() <= 1e-8, "k-point %d vs the oracle's solve" % k
    assert seen >= 1, "no stored oracle solve of a cfg 2 k-point found under tests/golden/"


# ------------------------------------------------------------------ batched multi-k entry points
def test_hpsi_batch_all_64_kpoints_of_cfg2(ks, oracle_mod):
    """ks_hpsi_batch over the whole 4x4x4 Monkhorst-Pack mesh of cfg 2 (Eq. 32 L507 per k): every element of
    every band of every k-point against the oracle's H psi, and against 64 single ks_hpsi calls."""
    ps = [I.make_problem(2, k) for k in range(64)]
    ctxs = [ks.Context.from_problem(p) for p in ps]
    psis = [_t(p.psi0) for p in ps]
    outs = ks.hpsi_batch(ctxs, psis)
    for k, (p, ctx) in enumerate(zip(ps, ctxs)):
        got = outs[k].cpu().numpy()
        ref = oracle_mod.Oracle.from_problem(p).hpsi(p.psi0)
        assert _rel(got, ref) <= HPSI_TOL and _elementwise_ok(got, ref), "k-point %d" % k
        one = ctx.hpsi(psis[k]).cpu().numpy()
        assert _rel(got, one) <= 1e-13, "k-point %d vs the single-k call" % k
    # the call is repeatable bit for bit (fixed summation orders, no atomics)
    again = ks.hpsi_batch(ctxs, psis)
    assert all(bool((a == b).all()) for a, b in zip(outs, again))


def test_hpsi_batch_ragged_and_edge_cases(ks, oracle_mod):
    import torch
    ps = [I.make_problem(2, k, nbands=nb) for k, nb in ((0, 5), (21, 32), (42, 1), (63, 17))]
    ctxs = [ks.Context.from_problem(p) for p in ps]
    psis = [_t(p.psi0) for p in ps]
    # ragged band counts, one empty entry, a group size that does not divide the batch, band slabs smaller than a block
    p5 = I.make_problem(2, 5, nbands=3)
    ctxs.append(ks.Context.from_problem(p5))
    ps.append(p5)
    psis.append(torch.empty((0, ctxs[4].npw), dtype=torch.complex128, device="cuda"))
    for ctx in ctxs:
        ctx.set_fft_batch(7)
    outs = ks.hpsi_batch(ctxs, psis)
    for k in range(4):
        ref = oracle_mod.Oracle.from_problem(ps[k]).hpsi(ps[k].psi0)
        got = outs[k].cpu().numpy()
        assert _rel(got, ref) <= HPSI_TOL and _elementwise_ok(got, ref)
    assert outs[4].shape[0] == 0
    assert ks.hpsi_batch([], []) == []
    # no projectors, local + kinetic only: bit-identical to the single-k path (same kernels' arithmetic, no GEMM)
    q = [I.make_problem(2, k, nbands=4, with_beta=False) for k in (3, 60)]
    cq = [ks.Context.from_problem(p) for p in q]
    tq = [_t(p.psi0) for p in q]
    oq = ks.hpsi_batch(cq, tq)
    for c, t, o in zip(cq, tq, oq):
        assert bool((c.hpsi(t) == o).all())
    # refused: a context twice, mixed grids, aliasing
    with pytest.raises(ks.KsError):
        ks.hpsi_batch([ctxs[0], ctxs[0]], [psis[0], psis[0]])
    other = ks.Context.from_problem(I.make_problem(0))
    with pytest.raises(ks.KsError):
        ks.hpsi_batch([ctxs[0], other], [psis[0], _t(I.make_problem(0).psi0)])
    with pytest.raises(ks.KsError):
        ks.hpsi_batch([ctxs[1]], [psis[1]], outs=[psis[1]])


def test_hpsi_batch_large_grid_cluster_path(ks, oracle_mod):
    """Two contexts on the 96 x 96 x 288 slab grid (different small spheres): the k-batched forward kernel runs as clusters of
    three CTAs with the descriptor picked by blockIdx.z."""
    ps = [I.make_problem(4, ecutwfc=e, grid=(96, 96, 288), nbands=nb, with_beta=False) for e, nb in ((3.0, 3), (6.0, 2))]
    ctxs = [ks.Context.from_problem(p) for p in ps]
    outs = ks.hpsi_batch(ctxs, [_t(p.psi0) for p in ps])
    for p, o in zip(ps, outs):
        ref = oracle_mod.Oracle.from_problem(p).hpsi(p.psi0)
        assert _rel(o.cpu().numpy(), ref) <= HPSI_TOL and _elementwise_ok(o.cpu().numpy(), ref)


def test_davidson_batch_cfg2(ks):
    """ks_davidson_batch on 16 k-points of cfg 2 (worker threads, one stream each) against single ks_davidson solves of
    the same contexts, the survey's printed values, and time reversal between k_i and k_{63-i}."""
    sel = [0, 1, 5, 21, 26, 31, 32, 37, 42, 58, 62, 63, 10, 53, 7, 56]
    ps = [I.make_problem(2, k) for k in sel]
    ctxs = [ks.Context.from_problem(p) for p in ps]
    rs = ks.davidson_batch(ctxs, [_t(p.psi0) for p in ps], tol=1e-8)
    eig = {}
    for k, p, ctx, r in zip(sel, ps, ctxs, rs):
        assert r["converged"] and float(r["resid"].max()) <= 1e-8
        eig[k] = r["eig"].cpu().numpy()
        if k in (0, 21, 63):
            one = ctx.davidson(_t(p.psi0), tol=1e-8)
            assert np.abs(one["eig"].cpu().numpy() - eig[k]).max() <= 1e-8
            assert one["iters"] == r["iters"] and one["band_applications"] == r["band_applications"]
    g = _gold()["cfg2"]
    for key in ("k_m38", "k_m18"):
        e = eig[g[key]["k_index"]]
        for i, name in ((0, "eps0"), (15, "eps15"), (16, "eps16"), (31, "eps31")):
            assert abs(e[i] - g[key][name]) <= 1e-8
    for a in sel:
        if 63 - a in eig:
            assert np.abs(eig[a] - eig[63 - a]).max() <= 1e-8


# ------------------------------------------------------------------ stand-ins for compute-sanitizer (profiles/r2_sanitizer.md)
def _disturber(stream, n):
    """a bandwidth-heavy kernel on another stream: changes which CTAs are co-resident and when"""
    import torch
    with torch.cuda.stream(stream):
        a = torch.empty(n, dtype=torch.float32, device="cuda")
        a.fill_(1.0)
        a.mul_(1.0001)
    return a


@pytest.mark.parametrize("which", ["cfg1_bg8", "cfg1_ragged31", "slab288_cluster", "cube128", "cfg2_kbatch", "slab288_kbatch"])
def test_hpsi_repeatability_stress(ks, which):
    """200 repeats of one block apply must give the same BITS every time (fixed summation orders, no atomics), also while
    another stream keeps the SMs and HBM busy: a shared-memory or cp.async hazard (k_x's barrier-free refill, the DSMEM
    exchange of the cluster kernel) would show up as a repeat that differs."""
    import torch
    if which == "cfg1_bg8":
        ps = [I.make_problem(1, nbands=64, with_beta=False)]
    elif which == "cfg1_ragged31":
        ps = [I.make_problem(1, nbands=31)]
    elif which == "slab288_cluster":
        ps = [I.make_problem(4, ecutwfc=12.0, grid=(96, 96, 288), nbands=6, with_beta=False)]
    elif which == "cube128":
        ps = [I.make_problem(3, ecutwfc=6.0, grid=(128, 128, 128), nbands=6, with_beta=False)]
    elif which == "cfg2_kbatch":
        ps = [I.make_problem(2, k, nbands=8) for k in (0, 21, 42, 63, 5)]
    else:
        ps = [I.make_problem(4, ecutwfc=e, grid=(96, 96, 288), nbands=3, with_beta=False) for e in (3.0, 6.0)]
    ctxs = [ks.Context.from_problem(p) for p in ps]
    psis = [_t(p.psi0) for p in ps]
    batch = which.endswith("kbatch")

    def apply():
        return ks.hpsi_batch(ctxs, psis) if batch else [ctxs[0].hpsi(psis[0])]

    first = [o.clone() for o in apply()]
    side = torch.cuda.Stream()
    keep = []
    for rep in range(200):
        if rep % 3 != 2:
            keep.append(_disturber(side, (1 + rep % 7) * (1 << 22)))
        outs = apply()
        for a, b in zip(first, outs):
            assert bool((a == b).all()), "repeat %d differs" % rep
        keep = keep[-2:]
    torch.cuda.synchronize()


def test_hpsi_guard_zones(ks):
    """psi / hpsi are slices of larger buffers; the borders hold a pattern that every entry point must leave alone."""
    import torch
    pat = complex(1.25e300, -7.5e-300)
    for ps, batch in (([I.make_problem(0)], False), ([I.make_problem(1, nbands=31)], False),
                      ([I.make_problem(2, k, nbands=nb) for k, nb in ((0, 5), (21, 32), (63, 17))], True),
                      ([I.make_problem(4, ecutwfc=3.0, grid=(96, 96, 288), nbands=3, with_beta=False)], False)):
        ctxs = [ks.Context.from_problem(p) for p in ps]
        G = 4096
        bufs_in, bufs_out, psis, outs = [], [], [], []
        for p in ps:
            n = p.nbands * p.npw
            bi = torch.full((n + 2 * G,), pat, dtype=torch.complex128, device="cuda")
            bo = torch.full((n + 2 * G,), pat, dtype=torch.complex128, device="cuda")
            bi[G:G + n] = _t(p.psi0).reshape(-1)
            bufs_in.append(bi); bufs_out.append(bo)
            psis.append(bi[G:G + n].view(p.nbands, p.npw)); outs.append(bo[G:G + n].view(p.nbands, p.npw))
        if batch:
            ks.hpsi_batch(ctxs, psis, outs)
        else:
            ctxs[0].hpsi(psis[0], out=outs[0])
        torch.cuda.synchronize()
        for p, bi, bo, o in zip(ps, bufs_in, bufs_out, outs):
            n = p.nbands * p.npw
            for b in (bi, bo):
                assert bool((b[:G] == pat).all()) and bool((b[G + n:] == pat).all()), "guard zone overwritten"
            assert bool((bi[G:G + n].view(p.nbands, p.npw) == _t(p.psi0)).all()), "input block modified"
            assert bool(torch.isfinite(o.real).all()) and float(o.abs().max()) < 1e6
