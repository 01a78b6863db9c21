"""Writes tests/golden/oracle_davidson_cfg<C>.json: the ORACLE's block-Davidson eigenvalues of a full-size config.

Calls only oracle/ and the seeded input generator (no CUDA code).  A full-size oracle solve takes minutes to hours of
CPU time (plain loops, OpenMP over bands), so its result is stored once and the GPU test compares against the file
(SURVEY.md §8(d) plan).  Usage:  python tests/golden/make_oracle_davidson.py <config> [k_index] [nbands] [--lapack GUARD SUBFACTOR]

With `nbands` the full-size problem (same cell, sphere, grid, projectors) is solved for its lowest `nbands` levels only,
start block drawn by the recipe with that nbands (inputs.make_problem(c, k, nbands=nbands)); the file is then
oracle_davidson_cfg<C>_nb<nbands>.json.  Configs with several k-points (cfg 2) write oracle_davidson_cfg<C>_k<k_index>.json.

--lapack GUARD SUBFACTOR: the one-off route SURVEY.md §8(d)(4) allows for the largest config: the same listing with
library primitives as steps (oracle/davidson_lapack.py: LAPACK eigh / QR, zgemm, the oracle's own H psi), GUARD extra
bands that are corrected but not waited for, subspace <= SUBFACTOR * (nbands + GUARD).  Converged eigenvalues do not
depend on the route; the stored iteration / band-application counts of such a run are NOT comparable with the GPU's.
"""
import json
import os
import sys
import time

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from paper_2501_08697_b200 import inputs as I  # noqa: E402
from oracle import kso  # noqa: E402


def main():
    argv = list(sys.argv[1:])
    lap = None
    if "--lapack" in argv:
        i = argv.index("--lapack")
        lap = (int(argv[i + 1]), int(argv[i + 2]))
        del argv[i:i + 3]
    c = int(argv[0])
    k = int(argv[1]) if len(argv) > 1 else 0
    nbo = int(argv[2]) if len(argv) > 2 else None
    route = "oracle/kso.cpp kso_davidson (DESIGN.md §3 listing)"
    t0 = time.time()
    if lap is None:
        p = I.make_problem(c, k, nbands=nbo)
        o = kso.Oracle.from_problem(p)
        r = o.davidson(p.psi0, tol=1e-8)
    else:
        from oracle.davidson_lapack import davidson_lapack
        nbt = I.config(c).nbands if nbo is None else nbo
        p = I.make_problem(c, k, nbands=nbt + lap[0])      # start block of nbands + GUARD vectors from the recipe
        o = kso.Oracle.from_problem(p)
        r = davidson_lapack(o, p.g2, p.psi0, nconv=nbt, tol=1e-8, max_sub_factor=lap[1],
                            log=lambda s: print(s, flush=True))
        p.nbands = nbt
        route = ("oracle/davidson_lapack.py (DESIGN.md §3 listing, LAPACK eigh/QR + zgemm as steps, oracle kso_hpsi; %d guard bands, "
                 "subspace <= %d x %d; iteration and band-application counts NOT comparable with the 2*nbands listing)"
                 % (lap[0], lap[1], nbt + lap[0]))
    wall = time.time() - t0
    out = {
        "_citation": "%s on BASELINE config %d, k-point %d, seed %d, tol 1e-8; "
                     "written by tests/golden/make_oracle_davidson.py" % (route, c, k, 1000 + c),
        "route": "listing" if lap is None else "lapack",
        "config": c, "k_index": k, "npw": int(p.npw), "nbands": int(p.nbands),
        "converged": bool(r["converged"]), "iterations": int(r["iters"]), "band_applications": int(r["nhpsi"]),
        "max_resid": float(r["resid"].max()), "wall_s": wall, "threads": kso.num_threads(),
        "eig": [float(x) for x in r["eig"]],
    }
    name = "oracle_davidson_cfg%d%s%s.json" % (c, "_k%d" % k if len(I.config(c).kpts) > 1 else "", "" if nbo is None else "_nb%d" % nbo)
    dst = os.path.join(os.path.dirname(os.path.abspath(__file__)), name)
    if os.environ.get("KSO_GOLDEN_OUT"):
        dst = os.environ["KSO_GOLDEN_OUT"]
    with open(dst, "w") as f:
        json.dump(out, f, indent=1)
    print("wrote", dst, "iterations", out["iterations"], "wall %.1f s" % wall, "threads", out["threads"])


if __name__ == "__main__":
    main()
