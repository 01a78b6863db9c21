"""Writes tests/golden/oracle_davidson_cfg<C>.json: the ORACLE's block-Davidson eigenvalues of a full-size config.

Calls only oracle/ and the seeded input generator (no CUDA code).  A full-size oracle solve takes minutes to hours of
CPU time (plain loops, OpenMP over bands), so its result is stored once and the GPU test compares against the file
(SURVEY.md §8(d) plan).  Usage:  python tests/golden/make_oracle_davidson.py 1 [k_index]
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
    c = int(sys.argv[1])
    k = int(sys.argv[2]) if len(sys.argv) > 2 else 0
    p = I.make_problem(c, k)
    o = kso.Oracle.from_problem(p)
    t0 = time.time()
    r = o.davidson(p.psi0, tol=1e-8)
    wall = time.time() - t0
    out = {
        "_citation": "oracle/kso.cpp kso_davidson (DESIGN.md §3 listing) on BASELINE config %d, k-point %d, seed %d, tol 1e-8; "
                     "written by tests/golden/make_oracle_davidson.py" % (c, k, 1000 + c),
        "config": c, "k_index": k, "npw": int(p.npw), "nbands": int(p.nbands),
        "converged": bool(r["converged"]), "iterations": int(r["iters"]), "band_applications": int(r["nhpsi"]),
        "max_resid": float(r["resid"].max()), "wall_s": wall, "threads": kso.num_threads(),
        "eig": [float(x) for x in r["eig"]],
    }
    dst = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_davidson_cfg%d.json" % c)
    if os.environ.get("KSO_GOLDEN_OUT"):
        dst = os.environ["KSO_GOLDEN_OUT"]
    with open(dst, "w") as f:
        json.dump(out, f, indent=1)
    print("wrote", dst, "iterations", out["iterations"], "wall %.1f s" % wall, "threads", out["threads"])


if __name__ == "__main__":
    main()
