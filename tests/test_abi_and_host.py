"""CPU-side tests of the boundary and the host logic (no GPU, no compute calls):
the C-ABI library loads and exports every symbol include/kspw.h declares, its pure host helpers agree bit for bit
with the oracle and the input generator, the product path fails loudly without a device, and the multi-rank
plumbing (world_size 2, gloo) shards units and aggregates device times the way bench.py reports them."""
import ctypes
import os
import re
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
from paper_2501_08697_b200 import inputs as I  # noqa: E402


@pytest.fixture(scope="module")
def lib():
    from paper_2501_08697_b200 import build
    return ctypes.CDLL(build.build())


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "kspw.h")).read()
    text = re.sub(r"/\*.*?\*/", " ", text, flags=re.S)
    return sorted(set(re.findall(r"\b(ks_[a-z0-9_]+)\s*\(", text)))


def test_header_symbols_are_exported(lib):
    names = _declared_symbols()
    assert len(names) >= 18 and "ks_create" in names and "ks_hpsi" in names and "ks_davidson" in names
    missing = [n for n in names if not hasattr(lib, n)]
    assert not missing, "declared in include/kspw.h but not exported by libkspw.so: %s" % missing


def test_binding_exports_match_header():
    from paper_2501_08697_b200 import kspw
    assert sorted(kspw.EXPORTS) == _declared_symbols()


def test_header_has_no_torch_or_cxx_types():
    text = open(os.path.join(ROOT, "include", "kspw.h")).read()
    assert 'extern "C"' in text
    for bad in ("torch", "at::", "std::", "template"):
        assert bad not in text


@pytest.mark.parametrize("c,k_index", [(0, 0), (2, 21), (2, 63), (4, 0)])
def test_pw_list_bit_exact_vs_generator(lib, c, k_index):
    """ks_pw_count / ks_pw_list are pure host helpers: the index work is compared bit for bit (readings C2, C3)."""
    p = I.make_problem(c, k_index, with_beta=False, with_vloc=False, nbands=1)
    cell = np.ascontiguousarray(p.cell, dtype=np.float64)
    kf = np.ascontiguousarray(p.k_frac, dtype=np.float64)
    n = ctypes.c_int(0)
    vp = ctypes.c_void_p
    lib.ks_pw_count.argtypes = [vp, vp, ctypes.c_double, vp]
    lib.ks_pw_list.argtypes = [vp, vp, ctypes.c_double, vp, vp]
    assert lib.ks_pw_count(cell.ctypes.data, kf.ctypes.data, float(p.ecutwfc), ctypes.addressof(n)) == 0
    assert n.value == p.npw
    mil = np.zeros((n.value, 3), dtype=np.int32)
    g2 = np.zeros(n.value, dtype=np.float64)
    assert lib.ks_pw_list(cell.ctypes.data, kf.ctypes.data, float(p.ecutwfc), mil.ctypes.data, g2.ctypes.data) == 0
    assert np.array_equal(mil, p.miller)
    assert np.abs(g2 - p.g2).max() <= 1e-14 * p.g2.max()    # floating point: a few ulp (different summation order)
    # canonical order: m1 slowest, m3 fastest, ascending
    key = (mil[:, 0].astype(np.int64) * 4096 + mil[:, 1]) * 4096 + mil[:, 2]
    assert (np.diff(key) > 0).all()


def test_bad_arguments_are_refused(lib):
    vp = ctypes.c_void_p
    lib.ks_pw_count.argtypes = [vp, vp, ctypes.c_double, vp]
    n = ctypes.c_int(0)
    cell = np.eye(3) * 10.0
    kf = np.zeros(3)
    assert lib.ks_pw_count(None, kf.ctypes.data, 10.0, ctypes.addressof(n)) < 0
    assert lib.ks_pw_count(cell.ctypes.data, kf.ctypes.data, -1.0, ctypes.addressof(n)) < 0
    lib.ks_npw.argtypes = [vp]
    assert lib.ks_npw(None) < 0
    lib.ks_last_error.argtypes = [vp]
    lib.ks_last_error.restype = ctypes.c_char_p
    assert lib.ks_last_error(None) is not None


def test_create_fails_loudly_without_a_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    from paper_2501_08697_b200 import kspw
    p = I.make_problem(0)
    with pytest.raises(kspw.KsError) as ei:
        kspw.Context.from_problem(p)
    assert ei.value.rc == -4 and "no CPU fallback" in str(ei.value)      # KS_ECUDA


def test_product_path_does_not_import_the_oracle():
    """Only tests/, __graft_entry__.smoke() and bench.py's oracle legs may touch oracle/."""
    pkg = os.path.join(ROOT, "paper_2501_08697_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in text.replace("oracle/", "").replace("the oracle", "").replace("oracle's", "") \
                    or f == "inputs.py", "%s mentions the oracle" % f
                assert "import oracle" not in text and "from oracle" not in text and "kso.h" not in text


def test_shard_units_partition():
    from paper_2501_08697_b200 import parallel as PL
    for n, w in ((64, 1), (64, 2), (64, 8), (64, 3), (5, 8)):
        parts = [PL.shard_units(n, r, w) for r in range(w)]
        assert sorted(sum(parts, [])) == list(range(n))
        assert max(len(x) for x in parts) - min(len(x) for x in parts) <= 1


_WORKER = r"""
import sys, os
sys.path.insert(0, %r)
from paper_2501_08697_b200 import parallel as PL
rank, world, local = PL.init("gloo")
assert world == 2
# k-point sharding of BASELINE config 2 (64 k-points): disjoint shares, one gather of 32 eigenvalues per k
mine = PL.shard_units(64, rank, world)
rows = {k: [k + 0.001 * b for b in range(32)] for k in mine}
PL.barrier()
table = PL.gather_rows(rows, 64, 32)
ms, e2e = PL.max_over_ranks([10.0 + 5.0 * rank, 3.0 - rank])     # each rank's own device time
value = PL.aggregate_throughput(160 * 10, world, ms)
if rank == 0:
    ok = all(abs(table[k][b] - (k + 0.001 * b)) < 1e-12 for k in range(64) for b in range(32))
    print("RESULT", len(mine), ok, ms, e2e, value)
PL.finalize()
"""


def test_world2_gloo_sharding_and_max_over_ranks(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(_WORKER % ROOT)
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), WORLD_SIZE="2", LOCAL_RANK=str(r), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT="29533", CUDA_VISIBLE_DEVICES="")
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=240) for p in procs]
    assert all(p.returncode == 0 for p in procs), outs
    line = [ln for ln in outs[0][0].splitlines() if ln.startswith("RESULT")][0].split()
    assert line[1] == "32" and line[2] == "True"
    assert float(line[3]) == 15.0 and float(line[4]) == 3.0          # MAX over ranks, element-wise
    assert abs(float(line[5]) - 2 * 1600 / 15.0e-3) < 1e-6           # whole-job units / slowest rank's time
