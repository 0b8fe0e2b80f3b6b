"""The CPU oracle under AddressSanitizer + UndefinedBehaviorSanitizer ("CPU oracle under
-fsanitize=address,undefined"), CPU only.

oracle/hec_oracle.c keeps fixed-size stack arrays (ORC_MAXN digits per element, ext_field F[ORC_MAXDEG] indexed by k);
this builds it with `gcc -fsanitize=address,undefined -fno-sanitize-recover` together with the small driver
oracle/hec_oracle_san_main.c, runs config 1 in full, a q = 9 batch (r = 2: extension degrees up to 6 over F_3, the
embedding search) and a q = 13, g = 4 slice with k up to 5 (one field beyond the genus, as the lambda oracle asks for),
and requires (i) a clean exit with nothing on stderr and (ii) the same numbers as the ordinary build."""
import os
import subprocess
from pathlib import Path

import numpy as np
import pytest

from oracle import hec_oracle as O
from paper_1805_11991_b200 import workloads as W

ORACLE = Path(O.__file__).resolve().parent


@pytest.fixture(scope="module")
def san_binary(tmp_path_factory):
    exe = tmp_path_factory.mktemp("san") / "hec_oracle_san"
    cmd = ["gcc", "-O1", "-g", "-std=c11", "-fopenmp", "-fsanitize=address,undefined", "-fno-sanitize-recover=all",
           "-fno-omit-frame-pointer", "-o", str(exe), str(ORACLE / "hec_oracle_san_main.c"), str(ORACLE / "hec_oracle.c")]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0 and "asan" in (r.stderr or "").lower() and "cannot find" in r.stderr:
        pytest.skip("libasan is not installed")
    assert r.returncode == 0, r.stderr
    return exe


def _edge_and_random_rows(q, g, n, seed):
    rng = np.random.default_rng(seed)
    rows = rng.integers(0, q, size=(n, 2 * g + 3), dtype=np.uint16)
    rows[: n // 2, 2 * g + 2] = 0                               # odd degree
    rows[: n // 2, 2 * g + 1] = rng.integers(1, q, size=n // 2)
    rows[n // 2:, 2 * g + 2] = rng.integers(1, q, size=n - n // 2)
    return np.concatenate([W.edge_rows(q, g), rows])


@pytest.mark.parametrize("name,q,p,r,g,k_hi", [("config1", 3, 3, 1, 2, 2), ("q9", 9, 3, 2, 3, 3), ("q13", 13, 13, 1, 4, 5)])
def test_oracle_is_clean_under_asan_and_ubsan(san_binary, tmp_path, name, q, p, r, g, k_hi):
    if name == "config1":
        rows = W.generate(W.CONFIGS[1])
    elif name == "q9":
        rows = _edge_and_random_rows(9, 3, 24, seed=91)
    else:
        rows = _edge_and_random_rows(13, 4, 0, seed=13)[5:8]   # k = 5: 371293 points per row under ASan
    fin, fout = tmp_path / "in.bin", tmp_path / "out.bin"
    np.ascontiguousarray(rows, dtype=np.uint16).tofile(fin)
    env = dict(os.environ, ASAN_OPTIONS="detect_leaks=1:abort_on_error=0", UBSAN_OPTIONS="print_stacktrace=1",
               OMP_NUM_THREADS="4")
    res = subprocess.run([str(san_binary), str(p), str(r), str(g), str(k_hi), str(fin), str(fout)],
                         capture_output=True, text=True, env=env, timeout=600)
    assert res.returncode == 0, res.stderr[-4000:]
    assert res.stderr.strip() == "", res.stderr[-4000:]
    n = len(rows)
    raw = np.fromfile(fout, dtype=np.uint8)
    cnt = raw[: 4 * n * k_hi].view(np.uint32).reshape(n, k_hi)
    r0 = raw[4 * n * k_hi: 8 * n * k_hi].view(np.uint32).reshape(n, k_hi)
    sf = raw[8 * n * k_hi:]
    ocnt, osf, _ = O.count(q, g, rows, k_hi=k_hi)
    assert (cnt == ocnt[:, :k_hi]).all() and (sf == osf).all()
    assert (r0 == O.roots(q, g, rows, k_hi=k_hi)).all()
