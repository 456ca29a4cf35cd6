"""The oracle under AddressSanitizer + UndefinedBehaviorSanitizer.

oracle/bg_oracle.c indexes fixed [MAXN+1][MAXN+1][MAXD] thread-local tables with the caller's n and d, and every
parity verdict of the GPU tests rests on it.  Here the same source is compiled with
-fsanitize=address,undefined -fno-sanitize-recover=all into a stand-alone driver (oracle/sanitize_main.c, argument
arrays are heap blocks of exactly the documented size) and run on the shapes that reach furthest: the survey's worked
examples, the largest shape n = d = 16 (with S = 2 states and the currents array), the smallest n = d = 4, a singular
point (a vanishing propagator: inv(0), status bit), inputs at and above p, a generic prime with the alternating
metric, and the 80-bit type.  A sanitizer report aborts the driver (non-zero exit); its results must equal the
normal -O2 library's bit for bit.
"""
import os
import shutil
import subprocess

import numpy as np
import pytest

import oracle
from paper_2502_07060_b200 import inputs

HERE = os.path.dirname(os.path.abspath(__file__))
ODIR = os.path.join(os.path.dirname(HERE), "oracle")


@pytest.fixture(scope="module")
def driver(tmp_path_factory):
    if not shutil.which("gcc"):
        pytest.skip("no gcc")
    exe = str(tmp_path_factory.mktemp("san") / "oracle_san")
    cmd = ["gcc", "-std=c11", "-O1", "-g", "-ffp-contract=off", "-fno-fast-math", "-fno-omit-frame-pointer",
           "-fsanitize=address,undefined", "-fno-sanitize-recover=all", "-Wall", "-Wextra",
           "-o", exe, os.path.join(ODIR, "sanitize_main.c"), os.path.join(ODIR, "bg_oracle.c"), "-lm"]
    r = subprocess.run(cmd, capture_output=True, text=True, cwd=ODIR)
    if r.returncode != 0 and "asan" in (r.stderr or "").lower():
        pytest.skip("this gcc has no sanitizer runtime: " + r.stderr[-200:])
    assert r.returncode == 0, r.stderr
    oracle.build()
    return exe


def _run(exe, tmp, field, mom, pol, metric=0, prime=0, want_currents=True):
    in_dt, out_dt = oracle._dtypes(field)
    mom = np.ascontiguousarray(mom, dtype=in_dt)
    pol = np.ascontiguousarray(pol, dtype=in_dt)
    batch, n, d = mom.shape
    S = pol.shape[1] if pol.ndim == 4 else 1
    fin, fout = str(tmp / "in.bin"), str(tmp / "out.bin")
    with open(fin, "wb") as f:
        f.write(np.array([field, metric, 0, n, d, batch, S, int(want_currents)], dtype=np.int32).tobytes())
        f.seek(8)
        f.write(np.uint32(prime).tobytes())
        f.seek(32)
        f.write(mom.tobytes())
        f.write(pol.tobytes())
    env = dict(os.environ, ASAN_OPTIONS="detect_leaks=0:abort_on_error=0", UBSAN_OPTIONS="print_stacktrace=1")
    r = subprocess.run([exe, fin, fout], capture_output=True, text=True, env=env, timeout=600)
    assert r.returncode == 0, f"sanitized oracle exited {r.returncode}:\n{r.stderr[-3000:]}"
    assert "runtime error" not in r.stderr and "AddressSanitizer" not in r.stderr, r.stderr[-3000:]
    raw = open(fout, "rb").read()
    w = np.dtype(out_dt).itemsize
    m = n - 1
    n_out = batch * S
    n_cur = n_out * m * m * d if want_currents else 0
    out = np.frombuffer(raw, dtype=out_dt, count=n_out).reshape(batch, S)
    cur = np.frombuffer(raw, dtype=out_dt, count=n_cur, offset=n_out * w).reshape(batch, S, m, m, d) if want_currents else None
    status = np.frombuffer(raw, dtype=np.uint32, count=batch, offset=(n_out + n_cur) * w)
    assert len(raw) == (n_out + n_cur) * w + 4 * batch
    # the normal library on the same inputs: bit for bit (same source, -O2 instead of -O1 -fsanitize, no contraction)
    ref = oracle.evaluate(field, mom, pol, metric, prime, want_currents=want_currents, want_status=True)
    r_out, r_cur, r_st = (ref[0], ref[1], ref[2]) if want_currents else (ref[0], None, ref[1])
    assert np.array_equal(out.view(np.uint8), np.ascontiguousarray(r_out).reshape(batch, S).view(np.uint8))
    if want_currents:
        assert np.array_equal(cur.view(np.uint8), np.ascontiguousarray(r_cur).reshape(cur.shape).view(np.uint8))
    assert np.array_equal(status, r_st)
    return out, status


def test_worked_examples(driver, tmp_path):
    """the survey's four worked examples (unphysical small integers; golden values in tests/golden)"""
    P = oracle.P31
    for n, d, want in [(4, 4, 509929092), (5, 6, 139101349), (6, 4, 1080021013), (8, 6, 1802767521)]:
        k = np.array([[((7 * i + 3 * mu + i * mu) % 11) - 5 for mu in range(d)] for i in range(n)])
        e = np.array([[((5 * i + 2 * mu + 3 * i * mu + 1) % 13) - 6 for mu in range(d)] for i in range(n)])
        out, _ = _run(driver, tmp_path, oracle.FP31, (k % P).astype(np.uint32)[None], (e % P).astype(np.uint32)[None])
        assert int(out[0, 0]) == want
        _run(driver, tmp_path, oracle.C128, k.astype(np.complex128)[None], e.astype(np.complex128)[None])


@pytest.mark.parametrize("field", [oracle.FP31, oracle.C128, oracle.C80])
def test_largest_and_smallest_shapes(driver, tmp_path, field):
    name = "fp31" if field == oracle.FP31 else "c128"
    for n, d, batch, S in [(16, 16, 2, 2), (4, 4, 3, 1), (16, 4, 1, 1), (4, 16, 2, 3)]:
        mom, pol, _ = inputs.make_state_inputs(name, n, d, batch, S, seed=3)
        _run(driver, tmp_path, field, mom, pol)


def test_singular_point_and_extreme_residues(driver, tmp_path):
    P = oracle.P31
    mom, pol, _ = inputs.make_fp_inputs(8, 6, 3, seed=9)
    mom = mom.copy()
    mom[1, 1] = mom[1, 0]                                  # k_2 = k_1 at point 1: P_{1,2}^2 = 4 k_1^2 = 0
    mom[2, 3] = P                                          # residues at and above p are reduced on load
    mom[2, 4, 0] = 0xFFFFFFFF
    pol[2, 0] = P - 1
    _, st = _run(driver, tmp_path, oracle.FP31, mom, pol)
    assert st[1] == 1 and st[0] == 0
    cm, cp, _ = inputs.make_complex_inputs(6, 4, 2, seed=9, helicities=(-1, -1, 1, 1, 1, 1))
    cm = cm.copy()
    cm[0, 1] = cm[0, 0]
    cm[1, 2] = 0.0                                         # k_3 = 0 exactly: P_{3,3}.. and J / 0 paths in floating point
    for field in (oracle.C128, oracle.C80):                # (k_1^2 is only ~1e-17 in doubles: no exact zero is claimed)
        _run(driver, tmp_path, field, cm, cp)


def test_generic_prime_alternating_metric_and_empty_batch(driver, tmp_path):
    prime = 2147483629
    mom, pol, _ = inputs.make_fp_inputs(7, 5, 2, seed=4, prime=prime, metric=1)
    _run(driver, tmp_path, oracle.FP31, mom, pol, metric=1, prime=prime)
    _run(driver, tmp_path, oracle.FP31, mom[:0], pol[:0], want_currents=False)
