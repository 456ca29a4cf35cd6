"""ctypes loader for the CPU oracle (oracle/bg_oracle.c).

TEST INFRASTRUCTURE: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this package.  It never imports
the CUDA package and shares no code with it.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "liboracle_bg.so")
_SRC = [os.path.join(_HERE, "bg_oracle.c"), os.path.join(_HERE, "bg_recursion.inc")]
_LIB = None

FP31, C128, C80 = 0, 1, 2
P31 = (1 << 31) - 1


def build(force: bool = False) -> str:
    """gcc -O2, FP contraction off so complex128 results are reproducible across hosts."""
    if not force and os.path.exists(_SO) and all(
            os.path.getmtime(_SO) >= os.path.getmtime(s) for s in _SRC):
        return _SO
    cmd = ["gcc", "-std=c11", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fPIC", "-shared",
           "-Wall", "-Wextra", "-o", _SO, _SRC[0], "-lm"]
    subprocess.run(cmd, check=True, cwd=_HERE)
    return _SO


def _lib():
    global _LIB
    if _LIB is None:
        build()
        lib = ctypes.CDLL(_SO)
        vp, i64, ci = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int
        lib.oracle_bg_currents.argtypes = [ci, ci, ci, i64, vp, vp, vp, vp, vp]
        lib.oracle_bg_currents.restype = ci
        lib.oracle_bg_amplitudes.argtypes = [ci, ci, ci, i64, vp, vp, vp, vp]
        lib.oracle_bg_amplitudes.restype = ci
        lib.oracle_bg_modulus.restype = ctypes.c_uint32
        lib.oracle_bg_evaluate.argtypes = [ci, ci, ctypes.c_uint32, ci, ci, i64, ci, vp, vp, vp, vp, vp]
        lib.oracle_bg_evaluate.restype = ci
        _LIB = lib
    return _LIB


def _dtypes(field: int):
    if field == FP31:
        return np.uint32, np.uint32
    if field == C128:
        return np.complex128, np.complex128
    if field == C80:
        return np.complex128, np.clongdouble
    raise ValueError("field must be FP31, C128 or C80")


MOSTLY_MINUS, ALTERNATING = 0, 1


def evaluate(field: int, momenta: np.ndarray, polarisations: np.ndarray, metric: int = MOSTLY_MINUS,
             prime: int = 0, want_currents: bool = False, want_status: bool = False, threads: int = 1):
    """The literal recursion for momenta [batch, n, d] and polarisations [batch, n, d] or, with S
    state configurations per momentum point (Eq.(4)), [batch, S, n, d].
    metric: MOSTLY_MINUS or ALTERNATING; prime (FP31 only): 0 for
    2^31-1, else any prime below 2^31.  Returns out [batch] / [batch, S] (and, on request,
    currents [batch, (S,) m, m, d] and status [batch]).  threads > 1 splits the batch into
    contiguous slices, one Python thread each (ctypes releases the GIL)."""
    in_dt, out_dt = _dtypes(field)
    mom = np.ascontiguousarray(momenta, dtype=in_dt)
    pol = np.ascontiguousarray(polarisations, dtype=in_dt)
    has_states = pol.ndim == 4
    if mom.ndim != 3 or pol.ndim not in (3, 4) or pol.shape[0] != mom.shape[0] or pol.shape[-2:] != mom.shape[1:]:
        raise ValueError("momenta must be [batch, n, d], polarisations [batch, n, d] or [batch, S, n, d]")
    batch, n, d = mom.shape
    S = pol.shape[1] if has_states else 1
    m = n - 1
    out = np.zeros((batch, S), dtype=out_dt)
    cur = np.zeros((batch, S, m, m, d), dtype=out_dt) if want_currents else None
    status = np.zeros(batch, dtype=np.uint32)
    lib = _lib()
    bad = []

    def run(b0, b1):
        if b1 > b0 and lib.oracle_bg_evaluate(
                field, metric, prime, n, d, b1 - b0, S, mom[b0:b1].ctypes.data, pol[b0:b1].ctypes.data,
                out[b0:b1].ctypes.data, None if cur is None else cur[b0:b1].ctypes.data,
                status[b0:b1].ctypes.data):
            bad.append(b0)

    if batch == 0:
        if lib.oracle_bg_evaluate(field, metric, prime, n, d, 0, S, None, None, None, None, None):
            bad.append(0)
    else:
        _sliced(batch, threads, run)
    if bad:
        raise ValueError("oracle rejected the arguments (need 4<=n<=16, 4<=d<=16, metric 0|1, prime < 2^31)")
    if not has_states:
        out = out[:, 0]
        cur = None if cur is None else cur[:, 0]
    res = [out]
    if want_currents:
        res.append(cur)
    if want_status:
        res.append(status)
    return res[0] if len(res) == 1 else tuple(res)


def orderings(field: int, momenta: np.ndarray, polarisations: np.ndarray, perms, metric: int = MOSTLY_MINUS,
              prime: int = 0, threads: int = 1) -> np.ndarray:
    """The colour-ordered amplitudes C(sigma(1), .., sigma(n)) of Eq.(5), for every
    row sigma of perms [K, n] (0-based legs): the literal recursion run once per ordering on the
    permuted inputs, nothing shared.  Returns out [batch, K] (or [batch, K, S] with a state axis)."""
    perms = np.asarray(perms)
    outs = [evaluate(field, momenta[:, list(s)], polarisations[..., list(s), :], metric, prime, threads=threads)
            for s in perms]
    return np.stack(outs, axis=1)


def amplitudes(field: int, momenta: np.ndarray, polarisations: np.ndarray,
               want_currents: bool = False, want_status: bool = False, threads: int = 1):
    """evaluate() with the mostly-minus metric, p = 2^31-1 and one state configuration"""
    return evaluate(field, momenta, polarisations, MOSTLY_MINUS, 0, want_currents, want_status, threads)


def _sliced(batch: int, threads: int, fn) -> None:
    """fn(b0, b1) on contiguous slices of [0, batch), one Python thread each"""
    if threads <= 1 or batch < 2 * threads:
        fn(0, batch)
        return
    bounds = [batch * t // threads for t in range(threads + 1)]
    ts = [threading.Thread(target=fn, args=(bounds[t], bounds[t + 1])) for t in range(threads)]
    for t in ts:
        t.start()
    for t in ts:
        t.join()


def modulus() -> int:
    return int(_lib().oracle_bg_modulus())
