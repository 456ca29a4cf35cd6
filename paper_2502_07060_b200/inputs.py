"""Seeded synthetic kinematics for the Berends-Giele hot path.

This module is the ONE piece shared by the CPU oracle (``oracle/``) and the CUDA
path (``csrc/``): it only *prepares inputs* (on-shell, momentum-conserving momenta
and transverse polarisation vectors).  It contains none of the method's arithmetic
(no currents, no vertices, no recursion) and imports neither side.

It stands in for the paper's host-side phase-space / state preparation, which
uses ``lips``/``syngular`` (§3) and is not available
here.  The recipe is the one BASELINE.json:configs states, made concrete in
SURVEY.md §8(d) and DESIGN.md §"Input recipe":

* every random number is a pure function of (seed, global point index, attempt,
  draw counter) through SplitMix64, so any slice ``[start, start+batch)`` of a
  workload can be generated independently (used for multi-GPU sharding);
* massless vectors come from light-cone data: p- = (sum p_perp^2) / (2 p+),
  Cartesian p^0 = p+ + p-/2, p^1 = p+ - p-/2, p^{2..d-1} = p_perp, metric
  diag(+,-,...,-);
* p_1..p_{n-2} free, K = -(p_1+..+p_{n-2}), q random massless,
  p_{n-1} = alpha q with alpha = K^2/(2 K.q), p_n = K - p_{n-1};
* generic polarisations eps_i = v_i - (v_i.p_i)/(r_i.p_i) r_i  (transverse,
  unnormalised), or, for d = 4 complex, spinor-helicity states eps_-/eps_+ built
  on the reference momentum r_i (used for the Parke-Taylor pin).
"""
from __future__ import annotations

import numpy as np

P31 = (1 << 31) - 1  # the prime of BASELINE.json:configs, p = 2^31 - 1

_U64 = np.uint64
_GOLDEN = _U64(0x9E3779B97F4A7C15)
_M1 = _U64(0xBF58476D1CE4E5B9)
_M2 = _U64(0x94D049BB133111EB)


def _mix64(z: np.ndarray) -> np.ndarray:
    """SplitMix64 output function (finaliser) on uint64 arrays, wrapping."""
    with np.errstate(over="ignore"):
        z = (z ^ (z >> _U64(30))) * _M1
        z = (z ^ (z >> _U64(27))) * _M2
        return z ^ (z >> _U64(31))


class _Stream:
    """Counter-based stream: draw c of point b, attempt a is
    mix64(key(seed, b, a) + (c+1)*GOLDEN).  Vectorised over points."""

    def __init__(self, seed: int, index: np.ndarray, attempt: np.ndarray):
        with np.errstate(over="ignore"):
            k = _mix64(np.full(index.shape, seed, dtype=_U64) + _GOLDEN)
            k = _mix64(k ^ (index.astype(_U64) * _M1 + _GOLDEN))
            k = _mix64(k ^ (attempt.astype(_U64) * _M2 + _GOLDEN))
        self.key = k
        self.counter = 0

    def u64(self, count: int) -> np.ndarray:
        """next `count` draws for every point -> uint64 [points, count]"""
        c = np.arange(self.counter + 1, self.counter + count + 1, dtype=_U64)
        self.counter += count
        with np.errstate(over="ignore"):
            return _mix64(self.key[:, None] + c[None, :] * _GOLDEN)


# ---------------------------------------------------------------------------
# metric
# ---------------------------------------------------------------------------
MOSTLY_MINUS, ALTERNATING = 0, 1


def metric_signs(d: int, metric: int = MOSTLY_MINUS) -> np.ndarray:
    """g_{mu mu}: diag(+,-,...,-) or Caravel's diag(+,-,+,-,...)"""
    g = np.ones(d, dtype=np.int64)
    if metric == MOSTLY_MINUS:
        g[1:] = -1
    elif metric == ALTERNATING:
        g[1::2] = -1
    else:
        raise ValueError("metric must be MOSTLY_MINUS or ALTERNATING")
    return g


# ---------------------------------------------------------------------------
# F_p helpers (input preparation only); P = the prime as np.uint64
# ---------------------------------------------------------------------------
def _fp_mul(a, b, P):
    return (a * b) % P  # operands < 2^31, product < 2^62 fits uint64


def _fp_sub(a, b, P):
    return (a + P - b) % P


def _fp_pow(a, e: int, P):
    r = np.ones_like(a)
    base = a.copy()
    while e:
        if e & 1:
            r = _fp_mul(r, base, P)
        base = _fp_mul(base, base, P)
        e >>= 1
    return r


def _fp_inv(a, P):
    return _fp_pow(a, int(P) - 2, P)


def _fp_dot(x, y, P, g):
    """Minkowski product with metric signs g, last axis = component."""
    t = _fp_mul(x, y, P)
    plus = t[..., g > 0].sum(axis=-1) % P
    minus = t[..., g < 0].sum(axis=-1) % P
    return _fp_sub(plus, minus, P)


def _fp_massless(plus, perp, P, g):
    """light-cone -> Cartesian massless vector. plus [..], perp [.., d-2] -> [.., d]:
    p0 = p+ + p-/2, p1 = p+ - p-/2 (g_00 = +, g_11 = - in both metrics, so p0^2 - p1^2 = 2 p+ p-),
    p- = -(sum_{mu>=2} g_mu p_mu^2) / (2 p+)"""
    sq = _fp_mul(perp, perp, P)
    gp = g[2:]
    perp2 = _fp_sub(sq[..., gp < 0].sum(axis=-1) % P, sq[..., gp > 0].sum(axis=-1) % P, P)
    minus = _fp_mul(perp2, _fp_inv(_fp_mul(_U64(2), plus, P), P), P)
    half = _fp_mul(minus, _U64((int(P) + 1) // 2), P)
    p0 = (plus + half) % P
    p1 = _fp_sub(plus, half, P)
    return np.concatenate([p0[..., None], p1[..., None], perp], axis=-1)


def _fp_generate(n: int, d: int, seed: int, index: np.ndarray, attempt: np.ndarray, P, g, helicities=None):
    """One attempt for every listed point. Returns mom, pol (uint64) and ok mask."""
    st = _Stream(seed, index, attempt)
    nb = index.shape[0]
    pm1 = _U64(int(P) - 1)
    mom = np.zeros((nb, n, d), dtype=_U64)
    raw = st.u64((n - 2) * (d - 1)).reshape(nb, n - 2, d - 1)
    plus = _U64(1) + raw[:, :, 0] % pm1                 # uniform in [1,p)
    perp = _U64(1) + raw[:, :, 1:] % pm1                # uniform in [1,p)
    mom[:, : n - 2] = _fp_massless(plus, perp, P, g)
    raw = st.u64(d - 1)
    q = _fp_massless(_U64(1) + raw[:, 0] % pm1, _U64(1) + raw[:, 1:] % pm1, P, g)
    ksum = mom[:, : n - 2].sum(axis=1) % P
    K = (P - ksum) % P
    K2 = _fp_dot(K, K, P, g)
    Kq = _fp_dot(K, q, P, g)
    ok = Kq != 0
    alpha = _fp_mul(K2, _fp_inv(_fp_mul(_U64(2), Kq, P), P), P)
    mom[:, n - 2] = _fp_mul(alpha[:, None], q, P)
    mom[:, n - 1] = _fp_sub(K, mom[:, n - 2], P)
    # polarisations: per leg v (d draws, uniform in F_p) then r (p+, p_perp in [1,p))
    raw = st.u64(n * (2 * d - 1)).reshape(nb, n, 2 * d - 1)
    v = raw[:, :, :d] % P
    r = _fp_massless(_U64(1) + raw[:, :, d] % pm1, _U64(1) + raw[:, :, d + 1:] % pm1, P, g)
    rp = _fp_dot(r, mom, P, g)
    ok &= (rp != 0).all(axis=1)
    if helicities is None:
        vp = _fp_dot(v, mom, P, g)
        coef = _fp_mul(vp, _fp_inv(rp, P), P)
        pol = _fp_sub(v, _fp_mul(coef[..., None], r, P), P)
    else:
        ops = FpOps(int(P))
        pol = np.zeros((nb, n, d), dtype=_U64)
        for i, h in enumerate(helicities):
            # spinors need M00 = p0 + p3 != 0 for k_i and r_i
            ok &= ((mom[:, i, 0] + mom[:, i, 3]) % P != 0) & ((r[:, i, 0] + r[:, i, 3]) % P != 0)
            pol[:, i] = helicity_polarisation(mom[:, i], r[:, i], int(h), ALTERNATING, ops)
    # reject points with a vanishing proper invariant P_{i,j}^2, 1<=i<j<=n-1, (i,j)!=(1,n-1)
    m = n - 1
    prefix = np.zeros((nb, m + 1, d), dtype=_U64)
    for j in range(1, m + 1):
        prefix[:, j] = (prefix[:, j - 1] + mom[:, j - 1]) % P
    for i in range(1, m + 1):
        for j in range(i + 1, m + 1):
            if i == 1 and j == m:
                continue
            Pij = _fp_sub(prefix[:, j], prefix[:, i - 1], P)
            ok &= _fp_dot(Pij, Pij, P, g) != 0
    return mom, pol, ok, r


def make_fp_inputs(n: int, d: int, batch: int, seed: int = 0, start: int = 0, prime: int = P31,
                   metric: int = MOSTLY_MINUS, helicities=None):
    """F_p workload slice [start, start+batch), p = `prime` (default 2^31-1).

    Returns (momenta, polarisations, info): uint32 arrays [batch, n, d] of canonical
    residues, all momenta outgoing; info = {"redraws": number of rejected attempts, "reference"}.
    Points with K.q = 0, r_i.p_i = 0 or a vanishing proper P_{i,j}^2 are redrawn
    deterministically with attempt+1.  helicities (d = 4, ALTERNATING metric
    only: the spinors of a (2,2)-signature vector are rational): spinor-helicity
    states on the reference momenta r_i instead of the generic transverse vectors."""
    if n < 4 or d < 3:
        raise ValueError("need n >= 4 and d >= 3")
    if helicities is not None and (d != 4 or metric != ALTERNATING or len(helicities) != n):
        raise ValueError("F_p helicity states need d == 4, the alternating metric and one sign per leg")
    P = _U64(prime)
    g = metric_signs(d, metric)
    index = np.arange(start, start + batch, dtype=_U64)
    mom = np.zeros((batch, n, d), dtype=np.uint32)
    pol = np.zeros((batch, n, d), dtype=np.uint32)
    ref = np.zeros((batch, n, d), dtype=np.uint32)
    todo = np.arange(batch)
    attempt = np.zeros(batch, dtype=_U64)
    redraws = 0
    chunk = 1 << 16
    while todo.size:
        nxt = []
        for c0 in range(0, todo.size, chunk):
            sel = todo[c0:c0 + chunk]
            m_, p_, ok, r_ = _fp_generate(n, d, seed, index[sel], attempt[sel], P, g, helicities)
            good = sel[ok]
            mom[good] = m_[ok].astype(np.uint32)
            pol[good] = p_[ok].astype(np.uint32)
            ref[good] = r_[ok].astype(np.uint32)
            nxt.append(sel[~ok])
        todo = np.concatenate(nxt) if nxt else np.zeros(0, dtype=np.int64)
        attempt[todo] += _U64(1)
        redraws += int(todo.size)
    return mom, pol, {"redraws": redraws, "reference": ref}


# ---------------------------------------------------------------------------
# complex128
# ---------------------------------------------------------------------------
def _c_uniform(raw: np.ndarray) -> np.ndarray:
    """uint64 [..., 2k] -> complex [..., k], re and im each (u>>11)*2^-52 - 1 in [-1,1)."""
    f = (raw >> _U64(11)).astype(np.float64) * (2.0 ** -52) - 1.0
    return f[..., 0::2] + 1j * f[..., 1::2]


def _c_dot(x, y, g=None):
    t = x * y
    if g is None:
        return t[..., 0] - t[..., 1:].sum(axis=-1)
    return (t * g).sum(axis=-1)


def _c_massless(plus, perp, g=None):
    if g is None:
        minus = (perp * perp).sum(axis=-1) / (2.0 * plus)
    else:
        minus = -((perp * perp) * g[2:]).sum(axis=-1) / (2.0 * plus)
    p0 = plus + 0.5 * minus
    p1 = plus - 0.5 * minus
    return np.concatenate([p0[..., None], p1[..., None], perp], axis=-1)


# ---------------------------------------------------------------------------
# spinor-helicity states in d = 4 (input preparation for the Parke-Taylor comparisons)
# ---------------------------------------------------------------------------
class ComplexOps:
    """complex128 arithmetic on arrays"""
    imag_unit = 1j

    def mul(self, a, b):
        return a * b

    def add(self, a, b):
        return a + b

    def sub(self, a, b):
        return a - b

    def div(self, a, b):
        return a / b

    def const(self, like, num, den=1):
        return np.full_like(like, num / den)


class FpOps:
    """arithmetic mod a prime on uint64 arrays of canonical residues"""
    imag_unit = None          # no sqrt(-1) is assumed: only the alternating metric's spinors exist

    def __init__(self, prime: int = P31):
        self.P = _U64(prime)

    def mul(self, a, b):
        return _fp_mul(a, b, self.P)

    def add(self, a, b):
        return (a + b) % self.P

    def sub(self, a, b):
        return _fp_sub(a, b, self.P)

    def div(self, a, b):
        return _fp_mul(a, _fp_inv(b, self.P), self.P)

    def const(self, like, num, den=1):
        v = num % int(self.P) * pow(den, int(self.P) - 2, int(self.P)) % int(self.P)
        return np.full_like(like, v)


_COMPLEX = ComplexOps()


def spinors(p: np.ndarray, metric: int = MOSTLY_MINUS, ops=_COMPLEX):
    """Holomorphic/antiholomorphic spinors of a massless 4-vector.

    mostly minus (complex only):  M = [[p0+p3, p1-i p2],[p1+i p2, p0-p3]]
    alternating diag(+,-,+,-):    M = [[p0+p3, p1+p2],[p1-p2, p0-p3]]   (the same matrix under
        p2 -> i p2, which maps one metric to the other; no i is left, so it also works over F_p)
    det M = p.p = 0, M = lam lamt^T with lam = (M00, M10), lamt = (1, M01/M00).
    Returns (lam [...,2], lamt [...,2])."""
    M00 = ops.add(p[..., 0], p[..., 3])
    if metric == MOSTLY_MINUS:
        M01 = p[..., 1] - 1j * p[..., 2]
        M10 = p[..., 1] + 1j * p[..., 2]
    else:
        M01 = ops.add(p[..., 1], p[..., 2])
        M10 = ops.sub(p[..., 1], p[..., 2])
    lam = np.stack([M00, M10], axis=-1)
    lamt = np.stack([ops.const(M00, 1), ops.div(M01, M00)], axis=-1)
    return lam, lamt


def spinor_bracket(a: np.ndarray, b: np.ndarray, ops=_COMPLEX) -> np.ndarray:
    """<ab> (or [ab] when fed lamt's) = a0 b1 - a1 b0."""
    return ops.sub(ops.mul(a[..., 0], b[..., 1]), ops.mul(a[..., 1], b[..., 0]))


def _bispinor_to_vector(N00, N01, N10, N11, metric=MOSTLY_MINUS, ops=_COMPLEX):
    half = ops.const(N00, 1, 2)
    if metric == MOSTLY_MINUS:
        return np.stack([(N00 + N11) / 2, (N01 + N10) / 2, (N10 - N01) / 2j, (N00 - N11) / 2], axis=-1)
    return np.stack([ops.mul(half, ops.add(N00, N11)), ops.mul(half, ops.add(N01, N10)),
                     ops.mul(half, ops.sub(N01, N10)), ops.mul(half, ops.sub(N00, N11))], axis=-1)


def helicity_polarisation(k: np.ndarray, r: np.ndarray, hel: int, metric: int = MOSTLY_MINUS,
                          ops=_COMPLEX) -> np.ndarray:
    """sqrt-free spinor-helicity states in d=4 (weights 1/2 * 2 as in Eq.(11)):
       eps_-(k;r) = vec(lam_k lamt_r^T) / [r k],  eps_+(k;r) = 2 vec(lam_r lamt_k^T) / <r k>.
    eps_+.eps_- = -1, eps_h.eps_h = 0, eps.k = 0."""
    lk, ltk = spinors(k, metric, ops)
    lr, ltr = spinors(r, metric, ops)
    if hel < 0:
        a, b, den, w = lk, ltr, spinor_bracket(ltr, ltk, ops), 1
    else:
        a, b, den, w = lr, ltk, spinor_bracket(lr, lk, ops), 2
    vec = _bispinor_to_vector(ops.mul(a[..., 0], b[..., 0]), ops.mul(a[..., 0], b[..., 1]),
                              ops.mul(a[..., 1], b[..., 0]), ops.mul(a[..., 1], b[..., 1]), metric, ops)
    scale = ops.div(ops.const(den, w), den)
    return ops.mul(vec, scale[..., None])


def make_complex_inputs(n: int, d: int, batch: int, seed: int = 0, start: int = 0,
                        helicities=None, metric: int = MOSTLY_MINUS):
    """complex128 workload slice.  Momenta: the light-cone/alpha construction with
    complex components (re, im uniform in [-1,1)).  Polarisations: generic transverse
    vectors (helicities=None) or, for d == 4, spinor-helicity states with the given
    signs (e.g. (-1,-1,+1,+1,+1,+1) for config 1) on random reference momenta r_i.
    No rejection.  Returns (mom, pol, info); info carries the
    reference momenta so tests can rebuild the spinors."""
    if n < 4 or d < 3:
        raise ValueError("need n >= 4 and d >= 3")
    if helicities is not None and (d != 4 or len(helicities) != n):
        raise ValueError("helicity states need d == 4 and one sign per leg")
    g = None if metric == MOSTLY_MINUS else metric_signs(d, metric).astype(np.float64)
    mom = np.zeros((batch, n, d), dtype=np.complex128)
    pol = np.zeros((batch, n, d), dtype=np.complex128)
    ref = np.zeros((batch, n, d), dtype=np.complex128)
    chunk = 1 << 16
    for c0 in range(0, batch, chunk):
        nb = min(chunk, batch - c0)
        index = np.arange(start + c0, start + c0 + nb, dtype=_U64)
        st = _Stream(seed, index, np.zeros(nb, dtype=_U64))
        raw = _c_uniform(st.u64(2 * (n - 2) * (d - 1))).reshape(nb, n - 2, d - 1)
        m_ = np.zeros((nb, n, d), dtype=np.complex128)
        m_[:, : n - 2] = _c_massless(raw[:, :, 0], raw[:, :, 1:], g)
        raw = _c_uniform(st.u64(2 * (d - 1)))
        q = _c_massless(raw[:, 0], raw[:, 1:], g)
        K = -m_[:, : n - 2].sum(axis=1)
        alpha = _c_dot(K, K, g) / (2.0 * _c_dot(K, q, g))
        m_[:, n - 2] = alpha[:, None] * q
        m_[:, n - 1] = K - m_[:, n - 2]
        raw = _c_uniform(st.u64(2 * n * (2 * d - 1))).reshape(nb, n, 2 * d - 1)
        v = raw[:, :, :d]
        r = _c_massless(raw[:, :, d], raw[:, :, d + 1:], g)
        if helicities is None:
            coef = _c_dot(v, m_, g) / _c_dot(r, m_, g)
            p_ = v - coef[..., None] * r
        else:
            p_ = np.zeros((nb, n, d), dtype=np.complex128)
            for i, h in enumerate(helicities):
                p_[:, i] = helicity_polarisation(m_[:, i], r[:, i], int(h), metric)
        mom[c0:c0 + nb], pol[c0:c0 + nb], ref[c0:c0 + nb] = m_, p_, r
    return mom, pol, {"redraws": 0, "reference": ref}


# ---------------------------------------------------------------------------
# the five workloads of BASELINE.json:configs
# ---------------------------------------------------------------------------
CONFIGS = {
    "cfg0": dict(n=4, d=4, field="fp31", batch=1 << 10, helicities=None),
    "cfg1": dict(n=6, d=4, field="c128", batch=1 << 20, helicities=(-1, -1, 1, 1, 1, 1)),
    "cfg2": dict(n=8, d=6, field="fp31", batch=1 << 20, helicities=None),
    "cfg3": dict(n=10, d=8, field="fp31", batch=1 << 18, helicities=None),
    "cfg4a": dict(n=12, d=6, field="fp31", batch=1 << 16, helicities=None),
    "cfg4b": dict(n=12, d=6, field="c128", batch=1 << 16, helicities=None),
}


def make_inputs(field: str, n: int, d: int, batch: int, seed: int = 0, start: int = 0,
                helicities=None, metric: int = MOSTLY_MINUS, prime: int = P31):
    if field == "fp31":
        return make_fp_inputs(n, d, batch, seed, start, prime, metric, helicities)
    if field == "c128":
        return make_complex_inputs(n, d, batch, seed, start, helicities, metric)
    raise ValueError(f"unknown field {field!r}")


def make_state_inputs(field: str, n: int, d: int, batch: int, states: int, seed: int = 0, start: int = 0,
                      metric: int = MOSTLY_MINUS, prime: int = P31):
    """S = `states` polarisation configurations per momentum point (the workload of the cut equation
    Eq.(4)): momenta [batch, n, d] of the seeded generator and polarisations
    [batch, S, n, d], every configuration transverse to the SAME momenta.  Configuration 0 is the
    generator's own; configuration s > 0 rebuilds eps_i = v_i - (v_i.p_i)/(r_i.p_i) r_i from the
    (v_i, r_i) of the generator run with seed + 7919 s (a point whose r_i.p_i vanishes over F_p keeps
    configuration 0's vector for that leg)."""
    mom, pol0, info = make_inputs(field, n, d, batch, seed, start, None, metric, prime)
    pol = np.empty((batch, states, n, d), dtype=pol0.dtype)
    pol[:, 0] = pol0
    g = metric_signs(d, metric)
    for s in range(1, states):
        _, pol_s, inf = make_inputs(field, n, d, batch, seed + 7919 * s, start, None, metric, prime)
        r = inf["reference"]
        if field == "fp31":
            P = _U64(prime)
            m64, v64, r64 = mom.astype(_U64), pol_s.astype(_U64), r.astype(_U64)
            rp = _fp_dot(r64, m64, P, g)
            coef = _fp_mul(_fp_dot(v64, m64, P, g), _fp_inv(rp, P), P)
            new = _fp_sub(v64, _fp_mul(coef[..., None], r64, P), P).astype(np.uint32)
            pol[:, s] = np.where((rp != 0)[..., None], new, pol0)
        else:
            gf = g.astype(np.float64)
            coef = _c_dot(pol_s, mom, gf) / _c_dot(r, mom, gf)
            pol[:, s] = pol_s - coef[..., None] * r
    return mom, pol, info


def make_config(name: str, batch: int | None = None, seed: int = 0, start: int = 0):
    c = CONFIGS[name]
    return make_inputs(c["field"], c["n"], c["d"], c["batch"] if batch is None else batch,
                       seed, start, c["helicities"])


def make_config_threaded(name: str, batch: int | None = None, seed: int = 0, start: int = 0,
                         threads: int | None = None, chunk: int = 1 << 13):
    """make_config() with the batch cut into chunks generated on a thread pool (numpy releases
    the GIL on the large array operations).  Every draw is a pure function of (seed, global
    point index), so the result is identical to the single-threaded call."""
    import os
    from concurrent.futures import ThreadPoolExecutor
    c = CONFIGS[name]
    batch = c["batch"] if batch is None else batch
    threads = threads or min(32, os.cpu_count() or 1)
    if batch <= chunk or threads <= 1:
        return make_config(name, batch, seed, start)
    offs = list(range(0, batch, chunk))
    with ThreadPoolExecutor(threads) as ex:
        parts = list(ex.map(lambda o: make_config(name, min(chunk, batch - o), seed, start + o), offs))
    mom = np.concatenate([p[0] for p in parts])
    pol = np.concatenate([p[1] for p in parts])
    info = {"redraws": sum(p[2]["redraws"] for p in parts)}
    return mom, pol, info
