"""Pins for the generalised oracle entry (oracle.evaluate): generic 31-bit primes, Caravel's
alternating metric diag(+,-,+,-,..) and S state configurations per momentum point
(Eq.(4)).  Everything here runs on CPU.

What fixes what:
* generic prime    -- exact rationals reduced mod p' (worked examples of tests/golden/ and random
                      rational points, final value AND every current), brute-force diagram sums mod
                      p', Ward / cyclicity / reflection / U(1) on generator points mod p';
* alternating      -- Parke-Taylor, Eq.(19), EXACTLY over F_p (the spinors of a (2,2)
  metric             signature vector are rational: the pin SURVEY.md 8(c) says needs this metric) and
                      over complex128; diagram sums and the rational cross-check typed with that
                      metric; the complex map q2 -> i q2 that turns one metric into the other;
* states           -- the S-configuration call equals S independent calls (no sharing in the oracle).
"""
import os
from fractions import Fraction

import numpy as np
import pytest

import independent as ind
from paper_2502_07060_b200 import inputs

P31 = ind.P31
# 2^31-19 (the largest prime below 2^31-1), 15*2^27+1 (= 1 mod 4), 2^30+3 (just above 2^30)
PRIMES = [2147483629, 2013265921, 1073741827]
GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "worked_examples.txt")


def test_the_test_primes_are_prime():
    for p in PRIMES + [P31]:
        assert ind.is_prime(p) and (1 << 30) < p < (1 << 31)
    assert not ind.is_prime(2147483647 - 2) and not ind.is_prime((1 << 30) + 1)


def _worked_inputs(n, d):
    k = [[((7 * i + 3 * mu + i * mu) % 11) - 5 for mu in range(d)] for i in range(n)]
    e = [[((5 * i + 2 * mu + 3 * i * mu + 1) % 13) - 6 for mu in range(d)] for i in range(n)]
    return k, e


def _golden_exact():
    rows = []
    with open(GOLDEN) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            n, d, num, den, _, _ = line.split()
            if num != "-":
                rows.append((int(n), int(d), Fraction(int(num), int(den))))
    return rows


# ------------------------------------------------------------------ generic primes
@pytest.mark.parametrize("prime", PRIMES)
def test_worked_examples_mod_other_primes(oracle_mod, prime):
    """the survey's exact rationals (tests/golden/worked_examples.txt) reduced mod p'"""
    for n, d, exact in _golden_exact():
        k, e = _worked_inputs(n, d)
        kf = (np.array(k) % prime).astype(np.uint32)[None]
        ef = (np.array(e) % prime).astype(np.uint32)[None]
        got = oracle_mod.evaluate(oracle_mod.FP31, kf, ef, prime=prime)
        assert int(got[0]) == ind.frac_to_fp(exact, prime)


@pytest.mark.parametrize("prime", PRIMES)
@pytest.mark.parametrize("metric", [0, 1])
def test_rational_points_mod_p_every_current(oracle_mod, prime, metric):
    rng = np.random.default_rng(99 + prime % 1000 + metric)
    for n, d in [(4, 4), (5, 5), (6, 4), (7, 6)]:
        kq = [[Fraction(int(a), int(b)) for a, b in zip(rng.integers(-9, 10, d), rng.integers(1, 6, d))]
              for _ in range(n)]
        eq = [[Fraction(int(a), int(b)) for a, b in zip(rng.integers(-9, 10, d), rng.integers(1, 6, d))]
              for _ in range(n)]
        if metric:
            with ind.alternating_metric():
                val, J, _ = ind.bg_python(kq, eq)
        else:
            val, J, _ = ind.bg_python(kq, eq)
        kf = np.array([[ind.frac_to_fp(x, prime) for x in v] for v in kq], dtype=np.uint32)[None]
        ef = np.array([[ind.frac_to_fp(x, prime) for x in v] for v in eq], dtype=np.uint32)[None]
        out, cur = oracle_mod.evaluate(oracle_mod.FP31, kf, ef, metric=metric, prime=prime, want_currents=True)
        assert int(out[0]) == ind.frac_to_fp(val, prime)
        for (i, j), vec in J.items():
            assert [int(x) for x in cur[0, i - 1, j - 1]] == [ind.frac_to_fp(x, prime) for x in vec]


@pytest.mark.parametrize("prime,metric", [(PRIMES[0], 0), (PRIMES[1], 1), (PRIMES[2], 0), (P31, 1)])
def test_bruteforce_diagrams(oracle_mod, prime, metric):
    """all planar cubic+quartic trees with the FULL three-gluon vertex, mod p', either metric"""
    F = ind.fp_class(prime)
    for n, d in [(4, 4), (5, 6), (6, 5)]:
        mom, pol, _ = inputs.make_fp_inputs(n, d, 3, seed=5, prime=prime, metric=metric)
        out = oracle_mod.evaluate(oracle_mod.FP31, mom, pol, metric=metric, prime=prime)
        for b in range(3):
            mf = [[F(x) for x in v] for v in mom[b]]
            pf = [[F(x) for x in v] for v in pol[b]]
            if metric:
                with ind.alternating_metric():
                    want = ind.diagram_sum(mf, pf).v
            else:
                want = ind.diagram_sum(mf, pf).v
            assert want == int(out[b])


@pytest.mark.parametrize("prime,metric", [(PRIMES[0], 0), (PRIMES[1], 0), (PRIMES[2], 1), (P31, 1)])
def test_identities(oracle_mod, prime, metric):
    """generator points are physical for (prime, metric); Ward, cyclicity, reflection, U(1) hold exactly"""
    n, d = 6, 6
    mom, pol, _ = inputs.make_fp_inputs(n, d, 12, seed=4, prime=prime, metric=metric)
    assert mom.max() < prime and pol.max() < prime
    g = inputs.metric_signs(d, metric)
    mo, po = mom.astype(object), pol.astype(object)
    assert not (mo.sum(axis=1) % prime).any()
    assert not ((mo * mo * g).sum(-1) % prime).any() and not ((mo * po * g).sum(-1) % prime).any()

    def amp(order, pl=pol):
        order = list(order)
        return oracle_mod.evaluate(oracle_mod.FP31, mom[:, order], pl[:, order], metric=metric,
                                   prime=prime).astype(np.int64)

    ident = list(range(n))
    a0 = amp(ident)
    assert np.count_nonzero(a0) == 12
    for g_ in range(n):
        p2 = pol.copy()
        p2[:, g_] = mom[:, g_]
        assert not amp(ident, p2).any()
    assert np.array_equal(amp(ident[2:] + ident[:2]), a0)
    assert np.array_equal(amp(ident[::-1]), a0)                     # n even: (-1)^n = +1
    tot = np.zeros(12, dtype=np.int64)
    for pos in range(n - 1):
        tot = (tot + amp(ident[1:][:pos] + [0] + ident[1:][pos:])) % prime
    assert not tot.any()


def test_prime_argument_default_and_mersenne(oracle_mod):
    mom, pol, _ = inputs.make_fp_inputs(6, 5, 16, seed=1)
    a = oracle_mod.amplitudes(oracle_mod.FP31, mom, pol)
    assert np.array_equal(a, oracle_mod.evaluate(oracle_mod.FP31, mom, pol, prime=P31))
    assert np.array_equal(a, oracle_mod.evaluate(oracle_mod.FP31, mom, pol, prime=0))
    with pytest.raises(ValueError):
        oracle_mod.evaluate(oracle_mod.FP31, mom, pol, metric=2)


# ------------------------------------------------------------------ alternating metric
def _parke_taylor_fp(lam, neg, prime):
    """2^(n-3) <ab>^4 / (<12>..<n1>) mod prime from integer spinors lam [n][2]"""
    n = len(lam)
    br = lambda x, y: (int(lam[x][0]) * int(lam[y][1]) - int(lam[x][1]) * int(lam[y][0])) % prime
    den = 1
    for i in range(n):
        den = den * br(i, (i + 1) % n) % prime
    return pow(2, n - 3, prime) * pow(br(*neg), 4, prime) % prime * pow(den, prime - 2, prime) % prime


@pytest.mark.parametrize("prime", [P31] + PRIMES)
@pytest.mark.parametrize("n,neg", [(4, (0, 1)), (5, (0, 1)), (5, (1, 3)), (6, (0, 1)), (6, (2, 5)), (7, (0, 3)),
                                   (8, (0, 1))])
def test_parke_taylor_exactly_over_fp(oracle_mod, prime, n, neg):
    """Eq.(19), with the alternating metric: spinors, states and the closed form are
    all rational, so the F_p oracle must reproduce the formula EXACTLY (i-free normalisation,
    DESIGN.md R2: out = 2^(n-3) <ab>^4 / (<12>...<n1>))"""
    hel = [1] * n
    for a in neg:
        hel[a] = -1
    mom, pol, _ = inputs.make_fp_inputs(n, 4, 24, seed=13, prime=prime, metric=1, helicities=hel)
    out = oracle_mod.evaluate(oracle_mod.FP31, mom, pol, metric=1, prime=prime)
    lam, _ = inputs.spinors(mom.astype(np.uint64), 1, inputs.FpOps(prime))
    assert np.count_nonzero(out) == 24
    for b in range(24):
        assert int(out[b]) == _parke_taylor_fp(lam[b], neg, prime)


def test_fp_helicity_states_satisfy_eq12():
    """(eps+, eps-) = -1, (eps, eps) = 0, (eps, k) = 0 exactly (Eq.(12))"""
    n = 5
    mom, pm, _ = inputs.make_fp_inputs(n, 4, 16, seed=3, metric=1, helicities=[-1] * n)
    _, pp, _ = inputs.make_fp_inputs(n, 4, 16, seed=3, metric=1, helicities=[1] * n)
    g = inputs.metric_signs(4, 1)
    dot = lambda x, y: (x.astype(object) * y.astype(object) * g).sum(-1) % P31
    assert (dot(pp, pm) == P31 - 1).all()
    for x in (pp, pm):
        assert not dot(x, x).any() and not dot(x, mom).any()


@pytest.mark.parametrize("n", [4, 6, 8])
def test_parke_taylor_complex_alternating(oracle_mod, n):
    hel = [-1, -1] + [1] * (n - 2)
    mom, pol, _ = inputs.make_complex_inputs(n, 4, 128, seed=11, helicities=hel, metric=1)
    out = oracle_mod.evaluate(oracle_mod.C128, mom, pol, metric=1)
    lam, _ = inputs.spinors(mom, 1)
    rel = np.array([abs(out[b] - ind.parke_taylor([tuple(lam[b, i]) for i in range(n)], (0, 1))) for b in range(128)])
    rel /= np.abs(out)
    assert np.median(rel) < 1e-12 and np.percentile(rel, 90) < 1e-10


def test_metrics_are_related_by_q2_to_i_q2(oracle_mod):
    """(q0,q1,q2,q3,..) with the alternating metric and (q0,q1,i q2,q3,i q4,..) with the mostly-minus
    one have the same products, hence the same amplitude (complex oracle)"""
    n, d = 6, 6
    mom, pol, _ = inputs.make_complex_inputs(n, d, 32, seed=2, metric=1)
    alt = oracle_mod.evaluate(oracle_mod.C128, mom, pol, metric=1)
    T = np.ones(d, dtype=np.complex128)
    T[2::2] = 1j
    mm = oracle_mod.evaluate(oracle_mod.C128, mom * T, pol * T, metric=0)
    assert np.all(np.abs(alt - mm) <= 1e-9 * np.abs(alt))
    assert not np.allclose(alt, oracle_mod.evaluate(oracle_mod.C128, mom, pol, metric=0))


# ------------------------------------------------------------------ state configurations
@pytest.mark.parametrize("field", ["fp31", "c128"])
def test_states_equal_independent_calls(oracle_mod, field):
    n, d, B, S = 6, 6, 9, 5
    f = oracle_mod.FP31 if field == "fp31" else oracle_mod.C128
    mom, pol0, _ = inputs.make_inputs(field, n, d, B, seed=1)
    pols = [pol0] + [inputs.make_inputs(field, n, d, B, seed=1 + s)[1] for s in range(1, S)]
    pol = np.stack(pols, axis=1)                                    # [B, S, n, d]
    out, cur, st = oracle_mod.evaluate(f, mom, pol, want_currents=True, want_status=True, threads=2)
    assert out.shape == (B, S) and cur.shape == (B, S, n - 1, n - 1, d)
    for s in range(S):
        o1, c1 = oracle_mod.amplitudes(f, mom, pols[s], want_currents=True)
        assert np.array_equal(out[:, s], o1) and np.array_equal(cur[:, s], c1)
    assert not st.any()


# ------------------------------------------------------------------ colour orderings
def test_orderings_are_independent_calls_and_obey_the_identities(oracle_mod):
    """oracle.orderings (Eq.(5)) = one literal evaluation per ordering; the sum over the
    n-1 insertions of leg 1 vanishes (U(1) decoupling), cyclic shifts agree"""
    n, d = 6, 5
    mom, pol, _ = inputs.make_fp_inputs(n, d, 10, seed=6)
    ident = list(range(n))
    perms = [ident, ident[2:] + ident[:2]] + [ident[1:][:pos] + [0] + ident[1:][pos:] for pos in range(n - 1)]
    out = oracle_mod.orderings(oracle_mod.FP31, mom, pol, perms)
    assert out.shape == (10, len(perms))
    for o, s in enumerate(perms):
        assert np.array_equal(out[:, o], oracle_mod.amplitudes(oracle_mod.FP31, mom[:, s], pol[:, s]))
    assert np.array_equal(out[:, 0], out[:, 1])
    assert not (out[:, 2:].astype(np.int64).sum(axis=1) % P31).any()
