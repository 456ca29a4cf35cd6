"""Pins for the CPU oracle (oracle/bg_oracle.c) -- everything here runs on CPU.

The oracle is the only thing the CUDA path is compared with, so it is pinned to
things other than itself: the paper's closed form (Parke-Taylor, Eq.(19)
PAPER.md:186), brute-force diagram sums with the FULL three-gluon vertex, the
identities a colour-ordered amplitude must obey (Ward PAPER.md:184, cyclicity,
reflection, U(1) decoupling), current conservation for every intermediate
current, an exact-rational evaluation reduced mod p (ties F_p to the complex
oracle), and the survey's worked examples (tests/golden/worked_examples.txt).
"""
import os
from fractions import Fraction

import numpy as np
import pytest

import independent as ind
from paper_2502_07060_b200 import inputs

P = ind.P31
GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "worked_examples.txt")


def _worked_inputs(n, d):
    k = [[((7 * i + 3 * mu + i * mu) % 11) - 5 for mu in range(d)] for i in range(n)]
    e = [[((5 * i + 2 * mu + 3 * i * mu + 1) % 13) - 6 for mu in range(d)] for i in range(n)]
    return k, e


def _golden_rows():
    rows = []
    with open(GOLDEN) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            n, d, num, den, modp, cval = line.split()
            rows.append((int(n), int(d), None if num == "-" else Fraction(int(num), int(den)),
                         int(modp), float(cval)))
    return rows


@pytest.mark.parametrize("row", _golden_rows(), ids=lambda r: f"n{r[0]}d{r[1]}")
def test_worked_examples(oracle_mod, row):
    n, d, exact, modp, cval = row
    k, e = _worked_inputs(n, d)
    kf = (np.array(k) % P).astype(np.uint32)[None]
    ef = (np.array(e) % P).astype(np.uint32)[None]
    assert int(oracle_mod.amplitudes(oracle_mod.FP31, kf, ef)[0]) == modp
    kc = np.array(k, dtype=np.complex128)[None]
    ec = np.array(e, dtype=np.complex128)[None]
    got = oracle_mod.amplitudes(oracle_mod.C128, kc, ec)[0]
    assert abs(got - cval) <= 1e-12 * abs(cval)
    got80 = oracle_mod.amplitudes(oracle_mod.C80, kc, ec)[0]
    assert abs(complex(got80) - cval) <= 1e-12 * abs(cval)
    # independent exact-rational re-derivation (third implementation)
    kq = [[Fraction(x) for x in v] for v in k]
    eq = [[Fraction(x) for x in v] for v in e]
    val, _, _ = ind.bg_python(kq, eq)
    if exact is not None:
        assert val == exact
    assert ind.frac_to_fp(val) == modp
    assert abs(float(val) - cval) <= 1e-12 * abs(cval)


# ----------------------------------------------------------------- Parke-Taylor
@pytest.mark.parametrize("n", [4, 5, 6, 7, 8])
@pytest.mark.parametrize("negpos", ["adjacent", "split", "wrap"])
def test_parke_taylor(oracle_mod, n, negpos):
    """Eq.(19): MHV amplitudes.  i-free normalisation (R2):
    out = 2^(n-3) <ab>^4 / (<12>...<n1>) with the sqrt-free states of inputs.py."""
    neg = {"adjacent": (0, 1), "split": (0, 2), "wrap": (1, n - 1)}[negpos]
    hel = [1] * n
    for a in neg:
        hel[a] = -1
    mom, pol, _ = inputs.make_complex_inputs(n, 4, 256, seed=11, helicities=hel)
    out = oracle_mod.amplitudes(oracle_mod.C128, mom, pol)
    truth = oracle_mod.amplitudes(oracle_mod.C80, mom, pol)
    lam, _ = inputs.spinors(mom)
    rel = np.empty(256)
    rel80 = np.empty(256)
    for b in range(256):
        pt = ind.parke_taylor([tuple(lam[b, i]) for i in range(n)], neg)
        rel[b] = abs(out[b] - pt) / abs(pt)
        rel80[b] = abs(complex(truth[b]) - pt) / abs(pt)
    # well-conditioned bulk: tight; ill-conditioned tail (high-order zero of the MHV
    # amplitude, R9) is bounded loosely
    assert np.median(rel) < 1e-12
    assert np.percentile(rel, 90) < 1e-10
    assert rel.max() < 1e-6
    assert np.median(rel80) < 1e-12


def test_helicity_states_are_what_the_formula_needs():
    """eps+.eps- = -1, eps.eps = 0, eps.k = 0 (Eq.(12))"""
    mom, pol_m, info = inputs.make_complex_inputs(5, 4, 32, seed=3, helicities=[-1] * 5)
    _, pol_p, _ = inputs.make_complex_inputs(5, 4, 32, seed=3, helicities=[1] * 5)

    def dot(x, y):
        return x[..., 0] * y[..., 0] - (x[..., 1:] * y[..., 1:]).sum(-1)

    assert np.allclose(dot(pol_p, pol_m), -1, atol=1e-9)
    assert np.allclose(dot(pol_p, pol_p), 0, atol=1e-9)
    assert np.allclose(dot(pol_m, pol_m), 0, atol=1e-9)
    assert np.allclose(dot(pol_p, mom), 0, atol=1e-9)
    assert np.allclose(dot(pol_m, mom), 0, atol=1e-9)


# ------------------------------------------------------------ diagram sums
@pytest.mark.parametrize("n,d", [(4, 4), (5, 4), (5, 6), (6, 4), (6, 6)])
def test_bruteforce_diagrams_fp(oracle_mod, n, d):
    assert ind.count_trees(n) == {4: 3, 5: 10, 6: 38}[n]
    mom, pol, _ = inputs.make_fp_inputs(n, d, 6, seed=5)
    out = oracle_mod.amplitudes(oracle_mod.FP31, mom, pol)
    for b in range(6):
        mf = [[ind.Fp(x) for x in v] for v in mom[b]]
        pf = [[ind.Fp(x) for x in v] for v in pol[b]]
        assert ind.diagram_sum(mf, pf).v == int(out[b])


@pytest.mark.parametrize("n,d", [(4, 4), (5, 6), (6, 4)])
def test_bruteforce_diagrams_complex(oracle_mod, n, d):
    mom, pol, _ = inputs.make_complex_inputs(n, d, 4, seed=6)
    out = oracle_mod.amplitudes(oracle_mod.C128, mom, pol)
    for b in range(4):
        val = ind.diagram_sum([list(v) for v in mom[b]], [list(v) for v in pol[b]])
        assert abs(val - out[b]) <= 1e-9 * abs(val)


def test_diagram_sum_needs_the_full_vertex():
    """sanity of the pin itself: on UNPHYSICAL inputs the full-vertex diagram sum and the
    reduced-V3 recursion differ (Eq.(7) assumes conserved currents, R4)"""
    k, e = _worked_inputs(4, 4)
    kq = [[ind.Fp(x) for x in v] for v in k]
    eq = [[ind.Fp(x) for x in v] for v in e]
    assert ind.diagram_sum(kq, eq).v != ind.bg_python(kq, eq)[0].v


# ------------------------------------------------------------ identities over F_p
def _amp_fp(oracle_mod, mom, pol, order):
    order = list(order)
    return oracle_mod.amplitudes(oracle_mod.FP31, mom[:, order], pol[:, order])


@pytest.mark.parametrize("n,d", [(4, 4), (5, 4), (6, 4), (6, 6), (7, 5), (8, 6)])
def test_ward_identity_fp(oracle_mod, n, d):
    """eps_g -> k_g gives exactly 0 for every leg g"""
    mom, pol, _ = inputs.make_fp_inputs(n, d, 16, seed=2)
    base = oracle_mod.amplitudes(oracle_mod.FP31, mom, pol)
    assert np.count_nonzero(base) > 0
    for g in range(n):
        p2 = pol.copy()
        p2[:, g] = mom[:, g]
        assert not oracle_mod.amplitudes(oracle_mod.FP31, mom, p2).any()


@pytest.mark.parametrize("n,d", [(4, 4), (5, 4), (6, 4), (6, 6), (7, 5), (8, 6)])
def test_cyclicity_reflection_u1_fp(oracle_mod, n, d):
    mom, pol, _ = inputs.make_fp_inputs(n, d, 16, seed=4)
    ident = list(range(n))
    a0 = _amp_fp(oracle_mod, mom, pol, ident).astype(np.int64)
    # cyclicity A(2..n,1) = A(1..n): exercises leg n being special in BG
    for shift in range(1, n):
        assert np.array_equal(_amp_fp(oracle_mod, mom, pol, ident[shift:] + ident[:shift]), a0)
    # reflection A(n..1) = (-1)^n A(1..n)
    refl = _amp_fp(oracle_mod, mom, pol, ident[::-1]).astype(np.int64)
    assert np.array_equal(refl, a0 if n % 2 == 0 else (P - a0) % P)
    # U(1) decoupling: leg 1 inserted at every position among (2..n-1), n fixed last
    tot = np.zeros(16, dtype=np.int64)
    rest = ident[1:]
    for pos in range(n - 1):
        order = rest[:pos] + [0] + rest[pos:]
        tot = (tot + _amp_fp(oracle_mod, mom, pol, order)) % P
    assert not tot.any()


@pytest.mark.parametrize("n,d", [(5, 4), (8, 6), (10, 8)])
def test_current_conservation_fp(oracle_mod, n, d):
    """P_{i,j} . J(i..j) = 0 for EVERY multi-gluon current incl. the top one:
    pins the intermediate currents, not only the final number"""
    mom, pol, _ = inputs.make_fp_inputs(n, d, 4, seed=8)
    out, cur = oracle_mod.amplitudes(oracle_mod.FP31, mom, pol, want_currents=True)
    m = n - 1
    for b in range(4):
        for i in range(m):
            for j in range(i + 1, m):
                Pij = [sum(int(x) for x in mom[b, i:j + 1, mu]) % P for mu in range(d)]
                Jij = [int(x) for x in cur[b, i, j]]
                s = (Pij[0] * Jij[0] - sum(a * c for a, c in zip(Pij[1:], Jij[1:]))) % P
                assert s == 0
                assert any(Jij)
        # and the single-gluon currents are the polarisations
        for i in range(m):
            assert np.array_equal(cur[b, i, i], pol[b, i])


def test_identities_complex(oracle_mod):
    n, d = 6, 6
    mom, pol, _ = inputs.make_complex_inputs(n, d, 32, seed=9)
    a0 = oracle_mod.amplitudes(oracle_mod.C128, mom, pol)
    scale = np.abs(a0)
    ident = list(range(n))
    cyc = oracle_mod.amplitudes(oracle_mod.C128, mom[:, ident[1:] + ident[:1]], pol[:, ident[1:] + ident[:1]])
    assert np.all(np.abs(cyc - a0) <= 1e-8 * scale)
    p2 = pol.copy()
    p2[:, 2] = mom[:, 2]
    ward = oracle_mod.amplitudes(oracle_mod.C128, mom, p2)
    assert np.median(np.abs(ward) / scale) < 1e-10


# ------------------------------------------------- cross-field homomorphism
@pytest.mark.parametrize("n,d", [(4, 4), (5, 5), (6, 4), (7, 6)])
def test_cross_field_homomorphism(oracle_mod, n, d):
    """rational inputs evaluated exactly (Fraction), reduced mod p == F_p oracle on the
    inputs mod p; float() of it == complex oracle.  Ties the two oracle fields together,
    so the Parke-Taylor pin (complex only) also constrains the F_p code path."""
    rng = np.random.default_rng(1234 + 10 * n + d)
    num = rng.integers(-9, 10, size=(n, d))
    den = rng.integers(1, 6, size=(n, d))
    kq = [[Fraction(int(a), int(b)) for a, b in zip(r, s)] for r, s in zip(num, den)]
    num2 = rng.integers(-9, 10, size=(n, d))
    den2 = rng.integers(1, 6, size=(n, d))
    eq = [[Fraction(int(a), int(b)) for a, b in zip(r, s)] for r, s in zip(num2, den2)]
    val, J, _ = ind.bg_python(kq, eq)
    kf = np.array([[ind.frac_to_fp(x) for x in v] for v in kq], dtype=np.uint32)[None]
    ef = np.array([[ind.frac_to_fp(x) for x in v] for v in eq], dtype=np.uint32)[None]
    out, cur = oracle_mod.amplitudes(oracle_mod.FP31, kf, ef, want_currents=True)
    assert int(out[0]) == ind.frac_to_fp(val)
    m = n - 1
    for i in range(1, m + 1):          # every intermediate current too
        for j in range(i, m + 1):
            assert [int(x) for x in cur[0, i - 1, j - 1]] == [ind.frac_to_fp(x) for x in J[i, j]]
    kc = np.array([[float(x) for x in v] for v in kq], dtype=np.complex128)[None]
    ec = np.array([[float(x) for x in v] for v in eq], dtype=np.complex128)[None]
    outc = oracle_mod.amplitudes(oracle_mod.C128, kc, ec)
    assert abs(outc[0] - float(val)) <= 1e-9 * abs(float(val))


# ------------------------------------------------- special / degenerate cases
def test_zero_invariant_sets_status_and_uses_inv0_eq_0(oracle_mod):
    """DESIGN.md R6: inv(0) := 0 and status bit0.  Make P_{1,2}^2 = 0 by k_2 = k_1 (massless)."""
    mom, pol, _ = inputs.make_fp_inputs(5, 4, 2, seed=1)
    mom = mom.copy()
    mom[0, 1] = mom[0, 0]
    out, cur, st = oracle_mod.amplitudes(oracle_mod.FP31, mom, pol, want_currents=True, want_status=True)
    assert st[0] == 1 and st[1] == 0
    assert not cur[0, 0, 1].any()          # J(1..2) = bracket * inv(0) = 0


def test_inputs_above_p_are_reduced(oracle_mod):
    mom, pol, _ = inputs.make_fp_inputs(4, 4, 4, seed=1)
    ref = oracle_mod.amplitudes(oracle_mod.FP31, mom, pol)
    big = mom.astype(np.uint64) + P
    assert big.max() < 2 ** 32
    assert np.array_equal(oracle_mod.amplitudes(oracle_mod.FP31, big.astype(np.uint32), pol), ref)


def test_bad_arguments(oracle_mod):
    z = np.zeros((1, 3, 4), dtype=np.uint32)
    with pytest.raises(ValueError):
        oracle_mod.amplitudes(oracle_mod.FP31, z, z)
    assert oracle_mod.modulus() == P
    e = np.zeros((0, 4, 4), dtype=np.uint32)
    assert oracle_mod.amplitudes(oracle_mod.FP31, e, e).shape == (0,)


def test_threads_give_identical_results(oracle_mod):
    mom, pol, _ = inputs.make_fp_inputs(6, 4, 257, seed=1)
    a = oracle_mod.amplitudes(oracle_mod.FP31, mom, pol, threads=1)
    b = oracle_mod.amplitudes(oracle_mod.FP31, mom, pol, threads=3)
    assert np.array_equal(a, b)


def test_multilinearity_in_polarisations(oracle_mod):
    """the amplitude is linear in each eps_i (what makes the unnormalised states of the
    generator legitimate)"""
    mom, pol, _ = inputs.make_fp_inputs(6, 6, 8, seed=12)
    a0 = oracle_mod.amplitudes(oracle_mod.FP31, mom, pol).astype(np.uint64)
    p3 = pol.astype(np.uint64)
    p3[:, 2] = (p3[:, 2] * 3) % P
    a3 = oracle_mod.amplitudes(oracle_mod.FP31, mom, p3.astype(np.uint32)).astype(np.uint64)
    assert np.array_equal(a3, (a0 * 3) % P)


def test_truth_type_is_extended_precision(oracle_mod):
    """rule R9 (oracle/rule.py) uses the long double instantiation as truth: it must carry a 64-bit
    mantissa and really differ from the double evaluation at rounding level"""
    from oracle import rule
    rule.assert_long_double_is_80_bit()
    mom, pol, _ = inputs.make_complex_inputs(8, 6, 64, seed=2)
    t = oracle_mod.amplitudes(oracle_mod.C80, mom, pol)
    dbl = oracle_mod.amplitudes(oracle_mod.C128, mom, pol)
    assert t.dtype == np.clongdouble
    rel = (np.abs(dbl.astype(np.clongdouble) - t) / np.abs(t)).astype(np.float64)
    assert (rel > 0).mean() > 0.9 and rel.max() < 1e-11 and np.median(rel) > 1e-18


def test_rule_r9_accepts_the_oracle_and_rejects_a_wrong_result(oracle_mod):
    from oracle import rule
    mom, pol, _ = inputs.make_complex_inputs(6, 4, 512, seed=3, helicities=(-1, -1, 1, 1, 1, 1))
    ref = rule.evaluate(mom, pol, threads=4)
    ok, st = rule.check(ref["dbl"], ref)
    assert ok.all() and st["fail"] == 0
    assert st["pass_by_1e-10"] + st["pass_by_16_e_d"] + st["pass_by_kappa_only"] == 512
    bad = ref["dbl"].copy()
    bad[7] *= 1 + 1e-6
    ok, st = rule.check(bad, ref)
    assert not ok[7] and st["fail"] >= 1
