"""Pins for oracle/states.py, the d-dimensional sqrt-free polarisation states of PAPER.md §2.3
(Eqs.(8)-(18)): the relations the paper itself tests in d = 4..10 (test_states.py):
transversality, orthonormality Eq.(12) and the completeness relations Eqs.(13)-(15), here EXACTLY
over F_p (alternating metric with p = 2^31-1; mostly-minus metric with a prime = 1 mod 4, where
sqrt(-1) exists) and to rounding over complex128.  A wrong sign, index or normalisation anywhere in
Eqs.(10),(16)-(18) breaks one of them."""
import numpy as np
import pytest

from oracle import states as st
from paper_2502_07060_b200 import inputs

P31 = inputs.P31
P_1MOD4 = 2013265921          # 15 * 2^27 + 1


def _massless(field, d, count, seed, metric, prime):
    """`count` massless d-vectors k and massless 4-vectors chi from the seeded generator"""
    mom, _, info = inputs.make_inputs(field, 4, d, count, seed=seed, metric=metric, prime=prime)
    ref4 = inputs.make_inputs(field, 4, 4, count, seed=seed + 1, metric=metric, prime=prime)[2]["reference"]
    return mom[:, 0], ref4[:, 0]


def _check_point(F, k, chi, metric, tol):
    d = len(k)
    eps, til = st.states(F, k, chi, metric)
    assert len(eps) == len(til) == d - 2
    kk = [F.num(x) for x in k]
    zero = lambda x: abs(x) <= tol if tol else x == 0
    eq = lambda a, b: zero(F.sub(a, b))
    g = [st.metric_sign(mu, metric) for mu in range(d)]
    assert zero(st.dot(F, kk, kk, metric))
    minus_one = F.sub(F.num(0), F.num(1))
    for x in range(d - 2):
        assert zero(st.dot(F, kk, eps[x], metric)) and zero(st.dot(F, kk, til[x], metric))      # transverse
        for y in range(d - 2):
            want = minus_one if x == y else F.num(0)                                            # Eq.(12)
            assert eq(st.dot(F, eps[x], til[y], metric), want), (x, y)
    assert eps[0] == til[1] and eps[1] == til[0]                                                # Eq.(18)
    # completeness, Eq.(13): sum_x eps_x^mu eps~_x^nu = -g^{mu nu} + (k^mu eta^nu + k^nu eta^mu)/(k, eta)
    if d == 4:
        eta = [F.num(x) for x in chi]
    else:
        eta = kk[:4] + [F.sub(F.num(0), x) for x in kk[4:]]                                     # Eq.(15)
    ike = F.inv(st.dot(F, kk, eta, metric))
    mu2 = st.dot(F, kk[:4], kk[:4], metric)
    for mu in range(d):
        for nu in range(d):
            lhs = F.num(0)
            for x in range(d - 2):
                lhs = F.add(lhs, F.mul(eps[x][mu], til[x][nu]))
            rhs = F.mul(F.add(F.mul(kk[mu], eta[nu]), F.mul(kk[nu], eta[mu])), ike)
            if mu == nu:
                rhs = F.sub(rhs, F.num(g[mu]))
            assert eq(lhs, rhs), (mu, nu)
            if d > 4:                                                                           # Eq.(14)
                if mu < 4 and nu < 4:
                    blk = F.mul(F.mul(kk[mu], kk[nu]), F.inv(mu2))
                elif mu >= 4 and nu >= 4:
                    blk = F.sub(F.num(0), F.mul(F.mul(kk[mu], kk[nu]), F.inv(mu2)))
                else:
                    blk = F.num(0)
                if mu == nu:
                    blk = F.sub(blk, F.num(g[mu]))
                assert eq(lhs, blk), (mu, nu)


@pytest.mark.parametrize("d", range(4, 11))
@pytest.mark.parametrize("metric,prime", [(st.ALTERNATING, P31), (st.ALTERNATING, P_1MOD4), (st.MOSTLY_MINUS, P_1MOD4)])
def test_states_fp_exact(d, metric, prime):
    F = st.FieldFp(prime)
    ks, chis = _massless("fp31", d, 6, 40 + d, metric, prime)
    for b in range(6):
        _check_point(F, [int(x) for x in ks[b]], [int(x) for x in chis[b]], metric, 0)


@pytest.mark.parametrize("d", range(4, 11))
@pytest.mark.parametrize("metric", [st.MOSTLY_MINUS, st.ALTERNATING])
def test_states_complex(d, metric):
    F = st.FieldComplex()
    ks, chis = _massless("c128", d, 6, 50 + d, metric, P31)
    for b in range(6):
        _check_point(F, [complex(x) for x in ks[b]], [complex(x) for x in chis[b]], metric, 1e-9)


def test_mostly_minus_needs_sqrt_minus_one():
    F = st.FieldFp(P31)                                 # 2^31-1 = 3 mod 4: no sqrt(-1)
    assert F.imag is None and st.FieldFp(P_1MOD4).imag ** 2 % P_1MOD4 == P_1MOD4 - 1
    ks, chis = _massless("fp31", 6, 1, 3, st.MOSTLY_MINUS, P31)
    with pytest.raises(ValueError):
        st.states(F, [int(x) for x in ks[0]], [int(x) for x in chis[0]], st.MOSTLY_MINUS)


def test_lower_dimensional_states_embed_trivially():
    """"eps_x^{mu > x+1} = 0, so that lower dimensional states are trivially embedded in higher
    dimensions": the first states of a d-vector with vanishing last component are the
    states of the (d-1)-vector"""
    F = st.FieldFp(P31)
    ks, chis = _massless("fp31", 7, 3, 9, st.ALTERNATING, P31)
    for b in range(3):
        k7 = [int(x) for x in ks[b]]
        chi = [int(x) for x in chis[b]]
        e7, t7 = st.states(F, k7, chi, st.ALTERNATING)
        for x in range(3, 5):                       # eps_4, eps_5 depend on k^4..k^{x+1} only
            assert all(v == 0 for v in e7[x][x + 3:])
        assert e7[3][4] == k7[5]                    # eps_4 = (0,0,0,0,k_5, -s_4 s_5 k_4, 0): Eq.(18)


def test_states_batch_shapes():
    ks, chis = _massless("c128", 6, 5, 1, st.MOSTLY_MINUS, P31)
    eps, til = st.states_batch("c128", ks, chis)
    assert eps.shape == til.shape == (5, 4, 6) and eps.dtype == np.complex128
    ks, chis = _massless("fp31", 8, 5, 1, st.ALTERNATING, P31)
    eps, til = st.states_batch("fp31", ks, chis, st.ALTERNATING)
    assert eps.shape == (5, 6, 8) and eps.dtype == np.uint32 and eps.max() < P31
