"""CPU oracle for the d-dimensional, square-root-free polarisation states of PAPER.md §2.3
(Eqs.(8)-(18)) -- SURVEY.md 8(f) row f1.

TEST INFRASTRUCTURE (see oracle/__init__.py): plain Python, one vector at a time, exact
Python integers mod p for F_p and Python complex for complex128; it shares nothing with
csrc/bg_states.cu.  Pinned in tests/test_oracle_states.py by the relations the paper itself
tests: orthonormality Eq.(12), transversality, and the completeness relations
Eqs.(13)-(15) for d = 4..10, exactly over F_p.

For a massless d-vector k and a massless 4-vector chi (embedded, Eq.(8)) the D-2 states are

    k_4d = (k^0..k^3),  mu^2 = (k_4d, k_4d),  kb = k_4d - mu^2/(2 (chi, k_4d)) chi      Eqs.(9),(10)
    eps_1 = <kb|gamma^mu|chi] / (2 [kb chi]),  eps_2 = [kb|gamma^mu|chi> / <kb chi>     Eq.(18)
    eps~_1 = eps_2, eps~_2 = eps_1
    eps_3 = kb - mu^2/(2 (chi, k_4d)) chi,  eps~_3 = eps_3 / mu^2                       Eq.(18)
    eps_4 = (0,0,0,0, k_5, -k_4, 0..),  eps~_4 = eps_4 / mu_6^2                          Eq.(18)
    eps_x (x >= 5) = (0,0,0,0, k_4 k_q, .., k_{q-1} k_q, -mu_q^2, 0..),  q = x + 1      Eq.(16)
    eps~_x = eps_x / (mu_q^2 mu_{q+1}^2),   mu_q^2 = k_4^2 + .. + k_{q-1}^2              Eq.(17)

Readings (R13-R15; the paper's text is garbled or silent here):
 R13 Eq.(10) prints (xi, k_4d) where (chi, k_4d) is meant (cf. Eq.(11)).  <a|gamma^mu|b] is the
     vector 2 vec(lam_a lamt_b^T) of the bispinor lam_a lamt_b^T, so that eps_1 = vec(lam_kb
     lamt_chi^T)/[kb chi] and eps_2 = 2 vec(lam_chi lamt_kb^T)/<kb chi>; (eps_1, eps_2) = -1.
     Spinor conventions as in paper_2502_07060_b200/inputs.py: M = lam lamt^T, lam = (M00, M10),
     lamt = (1, M01/M00), <ab> = a0 b1 - a1 b0.
 R14 Eq.(16) as printed (entries k_4 k_x .. k_{x-1} k_x, then -mu_{x+1}^2) is not transverse; with
     the state label x mapped to the position q = x + 1 of its last non-zero component (the
     paper's own "eps_x^{mu > x+1} = 0", and eps_4 of Eq.(11)) it reads (k_4 k_q, .., k_{q-1} k_q,
     -mu_q^2), which is transverse, has (eps_x, eps_x) = -mu_q^2 mu_{q+1}^2 and reproduces eps_4 up
     to the factor k_4 that Eq.(18) drops.  The sqrt-free split for x >= 5 (not printed) follows
     Eq.(18)'s pattern: eps_x unnormalised, eps~_x = eps_x / (mu_q^2 mu_{q+1}^2).
 R15 Alternating metric: with s_y = -g_yy for the extra dimensions y >= 4,
     mu_q^2 = sum_{y<q} s_y k_y^2, eps_x^q = -s_q mu_q^2, eps~_x = eps_x / (s_q mu_q^2 mu_{q+1}^2),
     eps_4 = (k_5, -s_4 s_5 k_4), eps~_4 = eps_4 / (s_4 s_5 mu_6^2) -- the unique choice that keeps
     transversality and (eps_x, eps~_x) = -1; for the mostly-minus metric all s_y = 1 and the
     formulas are the paper's.  The mostly-minus spinors contain i: over F_p they exist only
     when p = 1 mod 4 (sqrt(-1) in F_p); with the alternating metric they are rational.
"""
from __future__ import annotations

MOSTLY_MINUS, ALTERNATING = 0, 1


class FieldFp:
    """Python ints mod p"""

    def __init__(self, p: int):
        self.p = p
        self.imag = None
        if p % 4 == 1:                      # sqrt(-1) = g^((p-1)/4) for a quadratic non-residue g
            g = 2
            while pow(g, (p - 1) // 2, p) != p - 1:
                g += 1
            self.imag = pow(g, (p - 1) // 4, p)

    def num(self, x):
        return int(x) % self.p

    def add(self, a, b):
        return (a + b) % self.p

    def sub(self, a, b):
        return (a - b) % self.p

    def mul(self, a, b):
        return a * b % self.p

    def inv(self, a):
        if a % self.p == 0:
            raise ZeroDivisionError("singular configuration")
        return pow(a, self.p - 2, self.p)


class FieldComplex:
    imag = 1j

    def num(self, x):
        return complex(x)

    def add(self, a, b):
        return a + b

    def sub(self, a, b):
        return a - b

    def mul(self, a, b):
        return a * b

    def inv(self, a):
        return 1.0 / a


def metric_sign(mu: int, metric: int) -> int:
    if metric == MOSTLY_MINUS:
        return 1 if mu == 0 else -1
    return 1 if mu % 2 == 0 else -1


def dot(F, x, y, metric):
    s = F.num(0)
    for mu in range(len(x)):
        t = F.mul(x[mu], y[mu])
        s = F.add(s, t) if metric_sign(mu, metric) > 0 else F.sub(s, t)
    return s


def _spinors(F, p, metric):
    """lam, lamt of a massless 4-vector"""
    M00 = F.add(p[0], p[3])
    if metric == MOSTLY_MINUS:
        if F.imag is None:
            raise ValueError("the mostly-minus spinors need sqrt(-1) in the field (p = 1 mod 4)")
        ip2 = F.mul(F.num(F.imag), p[2])
        M01, M10 = F.sub(p[1], ip2), F.add(p[1], ip2)
    else:
        M01, M10 = F.add(p[1], p[2]), F.sub(p[1], p[2])
    return (M00, M10), (F.num(1), F.mul(M01, F.inv(M00)))


def _bracket(F, a, b):
    return F.sub(F.mul(a[0], b[1]), F.mul(a[1], b[0]))


def _vec(F, lam, lamt, metric):
    """the 4-vector of the bispinor lam lamt^T"""
    N00, N01, N10, N11 = (F.mul(lam[0], lamt[0]), F.mul(lam[0], lamt[1]), F.mul(lam[1], lamt[0]),
                          F.mul(lam[1], lamt[1]))
    half = F.inv(F.num(2))
    if metric == MOSTLY_MINUS:
        c2 = F.mul(F.sub(N10, N01), F.inv(F.mul(F.num(2), F.num(F.imag))))
    else:
        c2 = F.mul(half, F.sub(N01, N10))
    return [F.mul(half, F.add(N00, N11)), F.mul(half, F.add(N01, N10)), c2, F.mul(half, F.sub(N00, N11))]


def states(F, k, chi, metric=MOSTLY_MINUS):
    """k: d numbers (massless), chi: 4 numbers (massless in the 4-d block).  Returns (eps, eps_tilde):
    two lists of D-2 vectors of d numbers, eps[x-1] = eps_x."""
    d = len(k)
    k = [F.num(x) for x in k]
    chi = [F.num(x) for x in chi]
    zero = F.num(0)
    k4 = k[:4]
    mu2 = dot(F, k4, k4, metric)
    chik = dot(F, chi, k4, metric)
    c = F.mul(mu2, F.inv(F.mul(F.num(2), chik)))                      # mu^2 / (2 (chi, k_4d))
    kb = [F.sub(k4[mu], F.mul(c, chi[mu])) for mu in range(4)]         # Eq.(10)
    lk, ltk = _spinors(F, kb, metric)
    lc, ltc = _spinors(F, chi, metric)
    pad = [zero] * (d - 4)
    e1 = [F.mul(x, F.inv(_bracket(F, ltk, ltc))) for x in _vec(F, lk, ltc, metric)] + pad
    e2 = [F.mul(F.mul(F.num(2), x), F.inv(_bracket(F, lk, lc))) for x in _vec(F, lc, ltk, metric)] + pad
    eps, til = [e1, e2], [e2, e1]
    if d >= 5:
        e3 = [F.sub(kb[mu], F.mul(c, chi[mu])) for mu in range(4)] + pad
        imu2 = F.inv(mu2)
        eps.append(e3)
        til.append([F.mul(x, imu2) for x in e3])
    s = lambda y: -metric_sign(y, metric)                               # s_y = -g_yy
    musq = {4: zero}                                                    # mu_q^2 = sum_{4 <= y < q} s_y k_y^2
    for q in range(5, d + 1):
        t = F.mul(k[q - 1], k[q - 1])
        musq[q] = F.add(musq[q - 1], t) if s(q - 1) > 0 else F.sub(musq[q - 1], t)
    for q in range(5, d):                                               # state x = q - 1 = 4 .. d-2
        e = [zero] * d
        if q == 5:
            e[4] = k[5]
            e[5] = F.sub(zero, k[4]) if s(4) * s(5) > 0 else k[4]
            den = musq[6] if s(4) * s(5) > 0 else F.sub(zero, musq[6])
        else:
            for y in range(4, q):
                e[y] = F.mul(k[y], k[q])
            e[q] = F.sub(zero, musq[q]) if s(q) > 0 else musq[q]
            den = F.mul(musq[q], musq[q + 1])
            if s(q) < 0:
                den = F.sub(zero, den)
        iden = F.inv(den)
        eps.append(e)
        til.append([F.mul(x, iden) for x in e])
    return eps, til


def states_batch(field: str, mom, chi, metric=MOSTLY_MINUS, prime=(1 << 31) - 1):
    """mom [count, d], chi [count, 4] (numpy) -> eps, eps_tilde [count, d-2, d] (uint32 / complex128)"""
    import numpy as np
    F = FieldFp(prime) if field == "fp31" else FieldComplex()
    count, d = mom.shape
    dt = np.uint32 if field == "fp31" else np.complex128
    eps = np.zeros((count, d - 2, d), dtype=dt)
    til = np.zeros((count, d - 2, d), dtype=dt)
    for b in range(count):
        e, t = states(F, [x.item() for x in mom[b]], [x.item() for x in chi[b]], metric)
        eps[b] = np.array(e, dtype=object).astype(dt)
        til[b] = np.array(t, dtype=object).astype(dt)
    return eps, til
