"""Independent re-derivations used to PIN the oracle (tests only).

Nothing here is shared with oracle/ or with the CUDA path:

* `Fp`            exact arithmetic mod p with Python ints (a third number type);
* `diagram_sum`   brute-force sum over every planar tree diagram with cubic and
                  quartic vertices, each diagram evaluated separately with the FULL
                  symmetric three-gluon vertex (all momenta outgoing) -- not the
                  reduced V3 of Eq.(7) -- so it checks both the recursion's
                  bookkeeping and the current-conservation step hidden in Eq.(7)
                  (reading R4);
* `bg_python`     the recursion typed again in pure Python over any number type
                  (used with fractions.Fraction for the cross-field homomorphism);
* `parke_taylor`  Eq.(19), in the i-free normalisation of DESIGN.md R2.
"""
from __future__ import annotations

from fractions import Fraction

P31 = (1 << 31) - 1


class Fp:
    """exact arithmetic mod P with Python ints; subclasses made by fp_class(p) use another prime"""
    __slots__ = ("v",)
    P = P31

    def __init__(self, v):
        self.v = int(v) % self.P

    def __add__(self, o):
        return type(self)(self.v + _v(o))

    __radd__ = __add__

    def __sub__(self, o):
        return type(self)(self.v - _v(o))

    def __rsub__(self, o):
        return type(self)(_v(o) - self.v)

    def __mul__(self, o):
        return type(self)(self.v * _v(o))

    __rmul__ = __mul__

    def __neg__(self):
        return type(self)(-self.v)

    def __truediv__(self, o):
        return type(self)(self.v * pow(_v(o), self.P - 2, self.P))

    def __rtruediv__(self, o):
        return type(self)(_v(o) * pow(self.v, self.P - 2, self.P))

    def __eq__(self, o):
        return self.v == _v(o) % self.P

    def __repr__(self):
        return f"Fp({self.v} mod {self.P})"


def fp_class(p: int):
    """the same exact arithmetic modulo another prime (generic 31-bit primes)"""
    return type(f"Fp_{p}", (Fp,), {"P": p, "__slots__": ()})


def _v(o):
    return o.v if isinstance(o, Fp) else int(o)


def is_prime(n: int) -> bool:
    """deterministic Miller-Rabin for n < 3.3e24 (first 13 primes as bases)"""
    if n < 2:
        return False
    small = (2, 3, 5, 7, 11, 13, 17, 19, 23, 29, 31, 37, 41)
    for q in small:
        if n % q == 0:
            return n == q
    dd, r = n - 1, 0
    while dd % 2 == 0:
        dd //= 2
        r += 1
    for a in small:
        x = pow(a, dd, n)
        if x in (1, n - 1):
            continue
        for _ in range(r - 1):
            x = x * x % n
            if x == n - 1:
                break
        else:
            return False
    return True


def frac_to_fp(x: Fraction, p: int = P31) -> int:
    return x.numerator % p * pow(x.denominator % p, p - 2, p) % p


_ALTERNATING = False


class alternating_metric:
    """context manager: every product below uses diag(+,-,+,-,...) instead of the
    mostly-minus metric"""

    def __enter__(self):
        global _ALTERNATING
        self.prev, _ALTERNATING = _ALTERNATING, True

    def __exit__(self, *exc):
        global _ALTERNATING
        _ALTERNATING = self.prev


def mdot(x, y):
    s = x[0] * y[0]
    for mu in range(1, len(x)):
        minus = (mu % 2 == 1) if _ALTERNATING else True
        s = s - x[mu] * y[mu] if minus else s + x[mu] * y[mu]
    return s


def vadd(x, y):
    return [a + b for a, b in zip(x, y)]


def vsub(x, y):
    return [a - b for a, b in zip(x, y)]


def vscale(c, x):
    return [c * a for a in x]


# ------------------------------------------------------------------ diagrams
def _trees(i, j):
    """all planar trees with cubic/quartic vertices over the ordered legs i..j"""
    if i == j:
        return [("leaf", i)]
    out = []
    for k in range(i, j):
        for a in _trees(i, k):
            for b in _trees(k + 1, j):
                out.append(("v3", a, b))
    for k in range(i, j - 1):
        for l in range(k + 1, j):
            for a in _trees(i, k):
                for b in _trees(k + 1, l):
                    for c in _trees(l + 1, j):
                        out.append(("v4", a, b, c))
    return out


def count_trees(n):
    return len(_trees(1, n - 1))


def _eval(tree, mom, pol, root):
    """returns (off-shell current of this single diagram, its momentum)"""
    if tree[0] == "leaf":
        i = tree[1]
        return list(pol[i - 1]), list(mom[i - 1])
    subs = [_eval(t, mom, pol, False) for t in tree[1:]]
    if tree[0] == "v3":
        (A, P), (B, Q) = subs
        K = [-(a + b) for a, b in zip(P, Q)]            # all momenta outgoing: K+P+Q = 0
        # V3^{mu nu rho}(K,P,Q) = g^{nu rho}(P-Q)^mu + g^{rho mu}(Q-K)^nu + g^{mu nu}(K-P)^rho
        t1 = vscale(mdot(A, B), vsub(P, Q))
        t2 = vscale(mdot(vsub(Q, K), A), B)
        t3 = vscale(mdot(vsub(K, P), B), A)
        cur = vadd(vadd(t1, t2), t3)
        tot = vadd(P, Q)
    else:
        (A, P), (B, Q), (C, R) = subs
        cur = vsub(vsub(vscale(2 * mdot(A, C), B), vscale(mdot(A, B), C)), vscale(mdot(B, C), A))
        tot = vadd(vadd(P, Q), R)
    if not root:
        cur = vscale(1 / mdot(tot, tot), cur)
    return cur, tot


def diagram_sum(mom, pol):
    """mom, pol: n lists of d numbers (Fp, Fraction or complex).  Sum over diagrams of
    eps_n . (diagram), no propagator on the root line."""
    n = len(mom)
    total = None
    for t in _trees(1, n - 1):
        cur, _ = _eval(t, mom, pol, True)
        val = mdot(pol[n - 1], cur)
        total = val if total is None else total + val
    return total


# ------------------------------------------------------------- recursion again
def bg_python(mom, pol):
    n, d = len(mom), len(mom[0])
    m = n - 1
    zero = mom[0][0] - mom[0][0]
    P = {}
    J = {}
    for i in range(1, m + 1):
        acc = [zero] * d
        for j in range(i, m + 1):
            acc = vadd(acc, mom[j - 1])
            P[i, j] = acc
        J[i, i] = list(pol[i - 1])
    for L in range(2, m + 1):
        for i in range(1, m - L + 2):
            j = i + L - 1
            acc = [zero] * d
            for k in range(i, j):
                A, B, Pa, Q = J[i, k], J[k + 1, j], P[i, k], P[k + 1, j]
                acc = vadd(acc, vscale(mdot(A, B), vsub(Pa, Q)))
                acc = vadd(acc, vscale(2 * mdot(Q, A), B))
                acc = vsub(acc, vscale(2 * mdot(Pa, B), A))
            for k in range(i, j - 1):
                for l in range(k + 1, j):
                    A, B, C = J[i, k], J[k + 1, l], J[l + 1, j]
                    acc = vadd(acc, vscale(2 * mdot(A, C), B))
                    acc = vsub(acc, vscale(mdot(A, B), C))
                    acc = vsub(acc, vscale(mdot(B, C), A))
            if L < m:
                acc = vscale(1 / mdot(P[i, j], P[i, j]), acc)
            J[i, j] = acc
    return mdot(pol[n - 1], J[1, m]), J, P


# ------------------------------------------------------------- Parke-Taylor
def parke_taylor(lams, neg):
    """i-free MHV value for legs with holomorphic spinors lams (list of (l0,l1)),
    negative-helicity legs neg=(a,b) 0-based:  2^(n-3) <ab>^4 / (<12><23>...<n1>)."""
    n = len(lams)

    def br(x, y):
        return lams[x][0] * lams[y][1] - lams[x][1] * lams[y][0]

    den = 1.0
    for i in range(n):
        den = den * br(i, (i + 1) % n)
    a, b = neg
    return 2.0 ** (n - 3) * br(a, b) ** 4 / den
