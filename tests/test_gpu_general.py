"""Parity of the generalised CUDA path (bg_evaluate and friends) with the
CPU oracle: generic 31-bit primes (FpMont, Montgomery form inside the kernels), Caravel's alternating
metric, several primes per launch, and S state configurations per momentum point
(Eq.(4)).  F_p: bit-exact.  complex128: rule R9 (oracle/rule.py)."""
import numpy as np
import pytest

from paper_2502_07060_b200 import inputs

pytestmark = pytest.mark.gpu

P31 = inputs.P31
PRIMES = [2147483629, 2013265921, 1073741827]
# compiled bg_unit_kernel instances of FpMont / the alternating metric exist for the config shapes;
# the other shapes run bg_general_kernel
SHAPES = [(4, 4, 70), (8, 6, 133), (10, 8, 70), (12, 6, 40), (5, 5, 70), (7, 7, 45), (9, 4, 37), (16, 5, 33)]


@pytest.fixture(scope="module")
def bgl():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (there is no CPU fallback)")
    from paper_2502_07060_b200 import binding
    binding.load()
    return binding


def _gpu(bgl, mom, pol, metric=0, primes=(), want_status=False):
    import torch
    lead = 1 if primes else 0
    status = None
    if want_status:
        status = torch.zeros(mom.shape[:lead + 1], dtype=torch.int32, device="cuda")
    out = bgl.evaluate(bgl.to_device(mom), bgl.to_device(pol), metric=metric, primes=primes, status=status)
    torch.cuda.synchronize()
    if want_status:
        return bgl.to_numpy(out), status.cpu().numpy().astype(np.uint32)
    return bgl.to_numpy(out)


@pytest.mark.parametrize("metric", [0, 1])
@pytest.mark.parametrize("n,d,batch", SHAPES, ids=lambda v: str(v))
def test_generic_primes_bit_exact(bgl, oracle_mod, n, d, batch, metric):
    for prime in PRIMES:
        mom, pol, _ = inputs.make_fp_inputs(n, d, batch, seed=23, prime=prime, metric=metric)
        ref = oracle_mod.evaluate(oracle_mod.FP31, mom, pol, metric=metric, prime=prime, threads=8)
        got = _gpu(bgl, mom[None], pol[None], metric, (prime,))[0]
        assert got.max() < prime and np.array_equal(got, ref), (prime, metric)


@pytest.mark.parametrize("n,d", [(8, 6), (7, 7)])
def test_montgomery_with_the_mersenne_prime_equals_fp31(bgl, n, d):
    mom, pol, _ = inputs.make_fp_inputs(n, d, 100, seed=2)
    a = _gpu(bgl, mom, pol)
    b = _gpu(bgl, mom[None], pol[None], 0, (P31,))[0]
    assert np.array_equal(a, b)


@pytest.mark.parametrize("n,d", [(8, 6), (6, 5), (11, 7), (13, 4)])      # the last two: no compiled instance (bg_rt_kernel)
def test_several_primes_in_one_launch(bgl, oracle_mod, n, d):
    batch = 77
    primes = (PRIMES[0], PRIMES[2], P31, PRIMES[1])
    ins = [inputs.make_fp_inputs(n, d, batch, seed=31 + i, prime=p, metric=1) for i, p in enumerate(primes)]
    mom = np.stack([x[0] for x in ins])
    pol = np.stack([x[1] for x in ins])
    mom[1, 5, 1] = mom[1, 5, 0]                      # P_{1,2}^2 = 0 at point 5 of prime 1: status and inv(0) = 0
    got, st = _gpu(bgl, mom, pol, 1, primes, want_status=True)
    for q, p in enumerate(primes):
        ref, rst = oracle_mod.evaluate(oracle_mod.FP31, mom[q], pol[q], metric=1, prime=p, want_status=True)
        assert np.array_equal(got[q], ref) and np.array_equal(st[q], rst), p
    assert st[1, 5] == 1 and st.sum() == 1


def _extreme(kind, prime, shape, rng):
    if kind == "all_p-1":
        return np.full(shape, prime - 1, np.uint32), np.full(shape, prime - 1, np.uint32)
    if kind == "raw_above_p":
        hi = np.array([0xFFFFFFFF, 0xFFFFFFFE, prime, prime + 1, 2 * prime - 1, 2 * prime, 3 * prime], np.uint64)
        hi = hi[hi < 2 ** 32].astype(np.uint32)
        return rng.choice(hi, size=shape), rng.choice(hi, size=shape)
    pool = np.array([0, 1, 2, prime - 2, prime - 1, prime // 2, prime // 2 + 1, prime], np.uint32)
    pick = lambda: np.where(rng.random(shape) < 0.8, rng.choice(pool, size=shape),
                            rng.integers(0, prime, size=shape, dtype=np.uint32)).astype(np.uint32)
    return pick(), pick()


@pytest.mark.parametrize("metric", [0, 1])
@pytest.mark.parametrize("n,d", [(8, 6), (12, 6), (10, 8), (5, 16), (16, 4)])
def test_generic_primes_extreme_residues(bgl, oracle_mod, n, d, metric):
    """the headroom rules of FpMont (bg_field.cuh): worst-case residues, raw words above p"""
    rng = np.random.default_rng(5 + n + d)
    for prime in PRIMES + [P31]:
        for kind in ("all_p-1", "raw_above_p", "mixed"):
            mom, pol = _extreme(kind, prime, (40, n, d), rng)
            ref, rst = oracle_mod.evaluate(oracle_mod.FP31, mom, pol, metric=metric, prime=prime, want_status=True,
                                           threads=8)
            got, st = _gpu(bgl, mom[None], pol[None], metric, (prime,), want_status=True)
            assert np.array_equal(got[0], ref) and np.array_equal(st[0], rst), (prime, kind)


@pytest.mark.parametrize("n,d,batch", SHAPES, ids=lambda v: str(v))
def test_alternating_metric_fp31(bgl, oracle_mod, n, d, batch):
    mom, pol, _ = inputs.make_fp_inputs(n, d, batch, seed=29, metric=1)
    ref = oracle_mod.evaluate(oracle_mod.FP31, mom, pol, metric=1, threads=8)
    assert np.array_equal(_gpu(bgl, mom, pol, 1), ref)
    assert not np.array_equal(_gpu(bgl, mom, pol, 0), ref)


def test_parke_taylor_over_fp_on_the_gpu(bgl):
    """Eq.(19), exactly, straight from the kernels (alternating metric, d = 4)"""
    n, neg = 6, (0, 1)
    for prime, field_primes in ((P31, ()), (PRIMES[1], (PRIMES[1],))):
        mom, pol, _ = inputs.make_fp_inputs(n, 4, 200, seed=7, prime=prime, metric=1, helicities=(-1, -1, 1, 1, 1, 1))
        got = _gpu(bgl, mom[None], pol[None], 1, field_primes)[0] if field_primes else _gpu(bgl, mom, pol, 1)
        lam, _ = inputs.spinors(mom.astype(np.uint64), 1, inputs.FpOps(prime))
        for b in range(200):
            br = lambda x, y: (int(lam[b, x, 0]) * int(lam[b, y, 1]) - int(lam[b, x, 1]) * int(lam[b, y, 0])) % prime
            den = 1
            for i in range(n):
                den = den * br(i, (i + 1) % n) % prime
            want = 8 * pow(br(*neg), 4, prime) * pow(den, prime - 2, prime) % prime
            assert int(got[b]) == want


@pytest.mark.parametrize("n,d,batch,hel", [(6, 4, 200, (-1, -1, 1, 1, 1, 1)), (12, 6, 40, None), (7, 5, 45, None),
                                           (9, 8, 33, None)], ids=lambda v: str(v))
def test_alternating_metric_complex(bgl, oracle_mod, n, d, batch, hel):
    from oracle import rule
    mom, pol, _ = inputs.make_complex_inputs(n, d, batch, seed=3, helicities=hel, metric=1)
    got = _gpu(bgl, mom, pol, 1)
    dbl = oracle_mod.evaluate(oracle_mod.C128, mom, pol, metric=1, threads=8)
    truth = oracle_mod.evaluate(oracle_mod.C80, mom, pol, metric=1, threads=8).astype(np.clongdouble)
    # rule R9 with the alternating-metric oracle: kappa from the same oracle under seeded perturbations
    rng = np.random.default_rng(rule.SEED)
    kap = np.zeros(batch)
    for _ in range(rule.DRAWS):
        pm = mom * (1 + rule.EPS * (rng.standard_normal(mom.shape) + 1j * rng.standard_normal(mom.shape)))
        pp = pol * (1 + rule.EPS * (rng.standard_normal(pol.shape) + 1j * rng.standard_normal(pol.shape)))
        o = oracle_mod.evaluate(oracle_mod.C128, pm, pp, metric=1, threads=8)
        kap = np.maximum(kap, np.abs(o - dbl) / np.abs(dbl) / rule.EPS)
    ok, st = rule.check(got, {"truth": truth, "dbl": dbl, "kappa": kap})
    assert ok.all() and st["e_g"]["median"] < 1e-12, st


# ---- S state configurations per momentum point ----------------------------------------------------------
@pytest.mark.parametrize("n,d,batch,S", [(8, 6, 133, 4), (8, 6, 70, 16), (8, 6, 33, 1), (12, 6, 40, 3), (4, 4, 70, 2),
                                         (7, 5, 45, 5), (16, 4, 33, 2)], ids=lambda v: str(v))
def test_states_fp(bgl, oracle_mod, n, d, batch, S):
    import torch
    mom, pol, _ = inputs.make_state_inputs("fp31", n, d, batch, S, seed=11)
    mom = mom.copy()
    mom[3, 1] = mom[3, 0]                            # one singular point: status is per momentum point
    ref, rst = oracle_mod.evaluate(oracle_mod.FP31, mom, pol, want_status=True, threads=8)
    status = torch.zeros(batch, dtype=torch.int32, device="cuda")
    out = bgl.evaluate(bgl.to_device(mom), bgl.to_device(pol), status=status)
    torch.cuda.synchronize()
    assert out.shape == (batch, S)
    assert np.array_equal(bgl.to_numpy(out), ref)
    assert np.array_equal(status.cpu().numpy().astype(np.uint32), rst) and rst[3] == 1


def test_states_entry_point_and_generic_prime(bgl, oracle_mod):
    import torch
    n, d, batch, S = 8, 6, 70, 4
    mom, pol, _ = inputs.make_state_inputs("fp31", n, d, batch, S, seed=12)
    dm, dp = bgl.to_device(mom), bgl.to_device(pol)
    out = torch.empty((batch, S), dtype=torch.int32, device="cuda")
    rc = bgl.bg_amplitudes_states(bgl.FIELD_FP31, n, d, batch, S, dm.data_ptr(), dp.data_ptr(), out.data_ptr(), None,
                                  torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    assert rc == bgl.BG_OK
    assert np.array_equal(bgl.to_numpy(out), oracle_mod.evaluate(oracle_mod.FP31, mom, pol, threads=8))
    prime = PRIMES[0]
    mom, pol, _ = inputs.make_state_inputs("fp31", n, d, batch, S, seed=12, metric=1, prime=prime)
    got = bgl.to_numpy(bgl.evaluate(bgl.to_device(mom[None]), bgl.to_device(pol[None]), metric=1, primes=(prime,)))[0]
    torch.cuda.synchronize()
    assert np.array_equal(got, oracle_mod.evaluate(oracle_mod.FP31, mom, pol, metric=1, prime=prime, threads=8))


@pytest.mark.parametrize("n,d,batch,S", [(6, 4, 70, 4), (12, 6, 24, 3), (5, 5, 40, 2)], ids=lambda v: str(v))
def test_states_complex(bgl, oracle_mod, n, d, batch, S):
    import torch
    from oracle import rule
    mom, pol, _ = inputs.make_state_inputs("c128", n, d, batch, S, seed=13)
    out = bgl.to_numpy(bgl.evaluate(bgl.to_device(mom), bgl.to_device(pol)))
    torch.cuda.synchronize()
    for s in range(S):
        ps = np.ascontiguousarray(pol[:, s])
        ok, st = rule.check(out[:, s], rule.evaluate(mom, ps, threads=8))
        assert ok.all() and st["e_g"]["median"] < 1e-12, (s, st)


def test_generalised_argument_checks(bgl):
    import torch
    buf = torch.zeros(1 << 16, dtype=torch.int32, device="cuda")
    p = buf.data_ptr()
    ev = lambda pb, cur=None: bgl.bg_evaluate(pb, 8, p, p + 65536, p + 131072, cur, None, 0)
    assert ev(bgl.problem(0, 4, 4)) == bgl.BG_OK
    assert ev(bgl.problem(0, 4, 4, metric=2)) == bgl.BG_ERR_ARG
    assert ev(bgl.problem(0, 4, 4, states=0)) == bgl.BG_ERR_ARG
    assert ev(bgl.problem(0, 4, 4, primes=(PRIMES[0],))) == bgl.BG_ERR_ARG              # primes only with FPMONT
    assert ev(bgl.problem(2, 4, 4)) == bgl.BG_ERR_ARG                                   # FPMONT without a prime
    assert ev(bgl.problem(2, 4, 4, primes=(PRIMES[0] + 1,))) == bgl.BG_ERR_ARG          # even
    assert ev(bgl.problem(2, 4, 4, primes=((1 << 30) - 35,))) == bgl.BG_ERR_ARG         # below 2^30
    assert ev(bgl.problem(2, 4, 4, primes=(PRIMES[0],))) == bgl.BG_OK
    assert ev(bgl.problem(0, 4, 4, states=2), cur=p + 196608) == bgl.BG_ERR_ARG         # currents need S == 1
    torch.cuda.synchronize()


# ---- bg_state_sum: sum over states of the product of the trees of a cut (Eq.(4)) ---------------
def _state_sum_definition(amps, prime=None):
    """the plain definition, Python ints / long double: out[b] = sum_s prod_t amps[t][b][s]"""
    if prime is None:
        a = [x.astype(np.clongdouble) for x in amps]
        prod = a[0].copy()
        for x in a[1:]:
            prod = prod * x
        return prod.sum(axis=1)
    a = [x.astype(object) % prime for x in amps]          # raw words above p are reduced first
    prod = a[0]
    for x in a[1:]:
        prod = prod * x % prime
    return (prod.sum(axis=1) % prime).astype(np.uint32)


@pytest.mark.parametrize("trees,S,batch", [(1, 1, 70), (2, 16, 1000), (3, 4, 333), (8, 5, 65), (2, 8, 1001), (3, 32, 257),
                                           (2, 64, 100), (2, 128, 77), (2, 12, 99), (4, 256, 9)])
def test_state_sum_fp(bgl, trees, S, batch):
    import torch
    rng = np.random.default_rng(trees * 100 + S)
    for prime, arg in ((P31, 0), (PRIMES[1], PRIMES[1]), (PRIMES[2], PRIMES[2])):
        amps = [rng.integers(0, prime, size=(batch, S), dtype=np.uint32) for _ in range(trees)]
        amps[0][0, :] = prime - 1
        amps[-1][1, 0] = 0xFFFFFFFF                      # a raw word above p is reduced on load
        got = bgl.to_numpy(bgl.state_sum([bgl.to_device(a) for a in amps], prime=arg))
        torch.cuda.synchronize()
        assert np.array_equal(got, _state_sum_definition(amps, prime)), prime


def test_state_sum_complex_and_a_two_tree_cut(bgl, oracle_mod):
    """two trees sharing the state index, as in a two-particle cut: amplitudes from the kernels,
    summed by bg_state_sum, against the oracle's amplitudes summed by the definition"""
    import torch
    n, d, batch, S = 6, 6, 200, 4
    mom_l, pol_l, _ = inputs.make_state_inputs("c128", n, d, batch, S, seed=21)
    mom_r, pol_r, _ = inputs.make_state_inputs("c128", n, d, batch, S, seed=22)
    a_l = bgl.evaluate(bgl.to_device(mom_l), bgl.to_device(pol_l))
    a_r = bgl.evaluate(bgl.to_device(mom_r), bgl.to_device(pol_r))
    got = bgl.to_numpy(bgl.state_sum([a_l, a_r]))
    torch.cuda.synchronize()
    o_l = oracle_mod.evaluate(oracle_mod.C80, mom_l, pol_l, threads=8)
    o_r = oracle_mod.evaluate(oracle_mod.C80, mom_r, pol_r, threads=8)
    want = _state_sum_definition([o_l, o_r])
    scale = (np.abs(o_l) * np.abs(o_r)).sum(axis=1).astype(np.float64)
    assert np.all(np.abs(got - want).astype(np.float64) <= 1e-11 * scale)
    mom, pol, _ = inputs.make_state_inputs("fp31", n, d, batch, S, seed=23)
    a = bgl.evaluate(bgl.to_device(mom), bgl.to_device(pol))
    ref = oracle_mod.evaluate(oracle_mod.FP31, mom, pol, threads=8)
    got = bgl.to_numpy(bgl.state_sum([a, a]))
    torch.cuda.synchronize()
    assert np.array_equal(got, _state_sum_definition([ref, ref], P31))


def test_state_sum_argument_checks(bgl):
    import torch
    buf = torch.zeros(4096, dtype=torch.int32, device="cuda")
    p = buf.data_ptr()
    assert bgl.bg_state_sum(0, 0, 8, 4, [p, p + 1024], p + 2048) == bgl.BG_OK
    assert bgl.bg_state_sum(0, 0, 8, 0, [p], p + 2048) == bgl.BG_ERR_ARG
    assert bgl.bg_state_sum(0, 0, 8, 4, [p] * 9, p + 2048) == bgl.BG_ERR_ARG
    assert bgl.bg_state_sum(0, 0, 8, 4, [p, p + 2048], p + 2048) == bgl.BG_ERR_ARG        # aliasing
    assert bgl.bg_state_sum(2, 12, 8, 4, [p], p + 2048) == bgl.BG_ERR_ARG                 # not a 31-bit odd prime
    assert bgl.bg_state_sum(3, 0, 8, 4, [p], p + 2048) == bgl.BG_ERR_ARG
    assert bgl.bg_state_sum(0, 0, 0, 4, [p], p + 2048) == bgl.BG_OK
    torch.cuda.synchronize()


# ---- K colour orderings per point (Eq.(5)) -----------------------------------------------
def _perms(n, K, seed):
    """K orderings: the identity, the cyclic shift, the reflection, the U(1) insertions of leg 0, then random"""
    rng = np.random.default_rng(seed)
    ident = list(range(n))
    out = [ident, ident[1:] + ident[:1], ident[::-1]]
    out += [ident[1:][:pos] + [0] + ident[1:][pos:] for pos in range(n - 1)]
    while len(out) < K:
        out.append(list(rng.permutation(n - 1)) + [n - 1])
    return np.array(out[:max(K, n + 2)], dtype=np.uint8)


@pytest.mark.parametrize("n,d,batch", [(8, 6, 70), (6, 4, 133), (12, 6, 33), (7, 5, 45), (5, 7, 40), (11, 7, 20)], ids=lambda v: str(v))
def test_orderings_fp(bgl, oracle_mod, n, d, batch):
    import torch
    perms = _perms(n, 24, n)
    mom, pol, _ = inputs.make_fp_inputs(n, d, batch, seed=17)
    mom = mom.copy()
    mom[2, 2] = mom[2, 1]                             # k_2 = k_3 at point 2: singular in the orderings where they touch
    status = torch.zeros(batch, dtype=torch.int32, device="cuda")
    got = bgl.to_numpy(bgl.evaluate(bgl.to_device(mom), bgl.to_device(pol), orderings=perms, status=status))
    torch.cuda.synchronize()
    ref = oracle_mod.orderings(oracle_mod.FP31, mom, pol, perms, threads=8)
    assert got.shape == (batch, len(perms)) and np.array_equal(got, ref)
    st = status.cpu().numpy()
    assert st[2] == 1 and st.sum() == 1
    ok = np.arange(batch) != 2
    # what the colour-ordered amplitudes must obey (pins of the oracle, here straight from the kernels):
    g = got[ok].astype(np.int64)
    assert np.array_equal(g[:, 1], g[:, 0])                                              # cyclicity
    assert np.array_equal(g[:, 2], g[:, 0] if n % 2 == 0 else (P31 - g[:, 0]) % P31)     # reflection
    assert not (g[:, 3:3 + n - 1].sum(axis=1) % P31).any()                               # U(1) decoupling


def test_orderings_on_a_side_stream(bgl, oracle_mod):
    """evaluate(orderings=..., stream=s) with s NOT torch's current stream: the permutation table is a temporary
    of the call and must be uploaded on s (ordered before the kernel, its block reused only in s's order).  The
    current stream is kept busy and churns the allocator meanwhile, which is what exposed the table to reuse."""
    import torch
    n, d, batch = 8, 6, 4000
    perms = _perms(n, 24, n)
    mom, pol, _ = inputs.make_fp_inputs(n, d, batch, seed=23)
    dm, dp = bgl.to_device(mom), bgl.to_device(pol)
    ref = oracle_mod.orderings(oracle_mod.FP31, mom[:300], pol[:300], perms, threads=8)
    torch.cuda.synchronize()
    side = torch.cuda.Stream()
    for rep in range(5):
        big = torch.empty(1 << 26, dtype=torch.uint8, device="cuda")
        big.fill_(rep)                                             # long-running work on the current stream
        out = bgl.evaluate(dm, dp, orderings=perms, stream=side)
        junk = [torch.full((len(perms), n), 255, dtype=torch.uint8, device="cuda") for _ in range(8)]   # same size class
        side.synchronize()
        got = bgl.to_numpy(out)
        assert np.array_equal(got[:300], ref), rep
        del junk, big
    torch.cuda.synchronize()


# ---- orderings x states on the run-time-n tiled kernel (MULTI instantiation of bg_rt_kernel) ------------------------
RT_MULTI = [("fp31", 13, 5, 45, 3, 4, False),      # no compiled instance, one lane per point
            ("fp31", 16, 4, 33, 2, 0, False),      # states only (the caller's order)
            ("fp31", 16, 16, 20, 2, 3, False),     # two lanes per point (16-point tiles)
            ("fp31", 11, 7, 40, 1, 5, False),      # orderings only
            ("fp31", 8, 6, 70, 4, 6, True),        # compiled shapes, forced onto bg_rt_kernel
            ("fp31", 4, 4, 70, 3, 2, True),
            ("c128", 13, 4, 21, 2, 3, False), ("c128", 7, 5, 40, 2, 2, False), ("c128", 12, 6, 24, 2, 2, True)]


@pytest.mark.parametrize("field,n,d,batch,S,K,force", RT_MULTI, ids=lambda v: str(v))
def test_rt_kernel_orderings_and_states(bgl, oracle_mod, field, n, d, batch, S, K, force):
    """S state configurations x K colour orderings per point on shapes without a compiled instance run the tiled
    kernel (specialised == 4), not the one-thread-per-point fallback: bit-exact / rule R9 against the oracle, incl. a
    singular point (status per momentum point, OR over the orderings) and a ragged last tile."""
    import torch
    from oracle import rule
    f = bgl.FIELD_FP31 if field == "fp31" else bgl.FIELD_C128
    perms = _perms(n, K, min(n, K)) if K else None
    mom, pol, _ = inputs.make_state_inputs(field, n, d, batch, S, seed=29)
    mom = mom.copy()
    if field == "fp31":
        mom[3, 1] = mom[3, 0]
    if force:
        bgl.bg_set_kernel_override("rt", 0)
    try:
        pb = bgl.problem(f, n, d, states=S, n_orderings=0 if perms is None else len(perms),
                         orderings_ptr=None if perms is None else 4096)
        ki = bgl.bg_kernel_info_problem(pb)
        assert ki["specialised"] == 4, ki
        status = torch.zeros(batch, dtype=torch.int32, device="cuda")
        got = bgl.to_numpy(bgl.evaluate(bgl.to_device(mom), bgl.to_device(pol), orderings=perms, status=status))
        torch.cuda.synchronize()
    finally:
        bgl.bg_set_kernel_override("default", 0)
    ofield = oracle_mod.FP31 if field == "fp31" else oracle_mod.C128
    if perms is None:
        ref, rst = oracle_mod.evaluate(ofield, mom, pol, want_status=True, threads=8)
    else:
        ref = oracle_mod.orderings(ofield, mom, pol, perms, threads=8)
        rst = np.zeros(batch, np.uint32)
        for sg in perms:
            rst |= oracle_mod.evaluate(ofield, mom[:, list(sg)], pol[..., list(sg), :], want_status=True, threads=8)[1]
    assert got.shape == ref.shape
    if field == "fp31":
        assert np.array_equal(got, ref)
        assert np.array_equal(status.cpu().numpy().astype(np.uint32), rst) and rst[3] == 1
    else:
        g2, pol_s = got.reshape(batch, -1, S), pol
        for k in range(g2.shape[1]):
            sg = list(perms[k]) if perms is not None else list(range(n))
            for s_ in range(S):
                ok, st = rule.check(g2[:, k, s_], rule.evaluate(np.ascontiguousarray(mom[:, sg]),
                                                                np.ascontiguousarray(pol_s[:, s_][:, sg]), threads=8))
                assert ok.all() and st["e_g"]["median"] < 1e-12, (k, s_, st)


def test_orderings_entry_point_states_and_complex(bgl, oracle_mod):
    import torch
    from oracle import rule
    n, d, batch, S = 6, 6, 40, 3
    perms = _perms(n, 12, 3)
    mom, pol, _ = inputs.make_state_inputs("fp31", n, d, batch, S, seed=19)
    got = bgl.to_numpy(bgl.evaluate(bgl.to_device(mom), bgl.to_device(pol), orderings=perms))
    torch.cuda.synchronize()
    assert got.shape == (batch, len(perms), S)
    assert np.array_equal(got, oracle_mod.orderings(oracle_mod.FP31, mom, pol, perms, threads=8))
    # the named entry point
    dm, dp = bgl.to_device(mom), bgl.to_device(np.ascontiguousarray(pol[:, 0]))
    dperm = torch.from_numpy(perms).cuda()
    out = torch.empty((batch, len(perms)), dtype=torch.int32, device="cuda")
    rc = bgl.bg_amplitudes_orderings(bgl.FIELD_FP31, n, d, batch, len(perms), dperm.data_ptr(), dm.data_ptr(),
                                     dp.data_ptr(), out.data_ptr(), None, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    assert rc == bgl.BG_OK and np.array_equal(bgl.to_numpy(out), got[:, :, 0])
    # complex128 (cfg1 shape: bg_reg_kernel cannot loop over orderings, the two-lane tiled kernel runs)
    mom, pol, _ = inputs.make_complex_inputs(6, 4, 64, seed=5, helicities=(-1, -1, 1, 1, 1, 1))
    perms = _perms(6, 10, 4)
    got = bgl.to_numpy(bgl.evaluate(bgl.to_device(mom), bgl.to_device(pol), orderings=perms))
    torch.cuda.synchronize()
    for o, s in enumerate(perms):
        ok, st = rule.check(got[:, o], rule.evaluate(mom[:, list(s)], pol[:, list(s)], threads=8))
        assert ok.all(), (o, st)
