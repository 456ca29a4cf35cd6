"""Parity of the CUDA path (through the C ABI) with the CPU oracle, element by element.

F_p: bit-exact.  complex128: DESIGN.md reading R9, implemented ONCE in oracle/rule.py (also
used by smoke() and bench.py): with t the 80-bit oracle on the same double inputs,
e_g = |gpu - t|/|t|, e_d = |oracle_double - t|/|t| and kappa the condition number of the point
estimated by the oracle, every point must satisfy  e_g <= max(1e-10, 16 e_d, 64 kappa 2^-53);
the full-size tests record how many points needed which branch (gpurun_out/r9_stats.jsonl).
"""
import json
import os

import numpy as np
import pytest

from paper_2502_07060_b200 import inputs

pytestmark = pytest.mark.gpu

P = inputs.P31


@pytest.fixture(scope="module")
def bgl():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (there is no CPU fallback)")
    from paper_2502_07060_b200 import binding
    binding.load()
    return binding


@pytest.fixture
def select_kernel(bgl):
    """restrict the kernel selection for one test (bg_set_kernel_override), default again afterwards"""
    def choose(kind, warps=0):
        bgl.bg_set_kernel_override(kind, warps)
    yield choose
    bgl.bg_set_kernel_override("default", 0)


def _gpu_amplitudes(bgl, mom, pol, want_status=False):
    import torch
    dm, dp = bgl.to_device(mom), bgl.to_device(pol)
    status = torch.zeros(mom.shape[0], dtype=torch.int32, device="cuda") if want_status else None
    out = bgl.amplitudes(dm, dp, status=status)
    torch.cuda.synchronize()
    if want_status:
        return bgl.to_numpy(out), status.cpu().numpy().astype(np.uint32)
    return bgl.to_numpy(out)


def _rule(mom, pol, got, tag=None, threads=8):
    """-> (ok, stats) of rule R9; stats of tagged calls are appended to gpurun_out/r9_stats.jsonl"""
    from oracle import rule
    ok, stats = rule.check(got, rule.evaluate(mom, pol, threads=threads))
    out_dir = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "gpurun_out")
    if tag and os.path.isdir(out_dir):
        with open(os.path.join(out_dir, "r9_stats.jsonl"), "a") as f:
            f.write(json.dumps({"case": tag, **stats}) + "\n")
    return ok, stats


def _assert_rule(mom, pol, got, tag=None, threads=8):
    ok, st = _rule(mom, pol, got, tag, threads)
    assert ok.all(), f"{st['fail']} of {st['points']} points outside rule R9: {st}"
    assert st["e_g"]["median"] < 1e-12, st
    return st


# sizes span several 32-point tiles and a ragged tail
FP_SHAPES = [(4, 4, 1024), (8, 6, 517), (10, 8, 197), (12, 6, 133),     # the config shapes
             (5, 5, 99), (6, 4, 200), (7, 5, 77), (9, 7, 45), (5, 16, 40), (16, 4, 37), (13, 9, 35),
             (11, 4, 70), (11, 5, 45), (11, 6, 70), (11, 8, 40), (12, 4, 70), (12, 5, 45), (12, 8, 40)]


@pytest.mark.parametrize("n,d,batch", FP_SHAPES, ids=lambda v: str(v))
def test_fp_bit_exact(bgl, oracle_mod, n, d, batch):
    mom, pol, _ = inputs.make_fp_inputs(n, d, batch, seed=21)
    ref = oracle_mod.amplitudes(oracle_mod.FP31, mom, pol, threads=8)
    got = _gpu_amplitudes(bgl, mom, pol)
    assert got.dtype == np.uint32 and got.max() < P
    assert np.array_equal(got, ref)


C_SHAPES = [(6, 4, 515, (-1, -1, 1, 1, 1, 1)), (12, 6, 70, None), (5, 5, 99, None), (8, 6, 130, None),
            (4, 4, 64, (-1, 1, -1, 1)), (9, 10, 33, None),
            (15, 12, 21, None)]     # general kernel with fewer than 32 threads per block (15 KB per point)


@pytest.mark.parametrize("n,d,batch,hel", C_SHAPES, ids=lambda v: str(v))
def test_complex_within_rule(bgl, oracle_mod, n, d, batch, hel):
    mom, pol, _ = inputs.make_complex_inputs(n, d, batch, seed=22, helicities=hel)
    _assert_rule(mom, pol, _gpu_amplitudes(bgl, mom, pol))


@pytest.mark.parametrize("batch", [1, 31, 32, 33, 65])
def test_ragged_batches(bgl, oracle_mod, batch):
    mom, pol, _ = inputs.make_fp_inputs(8, 6, batch, seed=5)
    assert np.array_equal(_gpu_amplitudes(bgl, mom, pol), oracle_mod.amplitudes(oracle_mod.FP31, mom, pol))


def test_empty_batch_is_a_noop(bgl):
    assert bgl.bg_amplitudes(0, 8, 6, 0, 0, 0, 0, 0) == bgl.BG_OK


def test_unphysical_inputs_worked_examples(bgl):
    """the map is defined for arbitrary inputs (R4): survey worked examples"""
    for n, d, want in [(4, 4, 509929092), (5, 6, 139101349), (6, 4, 1080021013), (8, 6, 1802767521)]:
        k = np.array([[((7 * i + 3 * mu + i * mu) % 11) - 5 for mu in range(d)] for i in range(n)])
        e = np.array([[((5 * i + 2 * mu + 3 * i * mu + 1) % 13) - 6 for mu in range(d)] for i in range(n)])
        got = _gpu_amplitudes(bgl, (k % P).astype(np.uint32)[None], (e % P).astype(np.uint32)[None])
        assert int(got[0]) == want


def test_zero_invariant_status_and_value(bgl, oracle_mod):
    mom, pol, _ = inputs.make_fp_inputs(6, 4, 40, seed=3)
    mom = mom.copy()
    mom[7, 1] = mom[7, 0]          # P_{1,2}^2 = 0 at point 7
    mom[33, 3] = mom[33, 2]        # P_{3,4}^2 = 0 at point 33
    ref, rst = oracle_mod.amplitudes(oracle_mod.FP31, mom, pol, want_status=True)
    got, gst = _gpu_amplitudes(bgl, mom, pol, want_status=True)
    assert rst[7] == 1 and rst[33] == 1 and rst.sum() == 2
    assert np.array_equal(gst, rst)
    assert np.array_equal(got, ref)


def test_inputs_above_p_are_reduced(bgl, oracle_mod):
    mom, pol, _ = inputs.make_fp_inputs(5, 4, 64, seed=1)
    big_m = (mom.astype(np.uint64) + P).astype(np.uint32)
    big_p = (pol.astype(np.uint64) + P).astype(np.uint32)
    big_p[:, :, 0] = 0xFFFFFFFF                   # = 2p+1 = 1 mod p
    pol1 = pol.copy()
    pol1[:, :, 0] = 1
    ref = oracle_mod.amplitudes(oracle_mod.FP31, mom, pol1)
    assert np.array_equal(_gpu_amplitudes(bgl, big_m, big_p), ref)


@pytest.mark.parametrize("field,n,d", [("fp31", 8, 6), ("fp31", 5, 5), ("c128", 6, 4)])
def test_currents(bgl, oracle_mod, field, n, d):
    import torch
    mom, pol, _ = inputs.make_inputs(field, n, d, 70, seed=9)
    f = oracle_mod.FP31 if field == "fp31" else oracle_mod.C128
    ref, rcur = oracle_mod.amplitudes(f, mom, pol, want_currents=True)
    out, cur, st = bgl.currents(bgl.to_device(mom), bgl.to_device(pol))
    torch.cuda.synchronize()
    out, cur = bgl.to_numpy(out), bgl.to_numpy(cur)
    m = n - 1
    iu = np.triu_indices(m)
    if field == "fp31":
        assert np.array_equal(out, ref)
        assert np.array_equal(cur[:, iu[0], iu[1]], rcur[:, iu[0], iu[1]])
    else:
        _assert_rule(mom, pol, out)
        a, b = cur[:, iu[0], iu[1]], rcur[:, iu[0], iu[1]]
        assert np.all(np.abs(a - b) <= 1e-9 * (np.abs(b).max(axis=-1, keepdims=True)))
    assert not st.cpu().numpy().any()


@pytest.mark.parametrize("field,n,d,batch", [("fp31", 8, 6, 5000), ("c128", 6, 4, 3000)])
def test_host_entry_point(bgl, oracle_mod, field, n, d, batch):
    """bg_amplitudes_host: H2D, kernel, D2H pipelined in chunks (here 1024-point chunks)"""
    import torch
    mom, pol, _ = inputs.make_inputs(field, n, d, batch, seed=13)
    f = bgl.FIELD_FP31 if field == "fp31" else bgl.FIELD_C128
    ws = torch.empty(bgl.bg_host_workspace_bytes(f, n, d, 1024), dtype=torch.uint8, device="cuda")
    status = np.zeros(batch, dtype=np.uint32)
    out = bgl.amplitudes_host(mom, pol, workspace=ws, status=status)
    ref = oracle_mod.amplitudes(oracle_mod.FP31 if field == "fp31" else oracle_mod.C128, mom, pol, threads=8)
    if field == "fp31":
        assert np.array_equal(out, ref)
    else:
        _assert_rule(mom, pol, out)
    assert not status.any()


def test_error_codes(bgl):
    import torch
    buf = torch.zeros(4096, dtype=torch.int32, device="cuda")
    p = buf.data_ptr()
    assert bgl.bg_amplitudes(0, 3, 4, 8, p, p + 1024, p + 2048, 0) == bgl.BG_ERR_ARG      # n too small
    assert bgl.bg_amplitudes(0, 17, 4, 8, p, p + 1024, p + 2048, 0) == bgl.BG_ERR_ARG
    assert bgl.bg_amplitudes(0, 4, 3, 8, p, p + 1024, p + 2048, 0) == bgl.BG_ERR_ARG      # d too small
    assert bgl.bg_amplitudes(3, 4, 4, 8, p, p + 1024, p + 2048, 0) == bgl.BG_ERR_ARG      # field
    assert bgl.bg_amplitudes(2, 4, 4, 8, p, p + 1024, p + 2048, 0) == bgl.BG_ERR_ARG      # FPMONT needs a prime
    assert bgl.bg_amplitudes(0, 4, 4, -1, p, p + 1024, p + 2048, 0) == bgl.BG_ERR_ARG     # batch
    assert bgl.bg_amplitudes(0, 4, 4, 8, 0, p + 1024, p + 2048, 0) == bgl.BG_ERR_ARG      # null
    assert bgl.bg_amplitudes(0, 4, 4, 8, p + 4, p + 1024, p + 2048, 0) == bgl.BG_ERR_ARG  # misaligned
    assert bgl.bg_amplitudes(0, 4, 4, 8, p, p + 1024, p, 0) == bgl.BG_ERR_ARG             # aliasing
    assert bgl.bg_amplitudes(0, 4, 4, 8, p, p + 1024, p + 2048, 0) == bgl.BG_OK
    torch.cuda.synchronize()


def test_async_on_caller_stream(bgl, oracle_mod):
    import torch
    mom, pol, _ = inputs.make_fp_inputs(8, 6, 300, seed=17)
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        dm, dp = bgl.to_device(mom), bgl.to_device(pol)
        out = bgl.amplitudes(dm, dp, stream=s)
    s.synchronize()
    assert np.array_equal(bgl.to_numpy(out), oracle_mod.amplitudes(oracle_mod.FP31, mom, pol))


# ---- full-size workloads in the launch configuration bench.py times ------------------------------
@pytest.mark.parametrize("name", ["cfg0", "cfg2", "cfg3", "cfg4a"])
def test_full_size_fp_every_point(bgl, oracle_mod, name):
    """EVERY point of the F_p configs against the oracle (a few seconds on the host cores)"""
    mom, pol, _ = inputs.make_config_threaded(name)
    got = _gpu_amplitudes(bgl, mom, pol)
    ref = oracle_mod.amplitudes(oracle_mod.FP31, mom, pol, threads=os.cpu_count() or 8)
    assert np.array_equal(got, ref)
    assert got.max() < P and np.count_nonzero(got) > 0.99 * got.size


@pytest.mark.parametrize("name", ["cfg1", "cfg4b"])
def test_full_size_complex(bgl, oracle_mod, name):
    """EVERY point of both complex configs under rule R9 (2^20 n=6 points and 2^16 n=12 points are each some
    ten seconds of the 80-bit oracle on the host cores).  Branch statistics are recorded."""
    cfg = inputs.CONFIGS[name]
    mom, pol, _ = inputs.make_config_threaded(name)
    got = _gpu_amplitudes(bgl, mom, pol)
    assert np.isfinite(got.view(np.float64)).all()
    _assert_rule(mom, pol, got, tag=f"{name} default kernel, {cfg['batch']} points", threads=os.cpu_count() or 8)
    if name == "cfg1":   # config 1 is MHV: the whole batch can be checked against Parke-Taylor
        lam, _ = inputs.spinors(mom)
        br = lambda a, b: lam[:, a, 0] * lam[:, b, 1] - lam[:, a, 1] * lam[:, b, 0]
        den = np.ones(cfg["batch"], dtype=np.complex128)
        for i in range(6):
            den *= br(i, (i + 1) % 6)
        pt = 8.0 * br(0, 1) ** 4 / den                     # 2^(n-3) <12>^4 / (<12>...<61>)
        rel = np.abs(got - pt) / np.abs(pt)
        assert np.median(rel) < 1e-12 and np.mean(rel < 1e-9) > 0.995


# ---- every compiled kernel family / warps-per-tile variant (bg_set_kernel_override) --------------------
VARIANTS = [("fp31", 8, 6, "unit1", 4), ("fp31", 8, 6, "unit1", 6), ("fp31", 8, 6, "unit1", 2),
            ("fp31", 4, 4, "unit1", 1), ("fp31", 10, 8, "unit1", 8), ("fp31", 10, 8, "unit1", 4),
            ("fp31", 12, 6, "unit1", 8), ("fp31", 12, 6, "unit1", 16), ("fp31", 12, 6, "unit1", 4),
            ("fp31", 8, 6, "general", 0), ("fp31", 12, 6, "general", 0), ("c128", 6, 4, "general", 0),
            ("c128", 6, 4, "reg", 4), ("c128", 6, 4, "unit2", 2), ("c128", 6, 4, "unit2", 4),
            ("c128", 6, 4, "unit1", 2), ("c128", 6, 4, "unit1", 4),
            ("c128", 12, 6, "unit2", 16), ("c128", 12, 6, "unit2", 8), ("c128", 12, 6, "unit2", 4),
            # the shapes of the paper's own benchmarks (bg_inst_paper.cu)
            ("fp31", 6, 4, "unit1", 2), ("fp31", 8, 4, "unit1", 4), ("fp31", 9, 4, "unit1", 4), ("fp31", 6, 6, "unit1", 2),
            ("fp31", 9, 6, "unit1", 4), ("fp31", 6, 8, "unit1", 2), ("fp31", 8, 8, "unit1", 4), ("fp31", 9, 8, "unit1", 4),
            ("fp31", 6, 10, "unit1", 2), ("fp31", 9, 10, "unit1", 4), ("fp31", 5, 4, "unit1", 1), ("fp31", 7, 4, "unit1", 4),
            ("fp31", 10, 4, "unit1", 8), ("fp31", 4, 8, "unit1", 1), ("fp31", 5, 8, "unit1", 1), ("fp31", 7, 8, "unit1", 4),
            # the tiled kernel for a run-time n (bg_rt_kernel; 4 warps per tile for n <= 8, else 8): shapes with and
            # without a compiled instance, one and two lanes per point, odd d
            ("fp31", 8, 6, "rt", 4), ("fp31", 4, 4, "rt", 4), ("fp31", 13, 5, "rt", 8), ("fp31", 16, 4, "rt", 8),
            ("fp31", 5, 16, "rt", 4), ("fp31", 11, 9, "rt", 8), ("fp31", 16, 16, "rt", 8),
            ("c128", 6, 4, "rt", 4), ("c128", 12, 6, "rt", 8), ("c128", 7, 5, "rt", 4), ("c128", 13, 4, "rt", 8)]
KIND_ID = {"general": 0, "unit1": 1, "unit2": 2, "reg": 3, "rt": 4}


@pytest.mark.parametrize("field,n,d,kernel,w", VARIANTS, ids=lambda v: str(v))
def test_kernel_variants(bgl, oracle_mod, select_kernel, field, n, d, kernel, w):
    select_kernel(kernel, w)
    ki = bgl.bg_kernel_info(bgl.FIELD_FP31 if field == "fp31" else bgl.FIELD_C128, n, d)
    assert ki["specialised"] == KIND_ID[kernel] and (kernel == "general" or ki["threads_per_block"] == 32 * w)
    batch = 203                                              # six full tiles and a ragged one
    if field == "fp31":
        mom, pol, _ = inputs.make_fp_inputs(n, d, batch, seed=31)
        ref, rcur = oracle_mod.amplitudes(oracle_mod.FP31, mom, pol, threads=8, want_currents=True)
        out, cur, _ = bgl.currents(bgl.to_device(mom), bgl.to_device(pol))
        iu = np.triu_indices(n - 1)
        assert np.array_equal(bgl.to_numpy(out), ref)
        assert np.array_equal(bgl.to_numpy(cur)[:, iu[0], iu[1]], rcur[:, iu[0], iu[1]])
    else:
        mom, pol, _ = inputs.make_complex_inputs(n, d, batch, seed=31,
                                                 helicities=(-1, -1, 1, 1, 1, 1) if n == 6 else None)
        _assert_rule(mom, pol, _gpu_amplitudes(bgl, mom, pol))
        ref, rcur = oracle_mod.amplitudes(oracle_mod.C128, mom, pol, threads=8, want_currents=True)
        out, cur, _ = bgl.currents(bgl.to_device(mom), bgl.to_device(pol))
        iu = np.triu_indices(n - 1)
        a, b = bgl.to_numpy(cur)[:, iu[0], iu[1]], rcur[:, iu[0], iu[1]]
        assert np.all(np.abs(a - b) <= 1e-8 * (np.abs(b).max(axis=-1, keepdims=True)))


# ---- the whole grid n = 4..10 x d = 4..10 over F_p runs a compiled fast-path instance ------------------
@pytest.mark.parametrize("d", range(4, 11))
def test_fp_grid_fast_path(bgl, oracle_mod, d):
    for n in range(4, 11):
        assert bgl.bg_kernel_info(bgl.FIELD_FP31, n, d)["specialised"] >= 1, (n, d)
        mom, pol, _ = inputs.make_fp_inputs(n, d, 70, seed=41 + n)          # two full tiles and a ragged one
        ref = oracle_mod.amplitudes(oracle_mod.FP31, mom, pol, threads=8)
        assert np.array_equal(_gpu_amplitudes(bgl, mom, pol), ref), (n, d)


# ---- complex128: n = 4..10 at d = 4, 6, 8 run a compiled fast-path instance ------------------------------
@pytest.mark.parametrize("d", [4, 6, 8])
def test_complex_grid_fast_path(bgl, oracle_mod, d):
    for n in range(4, 11):
        assert bgl.bg_kernel_info(bgl.FIELD_C128, n, d)["specialised"] >= 1, (n, d)
        mom, pol, _ = inputs.make_complex_inputs(n, d, 40, seed=51 + n)     # two full 16-point tiles and a ragged one
        _assert_rule(mom, pol, _gpu_amplitudes(bgl, mom, pol))


# ---- extreme residues: the lazy-accumulation headroom (bg_field.cuh: kCap0 / kCapR / relief) -----------
# Uniformly random residues essentially never reach the worst-case operand magnitudes the headroom
# analysis is about, so these inputs do: all p-1, raw words above p (0xFFFFFFFE = 2p, 0xFFFFFFFF = 2p+1),
# p-1 alternating with 1, a seeded mix of {0, 1, 2, p-2, p-1, 2^30, 2^30+1, random}, and 4-dimensional
# physical states zero-padded to d (structural zeros: many dots are exactly 0 and p = neg(0) appears).
def _extreme_inputs(kind, n, d, batch):
    rng = np.random.default_rng(77 + n + d)
    shape = (batch, n, d)
    if kind == "all_p-1":
        return np.full(shape, P - 1, np.uint32), np.full(shape, P - 1, np.uint32)
    if kind == "raw_2p_and_2p+1":
        return np.full(shape, 0xFFFFFFFF, np.uint32), rng.choice(
            np.array([0xFFFFFFFE, 0xFFFFFFFF], np.uint32), size=shape)
    if kind == "p-1_alternating_1":
        a = np.where((np.arange(n * d).reshape(n, d) % 2) == 0, P - 1, 1).astype(np.uint32)
        b = np.where((np.arange(n * d).reshape(n, d) % 2) == 1, P - 1, 1).astype(np.uint32)
        return np.broadcast_to(a, shape).copy(), np.broadcast_to(b, shape).copy()
    if kind == "mixed":
        pool = np.array([0, 1, 2, P - 2, P - 1, 1 << 30, (1 << 30) + 1, P, 0xFFFFFFFF], np.uint32)
        pick = lambda: np.where(rng.random(shape) < 0.8, rng.choice(pool, size=shape),
                                rng.integers(0, P, size=shape, dtype=np.uint32)).astype(np.uint32)
        return pick(), pick()
    if kind == "4d_zero_padded":
        m4, p4, _ = inputs.make_fp_inputs(n, 4, batch, seed=61)
        mom = np.zeros(shape, np.uint32)
        pol = np.zeros(shape, np.uint32)
        mom[:, :, :4], pol[:, :, :4] = m4, p4
        return mom, pol
    raise ValueError(kind)


EXTREME_KINDS = ["all_p-1", "raw_2p_and_2p+1", "p-1_alternating_1", "mixed", "4d_zero_padded"]
EXTREME_CASES = [(8, 6, "unit1", 4), (8, 6, "unit1", 6), (8, 6, "unit1", 2), (8, 6, "general", 0),
                 (12, 6, "unit1", 8), (12, 6, "unit1", 16), (12, 6, "general", 0),
                 (10, 8, "unit1", 8), (10, 8, "unit1", 4), (10, 8, "general", 0),
                 (4, 4, "unit1", 1), (4, 4, "general", 0), (9, 10, "unit1", 4), (7, 5, "unit1", 4),
                 (5, 16, "general", 0), (16, 4, "general", 0), (16, 16, "general", 0),
                 (8, 6, "rt", 8), (13, 5, "rt", 8), (16, 4, "rt", 8), (5, 16, "rt", 8), (16, 16, "rt", 8)]


@pytest.mark.parametrize("n,d,kernel,w", EXTREME_CASES, ids=lambda v: str(v))
def test_fp_extreme_residues(bgl, oracle_mod, select_kernel, n, d, kernel, w):
    select_kernel(kernel, w)
    assert bgl.bg_kernel_info(bgl.FIELD_FP31, n, d)["specialised"] == KIND_ID[kernel]
    batch = 70
    iu = np.triu_indices(n - 1)
    for kind in EXTREME_KINDS:
        mom, pol = _extreme_inputs(kind, n, d, batch)
        ref, rcur, rst = oracle_mod.amplitudes(oracle_mod.FP31, mom, pol, threads=8, want_currents=True,
                                               want_status=True)
        out, cur, st = bgl.currents(bgl.to_device(mom), bgl.to_device(pol))
        assert np.array_equal(bgl.to_numpy(out), ref), kind
        assert np.array_equal(bgl.to_numpy(cur)[:, iu[0], iu[1]], rcur[:, iu[0], iu[1]]), kind
        assert np.array_equal(st.cpu().numpy().astype(np.uint32), rst), kind


def test_uncompiled_shapes_run_the_tiled_kernel_and_match_the_compiled_one(bgl, oracle_mod, select_kernel):
    """shapes without a compiled instance default to bg_rt_kernel (one state configuration, one ordering); on a
    compiled shape it gives the same residues as the compiled kernel, status words included"""
    assert bgl.bg_kernel_info(bgl.FIELD_FP31, 13, 5)["specialised"] == 4
    assert bgl.bg_kernel_info(bgl.FIELD_FP31, 8, 6)["specialised"] == 1
    mom, pol, _ = inputs.make_fp_inputs(10, 8, 1000, seed=5)
    mom[7, 1] = mom[7, 0]                                    # a vanishing invariant: inv(0) := 0, status bit 0
    dm, dp = bgl.to_device(mom), bgl.to_device(pol)
    import torch
    st0 = torch.zeros(1000, dtype=torch.int32, device="cuda")
    a = bgl.to_numpy(bgl.amplitudes(dm, dp, status=st0))
    select_kernel("rt", 0)
    st1 = torch.zeros(1000, dtype=torch.int32, device="cuda")
    b = bgl.to_numpy(bgl.amplitudes(dm, dp, status=st1))
    assert np.array_equal(a, b) and torch.equal(st0, st1) and int(st0[7]) == 1
