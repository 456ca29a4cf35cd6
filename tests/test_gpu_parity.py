"""Parity of the CUDA path (through the C ABI) with the CPU oracle, element by element.

F_p: bit-exact.  complex128: DESIGN.md reading R9 -- with t the 80-bit oracle on the same
double inputs, e_g = |gpu - t|/|t|, e_d = |oracle_double - t|/|t| and kappa the condition
number of the point estimated BY THE ORACLE (relative change of the double oracle's result
under random relative input perturbations of 1e-12, maximum of 4 draws, divided by 1e-12),
every point must satisfy  e_g <= max(1e-10, 16 e_d, 64 kappa 2^-53)  -- north_star's 1e-10
wherever a double evaluation can reach it at all; on ill-conditioned points (MHV amplitudes
near <12> -> 0) the GPU is held to the accuracy a backward-stable double evaluation has.
"""
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


def _gpu_amplitudes(bgl, mom, pol, want_status=False):
    import torch
    dm, dp = bgl.to_device(mom), bgl.to_device(pol)
    status = torch.zeros(mom.shape[0], dtype=torch.int32, device="cuda") if want_status else None
    out = bgl.amplitudes(dm, dp, status=status)
    torch.cuda.synchronize()
    if want_status:
        return bgl.to_numpy(out), status.cpu().numpy().astype(np.uint32)
    return bgl.to_numpy(out)


def _kappa(oracle_mod, mom, pol, dbl, draws=4, eps=1e-12):
    """condition number of each point, estimated with the double oracle alone"""
    rng = np.random.default_rng(1234)
    kap = np.zeros(mom.shape[0])

    def pert(a):
        return a * (1 + eps * (rng.standard_normal(a.shape) + 1j * rng.standard_normal(a.shape)))

    for _ in range(draws):
        o = oracle_mod.amplitudes(oracle_mod.C128, pert(mom), pert(pol), threads=8)
        kap = np.maximum(kap, np.abs(o - dbl) / np.abs(dbl) / eps)
    return kap


def _complex_rule(gpu, dbl, truth, kappa=None):
    t = truth.astype(np.clongdouble)
    scale = np.abs(t)
    e_g = (np.abs(gpu.astype(np.clongdouble) - t) / scale).astype(np.float64)
    e_d = (np.abs(dbl.astype(np.clongdouble) - t) / scale).astype(np.float64)
    tol = np.maximum(1e-10, 16 * e_d)
    if kappa is not None:
        tol = np.maximum(tol, 64 * kappa * 2.0 ** -53)
    return e_g <= tol, e_g, e_d


# sizes span several 32-point tiles and a ragged tail
FP_SHAPES = [(4, 4, 1024), (8, 6, 517), (10, 8, 197), (12, 6, 133),     # the config shapes
             (5, 5, 99), (6, 4, 200), (7, 5, 77), (9, 7, 45), (5, 16, 40), (16, 4, 37), (13, 9, 35)]


@pytest.mark.parametrize("n,d,batch", FP_SHAPES, ids=lambda v: str(v))
def test_fp_bit_exact(bgl, oracle_mod, n, d, batch):
    mom, pol, _ = inputs.make_fp_inputs(n, d, batch, seed=21)
    ref = oracle_mod.amplitudes(oracle_mod.FP31, mom, pol, threads=8)
    got = _gpu_amplitudes(bgl, mom, pol)
    assert got.dtype == np.uint32 and got.max() < P
    assert np.array_equal(got, ref)


C_SHAPES = [(6, 4, 515, (-1, -1, 1, 1, 1, 1)), (12, 6, 70, None), (5, 5, 99, None), (8, 6, 130, None),
            (4, 4, 64, (-1, 1, -1, 1)), (9, 10, 33, None)]


@pytest.mark.parametrize("n,d,batch,hel", C_SHAPES, ids=lambda v: str(v))
def test_complex_within_rule(bgl, oracle_mod, n, d, batch, hel):
    mom, pol, _ = inputs.make_complex_inputs(n, d, batch, seed=22, helicities=hel)
    dbl = oracle_mod.amplitudes(oracle_mod.C128, mom, pol, threads=8)
    truth = oracle_mod.amplitudes(oracle_mod.C80, mom, pol, threads=8)
    got = _gpu_amplitudes(bgl, mom, pol)
    ok, e_g, e_d = _complex_rule(got, dbl, truth, _kappa(oracle_mod, mom, pol, dbl))
    assert ok.all(), (f"worst e_g={e_g.max():.3e} (e_d there {e_d[e_g.argmax()]:.3e}); "
                      f"{(~ok).sum()} of {batch} points outside the rule")
    assert np.median(e_g) < 1e-12


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
        assert np.allclose(out, ref, rtol=1e-9)
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
        assert np.allclose(out, ref, rtol=1e-9)
    assert not status.any()


def test_error_codes(bgl):
    import torch
    buf = torch.zeros(4096, dtype=torch.int32, device="cuda")
    p = buf.data_ptr()
    assert bgl.bg_amplitudes(0, 3, 4, 8, p, p + 1024, p + 2048, 0) == bgl.BG_ERR_ARG      # n too small
    assert bgl.bg_amplitudes(0, 17, 4, 8, p, p + 1024, p + 2048, 0) == bgl.BG_ERR_ARG
    assert bgl.bg_amplitudes(0, 4, 3, 8, p, p + 1024, p + 2048, 0) == bgl.BG_ERR_ARG      # d too small
    assert bgl.bg_amplitudes(2, 4, 4, 8, p, p + 1024, p + 2048, 0) == bgl.BG_ERR_ARG      # field
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


# ---- full-size workloads in the launch configuration bench.py times, sampled -------------------
@pytest.mark.parametrize("name", ["cfg2", "cfg3", "cfg4a"])
def test_full_size_fp_sampled(bgl, oracle_mod, name):
    cfg = inputs.CONFIGS[name]
    mom, pol, _ = inputs.make_config(name)
    got = _gpu_amplitudes(bgl, mom, pol)
    rng = np.random.default_rng(0)
    idx = np.unique(np.concatenate([rng.integers(0, cfg["batch"], 4096),
                                    [0, 31, 32, cfg["batch"] - 33, cfg["batch"] - 1]]))
    ref = oracle_mod.amplitudes(oracle_mod.FP31, mom[idx], pol[idx], threads=8)
    assert np.array_equal(got[idx], ref)
    # property that holds at any size: canonical residues, and not degenerate
    assert got.max() < P and np.count_nonzero(got) > 0.99 * got.size


@pytest.mark.parametrize("name", ["cfg1", "cfg4b"])
def test_full_size_complex_sampled(bgl, oracle_mod, name):
    cfg = inputs.CONFIGS[name]
    mom, pol, _ = inputs.make_config(name)
    got = _gpu_amplitudes(bgl, mom, pol)
    rng = np.random.default_rng(1)
    idx = np.unique(np.concatenate([rng.integers(0, cfg["batch"], 4096), [0, cfg["batch"] - 1]]))
    dbl = oracle_mod.amplitudes(oracle_mod.C128, mom[idx], pol[idx], threads=8)
    truth = oracle_mod.amplitudes(oracle_mod.C80, mom[idx], pol[idx], threads=8)
    ok, e_g, e_d = _complex_rule(got[idx], dbl, truth, _kappa(oracle_mod, mom[idx], pol[idx], dbl))
    assert ok.all(), f"{(~ok).sum()} sampled points outside the rule, worst e_g={e_g.max():.3e}"
    assert np.isfinite(got.view(np.float64)).all()
    if name == "cfg1":   # config 1 is MHV: the whole batch can be checked against Parke-Taylor
        lam, _ = inputs.spinors(mom)
        br = lambda a, b: lam[:, a, 0] * lam[:, b, 1] - lam[:, a, 1] * lam[:, b, 0]
        den = np.ones(cfg["batch"], dtype=np.complex128)
        for i in range(6):
            den *= br(i, (i + 1) % 6)
        pt = 8.0 * br(0, 1) ** 4 / den                     # 2^(n-3) <12>^4 / (<12>...<61>)
        rel = np.abs(got - pt) / np.abs(pt)
        assert np.median(rel) < 1e-12 and np.mean(rel < 1e-9) > 0.995


# ---- every compiled kernel family / warps-per-tile variant (selection knobs BG_KERNEL, BG_SWEEP_W) ---
VARIANTS = [("fp31", 8, 6, "level", 4), ("fp31", 8, 6, "level", 6), ("fp31", 8, 6, "tile", 4),
            ("fp31", 4, 4, "level", 1), ("fp31", 4, 4, "tile", 1),
            ("fp31", 10, 8, "tile", 8), ("fp31", 12, 6, "tile", 16),
            ("c128", 6, 4, "level", 2), ("c128", 6, 4, "level", 4), ("c128", 6, 4, "tile", 4),
            ("c128", 6, 4, "tile", 2), ("fp31", 8, 6, "general", 0), ("c128", 6, 4, "general", 0),
            ("c128", 12, 6, "split", 16), ("c128", 6, 4, "split", 2), ("c128", 6, 4, "split", 4),
            ("c128", 6, 4, "reg", 4), ("fp31", 8, 6, "unit", 4),
            ("fp31", 10, 8, "unit", 8), ("fp31", 12, 6, "unit", 8),
            # the shapes of the paper's own benchmarks (bg_inst_paper.cu)
            ("fp31", 6, 4, "unit", 2), ("fp31", 8, 4, "unit", 4), ("fp31", 9, 4, "unit", 4), ("fp31", 6, 6, "unit", 2),
            ("fp31", 9, 6, "unit", 4), ("fp31", 6, 8, "unit", 2), ("fp31", 8, 8, "unit", 4), ("fp31", 9, 8, "unit", 4),
            ("fp31", 6, 10, "unit", 2), ("fp31", 9, 10, "unit", 4), ("fp31", 5, 4, "unit", 1), ("fp31", 7, 4, "unit", 4),
            ("fp31", 10, 4, "unit", 8), ("fp31", 4, 8, "unit", 1), ("fp31", 5, 8, "unit", 1), ("fp31", 7, 8, "unit", 4)]


@pytest.mark.parametrize("field,n,d,kernel,w", VARIANTS, ids=lambda v: str(v))
def test_kernel_variants(bgl, oracle_mod, monkeypatch, field, n, d, kernel, w):
    if kernel == "general":
        monkeypatch.setenv("BG_SWEEP_W", "0")               # the runtime-n kernel
    else:
        monkeypatch.setenv("BG_KERNEL", kernel)
        monkeypatch.setenv("BG_SWEEP_W", str(w))
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
        dbl = oracle_mod.amplitudes(oracle_mod.C128, mom, pol, threads=8)
        truth = oracle_mod.amplitudes(oracle_mod.C80, mom, pol, threads=8)
        ok, e_g, _ = _complex_rule(_gpu_amplitudes(bgl, mom, pol), dbl, truth, _kappa(oracle_mod, mom, pol, dbl))
        assert ok.all() and np.median(e_g) < 1e-12
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
        dbl = oracle_mod.amplitudes(oracle_mod.C128, mom, pol, threads=8)
        truth = oracle_mod.amplitudes(oracle_mod.C80, mom, pol, threads=8)
        ok, e_g, _ = _complex_rule(_gpu_amplitudes(bgl, mom, pol), dbl, truth, _kappa(oracle_mod, mom, pol, dbl))
        assert ok.all() and np.median(e_g) < 1e-12, (n, d, e_g.max())
