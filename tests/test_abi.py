"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every
symbol include/bg.h declares; the formula-only entry points agree with SURVEY.md §8(d).
No compute call is made here (no GPU)."""
import ctypes
import os
import re

import pytest

from paper_2502_07060_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return binding.load()


def test_every_declared_symbol_is_exported(lib):
    hdr = open(os.path.join(ROOT, "include", "bg.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(bg_[a-z0-9_]+)\s*\(", hdr))
    assert declared == set(binding.EXPORTS)
    raw = ctypes.CDLL(build.LIB)
    for name in declared:
        assert getattr(raw, name) is not None


def test_no_torch_types_in_the_header():
    hdr = open(os.path.join(ROOT, "include", "bg.h")).read()
    assert "torch" not in hdr.lower().replace("pytorch", "") and "at::" not in hdr


def test_constants(lib):
    assert binding.bg_modulus() == (1 << 31) - 1
    assert "sm_100a" in binding.bg_version()
    assert binding.bg_status_string(0) == "ok"
    assert "argument" in binding.bg_status_string(-1)


@pytest.mark.parametrize("n,d,field,mref,s3,s4,R,bytes_in", [
    (4, 4, 0, 143, 4, 1, 2, 128),
    (6, 4, 1, 940, 20, 15, 9, 768),
    (8, 6, 0, 4839, 56, 70, 20, 384),
    (10, 8, 0, 16510, 120, 210, 35, 640),
    (12, 6, 0, 26553, 220, 495, 54, 576),
    (12, 6, 1, 26553, 220, 495, 54, 2304),
])
def test_op_counts_match_the_survey_table(lib, n, d, field, mref, s3, s4, R, bytes_in):
    """M_ref = 6d C(n,3) + 6d C(n,4) + dR + 3(R-1) + dR + d"""
    oc = binding.bg_op_count(field, n, d)
    assert oc["mul_ref"] == mref
    assert (oc["splits3"], oc["splits4"], oc["propagators"]) == (s3, s4, R)
    assert oc["currents"] == n * (n - 1) // 2
    assert oc["bytes_in"] == bytes_in
    assert oc["mul_factored"] < oc["mul_ref"] or n <= 5


def test_kernel_info_and_bad_shapes(lib):
    ki = binding.bg_kernel_info(0, 8, 6)
    assert ki["specialised"] >= 1 and ki["points_per_block"] in (16, 32) and ki["threads_per_block"] % 32 == 0
    assert ki["smem_bytes_per_block"] <= 232448
    ki = binding.bg_kernel_info(0, 13, 5)                            # outside the compiled grid: run-time-n tiled kernel
    assert ki["specialised"] == 4 and ki["points_per_block"] == 32 and ki["threads_per_block"] == 256
    assert binding.bg_kernel_info(0, 16, 16)["points_per_block"] == 16   # two lanes per point: the 32-point tile is too large
    ki = binding.bg_kernel_info_problem(binding.problem(0, 13, 5, states=3))       # states / orderings on such a shape:
    assert ki["specialised"] == 4 and ki["points_per_block"] == 32                  # the MULTI instantiation of bg_rt_kernel
    assert binding.bg_kernel_info(1, 6, 4)["specialised"] == 3       # cfg1: bg_reg_kernel ...
    pb = binding.problem(1, 6, 4, states=4)
    assert binding.bg_kernel_info_problem(pb)["specialised"] == 2    # ... but not with several state configurations
    for metric in (0, 1):                                            # generic prime, both metrics: compiled cfg2 shape
        pb = binding.problem(binding.FIELD_FPMONT, 8, 6, metric=metric, primes=(2147483629,))
        assert binding.bg_kernel_info_problem(pb)["specialised"] == 1
    assert binding.bg_kernel_info_problem(binding.problem(0, 7, 7, metric=1))["specialised"] == 4
    big = binding.bg_kernel_info(1, 16, 16)          # largest record: fewer points per block
    assert 1 <= big["threads_per_block"] < 32
    for bad in [(0, 3, 4), (0, 17, 4), (0, 4, 3), (0, 4, 17), (3, 4, 4)]:
        with pytest.raises(binding.BgError):
            binding.bg_kernel_info(*bad)


def test_sweep_numbering_bound(lib):
    """K orderings x S state configurations per point are numbered in 32-bit arithmetic inside the kernels (times 16
    levels): the host refuses K * S >= 2^27 instead of letting the number overflow"""
    fake = 4096                                                      # never dereferenced by the host-side checks
    ok = binding.problem(0, 8, 6, states=4095, n_orderings=1 << 14, orderings_ptr=fake)      # K * S < 2^27
    assert binding.bg_kernel_info_problem(ok)["specialised"] >= 1
    with pytest.raises(binding.BgError):
        binding.bg_kernel_info_problem(binding.problem(0, 8, 6, states=65535, n_orderings=1 << 12, orderings_ptr=fake))
    with pytest.raises(binding.BgError):
        binding.bg_kernel_info_problem(binding.problem(0, 8, 6, states=8, n_orderings=1 << 24, orderings_ptr=fake))


@pytest.mark.timeout(120)
def test_composite_modulus_is_refused_not_hung(lib):
    """bg_states / bg_generate (mostly-minus metric, generic prime) need sqrt(-1) mod p and find it from a quadratic
    non-residue.  Primality is the caller's job; for the composite 32771^2 = 1 mod 4 no small g passes Euler's
    criterion, and the search must give up (BG_ERR_UNSUPPORTED) rather than spin on the host.  No launch happens."""
    p = 32771 * 32771
    assert (1 << 30) < p < (1 << 31) and p % 4 == 1
    fake = 4096
    rc = binding.bg_states(binding.FIELD_FPMONT, p, binding.METRIC_MOSTLY_MINUS, 4, 1, fake, fake + 256, fake + 512,
                           fake + 1024)
    assert rc == binding.BG_ERR_UNSUPPORTED
    rc = binding.bg_generate(binding.FIELD_FPMONT, p, binding.METRIC_MOSTLY_MINUS, 4, 4, 1, 0, 0, (1, 1, -1, -1),
                             fake, fake + 256)
    assert rc == binding.BG_ERR_UNSUPPORTED


DEFAULT_INSTANCES = [                                   # what cfg0, cfg2, cfg3, cfg4a, cfg4b and cfg1 launch by default
    "bg::bg_unit_kernel<bg::Fp31, 0, 4, 4, 1, 1, false>", "bg::bg_unit_kernel<bg::Fp31, 0, 8, 6, 4, 1, false>",
    "bg::bg_unit_kernel<bg::Fp31, 0, 10, 8, 8, 1, false>", "bg::bg_unit_kernel<bg::Fp31, 0, 12, 6, 8, 1, false>",
    "bg::bg_unit_kernel<bg::C128, 0, 12, 6, 12, 2, false>", "bg::bg_reg_kernel<bg::C128, 0, 6, 4>"]


def ptxas_entries():
    """{demangled kernel name: (stack bytes, spill stores, spill loads, registers)} from the build's ptxas -v log"""
    import shutil
    import subprocess
    log = os.path.join(build.CSRC, "ptxas.log")
    if not os.path.exists(log) or not shutil.which("c++filt"):
        pytest.skip("no ptxas.log (written by paper_2502_07060_b200.build) / c++filt")
    ents = re.findall(r"Compiling entry function '(\S+)' for 'sm_100a'\nptxas info\s*: Function properties for \S+\n"
                      r"\s*(\d+) bytes stack frame, (\d+) bytes spill stores, (\d+) bytes spill loads\n"
                      r"ptxas info\s*: Used (\d+) registers", open(log).read())
    names = subprocess.run(["c++filt"], input="\n".join(e[0] for e in ents), capture_output=True, text=True).stdout.split("\n")
    clean = lambda nm: re.sub(r"\((int|bool)\)", "", re.sub(r"^void ", "", nm.split("(bg::BgParams")[0].split("(bg::RtParams")[0]))
    return {clean(nm): tuple(int(x) for x in e[1:]) for nm, e in zip(names, ents)}


def test_default_kernels_do_not_spill(lib):
    """north_star asks for register spills as evidence: the six kernels the five configs launch by default keep
    everything in registers (no stack frame, no spill bytes) -- guarded here the way the uniform datapath is below.
    The instances that DO spill (none on a config's default path) are listed in DESIGN.md §6.6."""
    ents = ptxas_entries()
    assert len(ents) > 500
    for name in DEFAULT_INSTANCES:
        assert name in ents, (name, [k for k in ents if "8, 6, 4, 1" in k][:4])
        stack, st, ld, regs = ents[name]
        assert (stack, st, ld) == (0, 0, 0), (name, ents[name])
        assert regs <= 255
    # the run-time-n kernel over F_p (what shapes outside the compiled grid launch) may spill a few words of set-up /
    # loop state, not more (the complex128 instances at d >= 12 run at 255 registers and do spill: DESIGN.md §6.6)
    rt = {k: v for k, v in ents.items() if "bg_rt_kernel<bg::Fp31" in k or "bg_rt_kernel<bg::FpMont" in k}
    assert len(rt) >= 4 * 40
    worst = max((v[1] + v[2], k) for k, v in rt.items() if k.endswith("false>"))
    assert worst[0] <= 128, worst
    worst = max((v[1] + v[2], k) for k, v in rt.items() if k.endswith("true>"))
    assert worst[0] <= 256, worst


def test_host_workspace_formula(lib):
    w = binding.bg_host_workspace_bytes(0, 8, 6, 1024)
    assert w == 2 * (2 * 1024 * 48 * 4 + 1024 * 4 + 1024 * 4)
    assert binding.bg_host_workspace_bytes(0, 3, 6, 1024) == 0


def test_product_does_not_import_the_oracle():
    """the product path must not route through the oracle (or any CPU fallback)"""
    pkg = os.path.join(ROOT, "paper_2502_07060_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src, f
                assert "bg_oracle" not in src and "bg_recursion.inc" not in src, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".inc")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2502_07060_b200" not in src and "from paper_2502_07060_b200" not in src, f
            assert not re.search(r'#\s*include\s*[<"][^">]*(bg\.h|\.cuh)', src), f


def test_compile_time_schedules_are_valid(lib):
    """every splitting of every current exactly once, shared currents handed over consistently"""
    assert binding.bg_selftest_schedules() == 0


def test_headline_kernel_keeps_the_uniform_datapath(lib):
    """The sweep of the tiled kernel is a run-time loop over a table in constant memory: its control flow and
    table loads must sit on the uniform datapath (BRA.U / ULOP3 / LDCU).  ptxas drops that silently for innocent
    looking source changes (a run-time multiply on a table field, a named barrier, a select on a table flag:
    +4 % to +18 % at cfg2), so the SASS of the default instances is checked here."""
    import shutil
    import subprocess
    obj = os.path.join(build.CSRC, "bg_inst_default.o")
    tool = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    if not os.path.exists(obj) or not os.path.exists(tool):
        pytest.skip("no object file / cuobjdump")
    sass = subprocess.run([tool, "-sass", obj], capture_output=True, text=True, check=True).stdout
    kernels = re.split(r"\n\s*Function : ", sass)[1:]
    plain = [k for k in kernels if k.startswith("_ZN2bg14bg_unit_kernel") and "ELb0EEE" in k.split("\n", 1)[0]]
    assert plain, "no tiled kernel in the default table"
    for k in plain:
        name = k.split("\n", 1)[0]
        assert k.count("BRA.U") >= 5 and k.count("LDCU") >= 3, name
