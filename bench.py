#!/usr/bin/env python
"""bench.py -- throughput of the Berends-Giele hot path on B200 (BASELINE.json's metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config cfg2] [--impl reference]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 \
        --master-port P bench.py --gpus N --steps K --warmup W

A "step" is one pass of the whole hot path (SURVEY.md §8(a) rows a0-a6 = ONE kernel launch
through the C ABI, `bg_amplitudes`) over one batch of seeded synthetic kinematics.  The
headline workload is BASELINE.json configs[2] -- n=8 gluons, d=6, F_p (p=2^31-1), batch
2^20 -- the configuration north_star's target is quoted on; `--config` selects another.
With N GPUs every rank processes its own slice of N*batch points (points are independent:
no collective on the data path, "scaling": "weak").

Printed: ONE JSON line (rank 0) with the contract keys plus `roofline` (bound "alu": the
modmul-bound line of SURVEY.md §8(d) / DESIGN.md §Roofline), `cpu_baseline` (the oracle as
it stands, on this box's host cores, on a bounded sample), `e2e` (the same metric through
`bg_amplitudes_host` with pinned HOST buffers, H2D/D2H copies inside the timed region),
`clocks`, `gpu_launches`, `per_config` (short device-resident timings of the other BASELINE.json
configs, each with its own oracle timing and, for complex128, the branch statistics of tolerance
rule R9), `features` (the SURVEY.md 8(f) rows: state configurations, generic prime, alternating
metric, colour orderings, state sum, device generator and states, shapes without a compiled instance) and
`e2e_seeded` (seed -> amplitudes on the host with the generator on the device); N=1 only,
`--headline-only` skips them.
`--impl reference` times the CPU oracle alone (this tier's reference arm).
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

from paper_2502_07060_b200 import inputs  # noqa: E402

METRIC = "amplitudes_per_second"
UNIT = "amplitudes/s"
# a field multiplication is one IMAD.WIDE.U32 (32x32(+64) -> 64); on sm_100 it
# occupies the FMA-heavy pipe for 4 cycles per warp = 8 lanes per clock per SM sub-partition
# = 32 per SM (measured by the register-resident probe bg_peaks.cu: 30.6; ncu: pipe_fmaheavy).
# That pipe is the binding one for F_p, so the peak is 148 SMs x 32 per clock x max SM clock.
SM_COUNT = 148
WIDE_MUL_LANES_PER_CLK_PER_SM = 32
DFMA_LANES_PER_CLK_PER_SM = 64      # checked against the DFMA probe


def ncu_traffic(name: str):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the config's kernel, parsed from the
    committed `ncu --set full` summary that profiles/traffic.json names for it (None if there is none)"""
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.json")) as f:
            fn = json.load(f)[name]
        unit = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}
        tot = 0.0
        with open(os.path.join(ROOT, "profiles", fn)) as f:
            for line in f:
                t = line.split()
                if len(t) == 3 and t[0] in ("dram__bytes_read.sum", "dram__bytes_write.sum"):
                    tot += float(t[1]) * unit[t[2]]
        return {"bytes": tot, "source": "profiles/" + fn} if tot else None
    except Exception:  # noqa: BLE001
        return None


def log(*a):
    print(*a, file=sys.stderr, flush=True)


# ------------------------------------------------------------------------------- clocks
class ClockSampler:
    """samples SM clock and throttle reasons with NVML while the timed region runs"""

    def __init__(self, index: int, period: float = 0.01):
        self.samples, self.reasons, self.power = [], set(), []
        self.period, self._stop, self._thr = period, threading.Event(), None
        self.sm_max = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.sm_max = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception as e:  # noqa: BLE001
            log(f"[bench] NVML unavailable ({e}); clocks not sampled")
            self.nv = None

    _NAMES = {0x1: "gpu_idle", 0x2: "applications_clocks_setting", 0x4: "sw_power_cap", 0x8: "hw_slowdown",
              0x10: "sync_boost", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
              0x80: "hw_power_brake_slowdown", 0x100: "display_clock_setting"}

    def _run(self):
        nv = self.nv
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                for bit, name in self._NAMES.items():
                    if r & bit and name != "gpu_idle":
                        self.reasons.add(name)
                self.power.append(nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0)
            except Exception:  # noqa: BLE001
                pass
            self._stop.wait(self.period)

    def __enter__(self):
        if self.nv:
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()
        return self

    def __exit__(self, *exc):
        self._stop.set()
        if self._thr:
            self._thr.join()

    def summary(self) -> dict:
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.sm_max, "reasons": [], "samples": 0}
        return {"sm_mhz": statistics.median(self.samples), "sm_max_mhz": self.sm_max,
                "reasons": sorted(self.reasons), "samples": len(self.samples),
                "power_w_max": max(self.power) if self.power else None}


# ------------------------------------------------------------------------------- helpers
def op_counts(field: str, n: int, d: int) -> dict:
    """M_ref of SURVEY.md §8(d) by formula (the C library exports the same via bg_op_count;
    restated here so the reference arm needs no CUDA library)."""
    from math import comb
    m = n - 1
    R = m * (m - 1) // 2 - 1
    w = 4 if field == "fp31" else 16
    return {"mul_ref": 6 * d * comb(n, 3) + 6 * d * comb(n, 4) + d * R + 3 * (R - 1) + d * R + d,
            # what the kernels' factored form executes (bg.h: bg_opcount_t.mul_factored)
            "mul_exec": 6 * d * comb(n, 3) + 2 * d * comb(n, 4) + (R + 1) * (d + 1) + 2 * d * R + d + m * d + d * R +
            3 * (R - 1) + 38,
            "bytes": 2 * n * d * w + w}


def host_cores() -> int:
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:
        return os.cpu_count() or 1


def time_oracle(cfg_name: str, sample_points: int, cores: int, repeats: int = 1, start: int = 0):
    """the oracle as it stands, one thread per core over contiguous batch slices"""
    import oracle
    cfg = inputs.CONFIGS[cfg_name]
    mom, pol, _ = inputs.make_config_threaded(cfg_name, batch=sample_points, start=start)
    f = oracle.FP31 if cfg["field"] == "fp31" else oracle.C128
    oracle.amplitudes(f, mom[:256], pol[:256], threads=1)        # load the library
    ts = []
    for _ in range(repeats):
        t0 = time.perf_counter()
        oracle.amplitudes(f, mom, pol, threads=cores)
        ts.append(time.perf_counter() - t0)
    return ts


def pick_oracle_sample(cfg_name: str, cores: int, target_s: float) -> int:
    """sample size giving about target_s seconds of oracle wall time on `cores` threads"""
    probe = 256 * max(1, min(cores, 8))
    t = time_oracle(cfg_name, probe, cores)[0]
    pts = int(probe * target_s / max(t, 1e-6))
    full = inputs.CONFIGS[cfg_name]["batch"]
    return max(probe, min(full, 1 << max(8, pts.bit_length() - 1)))


# ------------------------------------------------------------------------------- reference arm
def run_reference(args) -> None:
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cores = host_cores()
    name = args.config
    cfg = inputs.CONFIGS[name]
    sample = args.oracle_points or pick_oracle_sample(name, cores, 2.0)
    total = args.steps + args.warmup
    ts = time_oracle(name, sample, cores, repeats=total)
    timed = ts[args.warmup:]
    ms = 1e3 * sum(timed) / len(timed)
    value = sample / (ms * 1e-3)
    desc = f"{sample} points of {name} per step (the first points of the seeded workload), {cores} threads"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "u32" if cfg["field"] == "fp31" else "f64",
        "data": "synthetic (seeded light-cone kinematics, DESIGN.md §Input recipe)",
        "config": {"workload": workload_name(name), "sample_points_per_step": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def workload_name(name: str) -> str:
    c = inputs.CONFIGS[name]
    fld = "F_p(p=2^31-1)" if c["field"] == "fp31" else "complex128"
    return f"{name}: n={c['n']} gluons, d={c['d']}, {fld}, batch {c['batch']} per GPU, seed 0"


# ------------------------------------------------------------------------------- GPU arm
def device_bench(binding, torch, name: str, batch: int, start: int, steps: int, warmup: int, dist):
    """device-resident timing of `steps` launches; returns dict"""
    cfg = inputs.CONFIGS[name]
    t0 = time.perf_counter()
    mom, pol, info = inputs.make_config_threaded(name, batch=batch, start=start)
    gen_s = time.perf_counter() - t0
    dm, dp = binding.to_device(mom), binding.to_device(pol)
    out = torch.empty(batch, dtype=dm.dtype, device="cuda")
    stream = torch.cuda.current_stream()
    field = binding.field_of(dm)
    n, d = cfg["n"], cfg["d"]

    def launch():
        rc = binding.bg_amplitudes(field, n, d, batch, dm.data_ptr(), dp.data_ptr(), out.data_ptr(),
                                   stream.cuda_stream)
        if rc != binding.BG_OK:
            raise RuntimeError(f"bg_amplitudes failed: {binding.bg_status_string(rc)}")

    for _ in range(warmup):
        launch()
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    evs = [torch.cuda.Event(enable_timing=True) for _ in range(steps + 1)]
    evs[0].record(stream)
    for k in range(steps):
        launch()
        evs[k + 1].record(stream)
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    total_ms = evs[0].elapsed_time(evs[-1])
    per = [evs[k].elapsed_time(evs[k + 1]) for k in range(steps)]
    return {"total_ms": total_ms, "per_launch_ms": per, "mom": mom, "pol": pol, "out": out,
            "gen_s": gen_s, "redraws": info.get("redraws", 0), "dm": dm, "dp": dp}


def e2e_bench(binding, torch, name: str, mom: np.ndarray, pol: np.ndarray, steps: int, warmup: int, dist):
    """bg_amplitudes_host on pinned host buffers: H2D + kernel + D2H inside the timed region"""
    cfg = inputs.CONFIGS[name]
    batch = mom.shape[0]
    field = binding.FIELD_FP31 if cfg["field"] == "fp31" else binding.FIELD_C128

    def pinned(a):
        t = torch.from_numpy(a.view(np.int32) if a.dtype == np.uint32 else a).pin_memory()
        return t, t.numpy()

    tm, hm = pinned(mom)
    tp, hp = pinned(pol)
    to = torch.empty(batch, dtype=tm.dtype).pin_memory()
    ho = to.numpy()
    chunk = min(batch, 1 << 17)
    ws = torch.empty(binding.bg_host_workspace_bytes(field, cfg["n"], cfg["d"], chunk), dtype=torch.uint8,
                     device="cuda")

    def call():
        rc = binding.bg_amplitudes_host(field, cfg["n"], cfg["d"], batch, hm.ctypes.data, hp.ctypes.data,
                                        ho.ctypes.data, None, ws.data_ptr(), ws.numel())
        if rc != binding.BG_OK:
            raise RuntimeError(f"bg_amplitudes_host failed: {binding.bg_status_string(rc)}")

    for _ in range(max(1, warmup)):
        call()
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    t0 = time.perf_counter()
    for _ in range(steps):
        call()                      # returns after the results are in host memory
    torch.cuda.synchronize()
    dt = time.perf_counter() - t0
    res = ho.view(np.uint32).copy() if cfg["field"] == "fp31" else ho.copy()
    return {"s_per_step": dt / steps, "h2d": int(mom.nbytes + pol.nbytes), "d2h": int(ho.nbytes), "out": res}


def time_device(torch, launch, steps: int, warmup: int = 3) -> float:
    """median duration in ms of `steps` launches (CUDA events on the current stream)"""
    stream = torch.cuda.current_stream()
    for _ in range(warmup):
        launch()
    torch.cuda.synchronize()
    evs = [torch.cuda.Event(enable_timing=True) for _ in range(steps + 1)]
    evs[0].record(stream)
    for k in range(steps):
        launch()
        evs[k + 1].record(stream)
    torch.cuda.synchronize()
    return statistics.median(evs[k].elapsed_time(evs[k + 1]) for k in range(steps))


def oracle_baseline(name: str, cores: int, target_s: float) -> dict:
    """the oracle as it stands on `cores` threads, on the first points of the config's workload"""
    sample = pick_oracle_sample(name, cores, target_s)
    t = time_oracle(name, sample, cores)[0]
    return {"value": sample / t, "unit": UNIT, "cores": cores, "kind": "naive oracle (literal Eq.(6), % p arithmetic, "
            "one Fermat inverse per propagator)", "sample": f"the first {sample} points of {name}, one pass, {t:.2f} s"}


def r9_report(name: str, got, points: int) -> dict:
    """branch statistics of tolerance rule R9 (oracle/rule.py) on the first `points` points of a complex config"""
    from oracle import rule
    mom, pol, _ = inputs.make_config_threaded(name, batch=points)
    ok, st = rule.check(got[:points], rule.evaluate(mom, pol, threads=host_cores()))
    st["all_pass"] = bool(ok.all())
    return st


def run_features(binding, torch, steps: int, sm_max_mhz: float | None = None) -> list:
    """SURVEY.md 8(f) rows, device-resident timings (inputs from the device generator)"""
    B = binding
    s = torch.cuda.current_stream().cuda_stream
    rows = []
    n, d = 8, 6
    prime = 2147483629                       # 2^31 - 19

    def ev(pb, batch, mom, pol, out):
        rc = B.bg_evaluate(pb, batch, mom.data_ptr(), pol.data_ptr(), out.data_ptr(), None, None, s)
        if rc != B.BG_OK:
            raise RuntimeError(B.bg_status_string(rc))

    def ok(rc):
        # a BG_ERR_* return comes back in microseconds: it must stop the run, not become a huge points/s row
        if rc != B.BG_OK:
            raise RuntimeError(B.bg_status_string(rc))

    def row(name, amps, ms, **kw):
        rows.append({"feature": name, "value": amps / (ms * 1e-3), "unit": UNIT, "kernel_ms_median": ms, **kw})

    clk_hz = (sm_max_mhz or 1965.0) * 1e6

    # f2: S state configurations per momentum point (Eq.(4)); the same 2^20 amplitudes per launch for every S
    for S in (1, 4, 16):
        batch = (1 << 20) // S
        mom, pol0, _ = B.generate(B.FIELD_FP31, n, d, batch, seed=0)
        pol = torch.stack([pol0] + [B.generate(B.FIELD_FP31, n, d, batch, seed=s_)[1] for s_ in range(1, S)],
                          dim=1).contiguous()
        out = torch.empty((batch, S), dtype=torch.int32, device="cuda")
        pb = B.problem(B.FIELD_FP31, n, d, states=S)
        ms = time_device(torch, lambda: ev(pb, batch, mom, pol, out), steps)
        row(f"f2 states: n=8 d=6 F_p, {batch} points x S={S}", batch * S, ms,
            input_bytes_per_amplitude=(1 + S) * n * d * 4 / S)
    del pol, pol0
    # f3: generic 31-bit prime (Montgomery), alternating metric, four primes in one launch
    batch = 1 << 20
    mom, pol, _ = B.generate(B.FIELD_FPMONT, n, d, batch, seed=0, prime=prime)
    out = torch.empty(batch, dtype=torch.int32, device="cuda")
    pb = B.problem(B.FIELD_FPMONT, n, d, primes=(prime,))
    row(f"f3 generic prime p=2^31-19 (Montgomery): n=8 d=6, 2^20 points", batch,
        time_device(torch, lambda: ev(pb, batch, mom, pol, out), steps))
    mom, pol, _ = B.generate(B.FIELD_FP31, n, d, batch, seed=0, metric=1)
    pb = B.problem(B.FIELD_FP31, n, d, metric=1)
    row("f3 alternating metric: n=8 d=6 F_p(2^31-1), 2^20 points", batch,
        time_device(torch, lambda: ev(pb, batch, mom, pol, out), steps))
    primes = (prime, 2013265921, 1073741827, (1 << 31) - 1)
    bq = 1 << 18
    gens = [B.generate(B.FIELD_FPMONT, n, d, bq, seed=0, prime=p) for p in primes]
    mom4 = torch.stack([g[0] for g in gens]).contiguous()
    pol4 = torch.stack([g[1] for g in gens]).contiguous()
    out4 = torch.empty((4, bq), dtype=torch.int32, device="cuda")
    pb = B.problem(B.FIELD_FPMONT, n, d, primes=primes)
    row("f3 four primes in one launch: n=8 d=6, 4 x 2^18 points", 4 * bq,
        time_device(torch, lambda: ev(pb, bq, mom4, pol4, out4), steps))
    del gens, mom4, pol4
    # f4: K colour orderings per point (Eq.(5))
    K, bo = 24, 1 << 15
    rng = np.random.default_rng(0)
    perms = np.array([list(rng.permutation(n - 1)) + [n - 1] for _ in range(K)], dtype=np.uint8)
    dperm = torch.from_numpy(perms).cuda()
    mom, pol, _ = B.generate(B.FIELD_FP31, n, d, bo, seed=0)
    outk = torch.empty((bo, K), dtype=torch.int32, device="cuda")
    pb = B.problem(B.FIELD_FP31, n, d, n_orderings=K, orderings_ptr=dperm.data_ptr())
    row(f"f4 colour orderings: n=8 d=6 F_p, 2^15 points x K={K}", bo * K,
        time_device(torch, lambda: ev(pb, bo, mom, pol, outk), steps))
    # shapes outside the compiled grid: the tiled kernel with a run-time n (bg_rt_kernel)
    for (gn, gd, gb) in ((13, 5, 1 << 15), (16, 4, 1 << 14)):
        mom, pol, _ = B.generate(B.FIELD_FP31, gn, gd, gb, seed=0)
        outg = torch.empty(gb, dtype=torch.int32, device="cuda")
        pb = B.problem(B.FIELD_FP31, gn, gd)
        ms = time_device(torch, lambda: ev(pb, gb, mom, pol, outg), max(3, steps // 4))
        oc = op_counts("fp31", gn, gd)
        row(f"uncompiled shape (run-time-n tiled kernel): n={gn} d={gd} F_p, {gb} points", gb, ms,
            roofline_frac=oc["mul_ref"] * gb / (ms * 1e-3) / (SM_COUNT * WIDE_MUL_LANES_PER_CLK_PER_SM * clk_hz),
            kernel=B.bg_kernel_info(B.FIELD_FP31, gn, gd))
    # ... and with S = 4 state configurations per point (the MULTI instantiation of bg_rt_kernel; until round 3 this
    # ran the one-thread-per-point fallback)
    gn, gd, gb, gS = 13, 5, 1 << 13, 4
    mom, pol0, _ = B.generate(B.FIELD_FP31, gn, gd, gb, seed=0)
    pol = torch.stack([pol0] + [B.generate(B.FIELD_FP31, gn, gd, gb, seed=s_)[1] for s_ in range(1, gS)], dim=1).contiguous()
    outg = torch.empty((gb, gS), dtype=torch.int32, device="cuda")
    pb = B.problem(B.FIELD_FP31, gn, gd, states=gS)
    ms = time_device(torch, lambda: ev(pb, gb, mom, pol, outg), max(3, steps // 4))
    oc = op_counts("fp31", gn, gd)
    row(f"uncompiled shape, S={gS} states (run-time-n tiled kernel): n={gn} d={gd} F_p, {gb} points", gb * gS, ms,
        roofline_frac=oc["mul_ref"] * gb * gS / (ms * 1e-3) / (SM_COUNT * WIDE_MUL_LANES_PER_CLK_PER_SM * clk_hz),
        kernel=B.bg_kernel_info_problem(pb))
    del pol, pol0
    # Eq.(4) state sum: HBM-bound
    T, S, bs = 2, 16, 1 << 20
    amps = [torch.randint(0, 2 ** 31 - 1, (bs, S), dtype=torch.int32, device="cuda") for _ in range(T)]
    outs = torch.empty(bs, dtype=torch.int32, device="cuda")
    ms = time_device(torch, lambda: ok(B.bg_state_sum(B.FIELD_FP31, 0, bs, S, [a.data_ptr() for a in amps],
                                                      outs.data_ptr(), s)), steps)
    rows.append({"feature": f"f2 state sum (Eq.(4)): {T} trees x S={S}, 2^20 points", "value": bs / (ms * 1e-3),
                 "unit": "points/s", "kernel_ms_median": ms, "hbm_GBs": (T * S + 1) * 4 * bs / (ms * 1e-3) / 1e9,
                 "hbm_frac": (T * S + 1) * 4 * bs / (ms * 1e-3) / 1e9 / hbm_peak()})
    # f1: generator and states on the device
    gb = 1 << 20
    mom = torch.empty((gb, n, d), dtype=torch.int32, device="cuda")
    pol = torch.empty_like(mom)
    ms = time_device(torch, lambda: ok(B.bg_generate(B.FIELD_FP31, 0, 0, n, d, gb, 0, 0, None, mom.data_ptr(),
                                                     pol.data_ptr(), None, None, s)), steps)
    rows.append({"feature": "f1 device generator: n=8 d=6 F_p, 2^20 points", "value": gb / (ms * 1e-3),
                 "unit": "points/s", "kernel_ms_median": ms, "hbm_frac": 2 * n * d * 4 * gb / (ms * 1e-3) / 1e9 / hbm_peak()})
    momA, _, refA, _ = B.generate(B.FIELD_FP31, n, d, 1 << 17, seed=0, metric=1, want_references=True)
    chi = B.generate(B.FIELD_FP31, n, 4, 1 << 17, seed=1, metric=1, want_references=True)[2]
    kv, cv = momA.reshape(-1, d), chi.reshape(-1, 4).contiguous()
    eps = torch.empty((kv.shape[0], d - 2, d), dtype=torch.int32, device="cuda")
    til = torch.empty_like(eps)
    ms = time_device(torch, lambda: ok(B.bg_states(B.FIELD_FP31, 0, 1, d, kv.shape[0], kv.data_ptr(), cv.data_ptr(),
                                                   eps.data_ptr(), til.data_ptr(), None, s)), steps)
    rows.append({"feature": "f1 device states (Eqs.(8)-(18)): d=6 alternating metric F_p, 2^20 vectors",
                 "value": kv.shape[0] / (ms * 1e-3), "unit": "vectors/s", "kernel_ms_median": ms})
    return rows


def seeded_e2e(binding, torch, name: str, steps: int) -> dict:
    """seed -> amplitudes in HOST memory: bg_generate + bg_amplitudes on the device, one D2H copy of the results
    per step (no input ever crosses the host link).  Wall clock, synchronised on both sides."""
    cfg = inputs.CONFIGS[name]
    B = binding
    n, d, batch = cfg["n"], cfg["d"], cfg["batch"]
    field = B.FIELD_FP31 if cfg["field"] == "fp31" else B.FIELD_C128
    dt = torch.int32 if cfg["field"] == "fp31" else torch.complex128
    mom = torch.empty((batch, n, d), dtype=dt, device="cuda")
    pol = torch.empty_like(mom)
    out = torch.empty(batch, dtype=dt, device="cuda")
    host = torch.empty(batch, dtype=dt).pin_memory()
    s = torch.cuda.current_stream().cuda_stream
    hel = cfg["helicities"]

    def step(k):
        rc = B.bg_generate(field, 0, 0, n, d, batch, 0, 0, hel, mom.data_ptr(), pol.data_ptr(), None, None, s)
        rc = rc or B.bg_amplitudes(field, n, d, batch, mom.data_ptr(), pol.data_ptr(), out.data_ptr(), s)
        if rc != B.BG_OK:
            raise RuntimeError(B.bg_status_string(rc))
        host.copy_(out, non_blocking=True)

    for k in range(2):
        step(k)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for k in range(steps):
        step(k)
    torch.cuda.synchronize()
    dt_s = (time.perf_counter() - t0) / steps
    return {"value": batch / dt_s, "unit": UNIT, "ms_per_step": dt_s * 1e3, "h2d_bytes_per_step": 0,
            "d2h_bytes_per_step": int(host.numel() * host.element_size()), "steps": steps,
            "api": "bg_generate (seeded kinematics on the device, SURVEY.md 8(f) f1) + bg_amplitudes + D2H of the results",
            "result": host.numpy().view(np.uint32).copy() if cfg["field"] == "fp31" else host.numpy().copy()}


def roofline(field: str, n: int, d: int, batch: int, kernel_ms: float, sm_max_mhz: float, probes: dict | None,
             traffic):
    oc = op_counts(field, n, d)
    clk = (sm_max_mhz or 1965.0) * 1e6
    if field == "fp31":
        peak = SM_COUNT * WIDE_MUL_LANES_PER_CLK_PER_SM * clk                            # field mul/s
        achieved = oc["mul_ref"] * batch / (kernel_ms * 1e-3)
        unit, what = "Gmul/s", ("M_ref field multiplications of the literal Eq.(6) evaluation per amplitude "
                                "(SURVEY.md §8(d)) x points / kernel time; peak = IMAD.WIDE.U32 issue rate "
                                "(8 lanes/clk/SMSP, FMA-heavy pipe) at max SM clock (DESIGN.md §7)")
    else:
        peak = SM_COUNT * DFMA_LANES_PER_CLK_PER_SM * clk                                # DFMA/s
        achieved = 4 * oc["mul_ref"] * batch / (kernel_ms * 1e-3)
        unit, what = "GDFMA/s", ("4 DFMA per complex multiply-add x M_ref x points / kernel time; peak = "
                                 "FP64-pipe issue rate at max SM clock (DESIGN.md §Roofline)")
    executed = (1 if field == "fp31" else 4) * oc["mul_exec"] * batch / (kernel_ms * 1e-3)
    r = {"bound": "alu", "achieved": achieved / 1e9, "peak": peak / 1e9, "unit": unit, "frac": achieved / peak,
         "traffic": None if traffic is None else traffic["bytes"],
         "traffic_source": None if traffic is None else traffic["source"],
         "basis": "frac = EFFECTIVE work: the literal Eq.(6) count M_ref (algorithmic, SURVEY.md 8(d)) / time / peak; "
                  "frac_executed = the multiplications the factored kernels actually issue (mul_exec) / time / peak, "
                  "i.e. multiplier-pipe utilisation",
         "executed": executed / 1e9, "frac_executed": executed / peak, "mul_exec_per_amplitude": oc["mul_exec"],
         "peak_source": "derived from unit counts and clock (DESIGN.md §7), confirmed by the on-box probe; MEASURED_PEAKS.json has no ALU peak",
         "what": what, "mul_ref_per_amplitude": oc["mul_ref"], "kernel_ms": kernel_ms,
         "hbm_frac": oc["bytes"] * batch / (kernel_ms * 1e-3) / 1e9 / hbm_peak()}
    if probes:
        key = "imad_wide_rz" if field == "fp31" else "dfma"       # the bare multiplier rate / the DFMA rate
        r["probe_peak"] = probes[key]["ops_per_s"] / 1e9
        r["frac_of_probe"] = achieved / probes[key]["ops_per_s"]
        r["frac_executed_of_probe"] = executed / probes[key]["ops_per_s"]
        if field == "fp31":
            # north_star's line: canonical Mersenne-31 modular multiplications per second (R_mm, measured)
            r["modmul_line_Gmodmul_s"] = probes["modmul"]["ops_per_s"] / 1e9
            r["frac_of_modmul_line"] = achieved / probes["modmul"]["ops_per_s"]
    return r


def hbm_peak() -> float:
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"])
    except Exception:  # noqa: BLE001
        return 6650.0


def run_gpu(args) -> None:
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the Berends-Giele path has no CPU fallback")
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    # BG_BENCH_SMOKE_SHARED_DEVICE=1: a code-path smoke test of the N > 1 branch on a box with fewer GPUs than
    # ranks (ranks share devices, rendezvous and reductions over gloo).  The ranks are independent -- no kernel
    # waits on another rank -- but the line is marked "shared_device" and is NOT a scaling measurement.
    shared = os.environ.get("BG_BENCH_SMOKE_SHARED_DEVICE") == "1" and local >= torch.cuda.device_count()
    if shared:
        local = local % torch.cuda.device_count()
    shared = shared or (os.environ.get("BG_BENCH_SMOKE_SHARED_DEVICE") == "1" and world > torch.cuda.device_count())
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist_mod
        if shared:
            dist_mod.init_process_group("gloo")
        else:
            dist_mod.init_process_group("nccl", device_id=torch.device("cuda", local))
        dist = dist_mod
    from paper_2502_07060_b200 import binding, measure, sharding
    binding.load()

    name = args.config
    cfg = inputs.CONFIGS[name]
    batch = args.batch or cfg["batch"]
    start, _ = sharding.weak_slice(rank, world, batch)   # rank r owns points [r*batch, (r+1)*batch)
    phys = torch.cuda.current_device()
    vis = os.environ.get("CUDA_VISIBLE_DEVICES")
    nvml_index = int(vis.split(",")[phys]) if vis and all(v.strip().isdigit() for v in vis.split(",")) else phys

    with ClockSampler(nvml_index) as clk:
        res = device_bench(binding, torch, name, batch, start, args.steps, args.warmup, dist)
    clocks = clk.summary()
    red_dev = "cpu" if shared else "cuda"                 # gloo reduces host tensors
    total_ms = torch.tensor([res["total_ms"]], dtype=torch.float64, device=red_dev)
    if dist is not None:
        dist.all_reduce(total_ms, op=dist.ReduceOp.MAX)
    total_ms = float(total_ms.item())
    ms_per_step = total_ms / args.steps
    value = world * batch / (ms_per_step * 1e-3)
    kernel_ms = sum(res["per_launch_ms"]) / len(res["per_launch_ms"])

    # end to end through the host entry point
    e2e_steps = max(3, min(args.steps, args.e2e_steps))
    e2e = e2e_bench(binding, torch, name, res["mom"], res["pol"], e2e_steps, min(args.warmup, 3), dist)
    e2e_t = torch.tensor([e2e["s_per_step"]], dtype=torch.float64, device=red_dev)
    if dist is not None:
        dist.all_reduce(e2e_t, op=dist.ReduceOp.MAX)
    e2e_value = world * batch / float(e2e_t.item())
    same = np.array_equal(e2e["out"], binding.to_numpy(res["out"])) if cfg["field"] == "fp31" else \
        bool(np.allclose(e2e["out"], binding.to_numpy(res["out"]), rtol=1e-12, atol=0))

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "u32" if cfg["field"] == "fp31" else "f64",
        "data": "synthetic (seeded light-cone kinematics, DESIGN.md §Input recipe)",
        "config": {"workload": workload_name(name), "n": cfg["n"], "d": cfg["d"], "field": cfg["field"],
                   "batch_per_gpu": batch, "global_batch": world * batch, "parallelism": f"dp{world} (batch sharding, "
                   "no collective)", "l2": "inputs (%.0f MB per step) exceed the 126 MB L2; no flush needed" %
                   ((res["mom"].nbytes + res["pol"].nbytes) / 1e6) if res["mom"].nbytes * 2 > 126e6 else
                   "inputs fit L2: a 256 MB buffer is NOT flushed between steps (arithmetic-bound kernel)",
                   "redraws": res["redraws"]},
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": e2e["h2d"], "d2h_bytes_per_step": e2e["d2h"],
                "steps": e2e_steps, "matches_device_path": same,
                "api": "bg_amplitudes_host (pinned host buffers, chunked H2D/kernel/D2H pipeline)"},
        "gpu_launches": args.steps,
        **({"shared_device": "SMOKE TEST of the N > 1 code path: the ranks shared GPUs; not a scaling number"}
           if shared else {}),
        "clocks": clocks,
        "kernel": binding.bg_kernel_info(binding.FIELD_FP31 if cfg["field"] == "fp31" else binding.FIELD_C128,
                                         cfg["n"], cfg["d"]),
    }

    if rank == 0:
        probes = None
        if not args.no_probes:
            probes = measure.measure_peaks(kinds=["imad_wide", "imad_wide_rz", "alu", "mix", "mix2", "mix3", "modmul", "dfma", "lds64"])
            line["pipe_probes_Gops"] = {k: round(v["ops_per_s"] / 1e9, 1) for k, v in probes.items()
                                        if isinstance(v, dict)}
            # SM sub-partition cycles per warp for one IMAD.WIDE (64-bit addend) + n ALU instructions:
            # independent pipes would give max(4, 2n); measured is additive
            smsp_hz = SM_COUNT * 4 * (clocks.get("sm_max_mhz") or 1965.0) * 1e6
            line["wide_plus_n_alu_cycles"] = {
                str(n): round(smsp_hz / (probes[k]["ops_per_s"] / (n + 1) / 32), 2)
                for n, k in ((1, "mix"), (2, "mix2"), (3, "mix3"))}
        line["roofline"] = roofline(cfg["field"], cfg["n"], cfg["d"], batch, kernel_ms, clocks.get("sm_max_mhz"),
                                    probes, ncu_traffic(name))
        if world == 1 and not args.headline_only:
            per = []
            for other in inputs.CONFIGS:
                if other == name:
                    continue
                oc = inputs.CONFIGS[other]
                r = device_bench(binding, torch, other, oc["batch"], 0, args.config_steps, 3, None)
                kms = statistics.median(r["per_launch_ms"])
                rl = roofline(oc["field"], oc["n"], oc["d"], oc["batch"], kms, clocks.get("sm_max_mhz"), probes, None)
                entry = {"workload": workload_name(other), "value": oc["batch"] / (kms * 1e-3), "unit": UNIT,
                         "kernel_ms_median": kms, "launches": args.config_steps,
                         "roofline_frac": rl["frac"], "roofline_frac_executed": rl["frac_executed"],
                         "roofline_unit": rl["unit"], "hbm_frac": rl["hbm_frac"],
                         "kernel": binding.bg_kernel_info(binding.FIELD_FP31 if oc["field"] == "fp31" else
                                                          binding.FIELD_C128, oc["n"], oc["d"])}
                if not args.no_cpu_baseline:
                    entry["cpu_baseline"] = oracle_baseline(other, host_cores(), 2.0)
                    if oc["field"] == "c128":
                        pts = min(oc["batch"], 1 << 17) if oc["n"] <= 6 else 4096
                        entry["parity_rule_R9"] = r9_report(other, binding.to_numpy(r["out"]), pts)
                per.append(entry)
                del r
            line["per_config"] = per
            line["features"] = run_features(binding, torch, args.config_steps, clocks.get("sm_max_mhz"))
            se = seeded_e2e(binding, torch, name, e2e_steps)
            se["matches_device_path"] = bool(np.array_equal(se.pop("result"), binding.to_numpy(res["out"]))) \
                if cfg["field"] == "fp31" else None
            line["e2e_seeded"] = se
        if world == 1 and not args.no_cpu_baseline:
            cores = host_cores()
            sample = args.oracle_points or pick_oracle_sample(name, cores, 10.0)
            t1 = time_oracle(name, sample, cores)[0]
            reps = max(1, min(64, int(10.0 / max(t1, 1e-3))))      # about 10 s of CPU work in total
            ts = [t1] + (time_oracle(name, sample, cores, repeats=reps - 1) if reps > 1 else [])
            t = sum(ts)
            line["cpu_baseline"] = {"value": sample * len(ts) / t, "unit": UNIT, "cores": cores, "kind": "oracle",
                                    "sample": f"the first {sample} points of {name} (same seeded workload), "
                                              f"{len(ts)} passes, {t:.1f} s on {cores} threads",
                                    "note": "the oracle is deliberately naive (literal Eq.(6), % p arithmetic, one "
                                            "Fermat inverse per propagator): a reported baseline, not a tuned CPU code"}
            t1c = time_oracle(name, 1 << 14, 1)[0]
            line["cpu_baseline"]["single_core"] = {"value": (1 << 14) / t1c, "unit": UNIT, "cores": 1,
                                                   "sample": f"the first 16384 points of {name}, {t1c:.2f} s"}
        print(json.dumps(line))
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="cfg2", choices=list(inputs.CONFIGS))
    ap.add_argument("--batch", type=int, default=0, help="points per GPU (default: the config's batch)")
    ap.add_argument("--e2e-steps", type=int, default=10)
    ap.add_argument("--config-steps", type=int, default=20, help="launches per secondary config")
    ap.add_argument("--oracle-points", type=int, default=0)
    ap.add_argument("--headline-only", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-probes", action="store_true")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        log("[bench] note: fewer than 3 warm-up steps requested")
    if args.impl == "reference":
        run_reference(args)
    else:
        run_gpu(args)


if __name__ == "__main__":
    main()
