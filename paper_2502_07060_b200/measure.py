"""Timing helpers used by bench.py: CUDA-event timing and the pipe-peak probes.

The Berends-Giele path is bound by the integer (F_p) and FP64 (complex128) issue
rates, which MEASURED_PEAKS.json does not carry; `measure_peaks()` measures them on
the box with the register-resident kernels of csrc/bg_peaks.cu.
"""
from __future__ import annotations

import statistics

from . import binding


def time_launches(fn, reps: int, stream=None):
    """list of per-launch durations in ms (CUDA events on the launching stream)"""
    import torch
    stream = stream or torch.cuda.current_stream()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(reps)]
    for a, b in ev:
        a.record(stream)
        fn()
        b.record(stream)
    stream.synchronize()
    return [a.elapsed_time(b) for a, b in ev]


def measure_peaks(kinds=None, sms: int | None = None, target_ms: float = 3.0, reps: int = 5) -> dict:
    """thread-operations per second for each probe kind (best of `reps`), plus the launch
    geometry.  One 'operation' = one instruction of the named kind per thread (for
    'modmul': one canonical Mersenne-31 modular multiplication; for 'mix': one IMAD.WIDE or
    one ALU instruction)."""
    import torch
    kinds = kinds or list(binding.PEAK_KINDS)
    props = torch.cuda.get_device_properties(0)
    sms = sms or props.multi_processor_count
    blocks, threads = sms * 8, 256
    sink = torch.zeros(blocks * threads, dtype=torch.int32, device="cuda")
    s = torch.cuda.current_stream().cuda_stream
    res = {"blocks": blocks, "threads": threads, "sms": sms}
    for kind in kinds:
        iters = 64
        ops = binding.bg_peak_probe(kind, iters, blocks, threads, sink.data_ptr(), s)   # warm-up
        torch.cuda.synchronize()
        t = min(time_launches(lambda: binding.bg_peak_probe(kind, iters, blocks, threads, sink.data_ptr(), s), 2))
        iters = max(64, int(iters * target_ms / max(t, 1e-3)))
        ops = binding.bg_peak_probe(kind, iters, blocks, threads, sink.data_ptr(), s)
        ts = time_launches(lambda: binding.bg_peak_probe(kind, iters, blocks, threads, sink.data_ptr(), s), reps)
        best = min(ts)
        res[kind] = {"ops_per_s": ops * blocks * threads / (best * 1e-3),
                     "ms_best": best, "ms_median": statistics.median(ts), "iters": iters}
    return res


def _main(argv=None) -> int:
    """python -m paper_2502_07060_b200.measure [--once ITERS] [kind ...]

    Prints the pipe-peak probes of this GPU as one JSON line (thread-operations per second per kind; kinds as in
    binding.PEAK_KINDS, default all).  --once ITERS launches every named probe exactly once with that many loop
    iterations and times nothing: the form to put under `ncu` when one wants the counters of a probe."""
    import argparse
    import json

    import torch
    ap = argparse.ArgumentParser(prog="python -m paper_2502_07060_b200.measure")
    ap.add_argument("kinds", nargs="*", default=None)
    ap.add_argument("--once", type=int, default=0, metavar="ITERS")
    args = ap.parse_args(argv)
    binding.load()
    kinds = args.kinds or list(binding.PEAK_KINDS)
    if args.once:
        sms = torch.cuda.get_device_properties(0).multi_processor_count
        blocks, threads = sms * 8, 256
        sink = torch.zeros(blocks * threads, dtype=torch.int32, device="cuda")
        s = torch.cuda.current_stream().cuda_stream
        ops = {k: binding.bg_peak_probe(k, args.once, blocks, threads, sink.data_ptr(), s) for k in kinds}
        torch.cuda.synchronize()
        print(json.dumps({"once": args.once, "blocks": blocks, "threads": threads, "ops_per_thread": ops}))
        return 0
    print(json.dumps(measure_peaks(kinds)))
    return 0


if __name__ == "__main__":
    raise SystemExit(_main())
