"""Thin ctypes binding of libbg_b200.so (include/bg.h) -- argument marshalling only.

Every step of the Berends-Giele path runs inside the CUDA kernels of the library;
PyTorch is used for device memory and streams, nothing else.  There is no CPU
fallback: if the library is missing or no CUDA device is present, calls raise.
The low-level functions carry the C names (bg_amplitudes, bg_currents, ...); the
`amplitudes()` / `currents()` helpers below only infer (field, n, d, batch) from
tensor shapes and allocate the output.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

from . import build as _build

FIELD_FP31, FIELD_C128, FIELD_FPMONT = 0, 1, 2
METRIC_MOSTLY_MINUS, METRIC_ALTERNATING = 0, 1
MAX_PRIMES = 8
KERNEL_KINDS = {"default": -1, "general": 0, "unit1": 1, "unit2": 2, "reg": 3, "rt": 4}
BG_OK, BG_ERR_ARG, BG_ERR_UNSUPPORTED, BG_ERR_CUDA, BG_ERR_TOO_LARGE = 0, -1, -2, -3, -4
PEAK_KINDS = {"imad_wide": 0, "imad": 1, "alu": 2, "mix": 3, "modmul": 4, "dfma": 5,
              "lds32": 6, "lds64": 7, "lds128": 8, "mix2": 9, "mix3": 10, "imad_wide_rz": 11}
P31 = (1 << 31) - 1

EXPORTS = ["bg_amplitudes", "bg_amplitudes_status", "bg_currents", "bg_evaluate", "bg_amplitudes_states",
           "bg_amplitudes_primes", "bg_amplitudes_orderings", "bg_state_sum", "bg_states", "bg_generate", "bg_amplitudes_host", "bg_host_workspace_bytes",
           "bg_amplitudes_host_noalloc", "bg_noalloc_max_batch", "bg_noalloc_scratch_bytes", "bg_modulus",
           "bg_status_string", "bg_version", "bg_op_count", "bg_kernel_info", "bg_kernel_info_problem",
           "bg_set_kernel_override", "bg_peak_probe", "bg_selftest_schedules"]


class BgError(RuntimeError):
    pass


class OpCount(ctypes.Structure):
    _fields_ = [(k, ctypes.c_int64) for k in
                ("currents", "propagators", "splits3", "splits4", "mul_v3", "mul_v4", "mul_other",
                 "mul_ref", "mul_factored", "bytes_in", "bytes_out")]


class Problem(ctypes.Structure):
    """bg_problem_t"""
    _fields_ = [("field", ctypes.c_int), ("metric", ctypes.c_int), ("n", ctypes.c_int), ("d", ctypes.c_int),
                ("states", ctypes.c_int), ("n_primes", ctypes.c_int), ("primes", ctypes.c_uint32 * MAX_PRIMES),
                ("n_orderings", ctypes.c_int), ("orderings", ctypes.c_void_p)]


def problem(field, n, d, metric=METRIC_MOSTLY_MINUS, states=1, primes=(), n_orderings=0, orderings_ptr=None) -> Problem:
    pb = Problem(field, metric, n, d, states, len(primes))
    for i, p in enumerate(primes):
        pb.primes[i] = p
    pb.n_orderings = n_orderings
    pb.orderings = orderings_ptr
    return pb


class KernelInfo(ctypes.Structure):
    _fields_ = [(k, ctypes.c_int) for k in
                ("specialised", "threads_per_block", "points_per_block", "smem_bytes_per_block",
                 "smem_bytes_per_point", "blocks_per_sm", "regs_per_thread")]


_LIB = None


def lib_path() -> str:
    return _build.LIB


def load(rebuild_if_stale: bool = False):
    """dlopen the in-tree library.  Fails loudly if it is not there."""
    global _LIB
    if _LIB is not None:
        return _LIB
    if rebuild_if_stale:
        _build.build()
    if not os.path.exists(_build.LIB):
        raise BgError(f"{_build.LIB} not built: run `python -m paper_2502_07060_b200.build` "
                      "(there is no CPU fallback)")
    lib = ctypes.CDLL(_build.LIB)
    vp, i64, ci, sz = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int, ctypes.c_size_t
    lib.bg_amplitudes.argtypes = [ci, ci, ci, i64, vp, vp, vp, vp]
    lib.bg_amplitudes_status.argtypes = [ci, ci, ci, i64, vp, vp, vp, vp, vp]
    lib.bg_currents.argtypes = [ci, ci, ci, i64, vp, vp, vp, vp, vp, vp]
    lib.bg_evaluate.argtypes = [ctypes.POINTER(Problem), i64, vp, vp, vp, vp, vp, vp]
    lib.bg_amplitudes_states.argtypes = [ci, ci, ci, i64, ci, vp, vp, vp, vp, vp]
    lib.bg_amplitudes_primes.argtypes = [ci, ci, ci, i64, ci, ctypes.POINTER(ctypes.c_uint32), vp, vp, vp, vp, vp]
    lib.bg_state_sum.argtypes = [ci, ctypes.c_uint32, i64, ci, ci, ctypes.POINTER(vp), vp, vp]
    lib.bg_state_sum.restype = ci
    lib.bg_states.argtypes = [ci, ctypes.c_uint32, ci, ci, i64, vp, vp, vp, vp, vp, vp]
    lib.bg_states.restype = ci
    lib.bg_generate.argtypes = [ci, ctypes.c_uint32, ci, ci, ci, i64, ctypes.c_uint64, i64, ctypes.c_char_p, vp, vp, vp,
                                vp, vp]
    lib.bg_generate.restype = ci
    lib.bg_amplitudes_orderings.argtypes = [ci, ci, ci, i64, ci, vp, vp, vp, vp, vp, vp]
    lib.bg_amplitudes_orderings.restype = ci
    lib.bg_kernel_info_problem.argtypes = [ctypes.POINTER(Problem), ctypes.POINTER(KernelInfo)]
    lib.bg_set_kernel_override.argtypes = [ci, ci]
    lib.bg_amplitudes_host.argtypes = [ci, ci, ci, i64, vp, vp, vp, vp, vp, sz]
    lib.bg_host_workspace_bytes.argtypes = [ci, ci, ci, i64]
    lib.bg_host_workspace_bytes.restype = sz
    lib.bg_amplitudes_host_noalloc.argtypes = [ci, ci, ci, i64, vp, vp, vp, vp, vp]
    lib.bg_amplitudes_host_noalloc.restype = ci
    lib.bg_noalloc_max_batch.argtypes = [ci, ci, ci]
    lib.bg_noalloc_max_batch.restype = i64
    lib.bg_noalloc_scratch_bytes.restype = sz
    lib.bg_modulus.restype = ctypes.c_uint32
    lib.bg_status_string.argtypes = [ci]
    lib.bg_status_string.restype = ctypes.c_char_p
    lib.bg_version.restype = ctypes.c_char_p
    lib.bg_op_count.argtypes = [ci, ci, ci, ctypes.POINTER(OpCount)]
    lib.bg_kernel_info.argtypes = [ci, ci, ci, ctypes.POINTER(KernelInfo)]
    lib.bg_peak_probe.argtypes = [ci, ci, ci, ci, vp, ctypes.POINTER(i64), vp]
    for name in ("bg_amplitudes", "bg_amplitudes_status", "bg_currents", "bg_amplitudes_host", "bg_evaluate",
                 "bg_amplitudes_states", "bg_amplitudes_primes", "bg_kernel_info_problem",
                 "bg_set_kernel_override", "bg_op_count", "bg_kernel_info", "bg_peak_probe"):
        getattr(lib, name).restype = ci
    _LIB = lib
    return lib


def _check(rc: int):
    if rc != BG_OK:
        raise BgError(f"libbg_b200: {load().bg_status_string(rc).decode()} ({rc})")


# ------------------------------------------------------------- C names, raw pointers
def bg_amplitudes(field, n, d, batch, momenta_ptr, polarisations_ptr, out_ptr, stream_ptr=0):
    return load().bg_amplitudes(field, n, d, batch, momenta_ptr, polarisations_ptr, out_ptr, stream_ptr)


def bg_amplitudes_status(field, n, d, batch, momenta_ptr, polarisations_ptr, out_ptr, status_ptr,
                         stream_ptr=0):
    return load().bg_amplitudes_status(field, n, d, batch, momenta_ptr, polarisations_ptr, out_ptr,
                                       status_ptr, stream_ptr)


def bg_currents(field, n, d, batch, momenta_ptr, polarisations_ptr, out_ptr, currents_ptr, status_ptr,
                stream_ptr=0):
    return load().bg_currents(field, n, d, batch, momenta_ptr, polarisations_ptr, out_ptr,
                              currents_ptr, status_ptr, stream_ptr)


def bg_evaluate(pb: Problem, batch, momenta_ptr, polarisations_ptr, out_ptr, currents_ptr=None, status_ptr=None,
                stream_ptr=0):
    return load().bg_evaluate(ctypes.byref(pb), batch, momenta_ptr, polarisations_ptr, out_ptr, currents_ptr,
                              status_ptr, stream_ptr)


def bg_amplitudes_states(field, n, d, batch, states, momenta_ptr, polarisations_ptr, out_ptr, status_ptr=None,
                         stream_ptr=0):
    return load().bg_amplitudes_states(field, n, d, batch, states, momenta_ptr, polarisations_ptr, out_ptr,
                                       status_ptr, stream_ptr)


def bg_amplitudes_primes(metric, n, d, batch, primes, momenta_ptr, polarisations_ptr, out_ptr, status_ptr=None,
                         stream_ptr=0):
    arr = (ctypes.c_uint32 * len(primes))(*primes)
    return load().bg_amplitudes_primes(metric, n, d, batch, len(primes), arr, momenta_ptr, polarisations_ptr,
                                       out_ptr, status_ptr, stream_ptr)


def bg_amplitudes_orderings(field, n, d, batch, n_orderings, orderings_ptr, momenta_ptr, polarisations_ptr, out_ptr,
                            status_ptr=None, stream_ptr=0):
    return load().bg_amplitudes_orderings(field, n, d, batch, n_orderings, orderings_ptr, momenta_ptr,
                                          polarisations_ptr, out_ptr, status_ptr, stream_ptr)


def bg_state_sum(field, prime, batch, states, amp_ptrs, out_ptr, stream_ptr=0):
    arr = (ctypes.c_void_p * len(amp_ptrs))(*amp_ptrs)
    return load().bg_state_sum(field, prime, batch, states, len(amp_ptrs), arr, out_ptr, stream_ptr)


def bg_states(field, prime, metric, d, count, momenta_ptr, chi_ptr, eps_ptr, eps_tilde_ptr, status_ptr=None,
              stream_ptr=0):
    return load().bg_states(field, prime, metric, d, count, momenta_ptr, chi_ptr, eps_ptr, eps_tilde_ptr, status_ptr,
                            stream_ptr)


def bg_generate(field, prime, metric, n, d, batch, seed, start, helicities, momenta_ptr, polarisations_ptr,
                references_ptr=None, redraws_ptr=None, stream_ptr=0):
    hel = None if helicities is None else bytes((int(h) & 0xFF) for h in helicities)
    return load().bg_generate(field, prime, metric, n, d, batch, seed, start, hel, momenta_ptr, polarisations_ptr,
                              references_ptr, redraws_ptr, stream_ptr)


def bg_set_kernel_override(kind=-1, warps=0):
    """kind: -1 / "default", or "general", "unit1", "unit2", "reg", "rt" (bg.h)"""
    return load().bg_set_kernel_override(KERNEL_KINDS[kind] if isinstance(kind, str) else kind, warps)


def bg_kernel_info_problem(pb: Problem) -> dict:
    ki = KernelInfo()
    _check(load().bg_kernel_info_problem(ctypes.byref(pb), ctypes.byref(ki)))
    return {k: int(getattr(ki, k)) for k, _ in KernelInfo._fields_}


def bg_amplitudes_host(field, n, d, batch, host_mom_ptr, host_pol_ptr, host_out_ptr, host_status_ptr,
                       workspace_ptr, workspace_bytes):
    return load().bg_amplitudes_host(field, n, d, batch, host_mom_ptr, host_pol_ptr, host_out_ptr,
                                     host_status_ptr, workspace_ptr, workspace_bytes)


def bg_host_workspace_bytes(field, n, d, chunk_points):
    return int(load().bg_host_workspace_bytes(field, n, d, chunk_points))


def bg_amplitudes_host_noalloc(field, n, d, batch, host_mom_ptr, host_pol_ptr, host_out_ptr, host_status_ptr,
                               stream_ptr=0):
    return load().bg_amplitudes_host_noalloc(field, n, d, batch, host_mom_ptr, host_pol_ptr, host_out_ptr,
                                             host_status_ptr, stream_ptr)


def bg_noalloc_max_batch(field, n, d):
    return int(load().bg_noalloc_max_batch(field, n, d))


def bg_noalloc_scratch_bytes():
    return int(load().bg_noalloc_scratch_bytes())


def bg_modulus():
    return int(load().bg_modulus())


def bg_version():
    return load().bg_version().decode()


def bg_status_string(rc):
    return load().bg_status_string(rc).decode()


def bg_op_count(field, n, d) -> dict:
    oc = OpCount()
    _check(load().bg_op_count(field, n, d, ctypes.byref(oc)))
    return {k: int(getattr(oc, k)) for k, _ in OpCount._fields_}


def bg_selftest_schedules() -> int:
    return int(load().bg_selftest_schedules())


def bg_kernel_info(field, n, d) -> dict:
    ki = KernelInfo()
    _check(load().bg_kernel_info(field, n, d, ctypes.byref(ki)))
    return {k: int(getattr(ki, k)) for k, _ in KernelInfo._fields_}


def bg_peak_probe(kind, iters, blocks, threads, sink_ptr, stream_ptr=0) -> int:
    ops = ctypes.c_int64(0)
    _check(load().bg_peak_probe(PEAK_KINDS[kind] if isinstance(kind, str) else kind, iters, blocks,
                                threads, sink_ptr, ctypes.byref(ops), stream_ptr))
    return int(ops.value)


# ------------------------------------------------------------- tensor helpers
def _torch():
    import torch
    if not torch.cuda.is_available():
        raise BgError("no CUDA device: the Berends-Giele path has no CPU fallback")
    return torch


def field_of(t) -> int:
    import torch
    if t.dtype in (torch.int32, torch.uint32):
        return FIELD_FP31
    if t.dtype == torch.complex128:
        return FIELD_C128
    raise BgError(f"unsupported dtype {t.dtype}: use uint32/int32 (F_p) or complex128")


def to_device(arr: np.ndarray, device="cuda"):
    """numpy [batch,n,d] uint32 / complex128 -> device tensor (F_p stored as int32 bits)"""
    torch = _torch()
    if arr.dtype == np.uint32:
        return torch.from_numpy(arr.view(np.int32)).to(device)
    return torch.from_numpy(np.ascontiguousarray(arr)).to(device)


def to_numpy(t) -> np.ndarray:
    import torch
    a = t.detach().cpu().numpy()
    return a.view(np.uint32) if t.dtype == torch.int32 else a


def _prep(momenta, polarisations):
    torch = _torch()
    if momenta.shape != polarisations.shape or momenta.dim() != 3:
        raise BgError("momenta and polarisations must both be [batch, n, d]")
    if momenta.dtype != polarisations.dtype or not momenta.is_cuda or not polarisations.is_cuda:
        raise BgError("momenta and polarisations must be CUDA tensors of the same dtype")
    if not (momenta.is_contiguous() and polarisations.is_contiguous()):
        raise BgError("inputs must be contiguous")
    batch, n, d = momenta.shape
    return torch, field_of(momenta), int(batch), int(n), int(d)


def amplitudes(momenta, polarisations, out=None, status=None, stream=None):
    """out[b] = eps_n . N(1..n-1) for every point of the batch (one kernel launch)."""
    torch, field, batch, n, d = _prep(momenta, polarisations)
    if out is None:
        out = torch.empty(batch, dtype=momenta.dtype, device=momenta.device)
    s = (stream or torch.cuda.current_stream(momenta.device)).cuda_stream
    with torch.cuda.device(momenta.device):
        if status is None:
            _check(bg_amplitudes(field, n, d, batch, momenta.data_ptr(), polarisations.data_ptr(),
                                 out.data_ptr(), s))
        else:
            _check(bg_amplitudes_status(field, n, d, batch, momenta.data_ptr(), polarisations.data_ptr(),
                                        out.data_ptr(), status.data_ptr(), s))
    return out


def evaluate(momenta, polarisations, metric=METRIC_MOSTLY_MINUS, primes=(), status=None, stream=None,
             orderings=None):
    """The generalised path (bg_evaluate).  momenta [B,n,d] (with primes: [P,B,n,d]); polarisations the same
    shape, or with a state axis [B,S,n,d] ([P,B,S,n,d]); orderings: None or a [K,n] array of leg permutations
    (Eq.(5)).  Returns out [B] / [B,S] / [B,K] / [B,K,S] (leading [P] with primes)."""
    torch = _torch()
    ord_dev = None
    launch = stream or torch.cuda.current_stream(momenta.device)
    if orderings is not None:
        o = np.ascontiguousarray(orderings, dtype=np.uint8)
        if o.ndim != 2 or o.shape[1] != momenta.shape[-2] or \
                not (np.sort(o, axis=1) == np.arange(o.shape[1], dtype=np.uint8)).all():
            raise BgError("orderings must be [K, n] permutations of 0..n-1")
        # the table is a temporary of this call: upload it ON the launch stream, so that the copy is ordered
        # before the kernel and the caching allocator hands the block out again only in that stream's order
        with torch.cuda.stream(launch):
            ord_dev = torch.from_numpy(o).to(momenta.device)
    lead = 1 if primes else 0
    if momenta.dim() != 3 + lead or polarisations.dim() not in (3 + lead, 4 + lead):
        raise BgError("bad tensor ranks for evaluate()")
    if not (momenta.is_cuda and polarisations.is_cuda and momenta.is_contiguous() and polarisations.is_contiguous()):
        raise BgError("inputs must be contiguous CUDA tensors")
    batch, n, d = (int(x) for x in momenta.shape[lead:])
    has_states = polarisations.dim() == 4 + lead
    states = int(polarisations.shape[lead + 1]) if has_states else 1
    field = FIELD_FPMONT if primes else field_of(momenta)
    if primes and (field_of(momenta) != FIELD_FP31 or momenta.shape[0] != len(primes)):
        raise BgError("with primes the inputs are uint32/int32 residues with a leading [len(primes)] axis")
    shape = ([len(primes)] if primes else []) + [batch] + ([ord_dev.shape[0]] if ord_dev is not None else []) + \
        ([states] if has_states else [])
    out = torch.empty(shape, dtype=momenta.dtype, device=momenta.device)
    out.record_stream(launch)
    pb = problem(field, n, d, metric, states, tuple(primes), 0 if ord_dev is None else int(ord_dev.shape[0]),
                 None if ord_dev is None else ord_dev.data_ptr())
    s = launch.cuda_stream
    with torch.cuda.device(momenta.device):
        _check(bg_evaluate(pb, batch, momenta.data_ptr(), polarisations.data_ptr(), out.data_ptr(), None,
                           None if status is None else status.data_ptr(), s))
    return out


def state_sum(amps, prime=0, stream=None):
    """out[b] = sum_s prod_t amps[t][b, s] (Eq.(4)) for a list of [batch, S] CUDA tensors"""
    torch = _torch()
    a0 = amps[0]
    if any(a.shape != a0.shape or a.dtype != a0.dtype or not a.is_cuda or not a.is_contiguous() for a in amps) \
            or a0.dim() != 2:
        raise BgError("amps must be contiguous CUDA tensors [batch, S] of one dtype")
    field = FIELD_FPMONT if prime else field_of(a0)
    out = torch.empty(a0.shape[0], dtype=a0.dtype, device=a0.device)
    s = (stream or torch.cuda.current_stream(a0.device)).cuda_stream
    with torch.cuda.device(a0.device):
        _check(bg_state_sum(field, prime, a0.shape[0], a0.shape[1], [a.data_ptr() for a in amps], out.data_ptr(), s))
    return out


def _dtype_of(field):
    import torch
    return torch.complex128 if field == FIELD_C128 else torch.int32


def generate(field, n, d, batch, seed=0, start=0, metric=METRIC_MOSTLY_MINUS, prime=0, helicities=None,
             want_references=False, stream=None):
    """seeded kinematics generated on the device (bg_generate): (momenta, polarisations[, references], redraws)"""
    torch = _torch()
    dt = _dtype_of(field)
    mom = torch.empty((batch, n, d), dtype=dt, device="cuda")
    pol = torch.empty((batch, n, d), dtype=dt, device="cuda")
    ref = torch.empty((batch, n, d), dtype=dt, device="cuda") if want_references else None
    redraws = torch.zeros(1, dtype=torch.int64, device="cuda")
    s = (stream or torch.cuda.current_stream()).cuda_stream
    _check(bg_generate(field, prime, metric, n, d, batch, seed, start, helicities, mom.data_ptr(), pol.data_ptr(),
                       None if ref is None else ref.data_ptr(), redraws.data_ptr(), s))
    return (mom, pol, ref, redraws) if want_references else (mom, pol, redraws)


def states(momenta, chi, metric=METRIC_MOSTLY_MINUS, prime=0, stream=None):
    """eps, eps_tilde [count, d-2, d] and status [count] for momenta [count, d], chi [count, 4] (bg_states)"""
    torch = _torch()
    count, d = momenta.shape
    field = FIELD_FPMONT if prime else field_of(momenta)
    eps = torch.empty((count, d - 2, d), dtype=momenta.dtype, device=momenta.device)
    til = torch.empty_like(eps)
    status = torch.zeros(count, dtype=torch.int32, device=momenta.device)
    s = (stream or torch.cuda.current_stream(momenta.device)).cuda_stream
    _check(bg_states(field, prime, metric, d, count, momenta.data_ptr(), chi.data_ptr(), eps.data_ptr(),
                     til.data_ptr(), status.data_ptr(), s))
    return eps, til, status


def currents(momenta, polarisations, stream=None):
    """returns (out [batch], currents [batch, m, m, d], status [batch] int32)"""
    torch, field, batch, n, d = _prep(momenta, polarisations)
    m = n - 1
    out = torch.empty(batch, dtype=momenta.dtype, device=momenta.device)
    cur = torch.zeros((batch, m, m, d), dtype=momenta.dtype, device=momenta.device)
    status = torch.zeros(batch, dtype=torch.int32, device=momenta.device)
    s = (stream or torch.cuda.current_stream(momenta.device)).cuda_stream
    with torch.cuda.device(momenta.device):
        _check(bg_currents(field, n, d, batch, momenta.data_ptr(), polarisations.data_ptr(),
                           out.data_ptr(), cur.data_ptr(), status.data_ptr(), s))
    return out, cur, status


def amplitudes_host_noalloc(momenta: np.ndarray, polarisations: np.ndarray, out=None, status=None, stream=None):
    """bg_amplitudes_host_noalloc on HOST arrays: for a caller that cannot allocate device memory (the device
    is already held by another framework's memory pool, or cudaMalloc's device-wide synchronisation is not
    acceptable where the call is made).  Nothing is allocated on the device, not by this wrapper either: the
    staging area is a fixed array inside the library, so the batch is limited to
    bg_noalloc_max_batch(field, n, d) points per call (BgError "batch exceeds ..." beyond it) and calls that
    overlap on the GPU race on that array.  Returns after the results are in `out` (and `status`)."""
    field = FIELD_FP31 if momenta.dtype == np.uint32 else FIELD_C128
    batch, n, d = momenta.shape
    if out is None:
        out = np.empty(batch, dtype=momenta.dtype)
    s = 0 if stream is None else stream.cuda_stream
    _check(bg_amplitudes_host_noalloc(field, n, d, batch, momenta.ctypes.data, polarisations.ctypes.data,
                                      out.ctypes.data, None if status is None else status.ctypes.data, s))
    return out


def amplitudes_host(momenta: np.ndarray, polarisations: np.ndarray, workspace=None, out=None,
                    status=None, chunk_points: int = 1 << 16):
    """End-to-end call on HOST arrays (numpy, ideally backed by pinned memory): H2D copies,
    kernel and D2H copies are pipelined inside the library."""
    torch = _torch()
    field = FIELD_FP31 if momenta.dtype == np.uint32 else FIELD_C128
    batch, n, d = momenta.shape
    if workspace is None:
        nbytes = bg_host_workspace_bytes(field, n, d, max(1024, min(chunk_points, batch)))
        workspace = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    if out is None:
        out = np.empty(batch, dtype=momenta.dtype)
    _check(bg_amplitudes_host(field, n, d, batch, momenta.ctypes.data, polarisations.ctypes.data,
                              out.ctypes.data, None if status is None else status.ctypes.data,
                              workspace.data_ptr(), workspace.numel()))
    return out
