"""Build libbg_b200.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2502_07060_b200.build [--force]
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")
LIB = os.path.join(HERE, "libbg_b200.so")
SOURCES = ["bg_api.cu", "bg_rt_host.cu", "bg_inst_default.cu", "bg_inst_fp_alt.cu", "bg_inst_c128_alt.cu", "bg_inst_paper.cu",
           "bg_inst_grid0.cu", "bg_inst_grid1.cu", "bg_inst_grid2.cu", "bg_inst_grid3.cu", "bg_inst_cgrid0.cu", "bg_inst_cgrid1.cu",
           "bg_inst_metric.cu", "bg_inst_mont.cu", "bg_inst_general_fp31.cu", "bg_inst_general_c128.cu",
           "bg_inst_general_mont.cu", "bg_inst_rt_fp31_mm.cu", "bg_inst_rt_fp31_alt.cu", "bg_inst_rt_c128_mm.cu", "bg_inst_rt_c128_alt.cu",
           "bg_inst_rt_mont_mm.cu", "bg_inst_rt_mont_alt.cu", "bg_state_sum.cu", "bg_states.cu", "bg_generate.cu", "bg_noalloc.cu", "bg_peaks.cu", "bg_selftest.cu"]
HEADERS = ["bg_field.cuh", "bg_common.cuh", "bg_schedule.cuh", "bg_tile.cuh", "bg_unit.cuh", "bg_reg.cuh",
           "bg_general.cuh", "bg_rt.cuh", "bg_inst_rt.cuh", "bg_rt_host.h", "bg_entries.h", "bg_inst_common.cuh", "bg_inst_general.cuh", "bg_states.cuh", "bg_host_util.h"]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
    "-Xcompiler", "-fPIC", "-Xptxas", "-v", "-Xptxas", "-warn-spills",
    # the schedules (bg_schedule.cuh) are found by constexpr dynamic programming, also in the host pass
    "-Xcompiler", "-fconstexpr-ops-limit=2000000000",
]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.join(INCLUDE, "bg.h"), __file__]
    return any(os.path.getmtime(p) > t for p in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    objs = []
    procs = []
    for src in SOURCES:
        obj = os.path.join(CSRC, src.replace(".cu", ".o"))
        objs.append(obj)
        cmd = [nvcc, *NVCC_FLAGS, "-c", os.path.join(CSRC, src), "-o", obj]
        procs.append((src, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
    log = []
    for src, p in procs:
        out, _ = p.communicate()
        log.append(out)
        if p.returncode != 0:
            sys.stderr.write(out)
            raise RuntimeError(f"nvcc failed on {src}")
    with open(os.path.join(CSRC, "ptxas.log"), "w") as f:
        f.write("\n".join(log))
    if verbose:
        print("\n".join(log))
    cmd = [nvcc, "-shared", "-o", LIB, *objs, "-gencode", "arch=compute_100a,code=sm_100a"]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
