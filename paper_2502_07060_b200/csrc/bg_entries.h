// bg_entries.h -- the table of compile-time (n, d) kernel instances, shared between bg_api.cu (which
// selects and launches) and the bg_inst_*.cu translation units (which instantiate the kernels).
#pragma once
#include <stddef.h>

struct SweepEntry {
    int field, n, d, w;      // w: warps per tile (bg_reg_kernel: independent warps per block)
    int kind;                // 0: bg_tile_kernel (table-driven loop over splittings), 1: bg_level_kernel (levels
                             // unrolled), 2: bg_split_kernel (table-driven, two lanes per point), 3: bg_reg_kernel
                             // (currents in registers, no barriers), 4: bg_unit_kernel (one body per number of
                             // 4-gluon splits)
    int tp;                  // points per block
    const void* func;
    size_t smem;
};

// first entry of a shape = the default; the others are selected with the tuning knobs BG_KERNEL
// (tile|level|split|reg|unit) and BG_SWEEP_W (warps per tile), read from the environment per call
const SweepEntry* bg_entries_default(int* count);     // bg_inst_default.cu
const SweepEntry* bg_entries_fp_alt(int* count);      // bg_inst_fp_alt.cu
const SweepEntry* bg_entries_c128_alt(int* count);    // bg_inst_c128_alt.cu
const SweepEntry* bg_entries_paper(int* count);       // bg_inst_paper.cu
const SweepEntry* bg_entries_grid0(int* count);       // bg_inst_grid0.cu
const SweepEntry* bg_entries_grid1(int* count);       // bg_inst_grid1.cu
const SweepEntry* bg_entries_grid2(int* count);       // bg_inst_grid2.cu
const SweepEntry* bg_entries_cgrid0(int* count);      // bg_inst_cgrid0.cu
const SweepEntry* bg_entries_cgrid1(int* count);      // bg_inst_cgrid1.cu
