// bg_entries.h -- the table of compile-time (field, metric, n, d) kernel instances, shared between
// bg_api.cu (which selects and launches) and the bg_inst_*.cu translation units (which instantiate
// the kernels; several units because the work lists of an instance sit in constant memory, a module
// has 64 KB of it, and nvcc compiles them in parallel).
#pragma once
#include <stddef.h>

enum BgKernelKind {
    BG_KIND_UNIT1 = 0,       // bg_unit_kernel, one lane per point, 32-point tiles
    BG_KIND_UNIT2 = 1,       // bg_unit_kernel, two lanes per point, 16-point tiles
    BG_KIND_REG = 2,         // bg_reg_kernel: currents in registers, no barriers (one state configuration only)
    BG_KIND_GENERAL = 3,     // bg_general_kernel: run-time n, one thread per point (not in the tables)
    BG_KIND_RT = 4           // bg_rt_kernel: the tiled kernel for a run-time n (not in the tables)
};

struct KernelEntry {
    int field, metric, n, d;
    int w;                   // warps per tile (bg_reg_kernel: independent warps per block)
    int kind;                // BgKernelKind
    int tp;                  // points per block
    const void* func;        // one state configuration, one ordering
    const void* func_multi;  // loops over orderings and state configurations; NULL: not available (bg_reg_kernel)
    size_t smem;             // dynamic shared memory of func
    size_t smem_multi;       // ... of func_multi (keeps the propagators in a table of their own)
};

// first entry of a shape = the default; the others are reachable through bg_set_kernel_override
#define BG_ENTRY_TABLES(X) X(default) X(fp_alt) X(c128_alt) X(paper) X(grid0) X(grid1) X(grid2) X(grid3) X(cgrid0) X(cgrid1) \
    X(metric) X(mont)
#define BG_DECLARE_TABLE(name) const KernelEntry* bg_entries_##name(int* count);
BG_ENTRY_TABLES(BG_DECLARE_TABLE)
#undef BG_DECLARE_TABLE

// bg_general_kernel<F, MET, D> for d = 4..16, one translation unit per field (bg_inst_general_*.cu);
// NULL if (metric, d) is out of range
// bg_rt_kernel<F, MET, D, W, S> for d = 4..16, W = 4 or 8 warps per tile, S = 1 or (even d) 2, one translation unit per
// field (bg_inst_rt_*.cu); NULL if out of range
inline int bg_rt_warps(int n) { return n <= 8 ? 4 : 8; }     // as the compiled instances (measured at cfg2, cfg3)
const void* bg_rt_kernel_ptr_fp31(int metric, int d, int s, int w, bool multi);
const void* bg_rt_kernel_ptr_c128(int metric, int d, int s, int w, bool multi);
const void* bg_rt_kernel_ptr_mont(int metric, int d, int s, int w, bool multi);
const void* bg_general_kernel_ptr_fp31(int metric, int d);
const void* bg_general_kernel_ptr_c128(int metric, int d);
const void* bg_general_kernel_ptr_mont(int metric, int d);
