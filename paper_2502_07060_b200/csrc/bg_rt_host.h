// bg_rt_host.h -- host side of bg_rt_kernel (bg_rt.cuh): the tile layout of a run-time n and its schedule, built
// once per shape by bg_api.cu and passed to every launch in the kernel's parameter block (bg::RtTables).
#pragma once
#include <stddef.h>

#include "bg_common.cuh"

struct RtHost {
    bg::RtLayout lay;
    int s;                         // lanes per point
    int threads, points_per_block;
    size_t smem;                   // dynamic shared memory per block
    bg::RtTables tab;              // ops, 4-gluon-split table, warp bounds, ranges
};

// layout and tables for elements of `eb` bytes moved in vector units of `u` elements, n gluons, d dimensions, s lanes
// per point (d % s == 0); multi: the layout of the MULTI instantiation (-1/P^2 in a table of its own instead of the U
// slots of the multi-gluon rows: with several orderings / state configurations per point the propagators outlive a
// sweep).  false if n is out of range.  The caller checks smem against the device limit.
bool bg_rt_make(int eb, int u, int n, int d, int s, bool multi, RtHost* out);
