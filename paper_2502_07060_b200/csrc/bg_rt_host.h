// bg_rt_host.h -- host side of bg_rt_kernel (bg_rt.cuh): the tile layout of a run-time n and its schedule as a
// packed table, built once per shape by bg_api.cu and copied to the device it is first used on.
#pragma once
#include <stddef.h>

#include <vector>

#include "bg_common.cuh"

struct RtHost {
    bg::RtLayout lay;
    int s;                         // lanes per point
    int threads, points_per_block;
    size_t smem;                   // dynamic shared memory per block
    std::vector<unsigned char> blob;   // FlatOp[nops] | quad[] | beg[W+1] | ranges[r], each 16-byte aligned
    size_t off_quad, off_beg, off_ranges;
};

// layout and tables for elements of `eb` bytes moved in vector units of `u` elements, n gluons, d dimensions, s lanes
// per point (d % s == 0); false if n is out of range.  The caller checks smem against the device limit.
bool bg_rt_make(int eb, int u, int n, int d, int s, RtHost* out);
