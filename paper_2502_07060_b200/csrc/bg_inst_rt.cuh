// bg_inst_rt.cuh -- bg_rt_kernel<F, MET, D, W, S> for d = 4..16 of one (field, metric) pair (W = kRtWarps warps per
// tile; S = 1 lane per point for every d, S = 2 for even d)
#pragma once
#include "../../include/bg.h"
#include "bg_entries.h"
#include "bg_rt.cuh"

namespace {

template <class F, int MET, int D>
const void* rt_for_s(int s)
{
    if (s == 1) return reinterpret_cast<const void*>(&bg::bg_rt_kernel<F, MET, D, kRtWarps, 1>);
    if constexpr (D % 2 == 0) {
        if (s == 2) return reinterpret_cast<const void*>(&bg::bg_rt_kernel<F, MET, D, kRtWarps, 2>);
    }
    return nullptr;
}

template <class F, int MET>
const void* rt_for_d(int d, int s)
{
    switch (d) {
#define BG_CASE(D) case D: return rt_for_s<F, MET, D>(s);
        BG_CASE(4) BG_CASE(5) BG_CASE(6) BG_CASE(7) BG_CASE(8) BG_CASE(9) BG_CASE(10)
        BG_CASE(11) BG_CASE(12) BG_CASE(13) BG_CASE(14) BG_CASE(15) BG_CASE(16)
#undef BG_CASE
    }
    return nullptr;
}

template <class F>
const void* rt_for(int metric, int d, int s)
{
    return metric == BG_METRIC_MOSTLY_MINUS ? rt_for_d<F, BG_METRIC_MOSTLY_MINUS>(d, s)
         : metric == BG_METRIC_ALTERNATING ? rt_for_d<F, BG_METRIC_ALTERNATING>(d, s) : nullptr;
}

}  // namespace
