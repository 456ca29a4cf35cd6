// bg_inst_rt.cuh -- bg_rt_kernel<F, MET, D, W, S, MULTI> for d = 4..16 of one (field, metric) pair (W = 4 or 8 warps
// per tile, chosen by n: bg_rt_warps(); S = 1 lane per point for every d, S = 2 for even d; MULTI: the loops over
// colour orderings and state configurations)
#pragma once
#include "../../include/bg.h"
#include "bg_entries.h"
#include "bg_rt.cuh"

namespace {

template <class F, int MET, int D, int W>
const void* rt_for_s(int s, bool multi)
{
    if (s == 1)
        return multi ? reinterpret_cast<const void*>(&bg::bg_rt_kernel<F, MET, D, W, 1, true>)
                     : reinterpret_cast<const void*>(&bg::bg_rt_kernel<F, MET, D, W, 1, false>);
    if constexpr (D % 2 == 0) {
        if (s == 2)
            return multi ? reinterpret_cast<const void*>(&bg::bg_rt_kernel<F, MET, D, W, 2, true>)
                         : reinterpret_cast<const void*>(&bg::bg_rt_kernel<F, MET, D, W, 2, false>);
    }
    return nullptr;
}

template <class F, int MET>
const void* rt_for_d(int d, int s, int w, bool multi)
{
    switch (d) {
#define BG_CASE(D) case D: return w == 4 ? rt_for_s<F, MET, D, 4>(s, multi) : w == 8 ? rt_for_s<F, MET, D, 8>(s, multi) : nullptr;
        BG_CASE(4) BG_CASE(5) BG_CASE(6) BG_CASE(7) BG_CASE(8) BG_CASE(9) BG_CASE(10)
        BG_CASE(11) BG_CASE(12) BG_CASE(13) BG_CASE(14) BG_CASE(15) BG_CASE(16)
#undef BG_CASE
    }
    return nullptr;
}

}  // namespace
