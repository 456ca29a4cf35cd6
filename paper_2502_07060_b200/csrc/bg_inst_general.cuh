// bg_inst_general.cuh -- bg_general_kernel<F, MET, D> for d = 4..16 of one (field, metric) pair
#pragma once
#include "../../include/bg.h"
#include "bg_entries.h"
#include "bg_general.cuh"

namespace {

template <class F, int MET>
const void* general_for_d(int d)
{
    switch (d) {
#define BG_CASE(D) case D: return reinterpret_cast<const void*>(&bg::bg_general_kernel<F, MET, D>);
        BG_CASE(4) BG_CASE(5) BG_CASE(6) BG_CASE(7) BG_CASE(8) BG_CASE(9) BG_CASE(10)
        BG_CASE(11) BG_CASE(12) BG_CASE(13) BG_CASE(14) BG_CASE(15) BG_CASE(16)
#undef BG_CASE
    }
    return nullptr;
}

}  // namespace
