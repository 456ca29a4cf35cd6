// bg_inst_common.cuh -- entry constructors used by the bg_inst_*.cu translation units
#pragma once
#include "../../include/bg.h"
#include "bg_entries.h"
#include "bg_reg.cuh"
#include "bg_unit.cuh"

namespace {

using bg::C128;
using bg::Fp31;
using bg::FpMont;
constexpr int MM = BG_METRIC_MOSTLY_MINUS, ALT = BG_METRIC_ALTERNATING;

// bg_unit_kernel with S lanes per point and W warps per tile
template <class F, int MET, int N, int D, int W, int S = 1>
KernelEntry unit_entry()
{
    return KernelEntry{F::kFieldId, MET, N, D, W, S == 1 ? BG_KIND_UNIT1 : BG_KIND_UNIT2, 32 / S,
                       reinterpret_cast<const void*>(&bg::bg_unit_kernel<F, MET, N, D, W, S, false>),
                       reinterpret_cast<const void*>(&bg::bg_unit_kernel<F, MET, N, D, W, S, true>),
                       bg::TileCfg<F, N, D, W, S, false>::SMEM_BYTES, bg::TileCfg<F, N, D, W, S, true>::SMEM_BYTES};
}
template <class F, int MET, int N, int D>
KernelEntry reg_entry()
{
    return KernelEntry{F::kFieldId, MET, N, D, bg::RegCfg<F, N, D>::WARPS, BG_KIND_REG, 16 * bg::RegCfg<F, N, D>::WARPS,
                       reinterpret_cast<const void*>(&bg::bg_reg_kernel<F, MET, N, D>), nullptr,
                       bg::RegCfg<F, N, D>::SMEM_BYTES, 0};
}

}  // namespace

#define BG_DEFINE_TABLE(name, ...)                                              \
    const KernelEntry* bg_entries_##name(int* count)                            \
    {                                                                           \
        static const KernelEntry table[] = {__VA_ARGS__};                       \
        *count = (int)(sizeof(table) / sizeof(table[0]));                       \
        return table;                                                           \
    }
