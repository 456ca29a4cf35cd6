// bg_inst_common.cuh -- entry constructors used by the bg_inst_*.cu translation units
#pragma once
#include "../../include/bg.h"
#include "bg_entries.h"
#include "bg_level.cuh"
#include "bg_reg.cuh"
#include "bg_split.cuh"
#include "bg_tile.cuh"
#include "bg_unit.cuh"

namespace {

using bg::C128;
using bg::Fp31;

template <class F, int N, int D, int W>
SweepEntry sweep_entry(int field)
{
    return SweepEntry{field, N, D, W, 0, 32, reinterpret_cast<const void*>(&bg::bg_tile_kernel<F, N, D, W>),
                      bg::TileCfg<F, N, D, W>::SMEM_BYTES};
}
template <class F, int N, int D, int W>
SweepEntry level_entry(int field)
{
    return SweepEntry{field, N, D, W, 1, 32, reinterpret_cast<const void*>(&bg::bg_level_kernel<F, N, D, W>),
                      bg::TileCfg<F, N, D, W>::SMEM_BYTES};
}
template <class F, int N, int D, int W>
SweepEntry split_entry(int field)
{
    return SweepEntry{field, N, D, W, 2, 16, reinterpret_cast<const void*>(&bg::bg_split_kernel<F, N, D, W, 2>),
                      bg::SplitCfg<F, N, D, W, 2>::SMEM_BYTES};
}
template <class F, int N, int D>
SweepEntry reg_entry(int field)
{
    return SweepEntry{field, N, D, bg::RegCfg<F, N, D>::WARPS, 3, 16 * bg::RegCfg<F, N, D>::WARPS,
                      reinterpret_cast<const void*>(&bg::bg_reg_kernel<F, N, D>), bg::RegCfg<F, N, D>::SMEM_BYTES};
}
template <class F, int N, int D, int W>
SweepEntry unit_entry(int field)
{
    return SweepEntry{field, N, D, W, 4, 32, reinterpret_cast<const void*>(&bg::bg_unit_kernel<F, N, D, W>),
                      bg::TileCfg<F, N, D, W>::SMEM_BYTES};
}

}  // namespace
