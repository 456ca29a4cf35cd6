// bg_inst_grid0.cu -- F_p instances of bg_unit_kernel filling the grid n = 4..10 x d = 4..10 (the dimensions
// the paper validates), part 1 of 3; split over files for build parallelism and
// the 64 KB of constant memory per module.
#include "bg_inst_common.cuh"

const SweepEntry* bg_entries_grid0(int* count)
{
    static const SweepEntry table[] = {
        unit_entry<Fp31, 4, 5, 1>(BG_FIELD_FP31),
        unit_entry<Fp31, 7, 5, 4>(BG_FIELD_FP31),
        unit_entry<Fp31, 10, 5, 8>(BG_FIELD_FP31),
        unit_entry<Fp31, 7, 6, 4>(BG_FIELD_FP31),
        unit_entry<Fp31, 5, 7, 1>(BG_FIELD_FP31),
        unit_entry<Fp31, 8, 7, 4>(BG_FIELD_FP31),
        unit_entry<Fp31, 4, 9, 1>(BG_FIELD_FP31),
        unit_entry<Fp31, 7, 9, 4>(BG_FIELD_FP31),
        unit_entry<Fp31, 10, 9, 8>(BG_FIELD_FP31),
        unit_entry<Fp31, 7, 10, 4>(BG_FIELD_FP31),
    };
    *count = (int)(sizeof(table) / sizeof(table[0]));
    return table;
}
