// bg_inst_grid2.cu -- F_p instances of bg_unit_kernel filling the grid n = 4..10 x d = 4..10 (the dimensions
// the paper validates), part 3 of 3; split over files for build parallelism and
// the 64 KB of constant memory per module.
#include "bg_inst_common.cuh"

const SweepEntry* bg_entries_grid2(int* count)
{
    static const SweepEntry table[] = {
        unit_entry<Fp31, 6, 5, 2>(BG_FIELD_FP31),
        unit_entry<Fp31, 9, 5, 4>(BG_FIELD_FP31),
        unit_entry<Fp31, 5, 6, 1>(BG_FIELD_FP31),
        unit_entry<Fp31, 4, 7, 1>(BG_FIELD_FP31),
        unit_entry<Fp31, 7, 7, 4>(BG_FIELD_FP31),
        unit_entry<Fp31, 10, 7, 8>(BG_FIELD_FP31),
        unit_entry<Fp31, 6, 9, 2>(BG_FIELD_FP31),
        unit_entry<Fp31, 9, 9, 4>(BG_FIELD_FP31),
        unit_entry<Fp31, 5, 10, 1>(BG_FIELD_FP31),
        unit_entry<Fp31, 10, 10, 8>(BG_FIELD_FP31),
    };
    *count = (int)(sizeof(table) / sizeof(table[0]));
    return table;
}
