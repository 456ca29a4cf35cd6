// bg_inst_grid1.cu -- F_p instances of bg_unit_kernel filling the grid n = 4..10 x d = 4..10 (the dimensions
// the paper validates), part 2 of 3; split over files for build parallelism and
// the 64 KB of constant memory per module.
#include "bg_inst_common.cuh"

const SweepEntry* bg_entries_grid1(int* count)
{
    static const SweepEntry table[] = {
        unit_entry<Fp31, 5, 5, 1>(BG_FIELD_FP31),
        unit_entry<Fp31, 8, 5, 4>(BG_FIELD_FP31),
        unit_entry<Fp31, 4, 6, 1>(BG_FIELD_FP31),
        unit_entry<Fp31, 10, 6, 8>(BG_FIELD_FP31),
        unit_entry<Fp31, 6, 7, 2>(BG_FIELD_FP31),
        unit_entry<Fp31, 9, 7, 4>(BG_FIELD_FP31),
        unit_entry<Fp31, 5, 9, 1>(BG_FIELD_FP31),
        unit_entry<Fp31, 8, 9, 4>(BG_FIELD_FP31),
        unit_entry<Fp31, 4, 10, 1>(BG_FIELD_FP31),
        unit_entry<Fp31, 8, 10, 4>(BG_FIELD_FP31),
    };
    *count = (int)(sizeof(table) / sizeof(table[0]));
    return table;
}
