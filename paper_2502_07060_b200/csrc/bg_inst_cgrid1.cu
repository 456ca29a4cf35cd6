// bg_inst_cgrid1.cu -- complex128 instances of bg_split_kernel (two lanes per point, 16-point tiles) for
// n = 4..10 at d = 4, 6, 8, part 2 of 2, so that these shapes do not fall to the general kernel.
#include "bg_inst_common.cuh"

const SweepEntry* bg_entries_cgrid1(int* count)
{
    static const SweepEntry table[] = {
        split_entry<C128, 5, 4, 2>(BG_FIELD_C128),
        split_entry<C128, 8, 4, 4>(BG_FIELD_C128),
        split_entry<C128, 10, 4, 8>(BG_FIELD_C128),
        split_entry<C128, 5, 6, 2>(BG_FIELD_C128),
        split_entry<C128, 7, 6, 4>(BG_FIELD_C128),
        split_entry<C128, 9, 6, 8>(BG_FIELD_C128),
        split_entry<C128, 4, 8, 2>(BG_FIELD_C128),
        split_entry<C128, 6, 8, 4>(BG_FIELD_C128),
        split_entry<C128, 8, 8, 4>(BG_FIELD_C128),
        split_entry<C128, 10, 8, 8>(BG_FIELD_C128),
    };
    *count = (int)(sizeof(table) / sizeof(table[0]));
    return table;
}
