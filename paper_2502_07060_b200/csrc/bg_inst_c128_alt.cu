// bg_inst_c128_alt.cu -- alternative complex128 instances for A/B runs (BG_KERNEL, BG_SWEEP_W)
#include "bg_inst_common.cuh"

const SweepEntry* bg_entries_c128_alt(int* count)
{
    static const SweepEntry table[] = {
        level_entry<C128, 6, 4, 2>(BG_FIELD_C128),
        level_entry<C128, 6, 4, 4>(BG_FIELD_C128),
        sweep_entry<C128, 6, 4, 4>(BG_FIELD_C128),
        sweep_entry<C128, 6, 4, 2>(BG_FIELD_C128),
        split_entry<C128, 6, 4, 2>(BG_FIELD_C128),
        split_entry<C128, 6, 4, 4>(BG_FIELD_C128),
    };
    *count = (int)(sizeof(table) / sizeof(table[0]));
    return table;
}
