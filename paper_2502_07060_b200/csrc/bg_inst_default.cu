// bg_inst_default.cu -- the kernel instances a call launches by default (chosen by measurement on B200)
#include "bg_inst_common.cuh"

const SweepEntry* bg_entries_default(int* count)
{
    static const SweepEntry table[] = {
        level_entry<Fp31, 8, 6, 4>(BG_FIELD_FP31),       // cfg2
        level_entry<Fp31, 4, 4, 1>(BG_FIELD_FP31),       // cfg0
        unit_entry<Fp31, 10, 8, 8>(BG_FIELD_FP31),       // cfg3
        unit_entry<Fp31, 12, 6, 8>(BG_FIELD_FP31),       // cfg4a
        reg_entry<C128, 6, 4>(BG_FIELD_C128),            // cfg1
        split_entry<C128, 12, 6, 16>(BG_FIELD_C128),     // cfg4b
    };
    *count = (int)(sizeof(table) / sizeof(table[0]));
    return table;
}
