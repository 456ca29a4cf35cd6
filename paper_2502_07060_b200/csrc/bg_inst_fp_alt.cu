// bg_inst_fp_alt.cu -- alternative F_p instances for A/B runs (BG_KERNEL, BG_SWEEP_W)
#include "bg_inst_common.cuh"

const SweepEntry* bg_entries_fp_alt(int* count)
{
    static const SweepEntry table[] = {
        sweep_entry<Fp31, 8, 6, 4>(BG_FIELD_FP31),
        sweep_entry<Fp31, 4, 4, 1>(BG_FIELD_FP31),
        level_entry<Fp31, 8, 6, 6>(BG_FIELD_FP31),
        unit_entry<Fp31, 8, 6, 4>(BG_FIELD_FP31),
        sweep_entry<Fp31, 10, 8, 8>(BG_FIELD_FP31),
        sweep_entry<Fp31, 12, 6, 16>(BG_FIELD_FP31),
    };
    *count = (int)(sizeof(table) / sizeof(table[0]));
    return table;
}
