// rumd_inst_wide.cuh -- the 512- and 768-thread instantiations of k_persist for ONE value of tp (included by
// rumd_inst_wide_tp*.cu; see rumd_dispatch.cuh).  Product code: shares nothing with oracle/.
#pragma once
#include "rumd_dispatch.cuh"
#include "rumd_persist.cuh"

// (not for the generic second-term kinds, COUL == 2: they keep blocks of 256 threads)
template <int TP, int COUL, bool ONE> static const void* persist_wide_fn()
{
    if constexpr (COUL < 2) return (const void*)&k_persist<TP, COUL, ONE, UnrollOf<TP>::value, false, 512>;
    else return nullptr;
}

template <int TP, int COUL, bool ONE> static const void* persist_wide3_fn()
{
    if constexpr (TP < 8 && COUL < 2) return (const void*)&k_persist<TP, COUL, ONE, UnrollOf<TP>::value, false, 768>;
    else return nullptr;
}

template <int TP> static void fill_wide_tables(const void* (*wide)[2], const void* (*wide3)[2])
{
    wide[0][0] = persist_wide_fn<TP, 0, false>();
    wide[0][1] = persist_wide_fn<TP, 0, true>();
    wide[1][0] = persist_wide_fn<TP, 1, false>();
    wide[1][1] = persist_wide_fn<TP, 1, true>();
    wide[2][0] = persist_wide_fn<TP, 2, false>();
    wide[2][1] = persist_wide_fn<TP, 2, true>();
    wide3[0][0] = persist_wide3_fn<TP, 0, false>();
    wide3[0][1] = persist_wide3_fn<TP, 0, true>();
    wide3[1][0] = persist_wide3_fn<TP, 1, false>();
    wide3[1][1] = persist_wide3_fn<TP, 1, true>();
    wide3[2][0] = persist_wide3_fn<TP, 2, false>();
    wide3[2][1] = persist_wide3_fn<TP, 2, true>();
}
