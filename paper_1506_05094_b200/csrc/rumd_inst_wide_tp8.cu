// one translation unit per tp: see rumd_dispatch.cuh
#include "rumd_inst_wide.cuh"
template <> void rumd_fill_wide<8>(const void* (*wide)[2], const void* (*wide3)[2]) { fill_wide_tables<8>(wide, wide3); }
