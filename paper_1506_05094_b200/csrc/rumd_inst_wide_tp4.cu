// one translation unit per tp: see rumd_dispatch.cuh
#include "rumd_inst_wide.cuh"
template <> void rumd_fill_wide<4>(const void* (*wide)[2], const void* (*wide3)[2]) { fill_wide_tables<4>(wide, wide3); }
