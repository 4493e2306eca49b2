// one translation unit per tp: see rumd_dispatch.cuh
#include "rumd_inst.cuh"
const KernelSet* rumd_kernels_tp8() { return kernel_set<8>(); }
