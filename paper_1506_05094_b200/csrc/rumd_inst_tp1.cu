// one translation unit per tp: see rumd_dispatch.cuh
#include "rumd_inst.cuh"
const KernelSet* rumd_kernels_tp1() { return kernel_set<1>(); }
