// rumd_dispatch.cuh -- the kernels that are templated on (tp, second-term kind, one-type) live in one translation
// unit per tp (rumd_inst_tp*.cu), so that the library builds in parallel; the host code (rumd_b200.cu) reaches
// them through this table.  Product code: shares nothing with oracle/.
#pragma once
#include "rumd_types.cuh"

// Listed pairs in flight per lane (the paper's one-ahead prefetch, P:108 item 4, generalised).  Measured on
// B200 (2 / 4 / 8 / 16 per lane): 8 is best while a lane has >= ~10 entries, 4 for the wide groups.
template <int TP> struct UnrollOf { static constexpr int value = TP >= 16 ? 4 : 8; };

// coul: 0 no second term, 1 Coulomb only, 2 any second-term kind of P:73;  one: a single particle type
struct KernelSet {
    const void* persist[3][2];  // k_persist<TP, coul, one, unroll, false>
    const void* persist_tile[3][2]; // k_persist<TP, coul, one, unroll, true> (tile method; null for tp > 8)
    const void* persist_wide[3][2]; // k_persist<TP, coul, one, unroll, false, 512>: blocks of 512 threads, one per SM (null for coul = 2)
    const void* persist_wide3[3][2]; // k_persist<TP, coul, one, unroll, false, 768>: blocks of 768 threads (tp < 8, coul < 2), one per SM
    const void* ensemble[3][2]; // k_ensemble<TP, coul, one>
    const void* force_fn[3][2]; // k_force<TP, coul, one, unroll>
    void (*force)(int coul, bool one, const Sys& S, int nblocks, int nthreads, cudaStream_t stream);
    void (*step)(int coul, bool one, bool energy, int nvt, const Sys& S, int nblocks, int nthreads, cudaStream_t stream);
    // tile method: pair forces out of shared memory (smem = dynamic shared bytes; returns the CUDA status)
    cudaError_t (*force_tile)(int coul, bool one, const Sys& S, int nblocks, size_t smem, cudaStream_t stream);
};

// the two wider instantiations of k_persist (512 and 768 threads per block) are compiled in translation units of their
// own (rumd_inst_wide_tp*.cu: twice the parallelism for the build); each defines this for its tp
template <int TP> void rumd_fill_wide(const void* (*wide)[2], const void* (*wide3)[2]);

const KernelSet* rumd_kernels_tp1();
const KernelSet* rumd_kernels_tp2();
const KernelSet* rumd_kernels_tp4();
const KernelSet* rumd_kernels_tp8();
const KernelSet* rumd_kernels_tp16();
const KernelSet* rumd_kernels_tp32();
