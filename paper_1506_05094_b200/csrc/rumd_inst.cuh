// rumd_inst.cuh -- instantiates every kernel templated on tp for ONE value of tp (included by rumd_inst_tp*.cu).
#pragma once
#include "rumd_dispatch.cuh"
#include "rumd_persist.cuh"
#include "rumd_ensemble.cuh"

template <int TP, int COUL, bool ONE>
static void launch_force_inst(const Sys& S, int nb, int nt, cudaStream_t st)
{
    k_force<TP, COUL, ONE, UnrollOf<TP>::value><<<nb, nt, 0, st>>>(S);
}

template <int TP, int COUL, bool ONE>
static void launch_step_inst(bool energy, int nvt, const Sys& S, int nb, int nt, cudaStream_t st)
{
    if (energy)
        k_step<TP, COUL, ONE, UnrollOf<TP>::value, true><<<nb, nt, 0, st>>>(S, nvt);
    else
        k_step<TP, COUL, ONE, UnrollOf<TP>::value, false><<<nb, nt, 0, st>>>(S, nvt);
}

template <int TP> static void force_tp(int coul, bool one, const Sys& S, int nb, int nt, cudaStream_t st)
{
    switch (coul * 2 + (one ? 1 : 0)) {
    case 0: launch_force_inst<TP, 0, false>(S, nb, nt, st); break;
    case 1: launch_force_inst<TP, 0, true>(S, nb, nt, st); break;
    case 2: launch_force_inst<TP, 1, false>(S, nb, nt, st); break;
    case 3: launch_force_inst<TP, 1, true>(S, nb, nt, st); break;
    case 4: launch_force_inst<TP, 2, false>(S, nb, nt, st); break;
    default: launch_force_inst<TP, 2, true>(S, nb, nt, st); break;
    }
}

template <int TP>
static void step_tp(int coul, bool one, bool energy, int nvt, const Sys& S, int nb, int nt, cudaStream_t st)
{
    switch (coul * 2 + (one ? 1 : 0)) {
    case 0: launch_step_inst<TP, 0, false>(energy, nvt, S, nb, nt, st); break;
    case 1: launch_step_inst<TP, 0, true>(energy, nvt, S, nb, nt, st); break;
    case 2: launch_step_inst<TP, 1, false>(energy, nvt, S, nb, nt, st); break;
    case 3: launch_step_inst<TP, 1, true>(energy, nvt, S, nb, nt, st); break;
    case 4: launch_step_inst<TP, 2, false>(energy, nvt, S, nb, nt, st); break;
    default: launch_step_inst<TP, 2, true>(energy, nvt, S, nb, nt, st); break;
    }
}

template <int TP, int COUL, bool ONE>
static cudaError_t launch_force_tile_inst(const Sys& S, int nb, size_t smem, cudaStream_t st)
{
    auto fn = &k_force_tile<TP, COUL, ONE>;
    cudaError_t e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    fn<<<nb, TILE_THREADS, smem, st>>>(S);
    return cudaSuccess;
}

template <int TP> static cudaError_t force_tile_tp(int coul, bool one, const Sys& S, int nb, size_t smem, cudaStream_t st)
{
    if constexpr (TP > 8) return cudaErrorInvalidValue; // the tile method takes tp <= 8 (chunks of 8 entries per lane)
    else
    switch (coul * 2 + (one ? 1 : 0)) {
    case 0: return launch_force_tile_inst<TP, 0, false>(S, nb, smem, st);
    case 1: return launch_force_tile_inst<TP, 0, true>(S, nb, smem, st);
    case 2: return launch_force_tile_inst<TP, 1, false>(S, nb, smem, st);
    case 3: return launch_force_tile_inst<TP, 1, true>(S, nb, smem, st);
    case 4: return launch_force_tile_inst<TP, 2, false>(S, nb, smem, st);
    default: return launch_force_tile_inst<TP, 2, true>(S, nb, smem, st);
    }
}

template <int TP, int COUL, bool ONE> static const void* persist_tile_fn()
{
    if constexpr (TP <= 8) return (const void*)&k_persist<TP, COUL, ONE, UnrollOf<TP>::value, true>;
    else return nullptr;
}

template <int TP> static const KernelSet* kernel_set()
{
    static const KernelSet ks = [] {
    KernelSet k = {
        {{(const void*)&k_persist<TP, 0, false, UnrollOf<TP>::value, false>, (const void*)&k_persist<TP, 0, true, UnrollOf<TP>::value, false>},
         {(const void*)&k_persist<TP, 1, false, UnrollOf<TP>::value, false>, (const void*)&k_persist<TP, 1, true, UnrollOf<TP>::value, false>},
         {(const void*)&k_persist<TP, 2, false, UnrollOf<TP>::value, false>, (const void*)&k_persist<TP, 2, true, UnrollOf<TP>::value, false>}},
        {{persist_tile_fn<TP, 0, false>(), persist_tile_fn<TP, 0, true>()},
         {persist_tile_fn<TP, 1, false>(), persist_tile_fn<TP, 1, true>()},
         {persist_tile_fn<TP, 2, false>(), persist_tile_fn<TP, 2, true>()}},
        {{nullptr, nullptr}, {nullptr, nullptr}, {nullptr, nullptr}}, // persist_wide, persist_wide3: filled below
        {{nullptr, nullptr}, {nullptr, nullptr}, {nullptr, nullptr}},
        {{(const void*)&k_ensemble<TP, 0, false, UnrollOf<TP>::value>, (const void*)&k_ensemble<TP, 0, true, UnrollOf<TP>::value>},
         {(const void*)&k_ensemble<TP, 1, false, UnrollOf<TP>::value>, (const void*)&k_ensemble<TP, 1, true, UnrollOf<TP>::value>},
         {(const void*)&k_ensemble<TP, 2, false, UnrollOf<TP>::value>, (const void*)&k_ensemble<TP, 2, true, UnrollOf<TP>::value>}},
        {{(const void*)&k_force<TP, 0, false, UnrollOf<TP>::value>, (const void*)&k_force<TP, 0, true, UnrollOf<TP>::value>},
         {(const void*)&k_force<TP, 1, false, UnrollOf<TP>::value>, (const void*)&k_force<TP, 1, true, UnrollOf<TP>::value>},
         {(const void*)&k_force<TP, 2, false, UnrollOf<TP>::value>, (const void*)&k_force<TP, 2, true, UnrollOf<TP>::value>}},
        &force_tp<TP>,
        &step_tp<TP>,
        &force_tile_tp<TP>,
    };
    rumd_fill_wide<TP>(k.persist_wide, k.persist_wide3);
    return k;
    }();
    return &ks;
}
