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

template <int TP> static const KernelSet* kernel_set()
{
    static const KernelSet ks = {
        {{(const void*)&k_persist<TP, 0, false, UnrollOf<TP>::value>, (const void*)&k_persist<TP, 0, true, UnrollOf<TP>::value>},
         {(const void*)&k_persist<TP, 1, false, UnrollOf<TP>::value>, (const void*)&k_persist<TP, 1, true, UnrollOf<TP>::value>},
         {(const void*)&k_persist<TP, 2, false, UnrollOf<TP>::value>, (const void*)&k_persist<TP, 2, true, UnrollOf<TP>::value>}},
        {{(const void*)&k_ensemble<TP, 0, false, UnrollOf<TP>::value>, (const void*)&k_ensemble<TP, 0, true, UnrollOf<TP>::value>},
         {(const void*)&k_ensemble<TP, 1, false, UnrollOf<TP>::value>, (const void*)&k_ensemble<TP, 1, true, UnrollOf<TP>::value>},
         {(const void*)&k_ensemble<TP, 2, false, UnrollOf<TP>::value>, (const void*)&k_ensemble<TP, 2, true, UnrollOf<TP>::value>}},
        &force_tp<TP>,
        &step_tp<TP>,
    };
    return &ks;
}
