// rumd_ensemble.cuh -- batched ensembles: many independent small systems in ONE launch (sm_100a).
// Product code: shares nothing with oracle/.
//
// P:63 points to "large ensembles of MD simulations of small systems" as the use of a GPU that a single small
// system cannot fill, and P:83 / P:363 leave multi-GPU as planned.  At N ~ 10^3 one system keeps a B200 busy
// for a few percent of its arithmetic: the time step is a chain of dependent latencies (k_persist: 4-5 us per
// step, 1.2 us of it the grid barrier).  Here every replica (same N, box, potentials and integrator; its own
// positions, velocities, list and thermostat) is run by ONE thread block for the whole rumd_run_steps(n):
// rebuild (N^2 build inside the block, or no list at all) -> fused force + leap-frog into the other position
// buffer -> __syncthreads.  No grid barrier, no inter-block traffic; blocks of different replicas overlap each
// other's latencies on an SM, and the grid is simply the number of replicas.
//
// Each block works on its own parameter block (a Sys whose pointers address the replica's slices), copied
// from global to shared memory at kernel start; the phases and the force loop are the ones of the
// single-system paths, so a replica's trajectory is bit-identical to the same system run alone in NVE.
#pragma once
#include "rumd_force.cuh"

#define ENS_THREADS 256
#ifndef ENS_MINB
#define ENS_MINB 3
#endif

#ifdef RUMD_MAIN_TU // non-template kernels: compiled once, in rumd_b200.cu
static __global__ void k_ens_reset(DevScalars* sc, int nrep)
{
    const int q = blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= nrep) return;
    DevScalars z;
    memset(&z, 0, sizeof(z));
    z.flag = 1u;
    sc[q] = z;
}

static __global__ void k_ens_request_rebuild(DevScalars* sc, int nrep)
{
    const int q = blockIdx.x * blockDim.x + threadIdx.x;
    if (q < nrep) sc[q].flag = 1u;
}
#endif // RUMD_MAIN_TU

// fixed-order block sum of a double (result valid in thread 0); s: ENS_THREADS / 32 doubles
__device__ __forceinline__ double ens_block_sum(double x, double* s)
{
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
    x = warp_sum(x);
    __syncthreads();
    if (lane == 0) s[wid] = x;
    __syncthreads();
    double a = 0.0;
    if (threadIdx.x == 0)
        for (int q = 0; q < nw; ++q) a += s[q];
    return a;
}

template <int TP, int COUL, bool ONE_TYPE, int UNROLL>
__global__ void __launch_bounds__(ENS_THREADS, ENS_MINB) k_ensemble(const Sys* __restrict__ systems, const int nsteps, const int nvt)
{
    __shared__ Sys R; // this replica's parameter block
    __shared__ float4 s_pp[4 * RUMD_MAXT * RUMD_MAXT];
    __shared__ float s_rcl2[RUMD_MAXT * RUMD_MAXT];
    __shared__ float4 s_tile[N2_TILE];
    __shared__ double s_red[ENS_THREADS / 32];
    __shared__ int s_moved, s_flag;
    __shared__ float s_ab[2];
    __shared__ double s_nh[4]; // xi, eta, xi_t, eta_t

    {
        const int* src = reinterpret_cast<const int*>(systems + blockIdx.x);
        int* dst = reinterpret_cast<int*>(&R);
        for (int q = threadIdx.x; q < (int)(sizeof(Sys) / sizeof(int)); q += blockDim.x) dst[q] = src[q];
    }
    __syncthreads();
    load_pair_table(R, s_pp);
    if (threadIdx.x < RUMD_MAXT * RUMD_MAXT) s_rcl2[threadIdx.x] = R.pp[threadIdx.x].rcl2;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
    DevScalars* sc = R.sc;
    int n_rebuilds = 0;
    float4* rc = R.r;
    float4* rn = R.r_alt;
    const int nvwarps = (R.N * TP + 31) / 32;
    if (threadIdx.x == 0) {
        s_moved = 0;
        s_flag = sc->flag != 0u;
        s_nh[0] = sc->xi;
        s_nh[1] = sc->eta;
        s_nh[2] = sc->xi_t;
        s_nh[3] = sc->eta_t;
    }
    __syncthreads();

    for (int k = 0; k < nsteps; ++k) {
        // ---------------------------------------------------------------- (rebuild if flag): N^2 build, in the block
        if (s_flag && R.method != 2) {
            ph_build_n2(R, rc, s_tile, s_rcl2, 0, 1, &sc->max_nbrs[0]);
            n_rebuilds += 1;
        }
        if (threadIdx.x == 0) { // leap-frog factors of this step (O6 / O7)
            float a = 1.0f, b = R.dt;
            if (nvt) {
                const double hx = 0.5 * s_nh[0] * R.dt_d;
                a = (float)((1.0 - hx) / (1.0 + hx));
                b = (float)(R.dt_d / (1.0 + hx));
            }
            s_ab[0] = a;
            s_ab[1] = b;
        }
        __syncthreads();
        const float a = s_ab[0], b = s_ab[1];

        // ---------------------------------------------------------------- A5 + A6 fused
        const bool last = k == nsteps - 1;
        double kt = 0.0, mv2 = 0.0, usum = 0.0, wsum = 0.0;
        bool moved = false;
        for (int vw = wid; vw < nvwarps; vw += nw) {
            const int vt = vw * 32 + lane;
            const int i = vt / TP;
            const int t = vt % TP;
            const bool have_i = i < R.N;
            float4 ri = make_float4(0.f, 0.f, 0.f, 0.f);
            int cnt = 0;
            if (have_i) {
                ri = rc[i];
                cnt = R.method == 2 ? 0 : R.num_nbrs[i];
            }
            float fx, fy, fz, u, w;
            if (last)
                force_any<TP, COUL, ONE_TYPE, UNROLL, false, true>(R, rc, s_pp, vw, i, t, have_i, ri, cnt, fx, fy, fz, u, w);
            else
                force_any<TP, COUL, ONE_TYPE, UNROLL, false, false>(R, rc, s_pp, vw, i, t, have_i, ri, cnt, fx, fy, fz, u, w);
            if (have_i && t == 0) {
                const float4 f = make_float4(fx, fy, fz, 0.5f * u);
                float4 v = R.v[i];
                int4 im = R.image[i];
                bool mv;
                double kti, mv2i;
                integrate_particle(R, a, b, ri, v, f, im, R.r_build[i], mv, kti, mv2i);
                rn[i] = ri;
                R.v[i] = v;
                R.image[i] = im;
                if (last) {
                    R.f[i] = f;
                    R.w[i] = 0.5f * w;
                    usum += (double)f.w;
                    wsum += (double)(0.5f * w);
                }
                moved |= mv && R.method != 2;
                kt += kti;
                mv2 += mv2i;
            }
        }
        if (__any_sync(FULLMASK, moved) && lane == 0) s_moved = 1;
        // ---------------------------------------------------------------- block sums, thermostat, flag
        const double bm = (nvt || last) ? ens_block_sum(mv2, s_red) : 0.0;
        const double bk = last ? ens_block_sum(kt, s_red) : 0.0;
        const double bu = last ? ens_block_sum(usum, s_red) : 0.0;
        const double bw = last ? ens_block_sum(wsum, s_red) : 0.0;
        __syncthreads();
        if (threadIdx.x == 0) {
            if (nvt) { // O7
                const double xi = s_nh[0];
                const double xin = xi + R.dt_d * R.omega2 * (bm / R.g / R.T0 - 1.0);
                s_nh[2] = xi;
                s_nh[3] = s_nh[1];
                s_nh[1] += 0.5 * R.dt_d * (xi + xin);
                s_nh[0] = xin;
            }
            if (last) {
                sc->K = bk;
                sc->mv2 = bm;
                sc->U = bu;
                sc->W = bw;
                if (!(bk == bk) || !(bu == bu)) sc->nonfinite = 1;
            }
            s_flag = s_moved; // O9 / P:270: rebuild before the next force evaluation
            s_moved = 0;
        }
        __syncthreads();
        float4* tmp = rc;
        rc = rn;
        rn = tmp;
    }
    if (rc != R.r)
        for (int i = threadIdx.x; i < R.N; i += blockDim.x) R.r[i] = rc[i];
    if (threadIdx.x == 0 && nsteps > 0) {
        sc->xi = s_nh[0];
        sc->eta = s_nh[1];
        sc->xi_t = s_nh[2];
        sc->eta_t = s_nh[3];
        sc->n_steps += nsteps;
        sc->n_rebuilds += n_rebuilds;
        sc->flag = s_flag ? 1u : 0u;
    }
}
