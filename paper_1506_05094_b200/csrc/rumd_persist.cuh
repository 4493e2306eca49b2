// rumd_persist.cuh -- A7: the whole run as ONE cooperative kernel (sm_100a).  Product code: shares nothing
// with oracle/.
//
// The paper keeps the host out of the time-step loop by launching its kernels every step and letting them
// exit early: "avoiding the overhead associated with communication between the GPU and CPU
// is important for the performance at small system sizes".  On B200 a dependent kernel launch inside a CUDA
// graph still costs ~1.2 us and an early-exit kernel ~0.7-1 us (measured), which is more than the
// arithmetic of a whole step at N ~ 10^3-10^4.  Here n time steps run inside one cooperative launch: a step
// is (rebuild phases if the displacement flag fired) -> fused pair-force + leap-frog update written to the
// OTHER position buffer (so nobody reads a position that was already advanced) -> one grid barrier.  The
// Nose-Hoover variable is advanced redundantly, identically, by every block from per-block fp64 partial sums
// added in a fixed order, so the run is bitwise reproducible and needs no second barrier.
#pragma once
#include "rumd_force.cuh"

#define PERSIST_SPIN_LIMIT (1u << 27)

__device__ __forceinline__ unsigned ld_acquire_u32(const unsigned* p)
{
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}

// Grid barrier over a monotone arrival counter (zeroed by the host before the launch).  Thread 0 of every
// block publishes the block's writes (fence), arrives, spins with acquire loads until all nblocks blocks of
// this epoch have arrived, and fences again (which also drops stale L1 lines of data other blocks rewrote).
// Returns false if the spin limit was hit (a block is missing: the kernel then winds down instead of hanging).
__device__ __forceinline__ bool grid_barrier(unsigned* counter, unsigned& epoch, unsigned nblocks, int* s_ok)
{
    __syncthreads();
    if (threadIdx.x == 0) {
        epoch += 1;
        __threadfence();
        atomicAdd(counter, 1u);
        const unsigned target = epoch * nblocks;
        unsigned spins = 0;
        bool ok = true;
        while (ld_acquire_u32(counter) < target) {
            if (++spins > PERSIST_SPIN_LIMIT) {
                ok = false;
                break;
            }
        }
        __threadfence();
        *s_ok = ok ? 1 : 0;
    }
    __syncthreads();
    return *s_ok != 0;
}

// Fixed-order block sum of one double per thread; result valid in every thread.  s_red: 33 doubles.
__device__ __forceinline__ double block_sum(double x, double* s_red)
{
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
    x = warp_sum(x);
    __syncthreads();
    if (lane == 0) s_red[wid] = x;
    __syncthreads();
    if (threadIdx.x == 0) {
        double a = 0.0;
        for (int q = 0; q < nw; ++q) a += s_red[q];
        s_red[32] = a;
    }
    __syncthreads();
    return s_red[32];
}

#define PB(call)                                                                                         \
    do {                                                                                                 \
        if (!grid_barrier(&S.sc->barrier, epoch, gridDim.x, &s_ok)) {                                    \
            if (threadIdx.x == 0) S.sc->nonfinite = 2;                                                   \
            return;                                                                                      \
        }                                                                                                \
    } while (0)

template <int TP, bool COUL, bool ONE_TYPE, int UNROLL>
__global__ void __launch_bounds__(512, 1) k_persist(const Sys S, const int nsteps, const int nvt)
{
    __shared__ float4 s_pp[3 * RUMD_MAXT * RUMD_MAXT];
    __shared__ float s_rcl2[RUMD_MAXT * RUMD_MAXT];
    __shared__ float4 s_tile[N2_TILE];
    __shared__ int s_warp[33];
    __shared__ double s_red[33];
    __shared__ int s_ok, s_moved;

    load_pair_table(S, s_pp);
    if (threadIdx.x < RUMD_MAXT * RUMD_MAXT) s_rcl2[threadIdx.x] = S.pp[threadIdx.x].rcl2;
    unsigned epoch = 0;
    const int first = blockIdx.x * blockDim.x + threadIdx.x, stride = gridDim.x * blockDim.x;
    const int lane = threadIdx.x & 31;
    DevScalars* sc = S.sc;

    // state every block carries identically (read before the first barrier, written back by block 0 at the end)
    const long long step0 = sc->n_steps;
    long long n_rebuilds = sc->n_rebuilds;
    bool flag = sc->flag != 0u;
    double xi = sc->xi, eta = sc->eta, xi_t = sc->xi_t, eta_t = sc->eta_t;
    float4* rc = S.r;     // positions r(t) of the current step
    float4* rn = S.r_alt; // where r(t+dt) goes
    const int nchunks = (S.grid.ncell + SCAN_CHUNK - 1) / SCAN_CHUNK;
    const long long nvt_threads = (long long)S.N * TP;
    __syncthreads();

    for (int k = 0; k < nsteps; ++k) {
        // ---------------------------------------------------------------- (rebuild if flag) A2 / A3 / A4
        if (flag) {
            int* max_slot = &sc->max_nbrs[n_rebuilds & 1];
            if (blockIdx.x == 0 && threadIdx.x == 0) sc->max_nbrs[(n_rebuilds + 1) & 1] = 0;
            if (sort_on_rebuild(S, n_rebuilds)) {
                ph_cell_assign(S, rc, first, stride);
                PB();
                if (nchunks <= 8) {
                    if (blockIdx.x == 0) ph_scan_single_block(S, s_warp);
                } else {
                    ph_scan_sums(S, s_warp, blockIdx.x, gridDim.x);
                    PB();
                    if (blockIdx.x == 0) ph_scan_blocks(S, s_warp);
                    PB();
                    ph_scan_apply(S, s_warp, blockIdx.x, gridDim.x);
                }
                PB();
                ph_cell_scatter(S, first, stride);
                PB();
                ph_cell_finish(S, first, stride);
                PB();
                ph_permute_gather(S, rc, first, stride);
                PB();
                ph_permute_store(S, rc, first, stride);
                PB();
            }
            if (S.method == 1)
                build_cell_dispatch(S, rc, s_rcl2, first, stride, max_slot);
            else
                ph_build_n2(S, rc, s_tile, s_rcl2, blockIdx.x, gridDim.x, max_slot);
            n_rebuilds += 1;
            PB();
        }

        // ---------------------------------------------------------------- A5 + A6 fused: forces, leap-frog
        float a, b;
        if (nvt) {
            const double hx = 0.5 * xi * S.dt_d;
            a = (float)((1.0 - hx) / (1.0 + hx));
            b = (float)(S.dt_d / (1.0 + hx));
        } else {
            a = 1.0f;
            b = S.dt;
        }
        const bool last = k == nsteps - 1;
        double kt = 0.0, mv2 = 0.0;
        bool moved = false;
        for (long long vt = first; vt - lane < nvt_threads; vt += stride) {
            const int i = (int)(vt / TP);
            const int t = (int)(vt % TP);
            const bool have_i = i < S.N;
            float4 ri = make_float4(0.f, 0.f, 0.f, 0.f);
            int cnt = 0;
            if (have_i) {
                ri = rc[i];
                cnt = S.num_nbrs[i];
            }
            float fx, fy, fz, u, w;
            force_group<TP, COUL, ONE_TYPE, UNROLL, false>(S, rc, s_pp, (int)(vt >> 5), i, t, ri, cnt, fx, fy, fz, u, w);
            if (have_i && t == 0) {
                const float4 f = make_float4(fx, fy, fz, 0.5f * u);
                float4 v = S.v[i];
                int4 im = S.image[i];
                bool mv;
                double kti, mv2i;
                integrate_particle(S, a, b, ri, v, f, im, S.r_build[i], mv, kti, mv2i);
                rn[i] = ri;
                S.v[i] = v;
                S.image[i] = im;
                if (last) { // forces / energies / virials of the LAST force evaluation are the outputs
                    S.f[i] = f;
                    S.w[i] = 0.5f * w;
                }
                moved |= mv;
                kt += kti;
                mv2 += mv2i;
            }
        }
        // per-block results: kinetic sums (needed every step for NVT, at the last step for the thermo read-out)
        if (threadIdx.x == 0) s_moved = 0;
        __syncthreads();
        if (moved) s_moved = 1;
        if (nvt || last) {
            const double bm = block_sum(mv2, s_red);
            const double bk = last ? block_sum(kt, s_red) : 0.0;
            if (threadIdx.x == 0) {
                double* p = S.partial + ((size_t)(k & 1) * gridDim.x + blockIdx.x) * 2;
                p[0] = bk;
                p[1] = bm;
            }
        }
        __syncthreads();
        if (threadIdx.x == 0 && s_moved) atomicMax(&sc->moved_step, step0 + k + 1);
        PB();

        // ---------------------------------------------------------------- after the barrier: next step's inputs
        flag = *((volatile long long*)&sc->moved_step) == step0 + k + 1; // O9 / P:270
        if (nvt || last) {
            const double* p = S.partial + (size_t)(k & 1) * gridDim.x * 2;
            double sm = 0.0, sk = 0.0;
            for (int q = threadIdx.x; q < (int)gridDim.x; q += blockDim.x) {
                sk += __ldcg(&p[2 * q]);
                sm += __ldcg(&p[2 * q + 1]);
            }
            sm = block_sum(sm, s_red);
            if (last) sk = block_sum(sk, s_red);
            if (nvt) { // O7: xi += dt w^2 (T_kin/T0 - 1), eta += dt/2 (xi_old + xi_new)
                const double xin = xi + S.dt_d * S.omega2 * (sm / S.g / S.T0 - 1.0);
                xi_t = xi;
                eta_t = eta;
                eta += 0.5 * S.dt_d * (xi + xin);
                xi = xin;
            }
            if (last && blockIdx.x == 0 && threadIdx.x == 0) {
                sc->K = sk;
                sc->mv2 = sm;
                if (!(sk == sk) || !(sm == sm)) sc->nonfinite = 1;
            }
        }
        float4* tmp = rc;
        rc = rn;
        rn = tmp;
    }

    // ---------------------------------------------------------------- wind down
    if (rc != S.r) // odd number of steps: the current positions sit in the alternate buffer
        for (int i = first; i < S.N; i += stride) S.r[i] = rc[i];
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        sc->xi = xi;
        sc->eta = eta;
        sc->xi_t = xi_t;
        sc->eta_t = eta_t;
        sc->n_steps = step0 + nsteps;
        sc->n_rebuilds = n_rebuilds;
        sc->flag = flag ? 1u : 0u;
        sc->pending = 0u;
    }
}
