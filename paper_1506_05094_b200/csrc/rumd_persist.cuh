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
#include "rumd_tile.cuh"

#ifndef PERSIST_THREADS
#define PERSIST_THREADS 256
#endif
#ifndef PERSIST_MINB
#define PERSIST_MINB 3
#endif
#define PERSIST_SPIN_LIMIT (1u << 24)

// Grid barrier.  Two monotone 64-bit arrival counters (zeroed by the host before the launch) are used in
// turn, so a block that is already arriving at the NEXT barrier never touches the counter a slow block is
// still polling.  Low word: arrivals; high word: how many arriving blocks reported "some particle moved more
// than skin/2" (O9) -- the displacement flag travels with the barrier and costs no extra round trip.
// Thread 0 of each block arrives with a release reduction (publishes the block's writes, which it has
// observed through the preceding __syncthreads) and polls with acquire loads (the compiler follows them by
// CCTL.IVALL, dropping stale L1 lines of data other blocks rewrote); the closing __syncthreads hands the
// ordering on to the rest of the block.  Returns false if the spin limit was hit (the kernel then winds
// down instead of hanging).  `any_moved`: did the high word change since this counter was last used.
struct BarrierState {
    unsigned n = 0;            // barriers passed so far
    unsigned seen_hi0 = 0, seen_hi1 = 0;
};

__device__ __forceinline__ bool barrier_arrive_wait(unsigned long long* counters, BarrierState& bs, unsigned nblocks,
                                                    bool moved, bool& any_moved)
{
    const unsigned p = bs.n & 1u;
    const unsigned target = ((bs.n >> 1) + 1u) * nblocks;
    bs.n += 1;
    unsigned long long* c = counters + p;
    const unsigned long long inc = 1ull | (moved ? (1ull << 32) : 0ull);
    asm volatile("red.release.gpu.global.add.u64 [%0], %1;" ::"l"(c), "l"(inc) : "memory");
    unsigned long long v;
    unsigned spins = 0;
    bool ok = true;
    for (;;) {
        asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(c) : "memory");
        if ((unsigned)v >= target) break;
        if (++spins > PERSIST_SPIN_LIMIT) {
            ok = false;
            break;
        }
    }
    const unsigned hi = (unsigned)(v >> 32);
    any_moved = hi != (p ? bs.seen_hi1 : bs.seen_hi0);
    if (p) bs.seen_hi1 = hi; else bs.seen_hi0 = hi;
    return ok;
}

// plain grid barrier between rebuild phases
#define PB()                                                                                             \
    do {                                                                                                 \
        __syncthreads();                                                                                 \
        if (threadIdx.x == 0) {                                                                          \
            bool any_;                                                                                   \
            s_ok = barrier_arrive_wait(sc->bar, bs, gridDim.x, false, any_) ? 1 : 0;                     \
        }                                                                                                \
        __syncthreads();                                                                                 \
        if (!s_ok) {                                                                                     \
            if (threadIdx.x == 0) sc->nonfinite = 2;                                                     \
            return;                                                                                      \
        }                                                                                                \
    } while (0)

// warp_sum over values that are zero except in every TP-th lane (lane 0 holds the total)
template <int TP> __device__ __forceinline__ double warp_sum_strided(double x)
{
#pragma unroll
    for (int o = 16; o >= TP; o >>= 1) x += __shfl_xor_sync(FULLMASK, x, o);
    return x;
}

// Fixed-order sum over the per-block partials of one step by ONE warp; every lane returns the total.
__device__ __forceinline__ double warp_sum_partials(const double* p, int n)
{
    double a = 0.0;
    for (int q = threadIdx.x & 31; q < n; q += 32) a += __ldcg(&p[2 * q]);
    return warp_sum(a);
}

// TILE: the instantiation for the tile method (RUMD_NB_TILE: halo in dynamic shared memory); the other methods share
// the TILE = false instantiation, whose register budget the tile code must not touch.
// NT: threads per block.  512 (one block per SM, up to 128 registers) is launched when blocks of 256 would need two per
// SM and 512 fit one: half the barrier arrivals and thermostat partials for the same 16 warps per SM (C1 7.75 -> 7.5 us);
// 768 (tp < 8, 85 registers) instead of three blocks of 256 per SM at large N.
template <int TP, int COUL, bool ONE_TYPE, int UNROLL, bool TILE, int NT = PERSIST_THREADS>
__global__ void __launch_bounds__(NT, NT > PERSIST_THREADS ? 1 : (TP == 8 && !TILE) ? 2 : PERSIST_MINB) k_persist(const Sys S, const int nsteps, const int nvt)
{
    __shared__ float4 s_pp[4 * RUMD_MAXT * RUMD_MAXT];
    __shared__ float s_rcl2[RUMD_MAXT * RUMD_MAXT];
    __shared__ float4 s_tile[N2_TILE];
    __shared__ int s_warp[33];
    __shared__ double s_redm[NT / 32], s_redk[NT / 32];
    __shared__ int s_ok, s_moved, s_flag;
    __shared__ float s_ab[2];
    __shared__ int s_ab_step; // s_ab holds the leap-frog factors of every step < s_ab_step
    __shared__ double s_nh[4];       // xi, eta, xi_t, eta_t: kept by lane 0 of warp 0 (identical in every block)
    __shared__ long long s_prof[6];  // cycle counters of block 0 / thread 0 (profiling runs only)
    extern __shared__ __align__(16) unsigned char tile_raw[]; // tile method only: halo positions + halo cell starts
    float4* s_pos = nullptr;
    unsigned short* s_hstart = nullptr;
    unsigned char* s_scratch = nullptr;
    if (TILE) tile_smem(S, tile_raw, s_pos, s_hstart, s_scratch);

    load_pair_table(S, s_pp);
    if (threadIdx.x < RUMD_MAXT * RUMD_MAXT) s_rcl2[threadIdx.x] = S.pp[threadIdx.x].rcl2;
    const int first = blockIdx.x * blockDim.x + threadIdx.x, stride = gridDim.x * blockDim.x;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
    DevScalars* sc = S.sc;
    BarrierState bs;

    // state every block carries identically (read before the first barrier, written back by block 0 at the end)
    const int n_rebuilds0 = (int)(sc->n_rebuilds & 0x3fffffff); // only its parity and value mod sort_interval matter
    int n_rebuilds = n_rebuilds0;
    bool flag = sc->flag != 0u;
    float4* rc = S.r;     // positions r(t) of the current step
    float4* rn = S.r_alt; // where r(t+dt) goes
    const int nchunks = (S.grid.ncell + SCAN_CHUNK - 1) / SCAN_CHUNK;
    const long long nvwarps = ((long long)S.N * TP + 31) / 32;
    const long long vw0 = nvwarps * blockIdx.x / gridDim.x, vw1 = nvwarps * (blockIdx.x + 1) / gridDim.x;
    if (threadIdx.x == 0) {
        s_moved = 0;
        s_ab[0] = 1.0f;
        s_ab[1] = S.dt;
        s_ab_step = nvt ? 0 : 0x7fffffff; // NVE: a = 1, b = dt for good
        s_nh[0] = sc->xi;
        s_nh[1] = sc->eta;
        s_nh[2] = sc->xi_t;
        s_nh[3] = sc->eta_t;
        for (int q = 0; q < 6; ++q) s_prof[q] = 0;
    }
    __syncthreads();
    // profiling (S.prof != nullptr): block 0 / thread 0 adds up SM cycles per phase
    const bool prof = S.prof != nullptr && blockIdx.x == 0 && threadIdx.x == 0;
    if (prof) s_prof[5] = clock64();
#define PROF_LAP(slot)                                                                                   \
    if (prof) {                                                                                          \
        const long long t_ = clock64();                                                                  \
        s_prof[slot] += t_ - s_prof[4];                                                                  \
        s_prof[4] = t_;                                                                                  \
    }

    for (int k = 0; k < nsteps; ++k) {
        if (prof) s_prof[4] = clock64();
        // ---------------------------------------------------------------- (rebuild if flag) A2 / A3 / A4
        if (flag && S.method != 2) { // (the "none" method keeps no list)
            int* max_slot = &sc->max_nbrs[n_rebuilds & 1];
            if (blockIdx.x == 0 && threadIdx.x == 0) {
                sc->max_nbrs[(n_rebuilds + 1) & 1] = 0;
                sc->build_queue = stride >> 5; // units 0 .. warps-1 are taken (the cell build is at least one grid barrier away)
            }
            const float4* rsrc = rc; // where the build reads the positions from
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
                ph_permute_gather_ranked(S, rc, first, stride);
                PB();
                // the copy back into the caller's arrays shares its phase with the build, which reads the
                // sorted positions from the scratch copy
                ph_permute_store(S, rc, first, stride);
                rsrc = S.tmp_r;
            }
            if (prof) s_prof[2] += clock64() - s_prof[4];
            if (TILE) {
                for (int t = blockIdx.x; t < S.ntiles; t += gridDim.x)
                    ph_build_tile(S, rsrc, t, s_pos, s_hstart, s_scratch, s_warp, s_rcl2, max_slot);
            } else if (S.method == 1)
            {
                // several units per warp: hand them out dynamically (see ph_build_cell); else one fixed pass
                const long long units = (((long long)S.N << S.build_tp_shift) + 31) >> 5;
                build_cell_dispatch(S, rsrc, s_rcl2, first, stride, max_slot, units >= 4LL * (stride >> 5) ? &sc->build_queue : nullptr);
            }
            else
                ph_build_n2(S, rsrc, s_tile, s_rcl2, blockIdx.x, gridDim.x, max_slot);
            n_rebuilds += 1;
            PB();
            if (blockIdx.x == 0 && threadIdx.x == 0) sc->last_max = __ldcg(max_slot);
        }
        PROF_LAP(0)

        // ---------------------------------------------------------------- Nose-Hoover factors of this step (O7)
        // One warp of EVERY block adds the previous step's per-block sums of m v^2 in the same fixed order and
        // advances xi identically; the other warps start on the forces and pick the factors up from shared
        // memory only when they integrate.
        if (nvt && wid == nw - 1) { // the LAST warp: with fewer virtual warps than warps (small N) it has no force work
            double sm = 0.0;
            if (k > 0) sm = warp_sum_partials(S.partial + (size_t)((k - 1) & 1) * gridDim.x * 2 + 1, gridDim.x);
            if (lane == 0) {
                double xi = s_nh[0];
                if (k > 0) {
                    const double xin = xi + S.dt_d * S.omega2 * (sm / S.g / S.T0 - 1.0); // xi += dt w^2 (T_kin/T0 - 1)
                    s_nh[2] = xi;
                    s_nh[3] = s_nh[1];
                    s_nh[1] += 0.5 * S.dt_d * (xi + xin);                               // eta += dt/2 (xi_old + xi_new)
                    s_nh[0] = xi = xin;
                }
                const double hx = 0.5 * xi * S.dt_d;
                ((volatile float*)s_ab)[0] = (float)((1.0 - hx) / (1.0 + hx));
                ((volatile float*)s_ab)[1] = (float)(S.dt_d / (1.0 + hx));
                __threadfence_block();
                *((volatile int*)&s_ab_step) = k + 1;
            }
        }

        // ---------------------------------------------------------------- A5 + A6 fused: forces, leap-frog
        const bool last = k == nsteps - 1;
        double kt = 0.0, mv2 = 0.0;
        bool moved = false;
        // leap-frog update of one particle from its force: the epilogue of both force paths
        auto advance = [&](int i, float4 ri, float fx, float fy, float fz, float u, float w, float4 v, int4 im, float4 rb) {
            while (*((volatile int*)&s_ab_step) <= k) {} // factors of step k published? (warp 0, above)
            __threadfence_block();
            const float a = ((volatile float*)s_ab)[0], b = ((volatile float*)s_ab)[1];
            const float4 f = make_float4(fx, fy, fz, 0.5f * u);
            bool mv;
            double kti, mv2i;
            integrate_particle(S, a, b, ri, v, f, im, rb, mv, kti, mv2i);
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
        };
        if constexpr (TILE) {
            // tile method: the block's tiles in turn -- halo into shared memory, forces of the owned particles out of
            // it, leap-frog
            for (int t = blockIdx.x; t < S.ntiles; t += gridDim.x) { // strided: every block gets its share of the (dearer) boundary tiles
                __syncthreads();
                tile_load_halo<false>(S, rc, t, s_pos);
                __syncthreads();
                auto done = [&](int i, bool lead, const float4& ri, float fx, float fy, float fz, float u, float w) {
                    if (lead) advance(i, ri, fx, fy, fz, u, w, S.v[i], S.image[i], S.r_build[i]);
                };
                if (last)
                    tile_force_own<TP, COUL, ONE_TYPE, false, true>(S, rc, t, s_pos, s_pp, done);
                else
                    tile_force_own<TP, COUL, ONE_TYPE, false, false>(S, rc, t, s_pos, s_pp, done);
            }
        } else
        // the N*TP/32 warps of work are split into gridDim.x contiguous, equally long chunks (spatial locality
        // inside a block, every SM equally loaded); the block's warps take the warps of its chunk in turn
        for (long long vw = vw0 + wid; vw < vw1; vw += nw) {
            const long long vt = vw * 32 + lane;
            const int i = (int)(vt / TP);
            const int t = (int)(vt % TP);
            const bool have_i = i < S.N;
            float4 ri = make_float4(0.f, 0.f, 0.f, 0.f);
            int cnt = 0;
            if (have_i) {
                ri = rc[i];
                cnt = S.method == 2 ? 0 : S.num_nbrs[i];
            }
            // Small systems (wide lane groups): the integrator's inputs are fetched BEFORE the force loop so that
            // their latency hides behind it; at tp < 8 the twelve registers cost more than the latency (measured).
            constexpr bool EARLY = TP >= 8;
            float4 v = make_float4(0.f, 0.f, 0.f, 1.f), rb = v;
            int4 im = make_int4(0, 0, 0, 0);
            if (EARLY && have_i && t == 0) {
                v = S.v[i];
                im = S.image[i];
                rb = S.r_build[i];
            }
            float fx, fy, fz, u, w;
            if (last) // energies and virials are outputs of the LAST force evaluation only
                force_any<TP, COUL, ONE_TYPE, UNROLL, false, true>(S, rc, s_pp, (int)vw, i, t, have_i, ri, cnt, fx, fy, fz, u, w);
            else
                force_any<TP, COUL, ONE_TYPE, UNROLL, false, false>(S, rc, s_pp, (int)vw, i, t, have_i, ri, cnt, fx, fy, fz, u, w);
            if (have_i && t == 0) {
                if (!EARLY) {
                    v = S.v[i];
                    im = S.image[i];
                    rb = S.r_build[i];
                }
                advance(i, ri, fx, fy, fz, u, w, v, im, rb);
            }
        }
        PROF_LAP(1)

        // ---------------------------------------------------------------- block sums, then the step's barrier
        {
            // (only the lanes with t == 0, every TP-th, hold a particle's contribution: the butterfly levels below TP
            // would add zeros; leaving them out gives the same bits and takes them off the step's critical path)
            const double wm = (nvt || last) ? warp_sum_strided<TP>(mv2) : 0.0;
            const double wk = last ? warp_sum_strided<TP>(kt) : 0.0;
            const bool wmoved = __any_sync(FULLMASK, moved);
            if (lane == 0) {
                s_redm[wid] = wm;
                s_redk[wid] = wk;
                if (wmoved) s_moved = 1;
            }
        }
        __syncthreads();
        if (threadIdx.x == 0) {
            if (nvt || last) {
                double bk = 0.0, bm = 0.0;
                for (int q = 0; q < nw; ++q) {
                    bk += s_redk[q];
                    bm += s_redm[q];
                }
                double* p = S.partial + ((size_t)(k & 1) * gridDim.x + blockIdx.x) * 2;
                p[0] = bk;
                p[1] = bm;
            }
            const bool mvd = s_moved != 0;
            s_moved = 0;
            bool any;
            s_ok = barrier_arrive_wait(sc->bar, bs, gridDim.x, mvd, any) ? 1 : 0;
            s_flag = any ? 1 : 0; // O9 / P:270: rebuild before the next force evaluation
        }
        __syncthreads();
        if (!s_ok) {
            if (threadIdx.x == 0) sc->nonfinite = 2;
            return;
        }
        flag = s_flag != 0;
        float4* tmp = rc;
        rc = rn;
        rn = tmp;
        PROF_LAP(3)
    }

    // ---------------------------------------------------------------- wind down
    if (rc != S.r) // odd number of steps: the current positions sit in the alternate buffer
        for (int i = first; i < S.N; i += stride) S.r[i] = rc[i];
    if (blockIdx.x == 0 && wid == 0 && nsteps > 0) {
        const double* p = S.partial + (size_t)((nsteps - 1) & 1) * gridDim.x * 2;
        const double sk = warp_sum_partials(p, gridDim.x);
        const double sm = warp_sum_partials(p + 1, gridDim.x);
        if (lane == 0) {
            if (nvt) {
                const double xi = s_nh[0];
                const double xin = xi + S.dt_d * S.omega2 * (sm / S.g / S.T0 - 1.0);
                s_nh[2] = xi;
                s_nh[3] = s_nh[1];
                s_nh[1] += 0.5 * S.dt_d * (xi + xin);
                s_nh[0] = xin;
            }
            sc->K = sk;
            sc->mv2 = sm;
            if (!(sk == sk) || !(sm == sm)) sc->nonfinite = 1;
            sc->xi = s_nh[0];
            sc->eta = s_nh[1];
            sc->xi_t = s_nh[2];
            sc->eta_t = s_nh[3];
            sc->n_steps += nsteps;
            sc->n_rebuilds += n_rebuilds - n_rebuilds0;
            sc->flag = flag ? 1u : 0u;
            sc->pending = 0u;
        }
    }
    if (prof) {
        S.prof[0] = s_prof[0];
        S.prof[1] = s_prof[1];
        S.prof[2] = s_prof[2];
        S.prof[3] = s_prof[3];
        S.prof[4] = 0;
        S.prof[5] = clock64() - s_prof[5];
        S.prof[6] = n_rebuilds - n_rebuilds0;
        S.prof[7] = gridDim.x;
    }
#undef PROF_LAP
}
