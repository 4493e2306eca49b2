// rumd_kernels.cuh -- sm_100a kernels of the RUMD hot path.  Product code: shares nothing with oracle/.
// "P:n" = PAPER.md line n; O*/S* = readings listed in DESIGN.md.
#pragma once
#include "rumd_types.cuh"

#define FULLMASK 0xffffffffu

// ------------------------------------------------------------------------------------------ helpers

// Minimum image of one coordinate difference (O1) without the fp32 cancellation error of
// (xi - xj) - L*nint(...): when |xi - xj| ~ L the plain difference is rounded at ulp(L) (3.8e-6 at
// L ~ 107).  Instead both operands are shifted by -+s*L/2 first (exact for every pair that can be inside a
// cutoff, Sterbenz), and the small numbers are subtracted.  h = L/2 exactly.
__device__ __forceinline__ float min_image(float xi, float xj, float h, float invL)
{
    const float MAGIC = 12582912.0f; // 1.5 * 2^23: (x + MAGIC) - MAGIC = nint(x) for |x| < 2^22
    float d0 = xi - xj;
    float s = __fadd_rn(__fmaf_rn(d0, invL, MAGIC), -MAGIC);
    float a = __fmaf_rn(-s, h, xi);
    float b = __fmaf_rn(s, h, xj);
    return a - b;
}

// Storage index of the k-th neighbour of particle i.  The list is tiled per warp of the force kernel: a
// warp owns ppw = 32/tp consecutive particles and in iteration `it` lane (pl*tp + t) reads entry
// k = it*tp + t of its particle pl -- so every warp-wide index load is ONE contiguous 128-byte line for any
// tp.  (The paper's column-major nbl[nvp*k + i], P:141-146 / P:167, is the tp = 1 case of this layout.)
__device__ __forceinline__ size_t nbl_index(const Sys& S, int i, int k)
{
    int g = i >> S.ppw_shift;
    int pl = i & ((1 << S.ppw_shift) - 1);
    int it = k >> S.tp_shift;
    int t = k & ((1 << S.tp_shift) - 1);
    return ((size_t)g * S.cap_it + it) * 32 + (pl << S.tp_shift) + t;
}

__device__ __forceinline__ int type_of(const float4& p) { return __float_as_int(p.w); }

__device__ __forceinline__ double warp_sum(double x)
{
#pragma unroll
    for (int o = 16; o; o >>= 1) x += __shfl_xor_sync(FULLMASK, x, o);
    return x;
}

// true iff this launch has rebuild work to do (the build kernel is "called at every timestep and
// checks ... whether there is anything to be done").
__device__ __forceinline__ bool rebuild_requested(const Sys& S) { return S.sc->flag != 0u; }

// sort on this rebuild?  cell method: always; n2 method: every sort_interval-th rebuild.
__device__ __forceinline__ bool sort_requested(const Sys& S)
{
    if (S.sc->flag == 0u) return false;
    if (S.method == 1) return true;
    return S.sort_interval > 0 && (S.sc->n_rebuilds % S.sort_interval) == 0;
}

__device__ __forceinline__ void cell_coords(const Sys& S, const float4& p, int& cx, int& cy, int& cz)
{
    // S17: c_k = floor((x_k + L_k/2) * n_k / L_k), clamped to [0, n_k - 1]
    cx = min(S.grid.n[0] - 1, max(0, (int)floorf((p.x + S.h[0]) * S.grid.scale[0])));
    cy = min(S.grid.n[1] - 1, max(0, (int)floorf((p.y + S.h[1]) * S.grid.scale[1])));
    cz = min(S.grid.n[2] - 1, max(0, (int)floorf((p.z + S.h[2]) * S.grid.scale[2])));
}

// ------------------------------------------------------------------------------------------ A2: N^2 build

// P:173-224 Fig. 4.  One WARP per particle i; j-positions staged through shared memory in tiles
// (P:184); the 32 lanes test 32 different j at once and slots are handed out by
// ballot + popc, so the row is in ascending-j order and the whole list is bitwise reproducible (the
// paper's atomicInc gives "an unspecified sequential order").  Early exit when no rebuild is
// requested.  Writes num_nbrs, positions at build and the overflow flag.
#define N2_WARPS 4
#define N2_TILE 256
__global__ void __launch_bounds__(N2_WARPS * 32) k_build_n2(const Sys S)
{
    if (!rebuild_requested(S)) return;
    __shared__ float4 tile[N2_TILE];
    __shared__ float s_rcl2[RUMD_MAXT * RUMD_MAXT];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    if (threadIdx.x < RUMD_MAXT * RUMD_MAXT) s_rcl2[threadIdx.x] = S.pp[threadIdx.x].rcl2;
    const int i = blockIdx.x * N2_WARPS + wid;
    const bool have_i = i < S.N;
    float4 ri = make_float4(0.f, 0.f, 0.f, 0.f);
    if (have_i) ri = S.r[i];
    const int trow = have_i ? type_of(ri) * S.ntypes : 0;
    int count = 0;
    for (int j0 = 0; j0 < S.N; j0 += N2_TILE) {
        __syncthreads();
        for (int t = threadIdx.x; t < N2_TILE; t += N2_WARPS * 32)
            if (j0 + t < S.N) tile[t] = S.r[j0 + t];
        __syncthreads();
        const int jend = min(N2_TILE, S.N - j0);
        for (int jj = lane; jj < ((jend + 31) & ~31); jj += 32) {
            bool acc = false;
            const int j = j0 + jj;
            if (jj < jend && have_i && j != i) {
                const float4 rj = tile[jj];
                const float dx = min_image(ri.x, rj.x, S.h[0], S.invL[0]);
                const float dy = min_image(ri.y, rj.y, S.h[1], S.invL[1]);
                const float dz = min_image(ri.z, rj.z, S.h[2], S.invL[2]);
                const float d2 = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, dx * dx));
                acc = d2 < s_rcl2[trow + type_of(rj)]; // strict <, per type pair
            }
            const unsigned m = __ballot_sync(FULLMASK, acc);
            if (acc) {
                const int k = count + __popc(m & ((1u << lane) - 1u));
                if (k < S.cap) S.nbl[nbl_index(S, i, k)] = j;
            }
            count += __popc(m);
        }
    }
    if (have_i && lane == 0) {
        S.num_nbrs[i] = min(count, S.cap);
        S.r_build[i] = ri;
        if (count > S.cap) S.sc->overflow = 1u;
        atomicMax(&S.sc->max_nbrs, count);
    }
}

// Bookkeeping that must happen once per step AFTER every rebuild kernel has read the flag: count the
// rebuild and clear the flag.  Runs as a 1-thread tail of the force kernel's first block (see k_force).
__device__ __forceinline__ void finish_rebuild(const Sys& S)
{
    if (S.sc->flag != 0u) {
        S.sc->n_rebuilds += 1;
        S.sc->flag = 0u;
    }
}

// ------------------------------------------------------------------------------------------ A3: cells + sort

// P:276 steps 1-3: cell of every particle, sort particles by cell, rearrange all particle data.  The paper
// calls Thrust; here it is a counting sort written out: (a) histogram with slot = atomicAdd, (b) three-phase
// exclusive scan, (c) scatter, (d) per-cell insertion sort of the (few) entries by old index, which removes
// the atomic's arbitrary order so that the particle order -- and with it every later fp32 sum -- is
// reproducible.  Cells are numbered along a Morton (Z-order) curve through the valid cells (zrank table,
// built once on the host): consecutive particles are spatially compact (BASELINE configs[3], S19).

__global__ void k_cell_assign(const Sys S)
{
    if (!sort_requested(S)) return;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= S.N) return;
    int cx, cy, cz;
    cell_coords(S, S.r[i], cx, cy, cz);
    const int z = S.zrank[(cz * S.grid.n[1] + cy) * S.grid.n[0] + cx];
    S.cell_of[i] = z;
    S.slot[i] = atomicAdd(&S.ccount[z], 1);
}

#define SCAN_THREADS 256
#define SCAN_ITEMS 8
#define SCAN_CHUNK (SCAN_THREADS * SCAN_ITEMS)

__device__ __forceinline__ int block_exclusive_scan(int x, int* s_warp, int& total)
{
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    int incl = x;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        int y = __shfl_up_sync(FULLMASK, incl, o);
        if (lane >= o) incl += y;
    }
    if (lane == 31) s_warp[wid] = incl;
    __syncthreads();
    if (wid == 0) {
        int v = lane < (SCAN_THREADS / 32) ? s_warp[lane] : 0;
        int vi = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            int y = __shfl_up_sync(FULLMASK, vi, o);
            if (lane >= o) vi += y;
        }
        if (lane < (SCAN_THREADS / 32)) s_warp[lane] = vi - v;
        if (lane == 31) s_warp[32] = vi;
    }
    __syncthreads();
    total = s_warp[32];
    const int res = incl - x + s_warp[wid];
    __syncthreads();
    return res;
}

// phase 1: per-chunk totals
__global__ void __launch_bounds__(SCAN_THREADS) k_scan_sums(const Sys S)
{
    if (!sort_requested(S)) return;
    __shared__ int s_warp[33];
    const int base = blockIdx.x * SCAN_CHUNK + threadIdx.x * SCAN_ITEMS;
    int x = 0;
#pragma unroll
    for (int q = 0; q < SCAN_ITEMS; ++q)
        if (base + q < S.grid.ncell) x += S.ccount[base + q];
    int total;
    block_exclusive_scan(x, s_warp, total);
    if (threadIdx.x == 0) S.blocksum[blockIdx.x] = total;
}

// phase 2: exclusive scan of the chunk totals (one block, loops if there are more than 256 chunks)
__global__ void __launch_bounds__(SCAN_THREADS) k_scan_blocks(const Sys S, int nchunks)
{
    if (!sort_requested(S)) return;
    __shared__ int s_warp[33];
    int carry = 0;
    for (int b0 = 0; b0 < nchunks; b0 += SCAN_THREADS) {
        const int b = b0 + threadIdx.x;
        const int x = b < nchunks ? S.blocksum[b] : 0;
        int total;
        const int e = block_exclusive_scan(x, s_warp, total);
        if (b < nchunks) S.blocksum[b] = carry + e;
        carry += total;
    }
}

// phase 3: exclusive scan inside each chunk + chunk offset -> first sorted slot of each Z-ordered cell
__global__ void __launch_bounds__(SCAN_THREADS) k_scan_apply(const Sys S)
{
    if (!sort_requested(S)) return;
    __shared__ int s_warp[33];
    const int base = blockIdx.x * SCAN_CHUNK + threadIdx.x * SCAN_ITEMS;
    int c[SCAN_ITEMS];
    int x = 0;
#pragma unroll
    for (int q = 0; q < SCAN_ITEMS; ++q) {
        c[q] = (base + q < S.grid.ncell) ? S.ccount[base + q] : 0;
        x += c[q];
    }
    int total;
    int e = block_exclusive_scan(x, s_warp, total) + S.blocksum[blockIdx.x];
#pragma unroll
    for (int q = 0; q < SCAN_ITEMS; ++q) {
        if (base + q < S.grid.ncell) S.cstart_z[base + q] = e;
        e += c[q];
    }
}

__global__ void k_cell_scatter(const Sys S)
{
    if (!sort_requested(S)) return;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= S.N) return;
    S.perm[S.cstart_z[S.cell_of[i]] + S.slot[i]] = i;
}

// One thread per cell: order its entries by old index (deterministic), publish cellStart / cellEnd under
// the row-major cell index the build kernel uses (here end is EXCLUSIVE, S20), clear the
// histogram for the next sort.
__global__ void k_cell_finish(const Sys S)
{
    if (!sort_requested(S)) return;
    const int z = blockIdx.x * blockDim.x + threadIdx.x;
    if (z >= S.grid.ncell) return;
    const int b = S.cstart_z[z], n = S.ccount[z];
    for (int a = 1; a < n; ++a) {
        const int key = S.perm[b + a];
        int q = a - 1;
        while (q >= 0 && S.perm[b + q] > key) {
            S.perm[b + q + 1] = S.perm[b + q];
            --q;
        }
        S.perm[b + q + 1] = key;
    }
    const int c = S.zinv[z];
    S.cell_start[c] = b;
    S.cell_end[c] = b + n;
    S.ccount[z] = 0;
}

// P:276 "rearrange all particle data into the sorted order": gather into scratch, then copy back (the
// caller owns the arrays, so the pointers cannot be swapped).
__global__ void k_permute_gather(const Sys S)
{
    if (!sort_requested(S)) return;
    const int d = blockIdx.x * blockDim.x + threadIdx.x;
    if (d >= S.N) return;
    const int src = S.perm[d];
    S.tmp_r[d] = S.r[src];
    S.tmp_v[d] = S.v[src];
    S.tmp_image[d] = S.image[src];
    S.tmp_id[d] = S.id[src];
}

__global__ void k_permute_store(const Sys S)
{
    if (!sort_requested(S)) return;
    const int d = blockIdx.x * blockDim.x + threadIdx.x;
    if (d >= S.N) return;
    S.r[d] = S.tmp_r[d];
    S.v[d] = S.tmp_v[d];
    S.image[d] = S.tmp_image[d];
    S.id[d] = S.tmp_id[d];
}

// ------------------------------------------------------------------------------------------ A4: cell build

// P:226-268 Fig. 5: one thread per (sorted) particle, 5x5x5 stencil of cells of edge >= (rc_max+skin)/2
// (P:278), periodic wrap (c + d + n) % n (needs n >= 5 per axis, S18), strict per-type-pair test
// (P:251-255), overflow flag, positions at build.  Rows come out in stencil order,
// which is fixed, so the list is reproducible.
__global__ void __launch_bounds__(128) k_build_cell(const Sys S)
{
    if (!rebuild_requested(S)) return;
    __shared__ float s_rcl2[RUMD_MAXT * RUMD_MAXT];
    if (threadIdx.x < RUMD_MAXT * RUMD_MAXT) s_rcl2[threadIdx.x] = S.pp[threadIdx.x].rcl2;
    __syncthreads();
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= S.N) return;
    const float4 ri = S.r[i];
    const int trow = type_of(ri) * S.ntypes;
    int cx, cy, cz;
    cell_coords(S, ri, cx, cy, cz);
    const int nx = S.grid.n[0], ny = S.grid.n[1], nz = S.grid.n[2];
    int count = 0;
    for (int dz = -2; dz <= 2; ++dz) {
        const int z = (cz + dz + nz) % nz;
        for (int dy = -2; dy <= 2; ++dy) {
            const int y = (cy + dy + ny) % ny;
            const int row = (z * ny + y) * nx;
            for (int dx = -2; dx <= 2; ++dx) {
                const int c = row + (cx + dx + nx) % nx;
                const int je = S.cell_end[c];
                for (int j = S.cell_start[c]; j < je; ++j) {
                    if (j == i) continue;
                    const float4 rj = __ldg(&S.r[j]);
                    const float ddx = min_image(ri.x, rj.x, S.h[0], S.invL[0]);
                    const float ddy = min_image(ri.y, rj.y, S.h[1], S.invL[1]);
                    const float ddz = min_image(ri.z, rj.z, S.h[2], S.invL[2]);
                    const float d2 = __fmaf_rn(ddz, ddz, __fmaf_rn(ddy, ddy, ddx * ddx));
                    if (d2 < s_rcl2[trow + type_of(rj)]) {
                        if (count < S.cap) S.nbl[nbl_index(S, i, count)] = j;
                        ++count;
                    }
                }
            }
        }
    }
    S.num_nbrs[i] = min(count, S.cap);
    S.r_build[i] = ri;
    if (count > S.cap) S.sc->overflow = 1u;
    atomicMax(&S.sc->max_nbrs, count);
}
