// rumd_kernels.cuh -- sm_100a neighbour-list kernels of the RUMD hot path (A2, A3, A4).  Product code: shares
// nothing with oracle/.  "P:n" = PAPER.md line n; O*/S* = readings listed in DESIGN.md.
//
// Every piece of work is written once as a __device__ "phase" over a virtual grid (first item, stride); the
// stand-alone __global__ kernels (one phase each, early exit when no rebuild is requested) and the
// persistent whole-run kernel (rumd_persist.cuh: all phases, grid barriers in between) both call the phases.
#pragma once
#include <type_traits>
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
__device__ __forceinline__ bool rebuild_requested(const Sys& S) { return S.sc->flag != 0u && S.method != 2; }

// sort on this rebuild?  cell method: always; n2 method: every sort_interval-th rebuild.
__device__ __forceinline__ bool sort_on_rebuild(const Sys& S, long long n_rebuilds)
{
    if (S.method == 1 || S.method == 3) return true; // cell and tile methods: at every rebuild
    return S.method == 0 && S.sort_interval > 0 && (n_rebuilds % S.sort_interval) == 0;
}
__device__ __forceinline__ bool sort_requested(const Sys& S)
{
    return S.sc->flag != 0u && sort_on_rebuild(S, S.sc->n_rebuilds);
}

__device__ __forceinline__ void cell_coords(const Sys& S, const float4& p, int& cx, int& cy, int& cz)
{
    // S17: c_k = floor((x_k + L_k/2) * n_k / L_k), clamped to [0, n_k - 1]
    cx = min(S.grid.n[0] - 1, max(0, (int)floorf((p.x + S.h[0]) * S.grid.scale[0])));
    cy = min(S.grid.n[1] - 1, max(0, (int)floorf((p.y + S.h[1]) * S.grid.scale[1])));
    cz = min(S.grid.n[2] - 1, max(0, (int)floorf((p.z + S.h[2]) * S.grid.scale[2])));
}

__device__ __forceinline__ float list_dist2(const Sys& S, const float4& ri, const float4& rj)
{
    const float dx = min_image(ri.x, rj.x, S.h[0], S.invL[0]);
    const float dy = min_image(ri.y, rj.y, S.h[1], S.invL[1]);
    const float dz = min_image(ri.z, rj.z, S.h[2], S.invL[2]);
    return __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, dx * dx));
}

// ------------------------------------------------------------------------------------------ tile geometry
// Tile method (RUMD_NB_TILE, rumd_tile.cuh): the cell grid of S17 is cut into nt[0] x nt[1] x nt[2] boxes of cells
// ("tiles", balanced widths: tile j of an axis with n cells covers cells [j n / nt, (j+1) n / nt)).  Particles are
// sorted TILE-MAJOR -- key = cells of all earlier tiles (tiles ordered z, y, x; x fastest) + row-major cell index
// inside the tile -- so that the particles a tile owns are ONE contiguous range and the cells of one x-row of a
// tile are contiguous too.
struct TileGeo {
    int x0, y0, z0, wx, wy, wz; // first cell and width per axis
    int cellbase;               // sort key of the tile's first cell
};

__device__ __forceinline__ TileGeo tile_geo(const Sys& S, int t)
{
    const int nx = S.grid.n[0], ny = S.grid.n[1], nz = S.grid.n[2];
    const int tx = t % S.nt[0], ty = (t / S.nt[0]) % S.nt[1], tz = t / (S.nt[0] * S.nt[1]);
    TileGeo g;
    g.x0 = tx * nx / S.nt[0];
    g.wx = (tx + 1) * nx / S.nt[0] - g.x0;
    g.y0 = ty * ny / S.nt[1];
    g.wy = (ty + 1) * ny / S.nt[1] - g.y0;
    g.z0 = tz * nz / S.nt[2];
    g.wz = (tz + 1) * nz / S.nt[2] - g.z0;
    // whole z-slabs of tiles below, whole rows of tiles at lower y in this slab, tiles at lower x in this row
    g.cellbase = g.z0 * ny * nx + g.wz * (g.y0 * nx + g.wy * g.x0);
    return g;
}

__device__ __forceinline__ int tile_of_cell(int c, int nt, int n) { return ((c + 1) * nt - 1) / n; }

__device__ __forceinline__ int tile_index_of_cell(const Sys& S, int cx, int cy, int cz)
{
    return (tile_of_cell(cz, S.nt[2], S.grid.n[2]) * S.nt[1] + tile_of_cell(cy, S.nt[1], S.grid.n[1])) * S.nt[0] +
           tile_of_cell(cx, S.nt[0], S.grid.n[0]);
}

__device__ __forceinline__ int tile_cell_key(const Sys& S, int cx, int cy, int cz)
{
    const TileGeo g = tile_geo(S, tile_index_of_cell(S, cx, cy, cz));
    return g.cellbase + ((cz - g.z0) * g.wy + (cy - g.y0)) * g.wx + (cx - g.x0);
}

// List rows of the tile method are addressed by a PADDED particle index, so that the rows of one tile start at a
// warp boundary: particle i of tile t (own range starting at o0) has row index pbase(t) + (i - o0).
__device__ __forceinline__ int tile_pbase(int o0, int t) { return ((o0 + 31) & ~31) + 32 * t; }

// Box lengths as a kernel sees them.  NVE / NVT: the constants of the parameter block.  NPT: the box is a device
// quantity that changes every step (DevScalars::box, rumd_npt.cuh).
struct Box {
    float L[3], h[3], invL[3];
};

__device__ __forceinline__ Box box_of_sys(const Sys& S)
{
    Box b;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        b.L[k] = S.L[k];
        b.h[k] = S.h[k];
        b.invL[k] = S.invL[k];
    }
    return b;
}

__device__ __forceinline__ Box box_of_doubles(const double* L)
{
    Box b;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        b.L[k] = (float)L[k];
        b.h[k] = 0.5f * b.L[k];
        b.invL[k] = (float)(1.0 / L[k]);
    }
    return b;
}

// ------------------------------------------------------------------------------------------ A2: N^2 build

// P:173-224 Fig. 4.  One WARP per particle i; j-positions staged through shared memory in tiles
// (P:184); the 32 lanes test 32 different j at once and slots are handed out by
// ballot + popc, so the row is in ascending-j order and the whole list is bitwise reproducible (the
// paper's atomicInc gives "an unspecified sequential order").  Writes num_nbrs, positions at build
// and the overflow flag.  Block-cooperative: `blk`/`nblk` = this block's index / block count
// in the virtual grid; blockDim.x must be a multiple of 32.  max_slot: &sc->max_nbrs[build & 1].
#define N2_TILE 256
template <bool NPT = false>
__device__ __forceinline__ void ph_build_n2(const Sys& S, const float4* r, float4* tile, const float* s_rcl2,
                                            int blk, int nblk, int* max_slot, const Box* bx = nullptr)
{
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
    const int ngroups = (S.N + nw - 1) / nw;
    for (int g = blk; g < ngroups; g += nblk) {
        const int i = g * nw + wid;
        const bool have_i = i < S.N;
        float4 ri = make_float4(0.f, 0.f, 0.f, 0.f);
        if (have_i) ri = r[i];
        const int trow = have_i ? type_of(ri) * S.ntypes : 0;
        int count = 0;
        for (int j0 = 0; j0 < S.N; j0 += N2_TILE) {
            __syncthreads();
            for (int t = threadIdx.x; t < N2_TILE; t += blockDim.x)
                if (j0 + t < S.N) tile[t] = r[j0 + t];
            __syncthreads();
            const int jend = min(N2_TILE, S.N - j0);
            for (int jj = lane; jj < ((jend + 31) & ~31); jj += 32) {
                bool acc = false;
                const int j = j0 + jj;
                if (jj < jend && have_i && j != i) {
                    const float4 rj = tile[jj];
                    float d2;
                    if (NPT) { // box read from device memory by the caller
                        const float dx = min_image(ri.x, rj.x, bx->h[0], bx->invL[0]);
                        const float dy = min_image(ri.y, rj.y, bx->h[1], bx->invL[1]);
                        const float dz = min_image(ri.z, rj.z, bx->h[2], bx->invL[2]);
                        d2 = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, dx * dx));
                    } else
                        d2 = list_dist2(S, ri, rj);
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
            atomicMax(max_slot, count);
        }
    }
}

// ------------------------------------------------------------------------------------------ A3: cells + sort

// P:276 steps 1-3: cell of every particle, sort particles by cell, rearrange all particle data.  The paper
// calls Thrust; here it is a counting sort written out: (a) histogram with slot = atomicAdd, (b) exclusive
// scan, (c) scatter, (d) ordering of the (few) entries of each cell by old index, which removes the
// atomic's arbitrary order so that the particle order -- and with it every later fp32 sum -- is
// reproducible.  Sort key of cell (x, y, z) = rowrank[z][y] * nx + x, where rowrank numbers the (y, z) cell
// columns along a 2-D Morton (Z-order) curve (table built once on the host): consecutive particles are
// spatially compact (BASELINE configs[3], S19) AND the cells of one x-row are contiguous in the sorted
// order, so the 5 x-neighbour cells of a stencil row are ONE particle range (cellStart of the first cell to
// cellStart of the cell after the last) -- the build then walks 25 ranges instead of 125 cells.

// Tile method: between rebuilds the integrator leaves coordinates that crossed a face UNWRAPPED (they stay within
// skin/2 of the box, O9), so that the periodic images fixed in a tile's halo at build time stay valid; the wrap into
// [-L/2, L/2) and the image counters (S7) are applied here, at the start of the next rebuild.
__device__ __forceinline__ void ph_cell_assign(const Sys& S, float4* r, int first, int stride)
{
    for (int i = first; i < S.N; i += stride) {
        int cx, cy, cz;
        float4 p = r[i];
        if (S.method == 3) {
            const float nx = rintf(p.x * S.invL[0]), ny = rintf(p.y * S.invL[1]), nz = rintf(p.z * S.invL[2]);
            if (nx != 0.f || ny != 0.f || nz != 0.f) {
                p.x = __fmaf_rn(-nx, S.L[0], p.x);
                p.y = __fmaf_rn(-ny, S.L[1], p.y);
                p.z = __fmaf_rn(-nz, S.L[2], p.z);
                int4 im = S.image[i];
                im.x += (int)nx;
                im.y += (int)ny;
                im.z += (int)nz;
                S.image[i] = im;
                r[i] = p;
            }
        }
        cell_coords(S, p, cx, cy, cz);
        const int z = S.method == 3 ? tile_cell_key(S, cx, cy, cz) : S.rowrank[cz * S.grid.n[1] + cy] * S.grid.n[0] + cx;
        S.cell_of[i] = z;
        S.slot[i] = atomicAdd(&S.ccount[z], 1);
    }
}

#define SCAN_THREADS 256
#define SCAN_ITEMS 8
#define SCAN_CHUNK (SCAN_THREADS * SCAN_ITEMS)

// Exclusive scan of one int per thread over the first SCAN_THREADS threads of the block (all threads of the
// block must call; threads >= SCAN_THREADS pass 0 and ignore the result).  s_warp: 33 ints.
__device__ __forceinline__ int block_exclusive_scan(int x, int* s_warp, int& total)
{
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    int incl = x;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        int y = __shfl_up_sync(FULLMASK, incl, o);
        if (lane >= o) incl += y;
    }
    if (lane == 31 && wid < SCAN_THREADS / 32) s_warp[wid] = incl;
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
    const int res = incl - x + (wid < SCAN_THREADS / 32 ? s_warp[wid] : 0);
    __syncthreads();
    return res;
}

// phase 1: per-chunk totals (block-cooperative over chunks)
__device__ __forceinline__ void ph_scan_sums(const Sys& S, int* s_warp, int blk, int nblk)
{
    const int nchunks = (S.grid.ncell + SCAN_CHUNK - 1) / SCAN_CHUNK;
    for (int c = blk; c < nchunks; c += nblk) {
        const int base = c * SCAN_CHUNK + threadIdx.x * SCAN_ITEMS;
        int x = 0;
        if (threadIdx.x < SCAN_THREADS) {
#pragma unroll
            for (int q = 0; q < SCAN_ITEMS; ++q)
                if (base + q < S.grid.ncell) x += S.ccount[base + q];
        }
        int total;
        block_exclusive_scan(x, s_warp, total);
        if (threadIdx.x == 0) S.blocksum[c] = total;
    }
}

// phase 2: exclusive scan of the chunk totals (ONE block)
__device__ __forceinline__ void ph_scan_blocks(const Sys& S, int* s_warp)
{
    const int nchunks = (S.grid.ncell + SCAN_CHUNK - 1) / SCAN_CHUNK;
    int carry = 0;
    for (int b0 = 0; b0 < nchunks; b0 += SCAN_THREADS) {
        const int b = b0 + threadIdx.x;
        const bool on = threadIdx.x < SCAN_THREADS && b < nchunks;
        const int x = on ? S.blocksum[b] : 0;
        int total;
        const int e = block_exclusive_scan(x, s_warp, total);
        if (on) S.blocksum[b] = carry + e;
        carry += total;
    }
    if (threadIdx.x == 0) S.cstart_z[S.grid.ncell] = S.N;
}

// phase 3: exclusive scan inside each chunk + chunk offset -> first sorted slot of each Z-ordered cell
__device__ __forceinline__ void ph_scan_apply(const Sys& S, int* s_warp, int blk, int nblk)
{
    const int nchunks = (S.grid.ncell + SCAN_CHUNK - 1) / SCAN_CHUNK;
    for (int ch = blk; ch < nchunks; ch += nblk) {
        const int base = ch * SCAN_CHUNK + threadIdx.x * SCAN_ITEMS;
        int c[SCAN_ITEMS];
        int x = 0;
#pragma unroll
        for (int q = 0; q < SCAN_ITEMS; ++q) {
            c[q] = (threadIdx.x < SCAN_THREADS && base + q < S.grid.ncell) ? S.ccount[base + q] : 0;
            x += c[q];
        }
        int total;
        int e = block_exclusive_scan(x, s_warp, total) + S.blocksum[ch];
        if (threadIdx.x < SCAN_THREADS) {
#pragma unroll
            for (int q = 0; q < SCAN_ITEMS; ++q) {
                if (base + q < S.grid.ncell) S.cstart_z[base + q] = e;
                e += c[q];
            }
        }
    }
}

// all three phases by ONE block (small grids: saves two grid barriers in the persistent kernel)
__device__ __forceinline__ void ph_scan_single_block(const Sys& S, int* s_warp)
{
    const int nchunks = (S.grid.ncell + SCAN_CHUNK - 1) / SCAN_CHUNK;
    int carry = 0;
    for (int ch = 0; ch < nchunks; ++ch) {
        const int base = ch * SCAN_CHUNK + threadIdx.x * SCAN_ITEMS;
        int c[SCAN_ITEMS];
        int x = 0;
#pragma unroll
        for (int q = 0; q < SCAN_ITEMS; ++q) {
            c[q] = (threadIdx.x < SCAN_THREADS && base + q < S.grid.ncell) ? S.ccount[base + q] : 0;
            x += c[q];
        }
        int total;
        int e = block_exclusive_scan(x, s_warp, total) + carry;
        if (threadIdx.x < SCAN_THREADS) {
#pragma unroll
            for (int q = 0; q < SCAN_ITEMS; ++q) {
                if (base + q < S.grid.ncell) S.cstart_z[base + q] = e;
                e += c[q];
            }
        }
        carry += total;
    }
    if (threadIdx.x == 0) S.cstart_z[S.grid.ncell] = S.N;
}

__device__ __forceinline__ void ph_cell_scatter(const Sys& S, int first, int stride)
{
    for (int i = first; i < S.N; i += stride) S.perm[S.cstart_z[S.cell_of[i]] + S.slot[i]] = i;
}

// P:276 "rearrange all particle data into the sorted order": gather into scratch, then copy back (the
// caller owns the arrays, so the pointers cannot be swapped).
// Step (d) and the gather in one pass: the particle in (unordered) slot d of the scatter finds its rank among
// the members of its cell by old index (cells hold a handful of particles) and moves its data to
// cellStart + rank; the first slot of a cell clears the cell's histogram entry for the next sort (empty cells
// are already 0).  cellStart is the scan output cstart_z[key]; cellEnd of a cell = cellStart of the
// next key (EXCLUSIVE, S20; cstart_z[ncell] = N).
__device__ __forceinline__ void ph_permute_gather_ranked(const Sys& S, const float4* r, int first, int stride)
{
    for (int d = first; d < S.N; d += stride) {
        const int src = S.perm[d];
        const int z = S.cell_of[src];
        const int b = S.cstart_z[z], n = S.cstart_z[z + 1] - b;
        int less = 0;
        for (int q = 0; q < n; ++q) less += S.perm[b + q] < src;
        if (d == b) S.ccount[z] = 0;
        const int dst = b + less;
        S.tmp_r[dst] = r[src];
        S.tmp_v[dst] = S.v[src];
        S.tmp_image[dst] = S.image[src];
        S.tmp_id[dst] = S.id[src];
    }
}

__device__ __forceinline__ void ph_permute_store(const Sys& S, float4* r, int first, int stride)
{
    for (int d = first; d < S.N; d += stride) {
        r[d] = S.tmp_r[d];
        S.v[d] = S.tmp_v[d];
        S.image[d] = S.tmp_image[d];
        S.id[d] = S.tmp_id[d];
    }
}

// ------------------------------------------------------------------------------------------ A4: cell build

// P:226-268 Fig. 5: 5x5x5 stencil of cells of edge >= (rc_max+skin)/2, periodic wrap of the cell
// coordinate (needs n >= 5 per axis, S18), strict per-type-pair test, overflow flag
// (P:256), positions at build.  The paper uses one thread per particle and notes that several
// threads per particle had "not been tried yet"; here G = 1..32 lanes share one particle: lane l
// takes stencil rows l, l+G, ... of the 25 (dy, dz) rows; a row's 5 x-cells are one contiguous particle range
// (two when the row wraps around the box in x).  The group walks its ranges in lock step and hands out list
// slots by ballot + popc, so rows of the list come out in the fixed order (round, position in range, lane)
// and the list is bitwise reproducible.  `first`/`stride` index the virtual grid of N*G threads.
// queue != nullptr: the warps take their units of 32 virtual threads from this device counter (which holds the number
// of warps of the grid when the phase starts) instead of the fixed stride.  A warp next to a face of the box walks the general stencil path for all its
// lanes, about twice the work of an interior one, and with ~9 units per warp at N = 10^6 the slowest warp of a fixed
// assignment finished 30 % after the average one (the others waited at the grid barrier).  The list does not depend
// on who builds a row.
template <int G>
__device__ __forceinline__ void ph_build_cell(const Sys& S, const float4* r, const float* s_rcl2, int first,
                                              int stride, int* max_slot, int* queue = nullptr)
{
    const int lane = threadIdx.x & 31;
    const int l = lane & (G - 1);
    const unsigned gmask = G == 32 ? FULLMASK : (((1u << G) - 1u) << (lane & ~(G - 1)));
    const unsigned lt = gmask & ((1u << lane) - 1u);
    const int nx = S.grid.n[0], ny = S.grid.n[1], nz = S.grid.n[2];
    const long long total = (long long)S.N * G;
    // dynamic assignment: the unit this warp works on next.  The first one is the warp's own index (the counter starts
    // at the number of warps: no burst of same-address atomics when the phase begins); the request for the one after is
    // in flight while the current one is worked on.
    int unit = first >> 5;
    for (long long vt = first;; vt += stride) {
        if (queue) {
            vt = (long long)unit * 32 + lane;
            if (vt - lane < total && lane == 0) unit = atomicAdd(queue, 1);
        }
        if (vt - lane >= total) break;
        const int i = (int)(vt / G);
        const bool have_i = i < S.N;
        float4 ri = make_float4(0.f, 0.f, 0.f, 0.f);
        if (have_i) ri = r[i];
        const int trow = have_i ? type_of(ri) * S.ntypes : 0;
        int cx = 0, cy = 0, cz = 0;
        if (have_i) cell_coords(S, ri, cx, cy, cz);
        // x extent of the stencil: main segment [x0, x1], wrapped segment [w0, w1] (empty if w0 > w1)
        const int x0 = max(cx - 2, 0), x1 = min(cx + 2, nx - 1);
        int w0 = 1, w1 = 0;
        if (cx - 2 < 0) {
            w0 = nx + cx - 2;
            w1 = nx - 1;
        } else if (cx + 2 >= nx) {
            w0 = 0;
            w1 = cx + 2 - nx;
        }
        int count = 0;
        const int isafe = have_i ? i : 0; // in-bounds stand-in for the masked slots of lanes past the last particle
        // warp-uniform fast path: no lane's stencil crosses a face of the box -> no wrapped x piece, no y / z shifts
        const bool interior = __all_sync(FULLMASK, !have_i || (cx >= 2 && cx + 2 < nx && cy >= 2 && cy + 2 < ny &&
                                                               cz >= 2 && cz + 2 < nz));
        // Minimum image without per-pair rounding work: all candidates of one range lie in cells reached with
        // the same periodic shift s in {-1, 0, +1} per axis (s != 0 where the stencil row, or the wrapped x
        // segment, crossed a face), and d = (x_i - s h) - (x_j + s h) is the exact nearest-image displacement
        // for every pair that can be inside the list cutoff (both brackets are exact, cf. min_image; needs
        // n >= 5 cells per axis, S18).  sxh: shift of the wrapped x segment; the main segment has none.
        const float sxh = cx - 2 < 0 ? -S.h[0] : S.h[0];
        // particle ranges of stencil row q (0..24): main [a.x, a.y) and wrapped [b.x, b.y); its y / z shifts
        auto ranges_of = [&](auto INT, int q, int2& a, int2& b, float& syh, float& szh) {
            a = b = make_int2(0, 0);
            syh = szh = 0.f;
            if (!have_i || q >= 25) return;
            int z = cz + q / 5 - 2, y = cy + q % 5 - 2;
            if (decltype(INT)::value) {
                const int* cs = S.cstart_z + S.rowrank[z * ny + y] * nx;
                a = make_int2(cs[cx - 2], cs[cx + 3]);
                return;
            }
            if (z < 0) {
                z += nz;
                szh = -S.h[2];
            } else if (z >= nz) {
                z -= nz;
                szh = S.h[2];
            }
            if (y < 0) {
                y += ny;
                syh = -S.h[1];
            } else if (y >= ny) {
                y -= ny;
                syh = S.h[1];
            }
            const int* cs = S.cstart_z + S.rowrank[z * ny + y] * nx;
            a = make_int2(cs[x0], cs[x1 + 1]);
            if (w0 <= w1) b = make_int2(cs[w0], cs[w1 + 1]);
        };
        // this particle's row of the tiled list: entry k at rowbase[(k >> tp_shift) * 32 + (k & (tp - 1))]
        int* rowbase = S.nbl + ((size_t)(i >> S.ppw_shift) * S.cap_it * 32 + ((i & ((1 << S.ppw_shift) - 1)) << S.tp_shift));
        const int tmask = (1 << S.tp_shift) - 1;
        // list cutoffs of this particle's type against every type (S4), held in registers
        const float c0 = s_rcl2[trow], c1 = s_rcl2[trow + 1], c2 = s_rcl2[trow + 2], c3 = s_rcl2[trow + 3];
        auto walk = [&](auto INT) {
        constexpr bool I = decltype(INT)::value;
        int2 na, nb;
        float nsy, nsz;
        ranges_of(INT, l, na, nb, nsy, nsz);
        for (int q0 = 0; q0 < 25; q0 += G) {
            const int2 a = na, b = nb;
            const float syh = nsy, szh = nsz;
            if (q0 + G < 25) ranges_of(INT, q0 + G + l, na, nb, nsy, nsz); // one-ahead prefetch of the next round's ranges
            const float ay = ri.y - syh, az = ri.z - szh;
            // the main piece of the row, then its x-wrapped piece (empty except next to the x faces)
#pragma unroll
            for (int piece = 0; piece < (I ? 1 : 2); ++piece) {
                const int start = piece == 0 ? a.x : b.x;
                const int n = piece == 0 ? a.y - a.x : b.y - b.x;
                const int nmax = __reduce_max_sync(FULLMASK, n);
                const float shx = piece == 0 ? 0.f : sxh;
                const float ax = ri.x - shx;
                // candidates in flight per lane: a stencil row holds 12-17 of them; 6 with several lanes per particle
                // (small N, latency bound: fewer dependent rounds), 4 with one lane (large N: fewer masked slots)
                constexpr int U = G == 1 ? 4 : 6;
                for (int it0 = 0; it0 < nmax; it0 += U) {
                    float4 rj[U];
                    int j[U];
#pragma unroll
                    for (int q = 0; q < U; ++q) {
                        j[q] = it0 + q < n ? start + it0 + q : isafe; // masked: gather the particle itself (n > 0 => have_i)
                        rj[q] = r[j[q]];
                    }
#pragma unroll
                    for (int q = 0; q < U; ++q) {
                        const float dx = piece == 0 ? ri.x - rj[q].x : ax - (rj[q].x + shx);
                        // interior: syh = szh = 0, the same values without the two additions
                        const float dy = I ? ri.y - rj[q].y : ay - (rj[q].y + syh);
                        const float dz = I ? ri.z - rj[q].z : az - (rj[q].z + szh);
                        const float d2 = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, dx * dx));
                        const int tj = type_of(rj[q]);
                        const float thr = S.ntypes <= 2 ? (tj ? c1 : c0) : (tj == 0 ? c0 : tj == 1 ? c1 : tj == 2 ? c2 : c3);
                        const bool acc = have_i && j[q] != i && d2 < thr;
                        if (G == 1) { // the lane owns the row: no slot negotiation
                            if (acc && count < S.cap) rowbase[((count >> S.tp_shift) << 5) + (count & tmask)] = j[q];
                            count += acc ? 1 : 0;
                        } else {
                            const unsigned m = __ballot_sync(FULLMASK, acc);
                            if (acc) {
                                const int k = count + __popc(m & lt);
                                if (k < S.cap) rowbase[((k >> S.tp_shift) << 5) + (k & tmask)] = j[q];
                            }
                            count += __popc(m & gmask);
                        }
                    }
                }
            }
        }
        };
        if (interior) walk(std::true_type{});
        else walk(std::false_type{});
        if (have_i && l == 0) {
            S.num_nbrs[i] = min(count, S.cap);
            S.r_build[i] = ri;
            if (count > S.cap) S.sc->overflow = 1u;
        }
        const int wmax = __reduce_max_sync(FULLMASK, count); // one atomic per warp, not per particle
        if (lane == 0) atomicMax(max_slot, wmax);
        if (queue) unit = __shfl_sync(FULLMASK, unit, 0);
    }
}

__device__ __forceinline__ void build_cell_dispatch(const Sys& S, const float4* r, const float* s_rcl2, int first,
                                                    int stride, int* max_slot, int* queue = nullptr)
{
    switch (S.build_tp_shift) {
    case 0: ph_build_cell<1>(S, r, s_rcl2, first, stride, max_slot, queue); break;
    case 1: ph_build_cell<2>(S, r, s_rcl2, first, stride, max_slot, queue); break;
    case 2: ph_build_cell<4>(S, r, s_rcl2, first, stride, max_slot, queue); break;
    case 3: ph_build_cell<8>(S, r, s_rcl2, first, stride, max_slot, queue); break;
    case 4: ph_build_cell<16>(S, r, s_rcl2, first, stride, max_slot, queue); break;
    default: ph_build_cell<32>(S, r, s_rcl2, first, stride, max_slot, queue); break;
    }
}

// ------------------------------------------------------------------------------------------ stand-alone kernels
// One phase each; every kernel exits at once when the device flag is clear, so the chain can be
// enqueued -- or baked into a CUDA graph -- every step without asking the host.

#define VGRID const int first = blockIdx.x * blockDim.x + threadIdx.x, stride = gridDim.x * blockDim.x

__device__ __forceinline__ int* max_slot_of(const Sys& S) { return &S.sc->max_nbrs[S.sc->n_rebuilds & 1]; }

#ifdef RUMD_MAIN_TU // non-template kernels: compiled once, in rumd_b200.cu
static __global__ void __launch_bounds__(128) k_build_n2(const Sys S)
{
    if (!rebuild_requested(S)) return;
    __shared__ float4 tile[N2_TILE];
    __shared__ float s_rcl2[RUMD_MAXT * RUMD_MAXT];
    if (threadIdx.x < RUMD_MAXT * RUMD_MAXT) s_rcl2[threadIdx.x] = S.pp[threadIdx.x].rcl2;
    __syncthreads();
    ph_build_n2(S, S.r, tile, s_rcl2, blockIdx.x, gridDim.x, max_slot_of(S));
}

static __global__ void __launch_bounds__(128) k_build_cell(const Sys S)
{
    if (!rebuild_requested(S)) return;
    __shared__ float s_rcl2[RUMD_MAXT * RUMD_MAXT];
    if (threadIdx.x < RUMD_MAXT * RUMD_MAXT) s_rcl2[threadIdx.x] = S.pp[threadIdx.x].rcl2;
    __syncthreads();
    VGRID;
    build_cell_dispatch(S, S.r, s_rcl2, first, stride, max_slot_of(S));
}

static __global__ void k_cell_assign(const Sys S)
{
    if (!sort_requested(S)) return;
    VGRID;
    ph_cell_assign(S, S.r, first, stride);
}

static __global__ void __launch_bounds__(SCAN_THREADS) k_scan_sums(const Sys S)
{
    if (!sort_requested(S)) return;
    __shared__ int s_warp[33];
    ph_scan_sums(S, s_warp, blockIdx.x, gridDim.x);
}

static __global__ void __launch_bounds__(SCAN_THREADS) k_scan_blocks(const Sys S)
{
    if (!sort_requested(S)) return;
    __shared__ int s_warp[33];
    ph_scan_blocks(S, s_warp);
}

static __global__ void __launch_bounds__(SCAN_THREADS) k_scan_apply(const Sys S)
{
    if (!sort_requested(S)) return;
    __shared__ int s_warp[33];
    ph_scan_apply(S, s_warp, blockIdx.x, gridDim.x);
}

static __global__ void __launch_bounds__(SCAN_THREADS) k_scan_single(const Sys S)
{
    if (!sort_requested(S)) return;
    __shared__ int s_warp[33];
    ph_scan_single_block(S, s_warp);
}

static __global__ void k_cell_scatter(const Sys S)
{
    if (!sort_requested(S)) return;
    VGRID;
    ph_cell_scatter(S, first, stride);
}

static __global__ void k_permute_gather(const Sys S)
{
    if (!sort_requested(S)) return;
    VGRID;
    ph_permute_gather_ranked(S, S.r, first, stride);
}

static __global__ void k_permute_store(const Sys S)
{
    if (!sort_requested(S)) return;
    VGRID;
    ph_permute_store(S, S.r, first, stride);
}
#endif // RUMD_MAIN_TU
