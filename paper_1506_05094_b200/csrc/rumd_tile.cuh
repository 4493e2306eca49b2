// rumd_tile.cuh -- the TILE method (RUMD_NB_TILE): list build and pair forces with the j-particles staged in
// shared memory (sm_100a).  Product code: shares nothing with oracle/.
//
// Why.  With the cell method every listed pair costs the force kernel one scattered 16-byte gather through L1
// (P:165 LOAD(); ncu at N = 10^6: L1 data stage 80 % busy, 14.5 sectors per request, 29 % of the FP32 peak) and
// every candidate of the build another one.  BASELINE north_star asks for "shared-memory tiling of j-particles".
// A broadcast tile (every i of a tile against every j of a tile) wastes 70-90 % of its pair evaluations at this
// cutoff (78 listed neighbours), so the list stays per particle -- but the positions it points into now live in
// SHARED memory:
//   * the cell grid (S17) is cut into tiles of <= 8 cells per axis; particles are sorted tile-major, a tile OWNS a
//     contiguous particle range and is worked on by one thread block;
//   * the block loads the tile's HALO -- all particles in the tile's cells plus two cells on every side (the 5x5x5
//     stencil of P:237-259 for every owned cell) -- once, coalesced, into shared memory: 3-12 loads per owned
//     particle instead of ~80-170 gathers;
//   * list entries are 16-bit HALO SLOT numbers (half the index stream of the int32 list), read eight at
//     a time (one 16-byte load per lane), and every gather is an LDS.128;
//   * the periodic image of a halo particle is fixed when the halo is laid out: a slot reached across a face holds
//     the half-shifted coordinate x - sign(x) L/2 (exact, cf. min_image) and a ghost bit per axis; the owning
//     particle then uses ITS half-shifted coordinate for that pair, so the displacement is bit for bit the one the
//     cell method computes.  To keep the fixed images valid the integrator does not wrap coordinates between
//     rebuilds (ph_cell_assign wraps them at the next rebuild; they stay within skin/2 of the box, O9);
//   * the build tests its candidates out of the same shared-memory halo (the 25 stencil rows of a particle are 25
//     contiguous slot ranges), so it issues no global gathers either.
#pragma once
#include "rumd_force.cuh"

#define TILE_WMAX 8                                                 // cells per tile edge, at most
#define TILE_HC_MAX ((TILE_WMAX + 4) * (TILE_WMAX + 4) * (TILE_WMAX + 4)) // halo cells of a tile, at most (1728)
#define TILE_THREADS 256
#define TILE_GHOST_SHIFT 28
#define TILE_IDX_MASK 0x0fffffff
#define TILE_FAR 1.0e15f // coordinate of the dummy slot: r^2 = 3e30 is finite and beyond every cutoff

// shared memory of a tile kernel: halo positions (hcap + 1 float4); kernels that build also hold the halo cell starts
// (16-bit) and, per warp of a 256-thread block, a candidate buffer and a row buffer (TILE_WARP_SCRATCH)
__host__ __device__ __forceinline__ size_t tile_smem_bytes_force(int hcap) { return (size_t)(hcap + 1) * 16; }
__host__ __device__ __forceinline__ size_t tile_smem_bytes(int hcap)
{
    return tile_smem_bytes_force(hcap) + (TILE_THREADS / 32) * ((512 + 384) * 2) + ((TILE_HC_MAX + 1) * 2 + 15) / 16 * 16;
}

// half shift toward the origin: x - sign(x) L/2, exact for |x| >= L/4 (Sterbenz), which every particle that can be
// paired across a face satisfies when L/2 >= 2 (rc + skin); in smaller boxes ulp(L/2) < 5e-7 bounds the error
__device__ __forceinline__ float half_shift(float x, float h) { return x - copysignf(h, x); }

// position of a halo slot as the pair loop wants it: half-shifted on the axes where the slot is a periodic image,
// .w = type | ghost bits << 8
__device__ __forceinline__ float4 tile_slot_value(const Sys& S, float4 p, unsigned gb)
{
    if (gb & 1u) p.x = half_shift(p.x, S.h[0]);
    if (gb & 2u) p.y = half_shift(p.y, S.h[1]);
    if (gb & 4u) p.z = half_shift(p.z, S.h[2]);
    p.w = __int_as_float(__float_as_int(p.w) | (int)(gb << 8));
    return p;
}

// Does this tile's halo touch a face of the box on axis k (then slots can be periodic images, and particles of
// the outermost cells can drift across the face)?  Bit k of the result.
__device__ __forceinline__ unsigned tile_wrap_axes(const Sys& S, const TileGeo& g)
{
    unsigned m = 0;
    if (g.x0 - 2 <= 0 || g.x0 + g.wx + 2 >= S.grid.n[0]) m |= 1u;
    if (g.y0 - 2 <= 0 || g.y0 + g.wy + 2 >= S.grid.n[1]) m |= 2u;
    if (g.z0 - 2 <= 0 || g.z0 + g.wz + 2 >= S.grid.n[2]) m |= 4u;
    return m;
}

// ------------------------------------------------------------------------------------------ halo, at build time
// Lays out the halo of tile t: slot order = halo cells (z, y, x; x fastest), particles of a cell in sorted order.
// Fills s_hstart[0 .. nhc] (first slot of every halo cell), halo_idx / halo_cnt in global memory and the slot
// values in shared memory.  Block-cooperative, blockDim.x >= SCAN_THREADS.
__device__ __forceinline__ void tile_layout_halo(const Sys& S, const float4* r, int t, const TileGeo& g, float4* s_pos,
                                                 unsigned short* s_hstart, int* s_warp)
{
    const int nx = S.grid.n[0], ny = S.grid.n[1], nz = S.grid.n[2];
    const int hx = g.wx + 4, hy = g.wy + 4, nhc = hx * hy * (g.wz + 4);
    auto cell_of_hc = [&](int hc, int& key, unsigned& gb) {
        int cx = g.x0 - 2 + hc % hx, cy = g.y0 - 2 + (hc / hx) % hy, cz = g.z0 - 2 + hc / (hx * hy);
        gb = 0;
        if (cx < 0) { cx += nx; gb |= 1u; } else if (cx >= nx) { cx -= nx; gb |= 1u; }
        if (cy < 0) { cy += ny; gb |= 2u; } else if (cy >= ny) { cy -= ny; gb |= 2u; }
        if (cz < 0) { cz += nz; gb |= 4u; } else if (cz >= nz) { cz -= nz; gb |= 4u; }
        key = tile_cell_key(S, cx, cy, cz);
    };
    {   // exclusive scan of the halo cells' populations (<= SCAN_CHUNK = 2048 cells: one pass)
        const int base = threadIdx.x * SCAN_ITEMS;
        int c[SCAN_ITEMS], x = 0;
#pragma unroll
        for (int q = 0; q < SCAN_ITEMS; ++q) {
            c[q] = 0;
            if (threadIdx.x < SCAN_THREADS && base + q < nhc) {
                int key;
                unsigned gb;
                cell_of_hc(base + q, key, gb);
                c[q] = S.cstart_z[key + 1] - S.cstart_z[key];
            }
            x += c[q];
        }
        int total;
        int e = block_exclusive_scan(x, s_warp, total);
        if (threadIdx.x < SCAN_THREADS) {
#pragma unroll
            for (int q = 0; q < SCAN_ITEMS; ++q) {
                if (base + q <= nhc) s_hstart[base + q] = (unsigned short)min(e, S.hcap); // (entry nhc = total)
                e += c[q];
            }
        }
        if (threadIdx.x == 0) {
            S.halo_cnt[t] = min(total, S.hcap);
            if (total > S.hcap) S.sc->overflow = 2u; // halo capacity exceeded: sticky, reported by rumd_get_thermo
        }
    }
    __syncthreads();
    int* hidx = S.halo_idx + (size_t)t * S.hcap;
    for (int hc = threadIdx.x; hc < nhc; hc += blockDim.x) {
        int key;
        unsigned gb;
        cell_of_hc(hc, key, gb);
        const int g0 = S.cstart_z[key], n = S.cstart_z[key + 1] - g0, s0 = s_hstart[hc];
        for (int p = 0; p < n; ++p) {
            const int slot = s0 + p;
            if (slot < S.hcap) {
                hidx[slot] = (g0 + p) | (int)(gb << TILE_GHOST_SHIFT);
                s_pos[slot] = tile_slot_value(S, r[g0 + p], gb);
            }
        }
    }
    if (threadIdx.x == 0) s_pos[S.hcap] = make_float4(TILE_FAR, TILE_FAR, TILE_FAR, 0.f);
    __syncthreads();
}

// ------------------------------------------------------------------------------------------ halo, every step
// Current positions of the tile's halo into shared memory (coalesced index read, mostly contiguous position reads).
template <bool NC>
__device__ __forceinline__ void tile_load_halo(const Sys& S, const float4* r, int t, float4* s_pos)
{
    const int nh = S.halo_cnt[t];
    const int* hidx = S.halo_idx + (size_t)t * S.hcap;
    constexpr int U = 4; // slots per thread in flight: index loads first, then the position loads they address
    for (int s0 = threadIdx.x; s0 < nh; s0 += U * blockDim.x) {
        int gi[U];
        float4 p[U];
#pragma unroll
        for (int q = 0; q < U; ++q) {
            const int slot = s0 + q * blockDim.x;
            gi[q] = slot < nh ? (NC ? __ldg(hidx + slot) : hidx[slot]) : 0;
        }
#pragma unroll
        for (int q = 0; q < U; ++q) p[q] = load_pos<NC>(r + (gi[q] & TILE_IDX_MASK));
#pragma unroll
        for (int q = 0; q < U; ++q) {
            const int slot = s0 + q * blockDim.x;
            if (slot < nh) s_pos[slot] = tile_slot_value(S, p[q], (unsigned)gi[q] >> TILE_GHOST_SHIFT);
        }
    }
    if (threadIdx.x == 0) s_pos[S.hcap] = make_float4(TILE_FAR, TILE_FAR, TILE_FAR, 0.f);
}

// ------------------------------------------------------------------------------------------ list layout
// Entry k of the list row with padded particle index v (tile_pbase): rows are tiled per warp of the force kernel
// as in the cell method, in CHUNKS of eight 16-bit entries = one uint4 per lane and iteration.  With tp lanes per
// particle, chunk c of a particle belongs to its lane c % tp, iteration c / tp.
__device__ __forceinline__ size_t tile_entry_index(const Sys& S, int v, int k)
{
    const int w = v >> S.ppw_shift, pl = v & ((1 << S.ppw_shift) - 1);
    const int c = k >> 3, tl = c & ((1 << S.tp_shift) - 1), it = c >> S.tp_shift;
    return ((((size_t)w * S.cap_it8 + it) << 5) + (pl << S.tp_shift) + tl) * 8 + (k & 7);
}

// ------------------------------------------------------------------------------------------ A4 from shared memory
// P:226-268 Fig. 5 on the staged halo, one WARP per owned cell.  All particles of a cell share the 5x5x5 stencil
// (P:237-259): its 25 x-rows are 25 contiguous slot ranges, which the warp first writes out as one flat candidate
// list in shared memory (~300 slots); then, for each particle of the cell in turn, the 32 lanes test 32 consecutive
// candidates at a time -- the candidate positions are read with consecutive-slot LDS.128 (no bank conflicts), the
// particle's position is a broadcast read, no lane idles on a short row and no two lanes diverge.  List slots are
// handed out by ballot + popc in candidate order: the list is bitwise reproducible (the paper's atomicInc gives "an
// unspecified sequential order").  Strict per-type-pair test.  GH: the tile has periodic-image
// slots (block-uniform).  s_cand: TILE_CAND_MAX 16-bit slots per warp.
#define TILE_CAND_MAX 512 // candidate slots per warp buffer (a 5x5x5 stencil holds ~300 at liquid densities), a multiple of 64
#define TILE_ROW_MAX 384  // list entries staged per particle (>= the list capacity the tile method accepts)
#define TILE_WARP_SCRATCH ((TILE_CAND_MAX + TILE_ROW_MAX) * 2) // bytes per warp
template <bool GH>
__device__ __forceinline__ void tile_build_rows(const Sys& S, int t, const TileGeo& g, const float4* s_pos,
                                                const unsigned short* s_hstart, unsigned char* s_scratch,
                                                const float* s_rcl2, int* max_slot)
{
    const int hx = g.wx + 4, hy = g.wy + 4;
    const int o0 = S.cstart_z[g.cellbase];
    const int pbase = tile_pbase(o0, t);
    uint4* list4 = reinterpret_cast<uint4*>(S.nbl);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
    const unsigned lt = (1u << lane) - 1u;
    unsigned short* s_cand = reinterpret_cast<unsigned short*>(s_scratch + wid * TILE_WARP_SCRATCH);
    unsigned short* s_row = s_cand + TILE_CAND_MAX; // 16-byte aligned: read back as uint4 chunks
    const int tmask = (1 << S.tp_shift) - 1;
    const int ncell_own = g.wx * g.wy * g.wz;
    const int rowcap = min(S.cap, TILE_ROW_MAX);
    int wmax = 0;
    for (int oc = wid; oc < ncell_own; oc += nw) { // own cells in key order: key = cellbase + oc
        const int lx = oc % g.wx + 2, ly = (oc / g.wx) % g.wy + 2, lz = oc / (g.wx * g.wy) + 2;
        const int hc = (lz * hy + ly) * hx + lx;
        const int s_first = s_hstart[hc], np = s_hstart[hc + 1] - s_first;
        if (np <= 0) continue;
        const int g_first = S.cstart_z[g.cellbase + oc];
        // slot ranges of the 25 stencil rows, one per lane; their running offsets in the flat candidate list
        int a = 0, len = 0;
        if (lane < 25) {
            const int row = ((lz + lane / 5 - 2) * hy + (ly + lane % 5 - 2)) * hx + lx;
            a = s_hstart[row - 2];
            len = s_hstart[row + 3] - a;
            if (len > TILE_CAND_MAX) { // > 512 particles in five cells: not a liquid; reported like a halo overflow
                len = TILE_CAND_MAX;
                S.sc->overflow = 2u;
            }
        }
        int off = len; // inclusive scan
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int y = __shfl_up_sync(FULLMASK, off, o);
            if (lane >= o) off += y;
        }
        const int total = __shfl_sync(FULLMASK, off, 31);
        off -= len;
        const bool one_batch = total <= TILE_CAND_MAX; // (nearly always: then the list is written once per cell)
        for (int p = 0; p < np; ++p) {
            const int self = s_first + p;
            const float4 ri = s_pos[self]; // broadcast read; own cells are never periodic images
            const float ax = half_shift(ri.x, S.h[0]), ay = half_shift(ri.y, S.h[1]), az = half_shift(ri.z, S.h[2]);
            const float* thr_of = s_rcl2 + type_of(ri) * S.ntypes; // list cutoffs of this particle's type (S4)
            const bool one_type = S.ntypes == 1;
            const float thr_one = s_rcl2[0];
            int count = 0;
            for (int row0 = 0; row0 < 25;) {
                // the batch of rows [row0, row1) that fits the candidate buffer
                const int off0 = __shfl_sync(FULLMASK, off, row0);
                const bool fits = lane >= row0 && lane < 25 && off + len - off0 <= TILE_CAND_MAX;
                const int row1 = row0 + max(1, __popc(__ballot_sync(FULLMASK, fits)));
                const int btotal = __shfl_sync(FULLMASK, off + len, row1 - 1) - off0;
                if (p == 0 || !one_batch) {
                    __syncwarp();
                    if (lane >= row0 && lane < row1)
                        for (int j = 0; j < len; ++j) s_cand[off - off0 + j] = (unsigned short)(a + j);
                    // pad to a multiple of 64 with the far-away dummy slot: the passes below need no bounds checks
                    for (int n = btotal + lane; n < ((btotal + 63) & ~63); n += 32) s_cand[n] = (unsigned short)S.hcap;
                    __syncwarp();
                }
                // two passes of 32 candidates per iteration (two independent chains of shared-memory reads in flight)
                for (int n0 = 0; n0 < btotal; n0 += 64) {
                    const int slot0 = s_cand[n0 + lane], slot1 = s_cand[n0 + 32 + lane];
                    const float4 p0 = s_pos[slot0], p1 = s_pos[slot1];
                    const int w0 = __float_as_int(p0.w), w1 = __float_as_int(p1.w);
                    const float dx0 = ((GH && (w0 & 0x100)) ? ax : ri.x) - p0.x, dx1 = ((GH && (w1 & 0x100)) ? ax : ri.x) - p1.x;
                    const float dy0 = ((GH && (w0 & 0x200)) ? ay : ri.y) - p0.y, dy1 = ((GH && (w1 & 0x200)) ? ay : ri.y) - p1.y;
                    const float dz0 = ((GH && (w0 & 0x400)) ? az : ri.z) - p0.z, dz1 = ((GH && (w1 & 0x400)) ? az : ri.z) - p1.z;
                    const float d20 = __fmaf_rn(dz0, dz0, __fmaf_rn(dy0, dy0, dx0 * dx0));
                    const float d21 = __fmaf_rn(dz1, dz1, __fmaf_rn(dy1, dy1, dx1 * dx1));
                    const float t0 = one_type ? thr_one : thr_of[GH ? (w0 & 0xff) : w0];
                    const float t1 = one_type ? thr_one : thr_of[GH ? (w1 & 0xff) : w1];
                    // strict <, per type pair; bitwise &: both sides are always evaluated, no branch
                    const bool acc0 = (slot0 != self) & (d20 < t0), acc1 = (slot1 != self) & (d21 < t1);
                    const unsigned m0 = __ballot_sync(FULLMASK, acc0), m1 = __ballot_sync(FULLMASK, acc1);
                    const int k0 = count + __popc(m0 & lt), k1 = count + __popc(m0) + __popc(m1 & lt);
                    if (acc0 && k0 < rowcap) s_row[k0] = (unsigned short)(slot0 << 4);
                    if (acc1 && k1 < rowcap) s_row[k1] = (unsigned short)(slot1 << 4);
                    count += __popc(m0) + __popc(m1);
                }
                row0 = row1;
            }
            // close the row: pad the last chunk with the far-away dummy slot (the force loop needs no masks), then
            // the chunks go out as 16-byte stores, chunk c to (iteration c / tp, lane c % tp of the particle)
            const int i = g_first + p;
            const int kept = min(count, rowcap), nch = (kept + 7) >> 3;
            __syncwarp();
            if (kept + lane < nch * 8) s_row[kept + lane] = (unsigned short)(S.hcap << 4); // (at most 7 pads)
            __syncwarp();
            if (lane < nch || lane + 32 < nch) {
                const int v = pbase + (i - o0);
                const size_t base4 = (((size_t)(v >> S.ppw_shift) * S.cap_it8) << 5) + ((v & ((1 << S.ppw_shift) - 1)) << S.tp_shift);
                for (int c = lane; c < nch; c += 32)
                    list4[base4 + ((size_t)(c >> S.tp_shift) << 5) + (c & tmask)] = reinterpret_cast<const uint4*>(s_row)[c];
            }
            if (lane == 0) {
                S.num_nbrs[i] = kept;
                S.r_build[i] = ri;
                if (count > S.cap) S.sc->overflow = 1u;
            }
            wmax = max(wmax, count);
        }
    }
    if (lane == 0 && wmax > 0) atomicMax(max_slot, wmax);
}

// whole build of one tile by one block (halo layout, then the rows of the owned particles)
__device__ __forceinline__ void ph_build_tile(const Sys& S, const float4* r, int t, float4* s_pos, unsigned short* s_hstart,
                                              unsigned char* s_scratch, int* s_warp, const float* s_rcl2, int* max_slot)
{
    const TileGeo g = tile_geo(S, t);
    __syncthreads(); // the previous tile's rows are done with the shared arrays
    tile_layout_halo(S, r, t, g, s_pos, s_hstart, s_warp);
    if (tile_wrap_axes(S, g))
        tile_build_rows<true>(S, t, g, s_pos, s_hstart, s_scratch, s_rcl2, max_slot);
    else
        tile_build_rows<false>(S, t, g, s_pos, s_hstart, s_scratch, s_rcl2, max_slot);
}

// ------------------------------------------------------------------------------------------ A5 from shared memory
// P:110-171 Fig. 3 with the gathers served by shared memory.  One lane's share of a list row: per iteration ONE
// 16-byte load brings eight 16-bit slot numbers, eight LDS.128 fetch the positions, eight pairs are evaluated
// (the paper's one-ahead prefetch, P:108 item 4, eight deep).  Rows are padded with the far-away dummy slot, lanes
// that ran out of chunks read a chunk of dummies: no masks in the loop.  GH: some pair of this warp may be a
// periodic image -> the slot's ghost bits select between the particle's plain and half-shifted coordinate.
template <int COUL, bool ONE_TYPE, bool NC, bool ENERGY, bool GH>
__device__ __forceinline__ void tile_force_loop(const Sys& S, const float4* s_pos, const float4* s_pp, const uint4* chunks,
                                                int nch, int nch_w, const float4 ri, float& fx, float& fy, float& fz,
                                                float& u, float& w)
{
    const int trow = ONE_TYPE ? 0 : 4 * type_of(ri) * S.ntypes;
    float4 pf, pc, pe, px;
    pc = pe = px = make_float4(0.f, 0.f, 0.f, 0.f);
    if (ONE_TYPE) {
        pf = s_pp[0];
        if (COUL) pc = s_pp[1];
        if (ENERGY) pe = s_pp[2];
        if (COUL == 2) px = s_pp[3];
    }
    const float ax = half_shift(ri.x, S.h[0]), ay = half_shift(ri.y, S.h[1]), az = half_shift(ri.z, S.h[2]);
    // list entries are slot numbers times 16 (the byte offset of the slot: hcap <= 4095 keeps them in 16 bits)
    const unsigned dummy = (unsigned)(S.hcap << 4) * 0x00010001u;
    const unsigned char* sbase = reinterpret_cast<const unsigned char*>(s_pos);
    auto chunk = [&](int it) {
        uint4 e = make_uint4(dummy, dummy, dummy, dummy);
        if (it < nch) e = NC ? __ldg(chunks + (size_t)it * 32) : __ldcs(chunks + (size_t)it * 32);
        return e;
    };
    // two chunks in flight ahead of the one being worked on: the list streams from L2 / HBM
    uint4 e0 = chunk(0), e1 = chunk(1);
    for (int it = 0; it < nch_w; ++it) {
        const uint4 e = e0;
        e0 = e1;
        e1 = chunk(it + 2);
        const unsigned ew[4] = {e.x, e.y, e.z, e.w};
        float4 rj[8];
#pragma unroll
        for (int q = 0; q < 8; ++q)
            rj[q] = *reinterpret_cast<const float4*>(sbase + ((q & 1) ? (ew[q >> 1] >> 16) : (ew[q >> 1] & 0xffffu)));
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            const int wj = __float_as_int(rj[q].w);
            const float dx = ((GH && (wj & 0x100)) ? ax : ri.x) - rj[q].x;
            const float dy = ((GH && (wj & 0x200)) ? ay : ri.y) - rj[q].y;
            const float dz = ((GH && (wj & 0x400)) ? az : ri.z) - rj[q].z;
            if (!ONE_TYPE) {
                const int o = trow + 4 * (GH ? (wj & 0xff) : wj);
                pf = s_pp[o];
                if (COUL) pc = s_pp[o + 1];
                if (ENERGY) pe = s_pp[o + 2];
                if (COUL == 2) px = s_pp[o + 3];
            }
            pair_accumulate<COUL, ENERGY>(pf, pc, pe, px, true, dx, dy, dz, fx, fy, fz, u, w);
        }
    }
}

// Forces on the particles tile t owns (the block's warps take the tile's virtual warps of TP lanes per particle in
// turn); the halo must be in s_pos.  done(i, lead, ri, fx, fy, fz, u, w) is called by every lane with the particle's
// totals (u, w not yet halved); lead = this lane is lane 0 of an existing particle.
template <int TP, int COUL, bool ONE_TYPE, bool NC, bool ENERGY, class Done>
__device__ __forceinline__ void tile_force_own(const Sys& S, const float4* r, int t, const float4* s_pos, const float4* s_pp,
                                               Done&& done)
{
    const TileGeo g = tile_geo(S, t);
    const int o0 = S.cstart_z[g.cellbase], o1 = S.cstart_z[g.cellbase + g.wx * g.wy * g.wz];
    const bool gh_tile = tile_wrap_axes(S, g) != 0u;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
    const int nvw = ((o1 - o0) * TP + 31) >> 5;
    const size_t w0 = (size_t)(tile_pbase(o0, t) >> S.ppw_shift);
    for (int vw = wid; vw < nvw; vw += nw) {
        const int vt = vw * 32 + lane;
        const int i = o0 + vt / TP, tl = vt % TP;
        const bool have_i = i < o1;
        float4 ri = make_float4(0.f, 0.f, 0.f, 0.f);
        int nch = 0;
        if (have_i) {
            ri = load_pos<NC>(r + i);
            const int c = (S.num_nbrs[i] + 7) >> 3;          // chunks of the row; lane tl owns chunks tl, tl + TP, ...
            nch = max(0, (c - tl + TP - 1) / TP);
        }
        const int nch_w = __reduce_max_sync(FULLMASK, nch);
        const uint4* chunks = reinterpret_cast<const uint4*>(S.nbl) + (((w0 + vw) * S.cap_it8) << 5) + lane;
        float fx = 0.f, fy = 0.f, fz = 0.f, u = 0.f, w = 0.f;
        // a particle further than rc_max + 2 skin from every face has no listed neighbour across a face (O9)
        const bool interior = fabsf(ri.x) < S.hin[0] && fabsf(ri.y) < S.hin[1] && fabsf(ri.z) < S.hin[2];
        if (gh_tile && __any_sync(FULLMASK, have_i && !interior))
            tile_force_loop<COUL, ONE_TYPE, NC, ENERGY, true>(S, s_pos, s_pp, chunks, nch, nch_w, ri, fx, fy, fz, u, w);
        else
            tile_force_loop<COUL, ONE_TYPE, NC, ENERGY, false>(S, s_pos, s_pp, chunks, nch, nch_w, ri, fx, fy, fz, u, w);
#pragma unroll
        for (int o = TP / 2; o; o >>= 1) {
            fx += __shfl_xor_sync(FULLMASK, fx, o);
            fy += __shfl_xor_sync(FULLMASK, fy, o);
            fz += __shfl_xor_sync(FULLMASK, fz, o);
            if (ENERGY) {
                u += __shfl_xor_sync(FULLMASK, u, o);
                w += __shfl_xor_sync(FULLMASK, w, o);
            }
        }
        done(i, have_i && tl == 0, ri, fx, fy, fz, u, w);
    }
}

// ------------------------------------------------------------------------------------------ stand-alone kernels

// carve the dynamic shared memory of a tile kernel
__device__ __forceinline__ void tile_smem(const Sys& S, unsigned char* raw, float4*& s_pos, unsigned short*& s_hstart,
                                          unsigned char*& s_scratch)
{
    s_pos = reinterpret_cast<float4*>(raw);
    s_scratch = raw + (size_t)(S.hcap + 1) * 16;                                      // 16-byte aligned
    s_hstart = reinterpret_cast<unsigned short*>(s_scratch + (TILE_THREADS / 32) * TILE_WARP_SCRATCH);
}

// A5 of the tile method as its own kernel (rumd_compute_forces, the per-step path, rumd_time_force): one block per
// tile (the grid strides when it is smaller), forces / energies / virials of the owned particles into f, w.
template <int TP, int COUL, bool ONE_TYPE>
__global__ void __launch_bounds__(TILE_THREADS) k_force_tile(const Sys S)
{
    extern __shared__ __align__(16) unsigned char tile_raw[];
    __shared__ float4 s_pp[4 * RUMD_MAXT * RUMD_MAXT];
    float4* s_pos = reinterpret_cast<float4*>(tile_raw);
    load_pair_table(S, s_pp);
    if (blockIdx.x == 0 && threadIdx.x == 0) finish_rebuild(S);
    for (int t = blockIdx.x; t < S.ntiles; t += gridDim.x) {
        __syncthreads();
        tile_load_halo<true>(S, S.r, t, s_pos);
        __syncthreads();
        tile_force_own<TP, COUL, ONE_TYPE, true, true>(S, S.r, t, s_pos, s_pp,
            [&](int i, bool lead, const float4&, float fx, float fy, float fz, float u, float w) {
                if (lead) {
                    S.f[i] = make_float4(fx, fy, fz, 0.5f * u); // P:160 "compensate for double counting"
                    S.w[i] = 0.5f * w;
                }
            });
    }
}

#ifdef RUMD_MAIN_TU // non-template kernels: compiled once, in rumd_b200.cu
static __global__ void __launch_bounds__(TILE_THREADS) k_build_tile(const Sys S)
{
    if (!rebuild_requested(S)) return;
    extern __shared__ __align__(16) unsigned char tile_raw[];
    __shared__ float s_rcl2[RUMD_MAXT * RUMD_MAXT];
    __shared__ int s_warp[33];
    float4* s_pos;
    unsigned short* s_hstart;
    unsigned char* s_scratch;
    tile_smem(S, tile_raw, s_pos, s_hstart, s_scratch);
    if (threadIdx.x < RUMD_MAXT * RUMD_MAXT) s_rcl2[threadIdx.x] = S.pp[threadIdx.x].rcl2;
    for (int t = blockIdx.x; t < S.ntiles; t += gridDim.x)
        ph_build_tile(S, S.r, t, s_pos, s_hstart, s_scratch, s_warp, s_rcl2, max_slot_of(S));
}

// Row-major export of the tile method's list in SLOT numbering of the particles (inspection / parity tests): the
// tile of a particle follows from its position at the build, its entries are halo slots of that tile.
static __global__ void k_export_nbl_tile(const Sys S, int* count, int* list, int rowcap)
{
    const int i = blockIdx.x;
    int cx, cy, cz;
    cell_coords(S, S.r_build[i], cx, cy, cz);
    const int t = tile_index_of_cell(S, cx, cy, cz);
    const TileGeo g = tile_geo(S, t);
    const int v = tile_pbase(S.cstart_z[g.cellbase], t) + (i - S.cstart_z[g.cellbase]);
    const int c = S.num_nbrs[i];
    const unsigned short* l16 = reinterpret_cast<const unsigned short*>(S.nbl);
    if (threadIdx.x == 0) count[i] = c;
    for (int k = threadIdx.x; k < rowcap; k += blockDim.x)
        list[(size_t)i * rowcap + k] = k < c ? (S.halo_idx[(size_t)t * S.hcap + (l16[tile_entry_index(S, v, k)] >> 4)] & TILE_IDX_MASK) : -1;
}
#endif // RUMD_MAIN_TU
