// rumd_force.cuh -- A5 pair force / energy / virial kernel and A6 integrator (sm_100a).
// Product code: shares nothing with oracle/.
#pragma once
#include "rumd_kernels.cuh"

// ------------------------------------------------------------------------------------------ pair function

// O3/O4/O5 for one listed pair: adds f_SF(r) d/r to (fx,fy,fz) and -- only when ENERGY -- u_SF to u and
// r f_SF to w (the halving of u and w is done once per particle).  Every term applies its own cutoff
// (S5, strict <, S3).  Branch-free: a warp almost never has all 32 pairs outside the cutoff, so the terms are
// computed for every pair and selected.  1/r^2 = MUFU.RCP(r^2) (1 ulp; the r^-14 force term amplifies it 7-fold
// to < 1e-6 relative per pair, two orders inside the 1e-4 rms|F| bar) and 1/r = MUFU.RSQ(r^2) (2 ulp; used
// only in the small shifted-force terms and the Coulomb term): no Newton steps.
//   pf = (12 c12, 6 c6, rc_lj^2, fc_lj)   pc = (a, rc_2^2, fc_2, -)   pe = (c12, c6, k0_lj, k0_2)
//   px = (-, kind of the second term, p1, p2)
// The second term (COUL instantiations) is Coulomb a/r or one of the other pair potentials of P:73: IPL
// a r^-n, Yukawa a exp(-r/b)/r, Gaussian core a exp(-(r/b)^2), Buckingham a exp(-r/b) - c/r^6; the kind is the
// same for all pairs of one type pair, so the switch diverges only between type pairs.
__device__ __forceinline__ float __frcp_approx(float x)
{
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// MUFU.RSQ alone: rsqrtf() wraps it in four instructions of denormal handling, and r^2 is never denormal here
__device__ __forceinline__ float __frsqrt_approx(float x)
{
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

template <int COUL, bool ENERGY>
__device__ __forceinline__ void pair_accumulate(const float4 pf, const float4 pc, const float4 pe, const float4 px, bool ok,
                                                float dx, float dy, float dz, float& fx, float& fy, float& fz,
                                                float& u, float& w)
{
    const float r2 = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, dx * dx));
    const float y = __frsqrt_approx(r2);
    const float rinv2 = __frcp_approx(r2);
    const float rinv6 = rinv2 * rinv2 * rinv2;
    const float r = r2 * y;
    const bool in_lj = ok && r2 < pf.z;
    // f_SF / r = (12 c12 r^-12 - 6 c6 r^-6) r^-2 - fc / r
    float fr = __fmaf_rn(rinv6 * rinv2, __fmaf_rn(pf.x, rinv6, -pf.y), -pf.w * y);
    fr = in_lj ? fr : 0.f;
    float uu = 0.f;
    if (ENERGY) { // u_SF = c12 r^-12 - c6 r^-6 + fc r - k0
        uu = __fmaf_rn(rinv6, __fmaf_rn(pe.x, rinv6, -pe.y), __fmaf_rn(pf.w, r, -pe.z));
        uu = in_lj ? uu : 0.f;
    }
    if (COUL) {
        const bool in_c = ok && r2 < pc.y;
        float ux, fx_r; // raw u and f / r of the second term
        switch (COUL == 1 ? 0 : __float_as_int(px.y)) { // COUL == 1: every second term is Coulomb, no switch
        default: // Coulomb: u = a / r
            ux = pc.x * y;
            fx_r = ux * rinv2;
            break;
        case 1: // inverse power law: u = a r^-n, n = p1
            ux = pc.x * exp2f(-0.5f * px.z * __log2f(r2));
            fx_r = px.z * ux * rinv2;
            break;
        case 2: // Yukawa: u = a exp(-r / b) / r, p1 = 1 / b;  f = u (1/r + 1/b)
            ux = pc.x * __expf(-r * px.z) * y;
            fx_r = ux * (y + px.z) * y;
            break;
        case 3: // Gaussian core: u = a exp(-(r/b)^2), p1 = 1 / b^2;  f = 2 r u / b^2
            ux = pc.x * __expf(-r2 * px.z);
            fx_r = 2.0f * px.z * ux;
            break;
        case 4: { // Buckingham: u = a exp(-r / b) - c r^-6, p1 = 1 / b, p2 = c;  f = (a/b) e^(-r/b) - 6 c r^-7
            const float e = pc.x * __expf(-r * px.z), c6 = px.w * rinv6;
            ux = e - c6;
            fx_r = __fmaf_rn(e * px.z, r, -6.0f * c6) * rinv2;
            break;
        }
        case 5: { // generalized LJ: u = A r^-m - B r^-n, m = p1, n = p2, B in the (unused) 12-6 slot pf.x
            const float l = -0.5f * __log2f(r2);
            const float tm = pc.x * exp2f(px.z * l), tn = pf.x * exp2f(px.w * l);
            ux = tm - tn;
            fx_r = __fmaf_rn(px.z, tm, -px.w * tn) * rinv2;
            break;
        }
        case 6: { // Girifalco: s = r / d (p2 = 1 / d), alpha = a, beta = p1; f = -(1/d) du/ds
            const float s = r * px.w, is = __frcp_approx(s), im = __frcp_approx(s - 1.0f), ip = __frcp_approx(s + 1.0f);
            const float is2 = is * is, is4 = is2 * is2, im3 = im * im * im, ip3 = ip * ip * ip;
            const float im9 = im3 * im3 * im3, ip9 = ip3 * ip3 * ip3, is10 = is4 * is4 * is2;
            ux = -pc.x * __fmaf_rn(is, im3 + ip3, -2.0f * is4) + px.z * __fmaf_rn(is, im9 + ip9, -2.0f * is10);
            const float d3 = is2 * ((4.0f * s - 1.0f) * im3 * im + (4.0f * s + 1.0f) * ip3 * ip) - 8.0f * is4 * is;
            const float d9 = is2 * ((10.0f * s - 1.0f) * im9 * im + (10.0f * s + 1.0f) * ip9 * ip) - 20.0f * is10 * is;
            fx_r = (px.z * d9 - pc.x * d3) * px.w * y; // -du/ds = beta d9 - alpha d3
            break;
        }
        case 7: { // Dzugutov: x = r / sigma (p1 = 1 / sigma); both pieces vanish with all derivatives at their edge
            const float x = r * px.z, ix2 = __frcp_approx(x * x), ix4 = ix2 * ix2, ix8 = ix4 * ix4, ix16 = ix8 * ix8;
            const float t1 = __frcp_approx(fminf(x - (float)DZ_a, -1e-6f)), t2 = __frcp_approx(fminf(x - (float)DZ_b, -1e-6f));
            const float e1 = x < (float)DZ_a ? (float)DZ_A * __expf((float)DZ_c * t1) : 0.f;
            const float e2 = x < (float)DZ_b ? (float)DZ_B * __expf((float)DZ_d * t2) : 0.f;
            const float g = ix16 - (float)DZ_B;
            ux = pc.x * __fmaf_rn(g, e1, e2);
            const float du = e1 * (-16.0f * ix16 * x * ix2 - g * (float)DZ_c * t1 * t1) - e2 * (float)DZ_d * t2 * t2;
            fx_r = -pc.x * du * px.z * y;
            break;
        }
        }
        fr += in_c ? __fmaf_rn(-pc.z, y, fx_r) : 0.f;                     // f / r - fc / r
        if (ENERGY) uu += in_c ? ux + __fmaf_rn(pc.z, r, -pe.w) : 0.f; // u + fc r - k0
    }
    fx = __fmaf_rn(fr, dx, fx);
    fy = __fmaf_rn(fr, dy, fy);
    fz = __fmaf_rn(fr, dz, fz);
    if (ENERGY) {
        u += uu;
        w = __fmaf_rn(fr, r2, w);
    }
}

// ------------------------------------------------------------------------------------------ A5: forces

// P:110-171 Fig. 3 (`Calcf_NBL_tp`): TP threads per particle stride the particle's neighbour row
// (P:143 `i = MyT; i += TPerPart`), positions gathered through the read-only path (P:165 LOAD()), partial
// sums reduced -- here by warp shuffles inside the TP-lane group instead of shared memory + __syncthreads
// --, lane 0 halves the energy.  Lane = (particle-in-warp)*TP + t; UNROLL listed pairs
// per lane are in flight at once (the paper's one-ahead index prefetch, P:108 item 4, generalised).
//
// force_group: the partial sums of one lane, then the butterfly over its TP-lane group; on return every lane
// of the group holds the particle's totals (u and w NOT yet halved; only computed when ENERGY).  vwarp =
// index of this warp in the virtual grid of N*TP threads.  NC = true: list and positions are read-only for
// the whole kernel, loads go through ld.global.nc; NC = false (persistent kernel, which rewrites both):
// coherent loads, the index stream marked evict-first.  All 32 lanes of the warp must call.
//
// Minimum image: a particle further than rc_max + 2 skin from every face of the box cannot have a listed
// neighbour across a periodic boundary (the pair was within rc + skin at the build and neither particle has
// moved more than skin/2 since, O9), so when this holds for ALL particles of the warp (WRAP = false) the
// displacement is the plain difference; otherwise the exact shifted form of min_image is used.
template <bool NC> __device__ __forceinline__ int load_idx(const int* p) { return NC ? __ldg(p) : __ldcs(p); }
template <bool NC> __device__ __forceinline__ float4 load_pos(const float4* p) { return NC ? __ldg(p) : *p; }

// PRE: the index loads of iteration 0 were issued by the caller before it knew the row length (jpre)
// TWO: the system has exactly two particle types and COUL < 2 (Kob-Andersen, the charged mixture): the two parameter
// records a lane can need -- (type of i, 0) and (type of i, 1) -- sit in registers and each pair SELECTS between them by
// its neighbour's type.  The table lookup it replaces costs one LDS.128 per record and pair, i.e. four cycles of the
// SM's load/store data path each, as many as the position gather itself needs at best (ncu: that path, not FP32
// issue, bounds the kernel); a select is one ALU instruction per register.
template <int TP, int COUL, bool ONE_TYPE, int UNROLL, bool NC, bool ENERGY, bool WRAP, bool MASKED, bool PRE = false, bool TWO = false>
__device__ __forceinline__ void force_loop(const Sys& S, const float4* r, const float4* s_pp, const int* base,
                                           int it_begin, int nit, int it_end, const float4 ri, float& fx, float& fy,
                                           float& fz, float& u, float& w, const int* jpre = nullptr)
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
    float4 pf0, pc0, pe0, pf1, pc1, pe1; // TWO: records of (type of i, 0) and (type of i, 1)
    pf0 = pc0 = pe0 = pf1 = pc1 = pe1 = make_float4(0.f, 0.f, 0.f, 0.f);
    if (TWO) {
        pf0 = s_pp[trow];
        pf1 = s_pp[trow + 4];
        if (COUL) {
            pc0 = s_pp[trow + 1];
            pc1 = s_pp[trow + 5];
        }
        if (ENERGY) {
            pe0 = s_pp[trow + 2];
            pe1 = s_pp[trow + 6];
        }
    }
    const float hx = S.h[0], hy = S.h[1], hz = S.h[2];
    const float ix = S.invL[0], iy = S.invL[1], iz = S.invL[2];
    for (int it = it_begin; it < it_end; it += UNROLL) {
        int j[UNROLL];
        bool ok[UNROLL];
        float4 rj[UNROLL];
#pragma unroll
        for (int q = 0; q < UNROLL; ++q) {
            ok[q] = !MASKED || (it + q) < nit;
            if (PRE && it == 0)
                j[q] = ok[q] ? jpre[q] : 0;
            else
                j[q] = ok[q] ? load_idx<NC>(base + (size_t)(it + q) * 32) : 0; // masked lanes gather slot 0 (always valid)
        }
#pragma unroll
        for (int q = 0; q < UNROLL; ++q) rj[q] = load_pos<NC>(&r[j[q]]);
#pragma unroll
        for (int q = 0; q < UNROLL; ++q) {
            float dx, dy, dz;
            if (WRAP) {
                dx = min_image(ri.x, rj[q].x, hx, ix);
                dy = min_image(ri.y, rj[q].y, hy, iy);
                dz = min_image(ri.z, rj[q].z, hz, iz);
            } else {
                dx = ri.x - rj[q].x;
                dy = ri.y - rj[q].y;
                dz = ri.z - rj[q].z;
            }
            if (TWO) {
                const bool b = type_of(rj[q]) != 0;
                pf = make_float4(b ? pf1.x : pf0.x, b ? pf1.y : pf0.y, b ? pf1.z : pf0.z, b ? pf1.w : pf0.w);
                if (COUL) pc = make_float4(b ? pc1.x : pc0.x, b ? pc1.y : pc0.y, b ? pc1.z : pc0.z, 0.f);
                if (ENERGY) pe = make_float4(b ? pe1.x : pe0.x, b ? pe1.y : pe0.y, b ? pe1.z : pe0.z, b ? pe1.w : pe0.w);
            } else if (!ONE_TYPE) {
                const int o = trow + 4 * type_of(rj[q]);
                pf = s_pp[o];
                if (COUL) pc = s_pp[o + 1];
                if (ENERGY) pe = s_pp[o + 2];
                if (COUL == 2) px = s_pp[o + 3];
            }
            pair_accumulate<COUL, ENERGY>(pf, pc, pe, px, ok[q], dx, dy, dz, fx, fy, fz, u, w);
        }
    }
}

template <int TP, int COUL, bool ONE_TYPE, int UNROLL, bool NC, bool ENERGY>
__device__ __forceinline__ void force_group(const Sys& S, const float4* r, const float4* s_pp, int vwarp, int i,
                                            int t, bool have_i, const float4 ri, int cnt, float& fx, float& fy,
                                            float& fz, float& u, float& w)
{
    const int lane = threadIdx.x & 31;
    const int* base = S.nbl + (size_t)vwarp * S.cap_it * 32 + lane;
    // Small systems (wide lane groups, persistent kernel): a time step is a chain of dependent L2 round trips, so the
    // first UNROLL list entries of every lane are requested BEFORE the row length is known (the row is allocated up
    // to the capacity; what lies beyond the length is masked below and never dereferenced).
    constexpr bool PRE = TP >= 8 && !NC;
    int jpre[UNROLL];
    if (PRE) {
#pragma unroll
        for (int q = 0; q < UNROLL; ++q) jpre[q] = q < S.cap_it ? load_idx<NC>(base + (size_t)q * 32) : 0;
    }
    int nit = (cnt - t + TP - 1) / TP; // entries t, t+TP, ... < cnt
    if (nit < 0) nit = 0;
    const int nit_w = __reduce_max_sync(FULLMASK, nit);
    fx = fy = fz = u = w = 0.f;
    // iterations every lane of the warp has (no masks needed), then the ragged tail
    const int nit_all = __reduce_min_sync(FULLMASK, have_i ? nit : 0) / UNROLL * UNROLL;
    const bool interior = fabsf(ri.x) < S.hin[0] && fabsf(ri.y) < S.hin[1] && fabsf(ri.z) < S.hin[2];
    const bool wrap = __any_sync(FULLMASK, have_i && !interior);
    constexpr bool CAN2 = !ONE_TYPE && COUL < 2; // two-type systems: parameter records in registers (force_loop, TWO)
    if (CAN2 && S.ntypes == 2) {
        if (wrap) {
            force_loop<TP, COUL, ONE_TYPE, UNROLL, NC, ENERGY, true, false, PRE, CAN2>(S, r, s_pp, base, 0, nit, nit_all, ri, fx, fy, fz, u, w, jpre);
            force_loop<TP, COUL, ONE_TYPE, UNROLL, NC, ENERGY, true, true, PRE, CAN2>(S, r, s_pp, base, nit_all, nit, nit_w, ri, fx, fy, fz, u, w, jpre);
        } else {
            force_loop<TP, COUL, ONE_TYPE, UNROLL, NC, ENERGY, false, false, PRE, CAN2>(S, r, s_pp, base, 0, nit, nit_all, ri, fx, fy, fz, u, w, jpre);
            force_loop<TP, COUL, ONE_TYPE, UNROLL, NC, ENERGY, false, true, PRE, CAN2>(S, r, s_pp, base, nit_all, nit, nit_w, ri, fx, fy, fz, u, w, jpre);
        }
    } else if (wrap) {
        force_loop<TP, COUL, ONE_TYPE, UNROLL, NC, ENERGY, true, false, PRE>(S, r, s_pp, base, 0, nit, nit_all, ri, fx, fy, fz, u, w, jpre);
        force_loop<TP, COUL, ONE_TYPE, UNROLL, NC, ENERGY, true, true, PRE>(S, r, s_pp, base, nit_all, nit, nit_w, ri, fx, fy, fz, u, w, jpre);
    } else {
        force_loop<TP, COUL, ONE_TYPE, UNROLL, NC, ENERGY, false, false, PRE>(S, r, s_pp, base, 0, nit, nit_all, ri, fx, fy, fz, u, w, jpre);
        force_loop<TP, COUL, ONE_TYPE, UNROLL, NC, ENERGY, false, true, PRE>(S, r, s_pp, base, nit_all, nit, nit_w, ri, fx, fy, fz, u, w, jpre);
    }
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
}

// P:371 "none" method: no neighbour list, lane t of the particle's TP lanes takes particles j = t, t + TP, ...
// of the WHOLE system (coalesced position loads), exact minimum image for every pair, self pair masked.  O(N^2)
// pair evaluations per step, but no list, no rebuilds and no index stream: wins for the smallest systems.
template <int TP, int COUL, bool ONE_TYPE, bool NC, bool ENERGY>
__device__ __forceinline__ void force_group_all(const Sys& S, const float4* r, const float4* s_pp, int i, int t,
                                                bool have_i, const float4 ri, float& fx, float& fy, float& fz,
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
    fx = fy = fz = u = w = 0.f;
    const float hx = S.h[0], hy = S.h[1], hz = S.h[2];
    const float ix = S.invL[0], iy = S.invL[1], iz = S.invL[2];
    constexpr int U = 4;
    for (int j0 = t; j0 < S.N; j0 += U * TP) {
        float4 rj[U];
        bool ok[U];
#pragma unroll
        for (int q = 0; q < U; ++q) {
            const int j = j0 + q * TP;
            ok[q] = have_i && j < S.N && j != i;
            rj[q] = load_pos<NC>(&r[j < S.N ? j : 0]);
        }
#pragma unroll
        for (int q = 0; q < U; ++q) {
            const float dx = min_image(ri.x, rj[q].x, hx, ix);
            const float dy = min_image(ri.y, rj[q].y, hy, iy);
            const float dz = min_image(ri.z, rj[q].z, hz, iz);
            if (!ONE_TYPE) {
                const int o = trow + 4 * type_of(rj[q]);
                pf = s_pp[o];
                if (COUL) pc = s_pp[o + 1];
                if (ENERGY) pe = s_pp[o + 2];
                if (COUL == 2) px = s_pp[o + 3];
            }
            pair_accumulate<COUL, ENERGY>(pf, pc, pe, px, ok[q], dx, dy, dz, fx, fy, fz, u, w);
        }
    }
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
}

// forces of one particle by whichever method is configured (warp-uniform choice)
template <int TP, int COUL, bool ONE_TYPE, int UNROLL, bool NC, bool ENERGY>
__device__ __forceinline__ void force_any(const Sys& S, const float4* r, const float4* s_pp, int vwarp, int i, int t,
                                          bool have_i, const float4 ri, int cnt, float& fx, float& fy, float& fz,
                                          float& u, float& w)
{
    if (S.method == 2)
        force_group_all<TP, COUL, ONE_TYPE, NC, ENERGY>(S, r, s_pp, i, t, have_i, ri, fx, fy, fz, u, w);
    else
        force_group<TP, COUL, ONE_TYPE, UNROLL, NC, ENERGY>(S, r, s_pp, vwarp, i, t, have_i, ri, cnt, fx, fy, fz, u, w);
}

// the pair table in shared memory: record of the ordered pair (a, b) at 4*(a*ntypes + b) (four float4)
__device__ __forceinline__ void load_pair_table(const Sys& S, float4* s_pp)
{
    const float4* src = reinterpret_cast<const float4*>(S.pp);
    for (int q = threadIdx.x; q < 4 * S.ntypes * S.ntypes; q += blockDim.x) s_pp[q] = src[q];
}

// Bookkeeping that must happen once per step AFTER every rebuild kernel has read the flag: count the
// rebuild, clear the flag and zero the max-length slot of the NEXT build.  1-thread tail of k_force.
__device__ __forceinline__ void finish_rebuild(const Sys& S)
{
    if (S.sc->flag != 0u) {
        if (S.method != 2) { // (the "none" method has no list: nothing was built)
            S.sc->last_max = S.sc->max_nbrs[S.sc->n_rebuilds & 1];
            S.sc->n_rebuilds += 1;
            S.sc->max_nbrs[S.sc->n_rebuilds & 1] = 0;
        }
        S.sc->flag = 0u;
    }
}

// The grid is sized to what is co-resident (a whole number of blocks per SM) and the N*TP/32 warps of work are cut
// into gridDim.x contiguous, equally long runs: no partial last wave (at N = 65536 the one-thread-per-lane grid was
// 1.7 waves), neighbouring particles stay on one SM.
template <int TP, int COUL, bool ONE_TYPE, int UNROLL>
__global__ void __launch_bounds__(1024, 1) k_force(const Sys S)
{
    __shared__ float4 s_pp[4 * RUMD_MAXT * RUMD_MAXT];
    load_pair_table(S, s_pp);
    __syncthreads();
    if (blockIdx.x == 0 && threadIdx.x == 0) finish_rebuild(S);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
    const long long nvwarps = ((long long)S.N * TP + 31) / 32;
    const long long vw0 = nvwarps * blockIdx.x / gridDim.x, vw1 = nvwarps * (blockIdx.x + 1) / gridDim.x;
    for (long long vw = vw0 + wid; vw < vw1; vw += nw) {
        const long long tid = vw * 32 + lane;
        const int i = (int)(tid / TP);
        const int t = (int)(tid % TP);
        const bool have_i = i < S.N;
        float4 ri = make_float4(0.f, 0.f, 0.f, 0.f);
        int cnt = 0;
        if (have_i) {
            ri = __ldg(&S.r[i]);
            cnt = S.method == 2 ? 0 : S.num_nbrs[i];
        }
        float fx, fy, fz, u, w;
        force_any<TP, COUL, ONE_TYPE, UNROLL, true, true>(S, S.r, s_pp, (int)vw, i, t, have_i, ri, cnt, fx, fy, fz, u, w);
        if (have_i && t == 0) {
            S.f[i] = make_float4(fx, fy, fz, 0.5f * u); // P:160 "compensate for double counting"
            S.w[i] = 0.5f * w;
        }
    }
}

// ------------------------------------------------------------------------------------------ A6: integrator

// O6 / O7 leap-frog step for one particle + wrap (S7) + displacement check (O9, S14).  Returns through
// kt / mv2 the particle's contributions to K(t) (O10) and sum m v(t+dt/2)^2.
//   NVE: a = 1, b = dt.   NVT: a = (1 - xi dt/2)/(1 + xi dt/2), b = dt/(1 + xi dt/2)  (O7 rearranged).
__device__ __forceinline__ void integrate_particle(const Sys& S, float a, float b, float4& r, float4& v,
                                                   const float4 f, int4& im, const float4 rb, bool& moved,
                                                   double& kt, double& mv2)
{
    const float m = v.w;
    const float bm = b / m;
    const float vx = __fmaf_rn(bm, f.x, a * v.x);
    const float vy = __fmaf_rn(bm, f.y, a * v.y);
    const float vz = __fmaf_rn(bm, f.z, a * v.z);
    const float hx = 0.5f * (v.x + vx), hy = 0.5f * (v.y + vy), hz = 0.5f * (v.z + vz);
    kt = 0.5 * (double)m * ((double)hx * hx + (double)hy * hy + (double)hz * hz);
    mv2 = (double)m * ((double)vx * vx + (double)vy * vy + (double)vz * vz);
    v.x = vx;
    v.y = vy;
    v.z = vz;
    float x = __fmaf_rn(S.dt, vx, r.x), y = __fmaf_rn(S.dt, vy, r.y), z = __fmaf_rn(S.dt, vz, r.z);
    // (tile method: no wrap between rebuilds, see ph_cell_assign)
    const bool wrap = S.method != 3;
    const float nx = wrap ? rintf(x * S.invL[0]) : 0.f, ny = wrap ? rintf(y * S.invL[1]) : 0.f,
                nz = wrap ? rintf(z * S.invL[2]) : 0.f;
    x = __fmaf_rn(-nx, S.L[0], x);
    y = __fmaf_rn(-ny, S.L[1], y);
    z = __fmaf_rn(-nz, S.L[2], z);
    im.x += (int)nx;
    im.y += (int)ny;
    im.z += (int)nz;
    r.x = x;
    r.y = y;
    r.z = z;
    const float dx = min_image(x, rb.x, S.h[0], S.invL[0]);
    const float dy = min_image(y, rb.y, S.h[1], S.invL[1]);
    const float dz = min_image(z, rb.z, S.h[2], S.invL[2]);
    moved = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, dx * dx)) > S.half_skin2; // strict > (S14)
}

__device__ __forceinline__ void nvt_factors(const Sys& S, bool nvt, float& a, float& b)
{
    if (nvt) {
        const double hx = 0.5 * S.sc->xi * S.dt_d;
        a = (float)((1.0 - hx) / (1.0 + hx));
        b = (float)(S.dt_d / (1.0 + hx));
    } else {
        a = 1.0f;
        b = S.dt;
    }
}

// Block-level tail shared by the split and the fused step kernels: fp64 block sums of (kt, mv2) ->
// partial[], then the LAST block to arrive (ticket) adds the partials in a fixed order, advances the
// thermostat (O7: xi += dt w^2 (T_kin/T0 - 1), eta += dt/2 (xi_old + xi_new)), publishes K, and turns this
// step's displacement result into the rebuild flag of the next step.  No host involvement.
template <int MAXWARPS>
__device__ __forceinline__ void step_tail(const Sys& S, bool nvt, double kt, double mv2, bool moved,
                                          int nblocks)
{
    __shared__ double s_k[MAXWARPS], s_m[MAXWARPS];
    __shared__ int s_moved;
    __shared__ bool s_last;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
    if (threadIdx.x == 0) s_moved = 0;
    __syncthreads();
    kt = warp_sum(kt);
    mv2 = warp_sum(mv2);
    if (__any_sync(FULLMASK, moved) && lane == 0) s_moved = 1;
    if (lane == 0) {
        s_k[wid] = kt;
        s_m[wid] = mv2;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        double a = 0.0, b = 0.0;
        for (int q = 0; q < nw; ++q) {
            a += s_k[q];
            b += s_m[q];
        }
        S.partial[2 * blockIdx.x] = a;
        S.partial[2 * blockIdx.x + 1] = b;
        if (s_moved) S.sc->pending = 1u;
        __threadfence();
        const unsigned tk = atomicAdd(&S.sc->ticket, 1u);
        s_last = (tk == (unsigned)nblocks - 1u);
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    double a = 0.0, b = 0.0;
    for (int q = threadIdx.x; q < nblocks; q += blockDim.x) {
        a += __ldcg(&S.partial[2 * q]);
        b += __ldcg(&S.partial[2 * q + 1]);
    }
    a = warp_sum(a);
    b = warp_sum(b);
    if (lane == 0) {
        s_k[wid] = a;
        s_m[wid] = b;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        a = 0.0;
        b = 0.0;
        for (int q = 0; q < nw; ++q) {
            a += s_k[q];
            b += s_m[q];
        }
        DevScalars* sc = S.sc;
        sc->K = a;
        sc->mv2 = b;
        if (nvt) {
            const double xi = sc->xi;
            const double xin = xi + S.dt_d * S.omega2 * (b / S.g / S.T0 - 1.0);
            sc->xi_t = xi;
            sc->eta_t = sc->eta;
            sc->eta += 0.5 * S.dt_d * (xi + xin);
            sc->xi = xin;
        }
        sc->n_steps += 1;
        unsigned pend = *((volatile unsigned*)&sc->pending);
        if (S.npt) { // rumd_npt.cuh: the kinetic kick of the strain rate, the new box, and the guards that go with it
            sc->nu_o += S.dt_d * S.cP * (1.0 + 3.0 / S.g) * b;
            double lmin = sc->box_next[0];
            for (int k = 0; k < 3; ++k) {
                // the list tolerates 0.1 skin of box change since its build (the displacement test uses 0.4 skin)
                if (fabs(sc->box_next[k] / sc->box_build[k] - 1.0) * (double)S.rcl_max > 0.1 * (double)S.skin) pend = 1u;
                sc->box[k] = sc->box_next[k];
                lmin = fmin(lmin, sc->box_next[k]);
            }
            if ((double)S.rcl_max > 0.5 * lmin) sc->nonfinite = 3; // the box shrank below 2 (rc_max + skin), O1
        }
        sc->flag = pend;
        sc->pending = 0u;
        sc->ticket = 0u;
        if (!(a == a) || !(b == b)) sc->nonfinite = 1;
    }
}

#define INT_THREADS 128
#ifdef RUMD_MAIN_TU // non-template kernels: compiled once, in rumd_b200.cu
static __global__ void __launch_bounds__(INT_THREADS) k_integrate(const Sys S, int nvt)
{
    float a, b;
    nvt_factors(S, nvt != 0, a, b);
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    double kt = 0.0, mv2 = 0.0;
    bool moved = false;
    if (i < S.N) {
        float4 r = S.r[i], v = S.v[i];
        int4 im = S.image[i];
        integrate_particle(S, a, b, r, v, S.f[i], im, S.r_build[i], moved, kt, mv2);
        S.r[i] = r;
        S.v[i] = v;
        S.image[i] = im;
    }
    step_tail<INT_THREADS / 32>(S, nvt != 0, kt, mv2, moved, gridDim.x);
}
#endif // RUMD_MAIN_TU

// A5 + A6 fused for the per-step path: forces of r(t) read from S.r, leap-frog update written to S.r_out
// (the OTHER position buffer: nobody reads a position that was already advanced), then the same block tail as
// k_integrate.  Saves the integrator's pass over r, v, f (~112 B per particle) and one launch per step.
// ENERGY: also write f, u, w (the step whose force evaluation is an output of the run).
template <int TP, int COUL, bool ONE_TYPE, int UNROLL, bool ENERGY>
__global__ void __launch_bounds__(1024, 1) k_step(const Sys S, int nvt)
{
    __shared__ float4 s_pp[4 * RUMD_MAXT * RUMD_MAXT];
    load_pair_table(S, s_pp);
    __syncthreads();
    if (blockIdx.x == 0 && threadIdx.x == 0) finish_rebuild(S);
    float a, b;
    nvt_factors(S, nvt != 0, a, b);
    const int tid = blockIdx.x * blockDim.x + threadIdx.x;
    const int i = tid / TP;
    const int t = tid % TP;
    const bool have_i = i < S.N;
    float4 ri = make_float4(0.f, 0.f, 0.f, 0.f);
    int cnt = 0;
    if (have_i) {
        ri = __ldg(&S.r[i]);
        cnt = S.method == 2 ? 0 : S.num_nbrs[i];
    }
    float fx, fy, fz, u, w;
    force_any<TP, COUL, ONE_TYPE, UNROLL, true, ENERGY>(S, S.r, s_pp, tid >> 5, i, t, have_i, ri, cnt, fx, fy, fz, u, w);
    double kt = 0.0, mv2 = 0.0;
    bool moved = false;
    if (have_i && t == 0) {
        const float4 f = make_float4(fx, fy, fz, 0.5f * u);
        float4 v = S.v[i];
        int4 im = S.image[i];
        integrate_particle(S, a, b, ri, v, f, im, S.r_build[i], moved, kt, mv2);
        S.r_out[i] = ri;
        S.v[i] = v;
        S.image[i] = im;
        if (ENERGY) {
            S.f[i] = f;
            S.w[i] = 0.5f * w;
        }
    }
    step_tail<32>(S, nvt != 0, kt, mv2, moved, gridDim.x);
}

// ------------------------------------------------------------------------------------------ small kernels

#ifdef RUMD_MAIN_TU // non-template kernels: compiled once, in rumd_b200.cu
static __global__ void k_request_rebuild(const Sys S)
{
    S.sc->flag = 1u;
    S.sc->pending = 0u;
    S.sc->max_nbrs[S.sc->n_rebuilds & 1] = 0;
    S.sc->overflow = 0u;
}

static __global__ void k_reset_scalars(const Sys S)
{
    DevScalars z;
    memset(&z, 0, sizeof(z));
    z.flag = 1u;
    for (int k = 0; k < 3; ++k) z.box[k] = z.box_next[k] = z.box_build[k] = (double)S.L[k];
    *S.sc = z;
}

// U = sum u_i, W = sum w_i in fp64, fixed order (single block).
static __global__ void __launch_bounds__(1024) k_thermo(const Sys S)
{
    __shared__ double s_u[32], s_w[32];
    double u = 0.0, w = 0.0;
    for (int i = threadIdx.x; i < S.N; i += blockDim.x) {
        u += (double)S.f[i].w;
        w += (double)S.w[i];
    }
    u = warp_sum(u);
    w = warp_sum(w);
    if ((threadIdx.x & 31) == 0) {
        s_u[threadIdx.x >> 5] = u;
        s_w[threadIdx.x >> 5] = w;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        u = 0.0;
        w = 0.0;
        for (int q = 0; q < 32; ++q) {
            u += s_u[q];
            w += s_w[q];
        }
        S.sc->U = u;
        S.sc->W = w;
        if (!(u == u) || !(w == w)) S.sc->nonfinite = 1;
    }
}

// Row-major export of the tiled list (inspection / parity tests).
static __global__ void k_export_nbl(const Sys S, int* count, int* list, int rowcap)
{
    const int i = blockIdx.x;
    const int c = S.method == 2 ? 0 : S.num_nbrs[i]; // the "none" method keeps no list
    if (threadIdx.x == 0) count[i] = c;
    for (int k = threadIdx.x; k < rowcap; k += blockDim.x)
        list[(size_t)i * rowcap + k] = k < c ? S.nbl[nbl_index(S, i, k)] : -1;
}

// snapshot / restore of (r, v, image, id)
static __global__ void k_copy_state(int N, const float4* r, const float4* v, const int4* im, const int* id, float4* r2,
                             float4* v2, int4* im2, int* id2)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    r2[i] = r[i];
    v2[i] = v[i];
    im2[i] = im[i];
    id2[i] = id[i];
}
#endif // RUMD_MAIN_TU
