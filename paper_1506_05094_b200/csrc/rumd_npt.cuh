// rumd_npt.cuh -- NPT integrator ("NPT [51]": Martyna, Tobias, Klein 1994, isotropic) on the per-step kernel
// path (sm_100a).  Product code: shares nothing with oracle/.
//
// The paper prints no equations of motion; reading S32 fixes them and their leap-frog form:
//     dr/dt = v + nu r,  dL/dt = nu L,  dv/dt = F/m - [xi + (1 + 3/g) nu] v,
//     dnu/dt = cP [ (1 + 3/g) sum m v^2 + W - 3 V P0 ],  cP = (2 pi / tau_P)^2 / ((g + 3) T0),
//     dxi/dt = w2 (sum m v^2 / (g T0) - 1)                                  (the thermostat of O7, on the particles)
// With a box that changes every step the box lengths cannot sit in the by-value parameter block: they live in
// DevScalars and every NPT kernel reads them from there.  A step is
//     (N^2 build if flag) -> k_force_npt (forces, u_i, w_i EVERY step: the virial drives the barostat)
//     -> k_npt_prepare (one block: W = sum w_i and sum m v(t-dt/2)^2 in a fixed order -> nu(t), friction and scale
//        factors, the next box)
//     -> k_integrate_npt (leap-frog update, r <- s r + dt sh v', wrap into the NEW box, displacement check)
//        whose last block advances xi, eta, nu and publishes the new box.
// Neighbour method: N^2 list or none (the cell grid of S17 is sized for a fixed box).  The list stays valid while
// every particle has moved less than 0.4 skin (not skin/2: the other 0.1 skin covers the change of the box since
// the build, which also raises the flag on its own when (L/L_build - 1)(rc_max + skin) exceeds 0.1 skin).
#pragma once
#include "rumd_force.cuh"

#ifdef RUMD_MAIN_TU
#define NPT_TP 8 // lanes per particle of the NPT force kernel

static __global__ void __launch_bounds__(128) k_build_n2_npt(const Sys S)
{
    if (!rebuild_requested(S)) return;
    __shared__ float4 tile[N2_TILE];
    __shared__ float s_rcl2[RUMD_MAXT * RUMD_MAXT];
    if (threadIdx.x < RUMD_MAXT * RUMD_MAXT) s_rcl2[threadIdx.x] = S.pp[threadIdx.x].rcl2;
    __syncthreads();
    const Box bx = box_of_doubles(S.sc->box);
    ph_build_n2<true>(S, S.r, tile, s_rcl2, blockIdx.x, gridDim.x, max_slot_of(S), &bx);
}

// A5 with the box read from device memory: NPT_TP lanes per particle stride its list row (any list layout, through
// nbl_index), or all particles with the "none" method; exact minimum image for every pair; energy and virial always.
template <int COUL, bool ONE_TYPE>
static __global__ void __launch_bounds__(256) k_force_npt(const Sys S)
{
    __shared__ float4 s_pp[4 * RUMD_MAXT * RUMD_MAXT];
    load_pair_table(S, s_pp);
    __syncthreads();
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        if (S.sc->flag != 0u)
            for (int k = 0; k < 3; ++k) S.sc->box_build[k] = S.sc->box[k]; // (the build that just ran used this box)
        finish_rebuild(S);
    }
    const Box bx = box_of_doubles(S.sc->box);
    const int tid = blockIdx.x * blockDim.x + threadIdx.x;
    const int i = tid / NPT_TP, t = tid % NPT_TP;
    const bool have_i = i < S.N;
    float4 ri = make_float4(0.f, 0.f, 0.f, 0.f);
    int cnt = 0;
    if (have_i) {
        ri = S.r[i];
        cnt = S.method == 2 ? S.N : S.num_nbrs[i];
    }
    const int trow = ONE_TYPE ? 0 : 4 * type_of(ri) * S.ntypes;
    float fx = 0.f, fy = 0.f, fz = 0.f, u = 0.f, w = 0.f;
    for (int k = t; k < cnt; k += NPT_TP) {
        const int j = S.method == 2 ? k : S.nbl[nbl_index(S, i, k)];
        const float4 rj = S.r[j];
        const float dx = min_image(ri.x, rj.x, bx.h[0], bx.invL[0]);
        const float dy = min_image(ri.y, rj.y, bx.h[1], bx.invL[1]);
        const float dz = min_image(ri.z, rj.z, bx.h[2], bx.invL[2]);
        const int o = ONE_TYPE ? 0 : trow + 4 * type_of(rj);
        pair_accumulate<COUL, true>(s_pp[o], COUL ? s_pp[o + 1] : make_float4(0.f, 0.f, 0.f, 0.f), s_pp[o + 2],
                                    COUL == 2 ? s_pp[o + 3] : make_float4(0.f, 0.f, 0.f, 0.f), j != i, dx, dy, dz, fx, fy,
                                    fz, u, w);
    }
#pragma unroll
    for (int o = NPT_TP / 2; o; o >>= 1) {
        fx += __shfl_xor_sync(FULLMASK, fx, o);
        fy += __shfl_xor_sync(FULLMASK, fy, o);
        fz += __shfl_xor_sync(FULLMASK, fz, o);
        u += __shfl_xor_sync(FULLMASK, u, o);
        w += __shfl_xor_sync(FULLMASK, w, o);
    }
    if (have_i && t == 0) {
        S.f[i] = make_float4(fx, fy, fz, 0.5f * u); // P:160 "compensate for double counting"
        S.w[i] = 0.5f * w;
    }
}

// fixed-order block sum of two doubles over 1024 threads (result in thread 0)
__device__ __forceinline__ void npt_block_sum2(double& a, double& b, double* s_a, double* s_b)
{
    a = warp_sum(a);
    b = warp_sum(b);
    if ((threadIdx.x & 31) == 0) {
        s_a[threadIdx.x >> 5] = a;
        s_b[threadIdx.x >> 5] = b;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        a = b = 0.0;
        for (int q = 0; q < (int)(blockDim.x >> 5); ++q) {
            a += s_a[q];
            b += s_b[q];
        }
    }
}

// Between the force evaluation and the leap-frog update: the two global sums the barostat needs, then every factor
// of this step (reading S32; same order of operations as the oracle).  One block.
static __global__ void __launch_bounds__(1024) k_npt_prepare(const Sys S)
{
    __shared__ double s_a[32], s_b[32];
    double W = 0.0, mv2 = 0.0;
    for (int i = threadIdx.x; i < S.N; i += blockDim.x) {
        W += (double)S.w[i];
        const float4 v = S.v[i];
        mv2 += (double)v.w * ((double)v.x * v.x + (double)v.y * v.y + (double)v.z * v.z);
    }
    npt_block_sum2(W, mv2, s_a, s_b);
    if (threadIdx.x == 0) {
        DevScalars* sc = S.sc;
        const double dt = S.dt_d, vol = sc->box[0] * sc->box[1] * sc->box[2];
        const double pos = S.cP * (W - 3.0 * vol * S.P0);
        const double nu = sc->nu_o + 0.5 * dt * pos;                                        // nu(t)
        const double nu_h = nu + 0.5 * dt * pos + 0.5 * dt * S.cP * (1.0 + 3.0 / S.g) * mv2; // strain rate of the drift
        const double gam = sc->xi + (1.0 + 3.0 / S.g) * nu;
        const double sh = exp(0.5 * nu_h * dt), s = sh * sh;
        sc->npt_a = (1.0 - 0.5 * gam * dt) / (1.0 + 0.5 * gam * dt);
        sc->npt_b = dt / (1.0 + 0.5 * gam * dt);
        sc->npt_s = s;
        sc->npt_sh = sh;
        sc->nu_t = nu;
        sc->vol_t = vol;
        sc->nu_o = nu + 0.5 * dt * pos; // the kinetic kick is added by the integrator's last block
        for (int k = 0; k < 3; ++k) sc->box_next[k] = s * sc->box[k];
        sc->W = W;
        if (!(W == W) || !(mv2 == mv2)) sc->nonfinite = 1;
    }
}

// A6 for NPT: v' = a v + b F/m, r' = s r + dt sh v', wrap into the new box, displacement check (0.4 skin, against
// the positions at the last build under the new box's minimum image); block sums -> step_tail, whose last block
// also advances nu and publishes the new box (S.npt branch).
static __global__ void __launch_bounds__(INT_THREADS) k_integrate_npt(const Sys S)
{
    const DevScalars* sc = S.sc;
    const float a = (float)sc->npt_a, b = (float)sc->npt_b, s = (float)sc->npt_s, dsh = (float)(S.dt_d * sc->npt_sh);
    const Box bn = box_of_doubles(sc->box_next);
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    double kt = 0.0, mv2 = 0.0;
    bool moved = false;
    if (i < S.N) {
        float4 r = S.r[i], v = S.v[i];
        const float4 f = S.f[i], rb = S.r_build[i];
        int4 im = S.image[i];
        const float m = v.w, bm = b / m;
        const float vx = __fmaf_rn(bm, f.x, a * v.x), vy = __fmaf_rn(bm, f.y, a * v.y), vz = __fmaf_rn(bm, f.z, a * v.z);
        const float hx = 0.5f * (v.x + vx), hy = 0.5f * (v.y + vy), hz = 0.5f * (v.z + vz);
        kt = 0.5 * (double)m * ((double)hx * hx + (double)hy * hy + (double)hz * hz);
        mv2 = (double)m * ((double)vx * vx + (double)vy * vy + (double)vz * vz);
        float x = __fmaf_rn(dsh, vx, s * r.x), y = __fmaf_rn(dsh, vy, s * r.y), z = __fmaf_rn(dsh, vz, s * r.z);
        const float nx = rintf(x * bn.invL[0]), ny = rintf(y * bn.invL[1]), nz = rintf(z * bn.invL[2]);
        x = __fmaf_rn(-nx, bn.L[0], x);
        y = __fmaf_rn(-ny, bn.L[1], y);
        z = __fmaf_rn(-nz, bn.L[2], z);
        im.x += (int)nx;
        im.y += (int)ny;
        im.z += (int)nz;
        const float dx = min_image(x, rb.x, bn.h[0], bn.invL[0]);
        const float dy = min_image(y, rb.y, bn.h[1], bn.invL[1]);
        const float dz = min_image(z, rb.z, bn.h[2], bn.invL[2]);
        moved = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, dx * dx)) > S.half_skin2; // (0.4 skin)^2 for NPT
        S.r[i] = make_float4(x, y, z, r.w);
        S.v[i] = make_float4(vx, vy, vz, m);
        S.image[i] = im;
    }
    step_tail<INT_THREADS / 32>(S, true, kt, mv2, moved, gridDim.x);
}
#endif // RUMD_MAIN_TU
