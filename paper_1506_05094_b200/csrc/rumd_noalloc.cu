// rumd_noalloc.cu -- rumd_forces_noalloc: ONE force / energy / virial evaluation (Fig. 3, O5) that allocates
// nothing.  Product code: shares nothing with oracle/.
//
// Why.  The handle API wants a caller-owned workspace (neighbour list P:101 / P:167, positions at build P:217,
// reduction partials) and rumd_create allocates pinned scalars and events.  Callers that cannot allocate at all -- code
// under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc -- get this variant of the pair-force
// kernel instead: the same N^2 list build (ph_build_n2, Fig. 4) and the same list force loop (force_group,
// tp = 8) as the handle path, with every piece of scratch in ONE file-scope device array of fixed size.  The caller
// passes only inputs (positions + types, box, pair parameters) and outputs (forces + u_i, w_i, four summary doubles).
//
// The scratch array is part of the library image: every GPU that loads librumd_b200.so holds NA_BYTES (8.2 MB)
// until the process exits.  ALL calls share it and it keeps the last call's contents: what must start at zero is
// cleared at the start of every call, on the call's stream.  Two calls that overlap on the GPU (different streams, no
// ordering between them) race on it.
//
// g_scratch below is a HOST-side stand-in for the device array in host code: its device address comes from
// cudaGetSymbolAddress, once per device, with that device current (scratch_of_current_device).
#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <mutex>

#include "../../include/rumd_b200.h"
#include "rumd_force.cuh"

#define NA_TP 8                                   // lanes per particle of the force kernel
#define NA_MAXN RUMD_NOALLOC_MAX_PARTICLES        // 8192
#define NA_CAP RUMD_NOALLOC_NBL_CAPACITY          // 256 list entries per particle
#define NA_THREADS 256
#define NA_MAXBLOCKS (NA_MAXN * NA_TP / NA_THREADS) // 256 blocks of the force kernel at most

// layout of the scratch array (byte offsets, all multiples of 256)
#define NA_OFF_NBL 0                                                   // int  [NA_MAXN * NA_CAP]  tiled list (nbl_index)
#define NA_OFF_NUM (NA_OFF_NBL + (size_t)NA_MAXN * NA_CAP * 4)         // int  [NA_MAXN]           list lengths
#define NA_OFF_RBUILD (NA_OFF_NUM + (size_t)NA_MAXN * 4)               // float4 [NA_MAXN]         positions at build
#define NA_OFF_PARTIAL (NA_OFF_RBUILD + (size_t)NA_MAXN * 16)          // double [2 * NA_MAXBLOCKS] block sums of u_i, w_i
#define NA_OFF_SC (NA_OFF_PARTIAL + (size_t)NA_MAXBLOCKS * 16)         // DevScalars               flags, ticket, max length
#define NA_BYTES (NA_OFF_SC + 512)
static_assert(sizeof(DevScalars) <= 512, "DevScalars outgrew its slot of the no-alloc scratch");
static_assert(NA_OFF_NUM % 256 == 0 && NA_OFF_RBUILD % 256 == 0 && NA_OFF_PARTIAL % 256 == 0 && NA_OFF_SC % 256 == 0,
              "scratch sections must stay 256-byte aligned");

static __device__ __align__(256) unsigned char g_scratch[NA_BYTES];

// ------------------------------------------------------------------------------------------ kernels

// A2 into the static list: one warp per particle, rows in ascending-j order (bitwise the list of the handle's n2 method)
static __global__ void __launch_bounds__(128) k_na_build(const Sys S)
{
    __shared__ float4 tile[N2_TILE];
    __shared__ float s_rcl2[RUMD_MAXT * RUMD_MAXT];
    if (threadIdx.x < RUMD_MAXT * RUMD_MAXT) s_rcl2[threadIdx.x] = S.pp[threadIdx.x].rcl2;
    __syncthreads();
    ph_build_n2(S, S.r, tile, s_rcl2, blockIdx.x, gridDim.x, &S.sc->max_nbrs[0]);
}

// A5 over the static list (force_group: the loop of k_force at tp = 8), then U = sum u_i and W = sum w_i: block sums in
// fp64 to the scratch, the last block to finish adds them in block order (fixed order: reproducible) and writes
// out4 = {U, W, longest list row, overflow flag}.
template <int COUL, bool ONE_TYPE>
static __global__ void __launch_bounds__(NA_THREADS) k_na_force(const Sys S, double* partial, double* out4)
{
    __shared__ float4 s_pp[4 * RUMD_MAXT * RUMD_MAXT];
    __shared__ double s_u[NA_THREADS / 32], s_w[NA_THREADS / 32];
    load_pair_table(S, s_pp);
    __syncthreads();
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int vwarp = blockIdx.x * (NA_THREADS / 32) + wid;
    const int tid = vwarp * 32 + lane;
    const int i = tid / NA_TP, t = tid % NA_TP;
    const bool have_i = i < S.N;
    float4 ri = make_float4(0.f, 0.f, 0.f, 0.f);
    int cnt = 0;
    if (have_i) {
        ri = __ldg(&S.r[i]);
        cnt = S.num_nbrs[i];
    }
    float fx, fy, fz, u, w;
    force_group<NA_TP, COUL, ONE_TYPE, 8, true, true>(S, S.r, s_pp, vwarp, i, t, have_i, ri, cnt, fx, fy, fz, u, w);
    double du = 0.0, dw = 0.0;
    if (have_i && t == 0) {
        const float ui = 0.5f * u, wi = 0.5f * w; // P:160 "compensate for double counting"
        S.f[i] = make_float4(fx, fy, fz, ui);
        S.w[i] = wi;
        du = (double)ui;
        dw = (double)wi;
    }
    du = warp_sum(du);
    dw = warp_sum(dw);
    if (lane == 0) {
        s_u[wid] = du;
        s_w[wid] = dw;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        double a = 0.0, b = 0.0;
        for (int q = 0; q < NA_THREADS / 32; ++q) {
            a += s_u[q];
            b += s_w[q];
        }
        partial[2 * blockIdx.x] = a;
        partial[2 * blockIdx.x + 1] = b;
        __threadfence();
        if (atomicAdd(&S.sc->ticket, 1u) == gridDim.x - 1) { // the last block to finish
            __threadfence();
            double U = 0.0, W = 0.0;
            for (unsigned q = 0; q < gridDim.x; ++q) {
                U += __ldcg(&partial[2 * q]);
                W += __ldcg(&partial[2 * q + 1]);
            }
            out4[0] = U;
            out4[1] = W;
            out4[2] = (double)S.sc->max_nbrs[0];
            out4[3] = S.sc->overflow != 0u ? 1.0 : 0.0;
            S.sc->ticket = 0u;
        }
    }
}

// ------------------------------------------------------------------------------------------ host side

static rumd_status na_fail(char* errbuf, size_t errbuf_len, rumd_status st, const char* fmt, ...)
{
    if (errbuf && errbuf_len > 0) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(errbuf, errbuf_len, fmt, ap);
        va_end(ap);
    }
    return st;
}

// Device address of g_scratch on the CURRENT device: looked up once per device (cudaGetSymbolAddress allocates
// nothing; the array came with the module), then cached.  In host code `g_scratch` itself is not a device address.
static cudaError_t scratch_of_current_device(unsigned char** out)
{
    static std::mutex mu;
    static unsigned char* ptr_of[64] = {nullptr};
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(mu);
    if (!ptr_of[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_scratch);
        if (e != cudaSuccess) return e;
        ptr_of[dev] = static_cast<unsigned char*>(p);
    }
    *out = ptr_of[dev];
    return cudaSuccess;
}

// the pair record of the kernels from the user's parameters: the LJ and the Coulomb part of refresh() in rumd_b200.cu
// (shifted force: f = f(r) - f(rc), u = u(r) - u(rc) + (r - rc) f(rc)), in double, rounded once
static void na_pair_params(const rumd_noalloc_pair& p, double skin, PairParams& q)
{
    memset(&q, 0, sizeof q);
    double rc = 0.0;
    if (p.rcut > 0.f) {
        const double s6 = std::pow((double)p.sigma, 6), c6 = 4.0 * p.epsilon * s6, c12 = c6 * s6;
        const double rcl = p.rcut, ri6 = std::pow(rcl, -6);
        const double uc = c12 * ri6 * ri6 - c6 * ri6;
        const double fc = (12 * c12 * ri6 * ri6 - 6 * c6 * ri6) / rcl;
        q.c12 = (float)c12;
        q.c6 = (float)c6;
        q.c12x12 = (float)(12.0 * c12);
        q.c6x6 = (float)(6.0 * c6);
        q.rc2_lj = (float)(rcl * rcl);
        q.fc_lj = (float)fc;
        q.k0_lj = (float)(uc + rcl * fc);
        rc = std::max(rc, rcl);
    }
    if (p.rcut_coulomb > 0.f) {
        const double a = p.kqq, rcc = p.rcut_coulomb;
        const double uraw = a / rcc, fraw = a / (rcc * rcc);
        q.qq = (float)a;
        q.rc2_c = (float)(rcc * rcc);
        q.fc_c = (float)fraw;
        q.k0_c = (float)(uraw + rcc * fraw);
        rc = std::max(rc, rcc);
    }
    q.rcl2 = (float)((rc + skin) * (rc + skin));
    q.rc2_max = (float)(rc * rc);
}

extern "C" rumd_status rumd_forces_noalloc(int n_particles, int n_types, const float box_lengths[3],
                                           const rumd_noalloc_pair* pairs, float skin, const void* d_r, void* d_f,
                                           void* d_w, void* d_out4, void* cuda_stream, char* errbuf, size_t errbuf_len)
{
    if (errbuf && errbuf_len > 0) errbuf[0] = 0;
    if (n_particles < 1)
        return na_fail(errbuf, errbuf_len, RUMD_ERR_INVALID_ARG, "n_particles = %d: need at least one particle", n_particles);
    if (n_particles > NA_MAXN)
        return na_fail(errbuf, errbuf_len, RUMD_ERR_INVALID_ARG,
                       "n_particles = %d exceeds RUMD_NOALLOC_MAX_PARTICLES = %d (the static scratch holds no more): use the handle API",
                       n_particles, NA_MAXN);
    if (n_types < 1 || n_types > RUMD_MAXT)
        return na_fail(errbuf, errbuf_len, RUMD_ERR_INVALID_ARG, "n_types = %d outside 1..%d", n_types, RUMD_MAXT);
    if (!box_lengths || !pairs || !d_r || !d_f || !d_w || !d_out4)
        return na_fail(errbuf, errbuf_len, RUMD_ERR_INVALID_ARG, "null pointer argument");
    if (((uintptr_t)d_r | (uintptr_t)d_f) & 15u || ((uintptr_t)d_w & 3u) || ((uintptr_t)d_out4 & 7u))
        return na_fail(errbuf, errbuf_len, RUMD_ERR_INVALID_ARG, "d_r / d_f must be 16-byte, d_out4 8-byte, d_w 4-byte aligned");
    if (!(skin >= 0.f) || !std::isfinite(skin))
        return na_fail(errbuf, errbuf_len, RUMD_ERR_INVALID_ARG, "skin = %g: need a finite value >= 0", (double)skin);

    Sys S;
    memset(&S, 0, sizeof S);
    bool any_coul = false;
    double rcm = 0.0;
    for (int a = 0; a < n_types; ++a)
        for (int b = 0; b < n_types; ++b) {
            const rumd_noalloc_pair& p = pairs[a * n_types + b];
            const rumd_noalloc_pair& pt = pairs[b * n_types + a];
            if (memcmp(&p, &pt, sizeof p) != 0)
                return na_fail(errbuf, errbuf_len, RUMD_ERR_INVALID_ARG, "pair parameters of (%d, %d) and (%d, %d) differ", a, b, b, a);
            if ((p.rcut > 0.f && !(p.sigma > 0.f && std::isfinite(p.epsilon) && std::isfinite(p.rcut))) ||
                (p.rcut_coulomb > 0.f && !(std::isfinite(p.kqq) && std::isfinite(p.rcut_coulomb))))
                return na_fail(errbuf, errbuf_len, RUMD_ERR_INVALID_ARG, "bad pair parameters for types (%d, %d)", a, b);
            na_pair_params(p, (double)skin, S.pp[a * n_types + b]);
            if (p.rcut > 0.f) rcm = std::max(rcm, (double)p.rcut);
            if (p.rcut_coulomb > 0.f) {
                rcm = std::max(rcm, (double)p.rcut_coulomb);
                any_coul = true;
            }
        }
    for (int k = 0; k < 3; ++k) {
        const double L = box_lengths[k];
        if (!(L > 0.0) || !std::isfinite(L))
            return na_fail(errbuf, errbuf_len, RUMD_ERR_INVALID_ARG, "box length %g on axis %d", L, k);
        if (rcm + skin > 0.5 * L) // O1: the minimum image must be unique for every listed pair
            return na_fail(errbuf, errbuf_len, RUMD_ERR_BOX_TOO_SMALL, "rc_max + skin = %g exceeds L/2 = %g on axis %d",
                           rcm + skin, 0.5 * L, k);
        S.L[k] = box_lengths[k];
        S.h[k] = 0.5f * box_lengths[k];
        S.invL[k] = (float)(1.0 / L);
        S.hin[k] = (float)(0.5 * L - (rcm + 2.0 * skin) - 1e-3);
    }

    unsigned char* scratch = nullptr;
    cudaError_t e = scratch_of_current_device(&scratch);
    if (e != cudaSuccess)
        return na_fail(errbuf, errbuf_len, RUMD_ERR_CUDA, "cudaGetSymbolAddress(static scratch) failed: %s", cudaGetErrorString(e));

    S.N = n_particles;
    S.Npad = (n_particles + 31) / 32 * 32;
    S.ntypes = n_types;
    S.cap = NA_CAP;
    S.cap_it = NA_CAP / NA_TP;
    S.tp_shift = 3; // log2(NA_TP)
    S.ppw_shift = 2;
    S.method = RUMD_NB_N2;
    S.skin = skin;
    S.rcl_max = (float)(rcm + skin);
    S.rc_margin = (float)(rcm + 2.0 * skin + 1e-3);
    S.r = static_cast<float4*>(const_cast<void*>(d_r)); // read only here
    S.f = static_cast<float4*>(d_f);
    S.w = static_cast<float*>(d_w);
    S.nbl = reinterpret_cast<int*>(scratch + NA_OFF_NBL);
    S.num_nbrs = reinterpret_cast<int*>(scratch + NA_OFF_NUM);
    S.r_build = reinterpret_cast<float4*>(scratch + NA_OFF_RBUILD);
    S.sc = reinterpret_cast<DevScalars*>(scratch + NA_OFF_SC);
    double* partial = reinterpret_cast<double*>(scratch + NA_OFF_PARTIAL);
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);

    // the scalars the kernels accumulate into (overflow flag, longest row, ticket) must start at zero
    e = cudaMemsetAsync(S.sc, 0, sizeof(DevScalars), stream);
    if (e != cudaSuccess) return na_fail(errbuf, errbuf_len, RUMD_ERR_CUDA, "cudaMemsetAsync failed: %s", cudaGetErrorString(e));
    const int build_blocks = std::min((n_particles + 3) / 4, 148 * 8);
    k_na_build<<<build_blocks, 128, 0, stream>>>(S);
    const int force_blocks = (n_particles * NA_TP + NA_THREADS - 1) / NA_THREADS;
    double* out4 = static_cast<double*>(d_out4);
    if (any_coul) {
        if (n_types == 1)
            k_na_force<1, true><<<force_blocks, NA_THREADS, 0, stream>>>(S, partial, out4);
        else
            k_na_force<1, false><<<force_blocks, NA_THREADS, 0, stream>>>(S, partial, out4);
    } else {
        if (n_types == 1)
            k_na_force<0, true><<<force_blocks, NA_THREADS, 0, stream>>>(S, partial, out4);
        else
            k_na_force<0, false><<<force_blocks, NA_THREADS, 0, stream>>>(S, partial, out4);
    }
    e = cudaGetLastError();
    if (e != cudaSuccess) return na_fail(errbuf, errbuf_len, RUMD_ERR_CUDA, "kernel launch failed: %s", cudaGetErrorString(e));
    return RUMD_OK;
}
