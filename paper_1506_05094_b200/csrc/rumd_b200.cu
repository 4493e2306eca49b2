// rumd_b200.cu -- host side of librumd_b200.so: C ABI (include/rumd_b200.h), workspace carving, launch
// chains, whole-timestep CUDA graphs and the Blackwell autotuner.  Product code: shares nothing with oracle/.
#define RUMD_MAIN_TU 1
#include "../../include/rumd_b200.h"
#include "rumd_dispatch.cuh"
#include "rumd_persist.cuh"
#include "rumd_ensemble.cuh"
#include "rumd_npt.cuh"

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <string>
#include <vector>

struct PotSlot {
    bool lj = false, coul = false;
    double eps = 0, sig = 0, rc_lj = 0, qq = 0, rc_c = 0; // qq: prefactor a of the second term
    int cut_lj = 0, cut_c = 0; // rumd_cutoff of each term
    int kind2 = 0;             // second term: rumd_pot_kind - 1 (0 Coulomb ... 7 Dzugutov)
    double b2 = 0, c2 = 0, d2 = 0; // its further parameters
};

struct GraphCache {
    cudaGraphExec_t exec = nullptr;
    int steps = 0;
    int kernels = 0;
};

struct rumd_system {
    int N = 0, ntypes = 0;  // N: particles of ONE system
    int nrep = 1;           // replicas (batched ensemble); the state arrays hold nrep * N particles
    Sys* d_systems = nullptr;     // ensemble: per-replica parameter blocks (in the workspace)
    DevScalars* ens_sc = nullptr; // ensemble: per-replica scalars (in the workspace)
    float box[3] = {0, 0, 0};
    cudaStream_t stream = nullptr;
    bool own_stream = false;
    Sys S;
    bool state_bound = false, ws_bound = false, integ_set = false;
    bool params_dirty = true;
    PotSlot pot[RUMD_MAXT][RUMD_MAXT];
    bool any_coul = false, any_generic = false; // a second term is set / one of them is not Coulomb
    int integ = 0;
    float dt = 0, T0 = 0, tau = 0;
    float P0 = 0, tauP = 0; // NPT: target pressure, barostat period
    rumd_tuning tune;
    int cap = 0;
    size_t nc_carved = 0;   // cells the bound workspace was carved (and its histogram zeroed) for
    void* ws = nullptr;
    size_t ws_bytes = 0;
    // snapshot area
    float4* snap_r = nullptr;
    float4* snap_v = nullptr;
    int4* snap_image = nullptr;
    int* snap_id = nullptr;
    DevScalars* snap_sc = nullptr;
    int grid_for[3] = {0, 0, 0}; // cell grid the device rowrank table was built for
    GraphCache graph_multi, graph_one;
    rumd_thermo* h_thermo = nullptr; // pinned
    DevScalars* h_sc = nullptr;      // pinned
    long long launches = 0;
    int int_blocks = 0;
    int num_sms = 148;
    int force_grid_for = -1, force_per_sm = 1; // co-resident blocks per SM of the stand-alone force kernel
    int persist_grid_for = -1; // tuning signature the cached persistent grid belongs to
    int persist_grid = 0, persist_threads = 0;
    long long* prof_buf = nullptr;
    std::string err;
};

static rumd_status fail(rumd_system* s, rumd_status st, const char* fmt, ...)
{
    if (s) {
        char buf[512];
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(buf, sizeof buf, fmt, ap);
        va_end(ap);
        s->err = buf;
    }
    return st;
}

#define CUDA_TRY(s, call)                                                                              \
    do {                                                                                               \
        cudaError_t e_ = (call);                                                                       \
        if (e_ != cudaSuccess)                                                                         \
            return fail((s), RUMD_ERR_CUDA, "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e_),    \
                        __FILE__, __LINE__);                                                           \
    } while (0)

static size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

static double rc_max_of(const rumd_system* s)
{
    double m = 0;
    for (int a = 0; a < s->ntypes; ++a)
        for (int b = 0; b < s->ntypes; ++b) {
            const PotSlot& p = s->pot[a][b];
            if (p.lj) m = std::max(m, p.rc_lj);
            if (p.coul) m = std::max(m, p.rc_c);
        }
    return m;
}

// S17 (+ a 1e-4 safety margin on the cell edge so that fp32 rounding of the cell coordinate cannot push a
// listed pair out of the 5x5x5 stencil): n_k = floor(L_k / (1.0001 (rc_max + skin)/2)).
static void grid_dims(const rumd_system* s, double skin, int n[3])
{
    const double edge = 0.5 * (rc_max_of(s) + skin) * 1.0001;
    for (int k = 0; k < 3; ++k) {
        n[k] = edge > 0 ? (int)std::floor(s->box[k] / edge) : 1;
        if (n[k] < 1) n[k] = 1;
        if (n[k] > 1024) n[k] = 1024;
    }
}

static size_t max_cells(const rumd_system* s)
{
    // upper bound over all skins >= 0 (skin = 0 gives the finest grid); used to size the workspace
    int n[3];
    const double edge = 0.5 * std::max(rc_max_of(s), 0.5) * 1.0001;
    size_t t = 1;
    for (int k = 0; k < 3; ++k) {
        n[k] = std::min(1024, std::max(1, (int)std::floor(s->box[k] / edge)));
        t *= (size_t)n[k];
    }
    return t;
}

// tile method: bounds used to size the workspace (refresh() checks the actual tiling against them)
static size_t tile_bound(const rumd_system* s) { return align_up((size_t)s->N, 32) / 32 - 1; } // tiles, at most
static size_t halo_slots_bound(const rumd_system* s) { return s->nrep > 1 ? 64 : 20 * (size_t)s->N + 65536; }

static uint32_t part1by1(uint32_t x) // spread the low 16 bits to the even bit positions
{
    x &= 0x0000ffff;
    x = (x ^ (x << 8)) & 0x00ff00ff;
    x = (x ^ (x << 4)) & 0x0f0f0f0f;
    x = (x ^ (x << 2)) & 0x33333333;
    x = (x ^ (x << 1)) & 0x55555555;
    return x;
}

// Carve the workspace.  Returns bytes needed; if base != nullptr also fills the pointers.
static size_t carve(rumd_system* s, char* base, int cap)
{
    // ensemble: every replica owns a slice of each particle array; list rows are padded per replica
    const size_t R = (size_t)s->nrep;
    const size_t N = (size_t)s->N * R, Npad = align_up((size_t)s->N, 32) * R;
    const size_t nc = max_cells(s);
    size_t off = 0;
    auto take = [&](size_t bytes) {
        size_t o = off;
        off = align_up(off + bytes, 256);
        return base ? (void*)(base + o) : (void*)nullptr;
    };
    Sys& S = s->S;
    void* p;
    p = take(sizeof(DevScalars)); if (base) S.sc = (DevScalars*)p;
    p = take(sizeof(DevScalars)); if (base) s->snap_sc = (DevScalars*)p;
    // (tile method: 16-bit entries, rows padded to a warp boundary per tile -> Npad + 32 (tiles + 1) rows of 2 cap
    // bytes, which fits this array as long as there are at most Npad / 32 - 1 tiles: tile_bound)
    p = take(Npad * (size_t)cap * 4); if (base) S.nbl = (int*)p;
    p = take(Npad * 4); if (base) S.num_nbrs = (int*)p;
    p = take(N * 16); if (base) S.r_build = (float4*)p;
    p = take(N * 16); if (base) S.r_alt = (float4*)p;
    p = take(N * 16); if (base) S.tmp_r = (float4*)p;
    p = take(N * 16); if (base) S.tmp_v = (float4*)p;
    p = take(N * 16); if (base) S.tmp_image = (int4*)p;
    p = take(N * 4); if (base) S.tmp_id = (int*)p;
    p = take(N * 16); if (base) s->snap_r = (float4*)p;
    p = take(N * 16); if (base) s->snap_v = (float4*)p;
    p = take(N * 16); if (base) s->snap_image = (int4*)p;
    p = take(N * 4); if (base) s->snap_id = (int*)p;
    p = take(N * 4); if (base) S.cell_of = (int*)p;
    p = take(N * 4); if (base) S.slot = (int*)p;
    p = take(N * 4); if (base) S.perm = (int*)p;
    p = take(nc * 4); if (base) S.ccount = (int*)p;
    p = take((nc + 1) * 4); if (base) S.cstart_z = (int*)p;
    p = take(nc * 4); if (base) S.rowrank = (int*)p;
    p = take((nc / SCAN_CHUNK + 2) * 4); if (base) S.blocksum = (int*)p;
    // (kt, mv2) per block: integrator kernel (N/128 blocks) or persistent kernel (2 sets x <= 4096 blocks)
    const size_t nblk = std::max<size_t>(N + 1, 2 * 4096); // the fused per-step kernel may run N blocks (pb = 1)
    p = take(nblk * 16); if (base) S.partial = (double*)p;
    p = take(8 * 8); if (base) s->prof_buf = (long long*)p;
    p = take(halo_slots_bound(s) * 4); if (base) S.halo_idx = (int*)p;
    p = take((tile_bound(s) + 1) * 4); if (base) S.halo_cnt = (int*)p;
    if (R > 1) {
        p = take(R * sizeof(Sys)); if (base) s->d_systems = (Sys*)p;
        p = take(R * sizeof(DevScalars)); if (base) s->ens_sc = (DevScalars*)p;
    }
    return off;
}

extern "C" const char* rumd_version(void) { return "rumd_b200 0.1 (sm_100a)"; }

extern "C" const char* rumd_last_error(const rumd_system* s) { return s ? s->err.c_str() : "null handle"; }

extern "C" long long rumd_launch_count(const rumd_system* s) { return s ? s->launches : 0; }

extern "C" rumd_status rumd_create(rumd_system** out, int n_particles, int n_types, const float box_lengths[3],
                                   void* cuda_stream)
{
    if (!out || !box_lengths || n_particles < 1 || n_types < 1 || n_types > RUMD_MAXT)
        return RUMD_ERR_INVALID_ARG;
    for (int k = 0; k < 3; ++k)
        if (!(box_lengths[k] > 0.f) || !std::isfinite(box_lengths[k])) return RUMD_ERR_INVALID_ARG;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
        cudaGetLastError();
        return RUMD_ERR_CUDA; // no CPU fallback
    }
    rumd_system* s = new rumd_system();
    memset(&s->S, 0, sizeof(Sys));
    s->N = n_particles;
    s->ntypes = n_types;
    s->stream = (cudaStream_t)cuda_stream;
    if (!s->stream) {
        // the legacy default stream cannot be captured into CUDA graphs: own a BLOCKING stream instead, which
        // stays implicitly ordered with the legacy default stream
        if (cudaStreamCreate(&s->stream) != cudaSuccess) {
            delete s;
            return RUMD_ERR_CUDA;
        }
        s->own_stream = true;
    }
    for (int k = 0; k < 3; ++k) {
        s->box[k] = box_lengths[k];
        s->S.L[k] = box_lengths[k]; // (k_reset_scalars seeds the device box from it, before the first refresh)
    }
    if (cudaMallocHost((void**)&s->h_thermo, sizeof(rumd_thermo)) != cudaSuccess ||
        cudaMallocHost((void**)&s->h_sc, sizeof(DevScalars)) != cudaSuccess) {
        delete s;
        return RUMD_ERR_CUDA;
    }
    {
        int dev = 0, sms = 0;
        if (cudaGetDevice(&dev) == cudaSuccess &&
            cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && sms > 0)
            s->num_sms = sms;
    }
    rumd_default_tuning(s, &s->tune);
    *out = s;
    return RUMD_OK;
}

static void drop_graphs(rumd_system* s)
{
    if (s->graph_multi.exec) cudaGraphExecDestroy(s->graph_multi.exec);
    if (s->graph_one.exec) cudaGraphExecDestroy(s->graph_one.exec);
    s->graph_multi = GraphCache();
    s->graph_one = GraphCache();
}

extern "C" rumd_status rumd_destroy(rumd_system* s)
{
    if (!s) return RUMD_ERR_INVALID_ARG;
    cudaStreamSynchronize(s->stream);
    drop_graphs(s);
    if (s->h_thermo) cudaFreeHost(s->h_thermo);
    if (s->h_sc) cudaFreeHost(s->h_sc);
    if (s->own_stream) cudaStreamDestroy(s->stream);
    delete s;
    return RUMD_OK;
}

// ---------------------------------------------------------------------------------------------- setters

static void ens_reset(rumd_system* s)
{
    if (s->nrep > 1 && s->ens_sc) {
        k_ens_reset<<<(s->nrep + 127) / 128, 128, 0, s->stream>>>(s->ens_sc, s->nrep);
        s->launches++;
    }
}

// Batched ensemble: the handle describes ONE system of n_particles; with n_replicas > 1 the state arrays
// hold n_replicas such systems back to back and rumd_run_steps advances all of them in one launch.
extern "C" rumd_status rumd_set_replicas(rumd_system* s, int n_replicas)
{
    if (!s) return RUMD_ERR_INVALID_ARG;
    if (n_replicas < 1 || (long long)n_replicas * s->N > (1LL << 30)) return fail(s, RUMD_ERR_INVALID_ARG, "bad replica count");
    if (s->state_bound || s->ws_bound) return fail(s, RUMD_ERR_NOT_READY, "set the replica count before binding state and workspace");
    s->nrep = n_replicas;
    s->params_dirty = true;
    return RUMD_OK;
}

extern "C" rumd_status rumd_bind_state(rumd_system* s, void* d_r, void* d_v, void* d_f, void* d_w, void* d_image,
                                       void* d_id)
{
    if (!s) return RUMD_ERR_INVALID_ARG;
    if (!d_r || !d_v || !d_f || !d_w || !d_image || !d_id) return fail(s, RUMD_ERR_INVALID_ARG, "null state pointer");
    if (((uintptr_t)d_r | (uintptr_t)d_v | (uintptr_t)d_f | (uintptr_t)d_image) & 15)
        return fail(s, RUMD_ERR_INVALID_ARG, "state arrays must be 16-byte aligned");
    s->S.r = (float4*)d_r;
    s->S.v = (float4*)d_v;
    s->S.f = (float4*)d_f;
    s->S.w = (float*)d_w;
    s->S.image = (int4*)d_image;
    s->S.id = (int*)d_id;
    s->state_bound = true;
    s->params_dirty = true;
    drop_graphs(s);
    if (s->ws_bound) {
        k_reset_scalars<<<1, 1, 0, s->stream>>>(s->S);
        s->launches++;
        ens_reset(s);
        CUDA_TRY(s, cudaGetLastError());
    }
    return RUMD_OK;
}

extern "C" size_t rumd_workspace_bytes(const rumd_system* s, int nbl_capacity)
{
    if (!s || nbl_capacity < 1) return 0;
    const int cap = (int)align_up((size_t)nbl_capacity, 32);
    return carve(const_cast<rumd_system*>(s), nullptr, cap);
}

extern "C" rumd_status rumd_bind_workspace(rumd_system* s, void* d_ws, size_t bytes, int nbl_capacity)
{
    if (!s || !d_ws || nbl_capacity < 1) return RUMD_ERR_INVALID_ARG;
    if ((uintptr_t)d_ws & 255) return fail(s, RUMD_ERR_INVALID_ARG, "workspace must be 256-byte aligned");
    const int cap = (int)align_up((size_t)nbl_capacity, 32);
    const size_t need = carve(s, nullptr, cap);
    if (bytes < need) return fail(s, RUMD_ERR_INVALID_ARG, "workspace too small: %zu < %zu", bytes, need);
    // keep the thermostat / counters across a re-bind (capacity doubling) when there was a workspace
    const bool had = s->ws_bound;
    DevScalars keep;
    if (had) {
        CUDA_TRY(s, cudaMemcpyAsync(&keep, s->S.sc, sizeof keep, cudaMemcpyDeviceToHost, s->stream));
        CUDA_TRY(s, cudaStreamSynchronize(s->stream));
    }
    carve(s, (char*)d_ws, cap);
    s->nc_carved = max_cells(s);
    s->ws = d_ws;
    s->ws_bytes = bytes;
    s->cap = cap;
    s->ws_bound = true;
    s->params_dirty = true;
    s->grid_for[0] = s->grid_for[1] = s->grid_for[2] = 0;
    drop_graphs(s);
    CUDA_TRY(s, cudaMemsetAsync(s->S.ccount, 0, s->nc_carved * 4, s->stream));
    CUDA_TRY(s, cudaMemsetAsync(s->S.num_nbrs, 0, align_up((size_t)s->N, 32) * (size_t)s->nrep * 4, s->stream));
    if (had) {
        keep.flag = 1u;
        keep.pending = 0u;
        keep.ticket = 0u;
        keep.overflow = 0u;
        keep.max_nbrs[0] = keep.max_nbrs[1] = 0;
        keep.last_max = 0;
        *s->h_sc = keep;
        CUDA_TRY(s, cudaMemcpyAsync(s->S.sc, s->h_sc, sizeof keep, cudaMemcpyHostToDevice, s->stream));
        CUDA_TRY(s, cudaStreamSynchronize(s->stream));
    } else {
        k_reset_scalars<<<1, 1, 0, s->stream>>>(s->S);
        s->launches++;
        ens_reset(s);
        CUDA_TRY(s, cudaGetLastError());
    }
    return RUMD_OK;
}

extern "C" rumd_status rumd_set_pair_potential(rumd_system* s, int ti, int tj, rumd_pot_kind kind,
                                               rumd_cutoff cutoff, const float* params, int n_params)
{
    if (!s || !params) return RUMD_ERR_INVALID_ARG;
    if (ti < 0 || tj < 0 || ti >= s->ntypes || tj >= s->ntypes) return fail(s, RUMD_ERR_INVALID_ARG, "type out of range");
    if (cutoff != RUMD_CUT_SHIFTED_FORCE && cutoff != RUMD_CUT_SHIFTED_POTENTIAL && cutoff != RUMD_CUT_NONE)
        return fail(s, RUMD_ERR_INVALID_ARG, "unknown cutoff method");
    for (int q = 0; q < n_params; ++q)
        if (!std::isfinite(params[q])) return fail(s, RUMD_ERR_INVALID_ARG, "non-finite parameter");
    for (int pass = 0; pass < 2; ++pass) {
        PotSlot& p = pass == 0 ? s->pot[ti][tj] : s->pot[tj][ti];
        if (kind == RUMD_POT_LJ_12_6) {
            if (n_params != 3) return fail(s, RUMD_ERR_INVALID_ARG, "LJ takes {epsilon, sigma, rcut}");
            p.lj = params[2] > 0.f;
            p.eps = params[0];
            p.sig = params[1];
            p.rc_lj = params[2];
            p.cut_lj = (int)cutoff;
            if (p.lj && !(p.sig > 0)) return fail(s, RUMD_ERR_INVALID_ARG, "sigma must be > 0");
        } else if (kind >= RUMD_POT_COULOMB && kind <= RUMD_POT_DZUGUTOV) {
            static const int n_of[8] = {2, 3, 3, 3, 4, 5, 4, 3}; // parameters incl. rcut, by kind - 1
            const int want = n_of[(int)kind - 1];
            if (n_params != want) return fail(s, RUMD_ERR_INVALID_ARG, "this potential takes %d parameters (see rumd_pot_kind)", want);
            const float rc = params[want - 1];
            p.coul = rc > 0.f;
            p.qq = params[0];
            p.rc_c = rc;
            p.cut_c = (int)cutoff;
            p.kind2 = (int)kind - 1;
            p.b2 = want >= 3 ? params[1] : 0.0;
            p.c2 = want >= 4 ? params[2] : 0.0;
            p.d2 = want >= 5 ? params[3] : 0.0;
            if (p.coul && (kind == RUMD_POT_YUKAWA || kind == RUMD_POT_GAUSSIAN_CORE || kind == RUMD_POT_BUCKINGHAM ||
                           kind == RUMD_POT_GEN_LJ || kind == RUMD_POT_DZUGUTOV) && !(p.b2 > 0))
                return fail(s, RUMD_ERR_INVALID_ARG, "the length parameter (second one) must be > 0");
            if (p.coul && kind == RUMD_POT_GEN_LJ && !(p.c2 > p.d2 && p.d2 > 0))
                return fail(s, RUMD_ERR_INVALID_ARG, "generalized LJ needs exponents m > n > 0");
            if (p.coul && kind == RUMD_POT_GIRIFALCO && !(p.c2 > 0 && rc > p.c2))
                return fail(s, RUMD_ERR_INVALID_ARG, "Girifalco needs a diameter d > 0 and rcut > d");
        } else
            return fail(s, RUMD_ERR_INVALID_ARG, "unknown potential kind");
    }
    s->params_dirty = true;
    return RUMD_OK;
}

extern "C" rumd_status rumd_set_integrator(rumd_system* s, rumd_integrator kind, float dt, float T, float tau)
{
    if (!s) return RUMD_ERR_INVALID_ARG;
    if (kind != RUMD_INT_NVE_LEAPFROG && kind != RUMD_INT_NVT_NOSE_HOOVER && kind != RUMD_INT_NPT_MTK)
        return fail(s, RUMD_ERR_INVALID_ARG, "unknown integrator");
    if (!(dt > 0.f) || !std::isfinite(dt)) return fail(s, RUMD_ERR_INVALID_ARG, "dt must be > 0");
    if (kind != RUMD_INT_NVE_LEAPFROG && !(T > 0.f)) return fail(s, RUMD_ERR_INVALID_ARG, "target temperature must be > 0");
    s->integ = (int)kind;
    s->dt = dt;
    s->T0 = T;
    s->tau = tau;
    s->integ_set = true;
    s->params_dirty = true;
    return RUMD_OK;
}

extern "C" rumd_status rumd_set_barostat(rumd_system* s, float target_P, float tau_P)
{
    if (!s) return RUMD_ERR_INVALID_ARG;
    if (!std::isfinite(target_P)) return fail(s, RUMD_ERR_INVALID_ARG, "target pressure must be finite");
    s->P0 = target_P;
    s->tauP = tau_P;
    s->params_dirty = true;
    return RUMD_OK;
}

// Untuned defaults (the paper's are n2 below N = 8000, pb = 32 / tp = 4 up to N = 10^4, else pb = 64 /
// tp = 1; these are the B200 counterparts: enough threads for 148 SMs at every N).
extern "C" rumd_status rumd_default_tuning(const rumd_system* s, rumd_tuning* t)
{
    if (!s || !t) return RUMD_ERR_INVALID_ARG;
    const int N = s->N;
    t->method = N <= 6000 ? RUMD_NB_N2 : RUMD_NB_CELL;
    t->tp = N <= 2048 ? 32 : N <= 16384 ? 8 : N <= 32768 ? 4 : N <= 131072 ? 2 : 1;
    t->pb = 256 / t->tp;
    t->skin = 0.3f;
    t->sort_interval = 0;
    t->use_graph = 1;
    t->steps_per_graph = 0;
    t->persistent = 1;
    t->build_tp = 0;
    t->tile = 0;
    return RUMD_OK;
}

static bool valid_tp(int tp) { return tp == 1 || tp == 2 || tp == 4 || tp == 8 || tp == 16 || tp == 32; }

extern "C" rumd_status rumd_set_tuning(rumd_system* s, const rumd_tuning* t)
{
    if (!s || !t) return RUMD_ERR_INVALID_ARG;
    if (t->method != RUMD_NB_N2 && t->method != RUMD_NB_CELL && t->method != RUMD_NB_NONE && t->method != RUMD_NB_TILE)
        return fail(s, RUMD_ERR_INVALID_ARG, "bad method");
    if (t->method == RUMD_NB_TILE && t->tp > 8) return fail(s, RUMD_ERR_INVALID_ARG, "the tile method takes tp <= 8");
    if (t->tile < 0 || t->tile > TILE_WMAX) return fail(s, RUMD_ERR_INVALID_ARG, "tile must be 0..%d cells", TILE_WMAX);
    if (!valid_tp(t->tp)) return fail(s, RUMD_ERR_INVALID_ARG, "tp must be 1,2,4,8,16 or 32");
    if (t->pb < 1 || (t->pb * t->tp) % 32 || t->pb * t->tp > 1024) return fail(s, RUMD_ERR_INVALID_ARG, "pb*tp must be a multiple of 32 and <= 1024");
    if (!(t->skin > 0.f) || !std::isfinite(t->skin)) return fail(s, RUMD_ERR_INVALID_ARG, "skin must be > 0");
    if (t->sort_interval < 0 || t->steps_per_graph < 0) return fail(s, RUMD_ERR_INVALID_ARG, "negative interval");
    if (t->build_tp != 0 && !valid_tp(t->build_tp)) return fail(s, RUMD_ERR_INVALID_ARG, "build_tp must be 0,1,2,4,8,16 or 32");
    s->tune = *t;
    s->params_dirty = true;
    return RUMD_OK;
}

extern "C" rumd_status rumd_get_tuning(const rumd_system* s, rumd_tuning* t)
{
    if (!s || !t) return RUMD_ERR_INVALID_ARG;
    *t = s->tune;
    return RUMD_OK;
}

// ---------------------------------------------------------------------------------------------- parameters

static int ilog2(int x)
{
    int l = 0;
    while ((1 << l) < x) ++l;
    return l;
}

// Recompute the by-value kernel parameter block (pair table, box, grid, tuning).  Host side, double precision.
static rumd_status refresh(rumd_system* s)
{
    if (!s->state_bound || !s->ws_bound) return fail(s, RUMD_ERR_NOT_READY, "state and workspace must be bound first");
    if (!s->params_dirty) return RUMD_OK;
    Sys& S = s->S;
    S.N = s->N;
    S.Npad = (int)align_up((size_t)s->N, 32);
    S.ntypes = s->ntypes;
    const rumd_tuning& t = s->tune;
    S.cap = s->cap;
    S.cap_it = s->cap / t.tp;
    S.tp_shift = ilog2(t.tp);
    S.ppw_shift = 5 - S.tp_shift;
    const double skin = t.skin;
    const double rcm = rc_max_of(s);
    for (int k = 0; k < 3; ++k) {
        S.L[k] = s->box[k];
        S.h[k] = 0.5f * s->box[k];
        S.invL[k] = (float)(1.0 / (double)s->box[k]);
        S.hin[k] = (float)(0.5 * (double)s->box[k] - (rcm + 2.0 * skin) - 1e-3);
        if (rcm + skin > 0.5 * (double)s->box[k])
            return fail(s, RUMD_ERR_BOX_TOO_SMALL, "rc_max + skin = %g exceeds L/2 = %g on axis %d", rcm + skin,
                        0.5 * s->box[k], k);
    }
    S.dt = s->dt;
    S.dt_d = (double)s->dt;
    S.half_skin2 = (float)(0.25 * skin * skin);
    S.T0 = s->T0 > 0 ? (double)s->T0 : 1.0;
    S.g = 3.0 * s->N - 3.0; // S10
    const double tau = s->tau;
    S.omega2 = (tau > 0 && std::isfinite(tau)) ? (2.0 * M_PI / tau) * (2.0 * M_PI / tau) : 0.0;
    S.sort_interval = t.sort_interval;
    S.method = t.method;
    S.npt = s->integ == RUMD_INT_NPT_MTK;
    S.P0 = s->P0;
    S.cP = 0.0;
    S.rc_margin = (float)(rcm + 2.0 * skin + 1e-3);
    S.rcl_max = (float)(rcm + skin);
    S.skin = (float)skin;
    if (S.npt) {
        if (t.method != RUMD_NB_N2 && t.method != RUMD_NB_NONE)
            return fail(s, RUMD_ERR_INVALID_ARG, "NPT needs the n2 or the none method (the cell grid is sized for a fixed box)");
        if (s->nrep > 1) return fail(s, RUMD_ERR_INVALID_ARG, "NPT is not available for a batched ensemble");
        const double tp = s->tauP;
        if (tp > 0 && std::isfinite(tp)) S.cP = (2.0 * M_PI / tp) * (2.0 * M_PI / tp) / ((S.g + 3.0) * S.T0);
        S.half_skin2 = (float)(0.16 * skin * skin); // 0.4 skin: 0.1 skin is kept for the change of the box (rumd_npt.cuh)
    }
    S.r_out = S.r;
    {   // lanes per particle of the cell build: several while the machine is not full, one at large N (measured)
        const int btp = t.build_tp > 0 ? t.build_tp : s->N <= 32768 ? 8 : 1;
        S.build_tp_shift = ilog2(btp);
    }
    s->any_coul = false;
    s->any_generic = false;
    memset(S.pp, 0, sizeof S.pp);
    for (int a = 0; a < s->ntypes; ++a)
        for (int b = 0; b < s->ntypes; ++b) {
            const PotSlot& p = s->pot[a][b];
            PairParams& q = S.pp[a * s->ntypes + b];
            double rc = 0;
            if (p.lj) {
                const double s6 = std::pow(p.sig, 6), c6 = 4 * p.eps * s6, c12 = c6 * s6;
                const double ri6 = std::pow(p.rc_lj, -6);
                // the kernel evaluates u = u(r) + fc r - k0 and f = f(r) - fc: shifted force fc = f(rc),
                // k0 = u(rc) + rc fc; shifted potential fc = 0, k0 = u(rc); no shift fc = k0 = 0
                const double uc = p.cut_lj == RUMD_CUT_NONE ? 0.0 : c12 * ri6 * ri6 - c6 * ri6;
                const double fc = p.cut_lj == RUMD_CUT_SHIFTED_FORCE ? (12 * c12 * ri6 * ri6 - 6 * c6 * ri6) / p.rc_lj : 0.0;
                q.c12 = (float)c12;
                q.c6 = (float)c6;
                q.c12x12 = (float)(12.0 * c12);
                q.c6x6 = (float)(6.0 * c6);
                q.rc2_lj = (float)(p.rc_lj * p.rc_lj);
                q.fc_lj = (float)fc;
                q.k0_lj = (float)(uc + p.rc_lj * fc);
                rc = std::max(rc, p.rc_lj);
            }
            if (p.coul) {
                // second term at the cutoff, in double: u(rc), f(rc) of the raw potential
                const double a = p.qq, b = p.b2, c = p.c2, rcc = p.rc_c;
                double uraw, fraw, p1 = 0.0, p2 = 0.0, amp = a;
                switch (p.kind2) {
                case 5: { // generalized LJ as A r^-m - B r^-n; B rides in the (unused) 12-6 slot of the pair
                    if (p.lj) return fail(s, RUMD_ERR_INVALID_ARG, "generalized LJ takes the place of the 12-6 term: a type pair has both");
                    const double m = c, n = p.d2, A = a * n * std::pow(b, m) / (m - n), B = a * m * std::pow(b, n) / (m - n);
                    uraw = A * std::pow(rcc, -m) - B * std::pow(rcc, -n);
                    fraw = (m * A * std::pow(rcc, -m) - n * B * std::pow(rcc, -n)) / rcc;
                    amp = A;
                    p1 = m;
                    p2 = n;
                    q.c12x12 = (float)B;
                    break;
                }
                case 6: { // Girifalco, s = r / d
                    const double sg = rcc / c, m = sg - 1.0, pl = sg + 1.0;
                    uraw = -a * (1.0 / (sg * std::pow(m, 3)) + 1.0 / (sg * std::pow(pl, 3)) - 2.0 / std::pow(sg, 4)) +
                           b * (1.0 / (sg * std::pow(m, 9)) + 1.0 / (sg * std::pow(pl, 9)) - 2.0 / std::pow(sg, 10));
                    const double du = -a * (-(4 * sg - 1) / (sg * sg * std::pow(m, 4)) - (4 * sg + 1) / (sg * sg * std::pow(pl, 4)) + 8.0 / std::pow(sg, 5)) +
                                      b * (-(10 * sg - 1) / (sg * sg * std::pow(m, 10)) - (10 * sg + 1) / (sg * sg * std::pow(pl, 10)) + 20.0 / std::pow(sg, 11));
                    fraw = -du / c;
                    p1 = b;
                    p2 = 1.0 / c;
                    break;
                }
                case 7: { // Dzugutov, x = r / sigma
                    const double x = rcc / b;
                    double uu = 0.0, du = 0.0;
                    if (x < DZ_a) {
                        const double e = std::exp(DZ_c / (x - DZ_a)), g = std::pow(x, -16.0) - DZ_B;
                        uu += DZ_A * g * e;
                        du += DZ_A * e * (-16.0 * std::pow(x, -17.0) - g * DZ_c / ((x - DZ_a) * (x - DZ_a)));
                    }
                    if (x < DZ_b) {
                        const double e = std::exp(DZ_d / (x - DZ_b));
                        uu += DZ_B * e;
                        du -= DZ_B * e * DZ_d / ((x - DZ_b) * (x - DZ_b));
                    }
                    uraw = a * uu;
                    fraw = -a * du / b;
                    p1 = 1.0 / b;
                    break;
                }
                case 1: uraw = a * std::pow(rcc, -b); fraw = b * a * std::pow(rcc, -b - 1.0); p1 = b; break;
                case 2: uraw = a * std::exp(-rcc / b) / rcc; fraw = uraw * (1.0 / rcc + 1.0 / b); p1 = 1.0 / b; break;
                case 3: uraw = a * std::exp(-(rcc / b) * (rcc / b)); fraw = 2.0 * rcc * uraw / (b * b); p1 = 1.0 / (b * b); break;
                case 4:
                    uraw = a * std::exp(-rcc / b) - c * std::pow(rcc, -6.0);
                    fraw = a / b * std::exp(-rcc / b) - 6.0 * c * std::pow(rcc, -7.0);
                    p1 = 1.0 / b;
                    p2 = c;
                    break;
                default: uraw = a / rcc; fraw = a / (rcc * rcc); break;
                }
                q.qq = (float)amp;
                q.rc2_c = (float)(rcc * rcc);
                const double ucc = p.cut_c == RUMD_CUT_NONE ? 0.0 : uraw;
                const double fcc = p.cut_c == RUMD_CUT_SHIFTED_FORCE ? fraw : 0.0;
                q.fc_c = (float)fcc;
                q.k0_c = (float)(ucc + rcc * fcc);
                const int kbits = p.kind2;
                memcpy(&q.kind2, &kbits, sizeof(int));
                q.p1 = (float)p1;
                q.p2 = (float)p2;
                rc = std::max(rc, p.rc_c);
                s->any_coul = true;
                if (p.kind2 != 0) s->any_generic = true;
            }
            q.rcl2 = (float)((rc + skin) * (rc + skin));
            q.rc2_max = (float)(rc * rc);
        }
    // cell grid + Morton rank table (S17, S19)
    int n[3];
    grid_dims(s, skin, n);
    const size_t ncell = (size_t)n[0] * n[1] * n[2];
    // the cell arrays were sized from the potentials in force when the workspace was bound: a shorter rc_max set
    // afterwards makes a finer grid than was carved
    if (ncell > s->nc_carved)
        return fail(s, RUMD_ERR_NOT_READY, "cell grid (%zu cells) outgrew the workspace (carved for %zu): re-bind the workspace after changing the potentials",
                    ncell, s->nc_carved);
    if (t.method == RUMD_NB_CELL && (n[0] < 5 || n[1] < 5 || n[2] < 5))
        return fail(s, RUMD_ERR_BOX_TOO_SMALL, "cell method needs >= 5 cells per axis (S18), have %dx%dx%d", n[0], n[1], n[2]);
    S.grid.n[0] = n[0];
    S.grid.n[1] = n[1];
    S.grid.n[2] = n[2];
    S.grid.ncell = (int)ncell;
    for (int k = 0; k < 3; ++k) S.grid.scale[k] = (float)((double)n[k] / (double)s->box[k]);
    if (n[0] != s->grid_for[0] || n[1] != s->grid_for[1] || n[2] != s->grid_for[2]) {
        // rank of every (y, z) cell column along a 2-D Morton curve (S19)
        const size_t nrows = (size_t)n[1] * n[2];
        std::vector<std::pair<uint32_t, int>> keys(nrows);
        for (int z = 0; z < n[2]; ++z)
            for (int y = 0; y < n[1]; ++y) {
                const int c = z * n[1] + y;
                keys[c] = {part1by1((uint32_t)y) | (part1by1((uint32_t)z) << 1), c};
            }
        std::sort(keys.begin(), keys.end());
        std::vector<int> rr(nrows);
        for (size_t q = 0; q < nrows; ++q) rr[keys[q].second] = (int)q;
        CUDA_TRY(s, cudaStreamSynchronize(s->stream));
        CUDA_TRY(s, cudaMemcpyAsync(S.rowrank, rr.data(), nrows * 4, cudaMemcpyHostToDevice, s->stream));
        CUDA_TRY(s, cudaStreamSynchronize(s->stream));
        s->grid_for[0] = n[0];
        s->grid_for[1] = n[1];
        s->grid_for[2] = n[2];
    }
    // tile method: cut the cell grid into tiles (balanced widths), size the shared-memory halo
    S.nt[0] = S.nt[1] = S.nt[2] = 1;
    S.ntiles = 0;
    S.hcap = 0;
    S.cap_it8 = 0;
    if (t.method == RUMD_NB_TILE) {
        if (s->nrep > 1) return fail(s, RUMD_ERR_INVALID_ARG, "replicas use the n2 or the none method (one block per replica)");
        if (t.tp > 8) return fail(s, RUMD_ERR_INVALID_ARG, "the tile method takes tp <= 8");
        if (s->N >= (1 << TILE_GHOST_SHIFT))
            return fail(s, RUMD_ERR_INVALID_ARG, "the tile method takes N < 2^28 (halo slots carry 28-bit particle indices)");
        const int T = t.tile > 0 ? t.tile : (s->N >= 500000 ? 6 : 4);
        size_t ntl = 1;
        double hcells = 1.0;
        for (int k = 0; k < 3; ++k) {
            // a tile plus its halo must stay narrower than the box (w + 4 <= n - 1): the periodic image of every
            // halo particle is then unambiguous, also after a drift of skin/2
            if (n[k] < 6)
                return fail(s, RUMD_ERR_BOX_TOO_SMALL, "tile method needs >= 6 cells per axis, have %dx%dx%d", n[0], n[1], n[2]);
            int ntk = std::max(1, (int)std::lround((double)n[k] / T));
            auto wmax = [&](int q) { return (n[k] + q - 1) / q; };
            while (wmax(ntk) > TILE_WMAX || wmax(ntk) + 5 > n[k]) ++ntk;
            S.nt[k] = ntk;
            ntl *= (size_t)ntk;
            hcells *= wmax(ntk) + 4;
        }
        if (ntl > tile_bound(s))
            return fail(s, RUMD_ERR_INVALID_ARG, "tile method: %zu tiles for %d particles (at most N/32 - 1): use a larger tile", ntl, s->N);
        const double mean = (double)s->N / (double)ncell * hcells;
        // 16-bit list entries hold the slot's byte offset in the shared-memory halo: 16 * slot <= 65535
        // (margin: 15 % + 4 Poisson sigmas; a liquid's density fluctuations on the scale of a halo are far smaller.  A
        // halo that does overflow raises the sticky overflow error of rumd_get_thermo.)
        const size_t hcap = std::min<size_t>(align_up((size_t)(1.15 * mean + 4.0 * std::sqrt(mean) + 32.0), 32), 4095);
        if ((double)hcap < 1.08 * mean + 3.0 * std::sqrt(mean))
            return fail(s, RUMD_ERR_INVALID_ARG, "tile method: a halo of ~%.0f particles does not fit 4095 slots: use a smaller tile", mean);
        if (ntl * hcap > halo_slots_bound(s))
            return fail(s, RUMD_ERR_INVALID_ARG, "tile method: %zu tiles x %zu halo slots exceed the workspace: use a larger tile", ntl, hcap);
        const int chunk = 8 * t.tp; // entries per list iteration of a particle's tp lanes
        const int cap_eff = std::min(s->cap, TILE_ROW_MAX) / chunk * chunk; // (rows are staged in shared memory by the build)
        if (cap_eff < chunk) return fail(s, RUMD_ERR_INVALID_ARG, "list capacity %d below one chunk of the tile method", s->cap);
        S.ntiles = (int)ntl;
        S.hcap = (int)hcap;
        S.cap = cap_eff;
        S.cap_it = cap_eff / t.tp;
        S.cap_it8 = cap_eff / chunk;
        cudaError_t e = cudaFuncSetAttribute(k_build_tile, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tile_smem_bytes(S.hcap));
        if (e != cudaSuccess) return fail(s, RUMD_ERR_CUDA, "tile method: %zu bytes of shared memory refused: %s", tile_smem_bytes(S.hcap), cudaGetErrorString(e));
    }
    s->int_blocks = (s->N + INT_THREADS - 1) / INT_THREADS;
    s->persist_grid_for = -1;
    if (s->nrep > 1) {
        if (t.method == RUMD_NB_CELL) return fail(s, RUMD_ERR_INVALID_ARG, "replicas use the n2 or the none method (one block per replica)");
        // per-replica parameter blocks: the same constants, pointers moved to the replica's slices
        std::vector<Sys> sys((size_t)s->nrep, S);
        const size_t n = (size_t)s->N, npad = (size_t)S.Npad;
        for (int q = 0; q < s->nrep; ++q) {
            Sys& Q = sys[(size_t)q];
            Q.r = S.r + q * n;
            Q.v = S.v + q * n;
            Q.f = S.f + q * n;
            Q.w = S.w + q * n;
            Q.image = S.image + q * n;
            Q.id = S.id + q * n;
            Q.r_out = Q.r;
            Q.r_alt = S.r_alt + q * n;
            Q.r_build = S.r_build + q * n;
            Q.nbl = S.nbl + q * npad * (size_t)S.cap;
            Q.num_nbrs = S.num_nbrs + q * npad;
            Q.sc = s->ens_sc + q;
            Q.prof = nullptr;
        }
        CUDA_TRY(s, cudaStreamSynchronize(s->stream));
        CUDA_TRY(s, cudaMemcpyAsync(s->d_systems, sys.data(), sys.size() * sizeof(Sys), cudaMemcpyHostToDevice, s->stream));
        CUDA_TRY(s, cudaStreamSynchronize(s->stream));
    }
    s->params_dirty = false;
    drop_graphs(s);
    // a list built with other parameters (skin, tp layout, method) is void
    k_request_rebuild<<<1, 1, 0, s->stream>>>(S);
    s->launches++;
    if (s->nrep > 1) {
        k_ens_request_rebuild<<<(s->nrep + 127) / 128, 128, 0, s->stream>>>(s->ens_sc, s->nrep);
        s->launches++;
    }
    CUDA_TRY(s, cudaGetLastError());
    return RUMD_OK;
}

// ---------------------------------------------------------------------------------------------- launch chains

// Kernel selection over (tp, second-term kind, one type): the instantiations live in one translation unit per tp
// (rumd_inst_tp*.cu, built in parallel) and are reached through their KernelSet.
static const KernelSet* kernels_of(const rumd_system* s)
{
    switch (s->tune.tp) {
    case 1: return rumd_kernels_tp1();
    case 2: return rumd_kernels_tp2();
    case 4: return rumd_kernels_tp4();
    case 8: return rumd_kernels_tp8();
    case 16: return rumd_kernels_tp16();
    default: return rumd_kernels_tp32();
    }
}
// second term of the pair potentials: 0 none, 1 Coulomb only (the hot path of configs[4]), 2 any kind of P:73
static int coul_of(const rumd_system* s) { return s->any_coul ? (s->any_generic ? 2 : 1) : 0; }
static bool one_of(const rumd_system* s) { return s->ntypes == 1; }

template <int COUL> static void launch_force_npt(rumd_system* s, int nb)
{
    if (s->ntypes == 1) k_force_npt<COUL, true><<<nb, 256, 0, s->stream>>>(s->S);
    else k_force_npt<COUL, false><<<nb, 256, 0, s->stream>>>(s->S);
}

static int launch_force(rumd_system* s)
{
    if (s->S.npt) { // box from device memory, energy and virial every step (rumd_npt.cuh)
        const int nb = (int)(((long long)s->N * NPT_TP + 255) / 256);
        switch ((s->any_coul ? (s->any_generic ? 2 : 1) : 0)) {
        case 0: launch_force_npt<0>(s, nb); break;
        case 1: launch_force_npt<1>(s, nb); break;
        default: launch_force_npt<2>(s, nb); break;
        }
        return 1;
    }
    if (s->tune.method == RUMD_NB_TILE) { // one block per tile, halo in shared memory
        kernels_of(s)->force_tile(coul_of(s), one_of(s), s->S, s->S.ntiles, tile_smem_bytes_force(s->S.hcap), s->stream);
        return 1;
    }
    const int tp = s->tune.tp, nthreads = s->tune.pb * tp;
    // one virtual warp per warp of the grid: the block scheduler balances better than equal static runs (measured:
    // 156 vs 168 us at N = 10^6)
    const long long nblocks = ((long long)s->N * tp + nthreads - 1) / nthreads;
    kernels_of(s)->force(coul_of(s), one_of(s), s->S, (int)nblocks, nthreads, s->stream);
    return 1;
}

static int persist_threads_of(const rumd_tuning&) { return PERSIST_THREADS; }

// n steps in ONE cooperative launch.  The grid is sized to cover N*tp virtual threads when it can be
// co-resident, else to the co-residency limit (the kernel strides).
static rumd_status launch_persistent(rumd_system* s, int nsteps)
{
    const bool tile = s->tune.method == RUMD_NB_TILE;
    const void* fn = (tile ? kernels_of(s)->persist_tile : kernels_of(s)->persist)[coul_of(s)][one_of(s) ? 1 : 0];
    if (!fn) return fail(s, RUMD_ERR_INVALID_ARG, "the tile method takes tp <= 8");
    int threads = persist_threads_of(s->tune);
    {   // blocks of 512 threads when blocks of 256 would need two per SM and 512 fit one per SM: half the
        // barrier arrivals and thermostat partial sums for the same warps per SM
        const void* wide = tile ? nullptr : kernels_of(s)->persist_wide[coul_of(s)][one_of(s) ? 1 : 0];
        const long long lanes = (long long)s->N * s->tune.tp;
        if (wide && (lanes + threads - 1) / threads > s->num_sms && (lanes + 2 * threads - 1) / (2 * threads) <= s->num_sms) {
            fn = wide;
            threads *= 2;
        } else {
            // more work than that (tp < 8, 80 registers): ONE block of 768 threads per SM instead of three of 256 -- a
            // third of the barrier arrivals, and the 24 warps of an SM work on consecutive particles (N = 10^6: 246 ->
            // 227 us per step, N = 131072: 50.7 -> 47.9)
            const void* wide3 = tile ? nullptr : kernels_of(s)->persist_wide3[coul_of(s)][one_of(s) ? 1 : 0];
            if (wide3 && (lanes + 2 * threads - 1) / (2 * threads) > s->num_sms) {
                fn = wide3;
                threads *= 3;
            }
        }
    }
    const size_t smem = tile ? tile_smem_bytes(s->S.hcap) : 0;
    const int sig = s->tune.tp * 4096 + threads + (s->any_coul ? 1 << 20 : 0) + (s->ntypes == 1 ? 1 << 21 : 0) +
                    (s->any_generic ? 1 << 22 : 0) + (tile ? 1 << 23 : 0);
    if (sig != s->persist_grid_for) { // (refresh() resets persist_grid_for whenever the tiling changes)
        if (tile) CUDA_TRY(s, cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        int per_sm = 0;
        CUDA_TRY(s, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, threads, smem));
        if (per_sm < 1) return fail(s, RUMD_ERR_CUDA, "persistent kernel does not fit an SM");
        // whole multiples of the SM count (every SM carries the same number of blocks; the kernel splits the
        // work into equal contiguous chunks per block), as many as the work can fill, at most what is co-resident
        const long long want = tile ? s->S.ntiles : ((long long)s->N * s->tune.tp + threads - 1) / threads;
        long long per = std::min<long long>(per_sm, (want + s->num_sms - 1) / s->num_sms);
        per = std::max<long long>(1, per);
        s->persist_grid = (int)std::min<long long>(per * s->num_sms, 4096);
        s->persist_threads = threads;
        s->persist_grid_for = sig;
    }
    CUDA_TRY(s, cudaMemsetAsync(s->S.sc->bar, 0, 2 * sizeof(unsigned long long), s->stream));
    int nvt = s->integ == RUMD_INT_NVT_NOSE_HOOVER;
    void* args[] = {(void*)&s->S, (void*)&nsteps, (void*)&nvt};
    CUDA_TRY(s, cudaLaunchCooperativeKernel(fn, dim3(s->persist_grid), dim3(s->persist_threads), args, smem, s->stream));
    s->launches += 1;
    return RUMD_OK;
}

// (rebuild if flag): every kernel of the chain exits at once when the device flag is clear, so the
// chain can be enqueued -- or baked into a graph -- every step without asking the host.
static int launch_rebuild_chain(rumd_system* s)
{
    const Sys& S = s->S;
    int n = 0;
    if (s->tune.method == RUMD_NB_NONE) return 0; // no list to rebuild
    const bool sorting = s->tune.method == RUMD_NB_CELL || s->tune.method == RUMD_NB_TILE || s->tune.sort_interval > 0;
    // Every phase strides over its items, so the grids are capped at a few blocks per SM: on the (many) steps
    // without a rebuild each kernel only reads the flag and exits, and that costs time per BLOCK.
    const int cap256 = s->num_sms * 8, cap128 = s->num_sms * 16;
    if (sorting) {
        const int nbp = std::min((s->N + 255) / 256, cap256);
        const int nchunks = (S.grid.ncell + SCAN_CHUNK - 1) / SCAN_CHUNK;
        k_cell_assign<<<nbp, 256, 0, s->stream>>>(S);
        if (nchunks <= 8) {
            k_scan_single<<<1, SCAN_THREADS, 0, s->stream>>>(S);
            n += 2;
        } else {
            k_scan_sums<<<std::min(nchunks, cap256), SCAN_THREADS, 0, s->stream>>>(S);
            k_scan_blocks<<<1, SCAN_THREADS, 0, s->stream>>>(S);
            k_scan_apply<<<std::min(nchunks, cap256), SCAN_THREADS, 0, s->stream>>>(S);
            n += 4;
        }
        k_cell_scatter<<<nbp, 256, 0, s->stream>>>(S);
        k_permute_gather<<<nbp, 256, 0, s->stream>>>(S);
        k_permute_store<<<nbp, 256, 0, s->stream>>>(S);
        n += 3;
    }
    if (s->S.npt)
        k_build_n2_npt<<<std::min((s->N + 3) / 4, cap128), 128, 0, s->stream>>>(S);
    else if (s->tune.method == RUMD_NB_TILE)
        k_build_tile<<<std::min(S.ntiles, cap256), TILE_THREADS, tile_smem_bytes(S.hcap), s->stream>>>(S);
    else if (s->tune.method == RUMD_NB_CELL) {
        const long long threads = (long long)s->N << S.build_tp_shift;
        k_build_cell<<<(unsigned)std::min<long long>((threads + 127) / 128, cap128), 128, 0, s->stream>>>(S);
    } else
        k_build_n2<<<std::min((s->N + 3) / 4, cap128), 128, 0, s->stream>>>(S);
    return n + 1;
}

static int launch_integrate(rumd_system* s)
{
    if (s->S.npt) {
        k_npt_prepare<<<1, 1024, 0, s->stream>>>(s->S);
        k_integrate_npt<<<s->int_blocks, INT_THREADS, 0, s->stream>>>(s->S);
        return 2;
    }
    k_integrate<<<s->int_blocks, INT_THREADS, 0, s->stream>>>(s->S, s->integ == RUMD_INT_NVT_NOSE_HOOVER);
    return 1;
}

static int launch_step(rumd_system* s)
{
    int n = launch_rebuild_chain(s);
    n += launch_force(s);
    n += launch_integrate(s);
    return n;
}

// entry points that only make sense for a single system
#define SINGLE_ONLY(s)                                                                                   \
    do {                                                                                                 \
        if ((s) && (s)->nrep > 1)                                                                        \
            return fail((s), RUMD_ERR_INVALID_ARG, "not available for a batched ensemble (replicas > 1)"); \
    } while (0)

static rumd_status ready(rumd_system* s, bool need_integ)
{
    if (!s) return RUMD_ERR_INVALID_ARG;
    if (need_integ && !s->integ_set) return fail(s, RUMD_ERR_NOT_READY, "integrator not set");
    return refresh(s);
}

extern "C" rumd_status rumd_build_nblist(rumd_system* s)
{
    SINGLE_ONLY(s);
    rumd_status st = ready(s, false);
    if (st != RUMD_OK) return st;
    k_request_rebuild<<<1, 1, 0, s->stream>>>(s->S);
    s->launches += 1 + launch_rebuild_chain(s);
    CUDA_TRY(s, cudaGetLastError());
    return RUMD_OK;
}

extern "C" rumd_status rumd_compute_forces(rumd_system* s)
{
    SINGLE_ONLY(s);
    rumd_status st = ready(s, false);
    if (st != RUMD_OK) return st;
    s->launches += launch_rebuild_chain(s);
    s->launches += launch_force(s);
    CUDA_TRY(s, cudaGetLastError());
    return RUMD_OK;
}

// Whole-timestep CUDA graph: `steps` time steps (each the full early-exit chain) captured once and replayed;
// removes the per-kernel launch cost that dominates at small N.
// Two fused steps: r -> r_alt -> r.  The second one runs on a copy of the parameter block with the two
// position buffers exchanged (its rebuild chain sorts and lists the positions where they currently are).
static int launch_step_pair(rumd_system* s, bool energy_on_second)
{
    const int tp = s->tune.tp, nthreads = s->tune.pb * tp;
    const int nblocks = (int)(((size_t)s->N * tp + nthreads - 1) / nthreads);
    Sys A = s->S;
    A.r_out = A.r_alt;
    Sys B = s->S;
    B.r = s->S.r_alt;
    B.r_out = s->S.r;
    int n = launch_rebuild_chain(s);
    const int nvt = s->integ == RUMD_INT_NVT_NOSE_HOOVER;
    kernels_of(s)->step(coul_of(s), one_of(s), false, nvt, A, nblocks, nthreads, s->stream);
    n += 1;
    const Sys keep = s->S;
    s->S = B; // the chain launchers read s->S
    n += launch_rebuild_chain(s);
    s->S = keep;
    kernels_of(s)->step(coul_of(s), one_of(s), energy_on_second, nvt, B, nblocks, nthreads, s->stream);
    n += 1;
    return n;
}

static rumd_status get_graph(rumd_system* s, GraphCache& gc, int steps, int* kernels_per_graph)
{
    if (gc.exec && gc.steps == steps) {
        *kernels_per_graph = gc.kernels;
        return RUMD_OK;
    }
    if (gc.exec) cudaGraphExecDestroy(gc.exec);
    gc = GraphCache();
    cudaGraph_t g = nullptr;
    CUDA_TRY(s, cudaStreamBeginCapture(s->stream, cudaStreamCaptureModeThreadLocal));
    int n = 0;
    if (steps % 2 == 0 && s->tune.method != RUMD_NB_TILE && !s->S.npt) // (tile method, NPT: no fused per-step kernel)
        for (int q = 0; q < steps; q += 2) n += launch_step_pair(s, q + 2 == steps);
    else
        for (int q = 0; q < steps; ++q) n += launch_step(s);
    cudaError_t e = cudaStreamEndCapture(s->stream, &g);
    if (e != cudaSuccess) return fail(s, RUMD_ERR_CUDA, "graph capture failed: %s", cudaGetErrorString(e));
    e = cudaGraphInstantiate(&gc.exec, g, 0);
    cudaGraphDestroy(g);
    if (e != cudaSuccess) return fail(s, RUMD_ERR_CUDA, "graph instantiate failed: %s", cudaGetErrorString(e));
    gc.steps = steps;
    gc.kernels = n;
    *kernels_per_graph = n;
    return RUMD_OK;
}

extern "C" rumd_status rumd_run_steps(rumd_system* s, long n)
{
    rumd_status st = ready(s, true);
    if (st != RUMD_OK) return st;
    if (n < 0) return fail(s, RUMD_ERR_INVALID_ARG, "negative step count");
    if (n == 0) return RUMD_OK;
    if (s->nrep > 1) { // batched ensemble: one block per replica runs the whole call
        for (long left = n; left > 0;) {
            int chunk = (int)std::min<long>(left, 1L << 20);
            int nvt = s->integ == RUMD_INT_NVT_NOSE_HOOVER;
            void* args[] = {(void*)&s->d_systems, (void*)&chunk, (void*)&nvt};
            CUDA_TRY(s, cudaLaunchKernel(kernels_of(s)->ensemble[coul_of(s)][one_of(s) ? 1 : 0], dim3(s->nrep), dim3(ENS_THREADS), args, 0,
                                         s->stream));
            s->launches += 1;
            left -= chunk;
        }
        return RUMD_OK;
    }
    if (s->tune.persistent && !s->S.npt) { // (NPT runs on the per-step kernels, rumd_npt.cuh)
        // one cooperative launch per <= 2^16 steps (keeps the 32-bit arrival count of the grid barrier in range)
        for (long left = n; left > 0;) {
            const int chunk = (int)std::min<long>(left, 1L << 16);
            st = launch_persistent(s, chunk);
            if (st != RUMD_OK) return st;
            left -= chunk;
        }
        return RUMD_OK;
    }
    if (!s->tune.use_graph) {
        for (long q = 0; q < n; ++q) s->launches += launch_step(s);
        CUDA_TRY(s, cudaGetLastError());
        return RUMD_OK;
    }
    int spg = s->tune.steps_per_graph > 0 ? s->tune.steps_per_graph : 32;
    long left = n;
    if (left >= spg) {
        int kpg = 0;
        st = get_graph(s, s->graph_multi, spg, &kpg);
        if (st != RUMD_OK) return st;
        while (left >= spg) {
            CUDA_TRY(s, cudaGraphLaunch(s->graph_multi.exec, s->stream));
            s->launches += kpg;
            left -= spg;
        }
    }
    if (left > 0) {
        int kpg = 0;
        st = get_graph(s, s->graph_one, 1, &kpg);
        if (st != RUMD_OK) return st;
        for (; left > 0; --left) {
            CUDA_TRY(s, cudaGraphLaunch(s->graph_one.exec, s->stream));
            s->launches += kpg;
        }
    }
    return RUMD_OK;
}

// ---------------------------------------------------------------------------------------------- read-back

extern "C" rumd_status rumd_export_nblist(rumd_system* s, void* d_count, void* d_list, int row_capacity)
{
    SINGLE_ONLY(s);
    rumd_status st = ready(s, false);
    if (st != RUMD_OK) return st;
    if (!d_count || !d_list || row_capacity < 1) return fail(s, RUMD_ERR_INVALID_ARG, "bad export arguments");
    if (s->tune.method == RUMD_NB_TILE)
        k_export_nbl_tile<<<s->N, 128, 0, s->stream>>>(s->S, (int*)d_count, (int*)d_list, row_capacity);
    else
        k_export_nbl<<<s->N, 128, 0, s->stream>>>(s->S, (int*)d_count, (int*)d_list, row_capacity);
    s->launches++;
    CUDA_TRY(s, cudaGetLastError());
    return RUMD_OK;
}

extern "C" rumd_status rumd_get_thermo(rumd_system* s, rumd_thermo* out)
{
    SINGLE_ONLY(s);
    rumd_status st = ready(s, false);
    if (st != RUMD_OK) return st;
    if (!out) return fail(s, RUMD_ERR_INVALID_ARG, "null output");
    k_thermo<<<1, 1024, 0, s->stream>>>(s->S);
    s->launches++;
    CUDA_TRY(s, cudaMemcpyAsync(s->h_sc, s->S.sc, sizeof(DevScalars), cudaMemcpyDeviceToHost, s->stream));
    CUDA_TRY(s, cudaStreamSynchronize(s->stream));
    CUDA_TRY(s, cudaGetLastError());
    const DevScalars& d = *s->h_sc;
    out->U = d.U;
    out->W = d.W;
    out->K = d.K;
    out->mv2 = d.mv2;
    out->xi = d.xi;
    out->eta = d.eta;
    double H = d.K + d.U;
    if (s->integ != RUMD_INT_NVE_LEAPFROG) { // O10
        // K and U belong to time t of the last step; xi, eta are already at t + dt, so H(t) uses the
        // values step_tail kept for time t (xi_t, eta_t).
        H += s->S.g * s->S.T0 * d.eta_t;
        if (s->S.omega2 > 0) H += 0.5 * s->S.g * s->S.T0 * d.xi_t * d.xi_t / s->S.omega2;
    }
    if (s->integ == RUMD_INT_NPT_MTK) { // reading S32: + P0 V(t) + Wb nu(t)^2 / 2, Wb = (g + 3) T0 / wP^2 = 1 / cP
        H += s->S.P0 * d.vol_t;
        if (s->S.cP > 0) H += 0.5 * d.nu_t * d.nu_t / s->S.cP;
    }
    out->H = H;
    out->n_steps = d.n_steps;
    out->n_rebuilds = d.n_rebuilds;
    // longest row of the last completed build; a list built by rumd_build_nblist whose force evaluation has not
    // run yet still owns the flag and its slot (a flag raised by the displacement check finds that slot zeroed)
    int max_nbrs = d.last_max;
    if (d.flag && d.max_nbrs[d.n_rebuilds & 1] > 0) max_nbrs = d.max_nbrs[d.n_rebuilds & 1];
    out->max_nbrs = max_nbrs;
    out->nbl_capacity = s->cap;
    out->overflow = (int)d.overflow;
    out->pad_ = 0;
    if (d.overflow == 2u)
        return fail(s, RUMD_ERR_NBL_OVERFLOW, "tile method: a tile's halo holds more than %d particles (density far from uniform): use a smaller tile or the cell method", s->S.hcap);
    if (d.overflow) return fail(s, RUMD_ERR_NBL_OVERFLOW, "neighbour list overflow: %d neighbours > capacity %d", max_nbrs, s->S.cap);
    if (d.nonfinite == 2) return fail(s, RUMD_ERR_CUDA, "persistent kernel: grid barrier timed out");
    if (d.nonfinite == 3) return fail(s, RUMD_ERR_BOX_TOO_SMALL, "NPT: the box shrank below 2 (rc_max + skin)");
    if (d.nonfinite) return fail(s, RUMD_ERR_NONFINITE, "non-finite energy");
    return RUMD_OK;
}

// Per-replica thermodynamic scalars of a batched ensemble; U, W, K refer to the last step of the last run.
extern "C" rumd_status rumd_get_thermo_replicas(rumd_system* s, rumd_thermo* out, int n_out)
{
    rumd_status st = ready(s, false);
    if (st != RUMD_OK) return st;
    if (s->nrep < 2) return fail(s, RUMD_ERR_INVALID_ARG, "no replicas: use rumd_get_thermo");
    if (!out || n_out < s->nrep) return fail(s, RUMD_ERR_INVALID_ARG, "output array too small");
    std::vector<DevScalars> h((size_t)s->nrep);
    CUDA_TRY(s, cudaMemcpyAsync(h.data(), s->ens_sc, h.size() * sizeof(DevScalars), cudaMemcpyDeviceToHost, s->stream));
    CUDA_TRY(s, cudaStreamSynchronize(s->stream));
    CUDA_TRY(s, cudaGetLastError());
    rumd_status worst = RUMD_OK;
    for (int q = 0; q < s->nrep; ++q) {
        const DevScalars& d = h[(size_t)q];
        rumd_thermo& o = out[q];
        o.U = d.U;
        o.W = d.W;
        o.K = d.K;
        o.mv2 = d.mv2;
        o.xi = d.xi;
        o.eta = d.eta;
        o.H = d.K + d.U;
        if (s->integ == RUMD_INT_NVT_NOSE_HOOVER) {
            o.H += s->S.g * s->S.T0 * d.eta_t;
            if (s->S.omega2 > 0) o.H += 0.5 * s->S.g * s->S.T0 * d.xi_t * d.xi_t / s->S.omega2;
        }
        o.n_steps = d.n_steps;
        o.n_rebuilds = d.n_rebuilds;
        o.max_nbrs = d.max_nbrs[0];
        o.nbl_capacity = s->cap;
        o.overflow = (int)d.overflow;
        o.pad_ = 0;
        if (d.overflow) worst = fail(s, RUMD_ERR_NBL_OVERFLOW, "neighbour list overflow in replica %d: %d neighbours > capacity %d", q, d.max_nbrs[0], s->cap);
        else if (d.nonfinite && worst == RUMD_OK) worst = fail(s, RUMD_ERR_NONFINITE, "non-finite energy in replica %d", q);
    }
    return worst;
}

extern "C" rumd_status rumd_get_box(rumd_system* s, double* box_out, double* nu_out)
{
    SINGLE_ONLY(s);
    rumd_status st = ready(s, false);
    if (st != RUMD_OK) return st;
    if (!box_out) return fail(s, RUMD_ERR_INVALID_ARG, "null output");
    CUDA_TRY(s, cudaMemcpyAsync(s->h_sc, s->S.sc, sizeof(DevScalars), cudaMemcpyDeviceToHost, s->stream));
    CUDA_TRY(s, cudaStreamSynchronize(s->stream));
    const bool npt = s->integ == RUMD_INT_NPT_MTK;
    for (int k = 0; k < 3; ++k) box_out[k] = npt ? s->h_sc->box[k] : (double)s->box[k];
    if (nu_out) *nu_out = npt ? s->h_sc->nu_o : 0.0;
    return RUMD_OK;
}

extern "C" rumd_status rumd_snapshot(rumd_system* s)
{
    SINGLE_ONLY(s);
    rumd_status st = ready(s, false);
    if (st != RUMD_OK) return st;
    const Sys& S = s->S;
    k_copy_state<<<(s->N + 255) / 256, 256, 0, s->stream>>>(s->N, S.r, S.v, S.image, S.id, s->snap_r, s->snap_v,
                                                           s->snap_image, s->snap_id);
    s->launches++;
    CUDA_TRY(s, cudaMemcpyAsync(s->snap_sc, S.sc, sizeof(DevScalars), cudaMemcpyDeviceToDevice, s->stream));
    CUDA_TRY(s, cudaGetLastError());
    return RUMD_OK;
}

extern "C" rumd_status rumd_restore(rumd_system* s)
{
    SINGLE_ONLY(s);
    rumd_status st = ready(s, false);
    if (st != RUMD_OK) return st;
    const Sys& S = s->S;
    k_copy_state<<<(s->N + 255) / 256, 256, 0, s->stream>>>(s->N, s->snap_r, s->snap_v, s->snap_image, s->snap_id,
                                                           S.r, S.v, S.image, S.id);
    CUDA_TRY(s, cudaMemcpyAsync(S.sc, s->snap_sc, sizeof(DevScalars), cudaMemcpyDeviceToDevice, s->stream));
    k_request_rebuild<<<1, 1, 0, s->stream>>>(S);
    s->launches += 2;
    CUDA_TRY(s, cudaGetLastError());
    return RUMD_OK;
}

extern "C" rumd_status rumd_upload_state(rumd_system* s, const void* h_r, const void* h_v, const void* h_image,
                                         const void* h_id)
{
    rumd_status st = ready(s, false);
    if (st != RUMD_OK) return st;
    const size_t N = (size_t)s->N * (size_t)s->nrep;
    if (h_r) { // the type in r.w indexes the pair table in every kernel: check it here, where it is cheap
        const int* bits = (const int*)h_r;
        for (size_t i = 0; i < N; ++i)
            if (bits[4 * i + 3] < 0 || bits[4 * i + 3] >= s->ntypes)
                return fail(s, RUMD_ERR_INVALID_ARG, "particle %zu has type %d, outside [0, %d)", i, bits[4 * i + 3], s->ntypes);
    }
    if (h_r) CUDA_TRY(s, cudaMemcpyAsync(s->S.r, h_r, N * 16, cudaMemcpyHostToDevice, s->stream));
    if (h_v) CUDA_TRY(s, cudaMemcpyAsync(s->S.v, h_v, N * 16, cudaMemcpyHostToDevice, s->stream));
    if (h_image) CUDA_TRY(s, cudaMemcpyAsync(s->S.image, h_image, N * 16, cudaMemcpyHostToDevice, s->stream));
    if (h_id) CUDA_TRY(s, cudaMemcpyAsync(s->S.id, h_id, N * 4, cudaMemcpyHostToDevice, s->stream));
    k_reset_scalars<<<1, 1, 0, s->stream>>>(s->S);
    s->launches++;
    ens_reset(s);
    CUDA_TRY(s, cudaGetLastError());
    return RUMD_OK;
}

extern "C" rumd_status rumd_download_state(rumd_system* s, void* h_r, void* h_v, void* h_f, void* h_w,
                                           void* h_image, void* h_id)
{
    rumd_status st = ready(s, false);
    if (st != RUMD_OK) return st;
    const size_t N = (size_t)s->N * (size_t)s->nrep;
    if (h_r) CUDA_TRY(s, cudaMemcpyAsync(h_r, s->S.r, N * 16, cudaMemcpyDeviceToHost, s->stream));
    if (h_v) CUDA_TRY(s, cudaMemcpyAsync(h_v, s->S.v, N * 16, cudaMemcpyDeviceToHost, s->stream));
    if (h_f) CUDA_TRY(s, cudaMemcpyAsync(h_f, s->S.f, N * 16, cudaMemcpyDeviceToHost, s->stream));
    if (h_w) CUDA_TRY(s, cudaMemcpyAsync(h_w, s->S.w, N * 4, cudaMemcpyDeviceToHost, s->stream));
    if (h_image) CUDA_TRY(s, cudaMemcpyAsync(h_image, s->S.image, N * 16, cudaMemcpyDeviceToHost, s->stream));
    if (h_id) CUDA_TRY(s, cudaMemcpyAsync(h_id, s->S.id, N * 4, cudaMemcpyDeviceToHost, s->stream));
    CUDA_TRY(s, cudaStreamSynchronize(s->stream));
    return RUMD_OK;
}

// One un-graphed step with events around each kernel class (launch-gap / share analysis at small N).
extern "C" rumd_status rumd_profile_step(rumd_system* s, float* ms_out, int* did_rebuild_out)
{
    SINGLE_ONLY(s);
    rumd_status st = ready(s, true);
    if (st != RUMD_OK) return st;
    if (!ms_out) return fail(s, RUMD_ERR_INVALID_ARG, "null output");
    CUDA_TRY(s, cudaMemcpyAsync(s->h_sc, s->S.sc, sizeof(DevScalars), cudaMemcpyDeviceToHost, s->stream));
    CUDA_TRY(s, cudaStreamSynchronize(s->stream));
    const int did = s->h_sc->flag != 0;
    cudaEvent_t ev[4] = {nullptr, nullptr, nullptr, nullptr};
    cudaError_t e = cudaSuccess;
    for (auto& x : ev)
        if (e == cudaSuccess) e = cudaEventCreate(&x);
    if (e == cudaSuccess) {
        cudaEventRecord(ev[0], s->stream);
        s->launches += launch_rebuild_chain(s);
        cudaEventRecord(ev[1], s->stream);
        s->launches += launch_force(s);
        cudaEventRecord(ev[2], s->stream);
        s->launches += launch_integrate(s);
        cudaEventRecord(ev[3], s->stream);
        e = cudaStreamSynchronize(s->stream);
    }
    if (e == cudaSuccess)
        for (int q = 0; q < 3 && e == cudaSuccess; ++q) e = cudaEventElapsedTime(&ms_out[q], ev[q], ev[q + 1]);
    for (auto& x : ev) // the events are destroyed on every path
        if (x) cudaEventDestroy(x);
    if (e == cudaSuccess) e = cudaGetLastError();
    if (e != cudaSuccess) return fail(s, RUMD_ERR_CUDA, "profile step failed: %s", cudaGetErrorString(e));
    ms_out[3] = 0.f;
    if (did_rebuild_out) *did_rebuild_out = did;
    return RUMD_OK;
}

// Average device time of ONE force-kernel launch (current tuning, current list): `reps` launches captured in
// a graph (no host launch gaps), bracketed by CUDA events on the library's stream.  The list must exist.
extern "C" rumd_status rumd_time_force(rumd_system* s, int reps, float* us_per_launch)
{
    SINGLE_ONLY(s);
    rumd_status st = ready(s, false);
    if (st != RUMD_OK) return st;
    if (reps < 1 || !us_per_launch) return fail(s, RUMD_ERR_INVALID_ARG, "bad arguments");
    cudaGraph_t g = nullptr;
    cudaGraphExec_t ex = nullptr;
    CUDA_TRY(s, cudaStreamBeginCapture(s->stream, cudaStreamCaptureModeThreadLocal));
    for (int q = 0; q < reps; ++q) launch_force(s);
    cudaError_t e = cudaStreamEndCapture(s->stream, &g);
    if (e != cudaSuccess) return fail(s, RUMD_ERR_CUDA, "graph capture failed: %s", cudaGetErrorString(e));
    e = cudaGraphInstantiate(&ex, g, 0);
    cudaGraphDestroy(g);
    if (e != cudaSuccess) return fail(s, RUMD_ERR_CUDA, "graph instantiate failed: %s", cudaGetErrorString(e));
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    cudaGraphLaunch(ex, s->stream); // warm-up
    cudaEventRecord(e0, s->stream);
    cudaGraphLaunch(ex, s->stream);
    cudaEventRecord(e1, s->stream);
    cudaError_t es = cudaStreamSynchronize(s->stream);
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaGraphExecDestroy(ex);
    s->launches += 2LL * reps;
    if (es != cudaSuccess) return fail(s, RUMD_ERR_CUDA, "force timing failed: %s", cudaGetErrorString(es));
    *us_per_launch = 1000.f * ms / (float)reps;
    return RUMD_OK;
}

// Where the time of the persistent kernel goes: runs n steps with the cycle counters of block 0 switched on.
extern "C" rumd_status rumd_profile_persistent(rumd_system* s, int nsteps, double* out8)
{
    SINGLE_ONLY(s);
    rumd_status st = ready(s, true);
    if (st != RUMD_OK) return st;
    if (nsteps < 1 || !out8) return fail(s, RUMD_ERR_INVALID_ARG, "bad arguments");
    CUDA_TRY(s, cudaMemsetAsync(s->prof_buf, 0, 64, s->stream));
    s->S.prof = s->prof_buf;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    cudaEventRecord(e0, s->stream);
    st = launch_persistent(s, nsteps);
    cudaEventRecord(e1, s->stream);
    s->S.prof = nullptr;
    long long h[8];
    cudaError_t e = cudaMemcpyAsync(h, s->prof_buf, 64, cudaMemcpyDeviceToHost, s->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s->stream);
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    if (st != RUMD_OK) return st;
    if (e != cudaSuccess) return fail(s, RUMD_ERR_CUDA, "profiling run failed: %s", cudaGetErrorString(e));
    // convert cycles to microseconds per step with the kernel's own total (cycles <-> event time)
    const double us_total = 1000.0 * ms, cyc_total = (double)h[5];
    for (int q = 0; q < 5; ++q) out8[q] = cyc_total > 0 ? (double)h[q] / cyc_total * us_total / nsteps : 0.0;
    out8[5] = us_total / nsteps;
    out8[6] = (double)h[6];
    out8[7] = (double)h[7];
    return RUMD_OK;
}

// FP32 peak as measured, not derived ("the builder should add an FFMA-chain microbenchmark and quote
// fractions against both the formula and the measured value").  Every thread runs 16 independent register-operand
// FFMA chains; 2 blocks of 1024 threads per SM (full occupancy), so the FMA pipes never wait on a dependency.
#define PEAK_CHAINS 16
static __global__ void __launch_bounds__(1024, 2) k_ffma_peak(float* out, int iters, float b0, float c0)
{
    float x[PEAK_CHAINS];
    const float b = b0 + 1e-9f * (float)threadIdx.x, c = c0 + 1e-9f * (float)blockIdx.x;
#pragma unroll
    for (int q = 0; q < PEAK_CHAINS; ++q) x[q] = (float)(threadIdx.x + q);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 4; ++u)
#pragma unroll
            for (int q = 0; q < PEAK_CHAINS; ++q) x[q] = __fmaf_rn(x[q], b, c);
    }
    float acc = 0.f;
#pragma unroll
    for (int q = 0; q < PEAK_CHAINS; ++q) acc += x[q];
    if (acc == 123.456f) out[0] = acc; // never true in practice: keeps the chains alive
}

// Measured FP32 FMA throughput of this GPU in TFLOP/s (2 flop per FFMA): best of `reps` launches timed with CUDA
// events on the library's stream.  scratch: any 4 writable device bytes are taken from the workspace.
extern "C" rumd_status rumd_measure_fp32_peak(rumd_system* s, int reps, double* tflops_out)
{
    if (!s || !tflops_out || reps < 1) return RUMD_ERR_INVALID_ARG;
    if (!s->ws_bound) return fail(s, RUMD_ERR_NOT_READY, "bind a workspace first");
    const int iters = 4096, blocks = 2 * s->num_sms, threads = 1024;
    const double flop = 2.0 * 4.0 * PEAK_CHAINS * (double)iters * (double)blocks * threads;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    cudaError_t e = cudaEventCreate(&e0);
    if (e == cudaSuccess) e = cudaEventCreate(&e1);
    double best = 0.0;
    for (int r = 0; r <= reps && e == cudaSuccess; ++r) { // launch 0 is the warm-up
        cudaEventRecord(e0, s->stream);
        k_ffma_peak<<<blocks, threads, 0, s->stream>>>((float*)s->prof_buf, iters, 0.999f, 0.001f);
        cudaEventRecord(e1, s->stream);
        e = cudaStreamSynchronize(s->stream);
        float ms = 0.f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
        if (e == cudaSuccess && r > 0 && ms > 0.f) best = std::max(best, flop / (ms * 1e-3) / 1e12);
        s->launches++;
    }
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    if (e != cudaSuccess) return fail(s, RUMD_ERR_CUDA, "fp32 peak measurement failed: %s", cudaGetErrorString(e));
    *tflops_out = best;
    return RUMD_OK;
}

// ---------------------------------------------------------------------------------------------- A8: autotuner

// One trial (every trial restarts from the same stored state): restore, warm up (includes the first
// build), time `steps` steps with CUDA events.  Returns steps per second, or 0 when the setting is not
// admissible (box too small for it, list overflow).
static double trial(rumd_system* s, const rumd_tuning& t, int steps)
{
    if (rumd_set_tuning(s, &t) != RUMD_OK) return 0.0;
    if (rumd_restore(s) != RUMD_OK) return 0.0;
    const int warm = std::max(8, steps / 4);
    if (rumd_run_steps(s, warm) != RUMD_OK) return 0.0;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    cudaEventRecord(e0, s->stream);
    rumd_status st = rumd_run_steps(s, steps);
    cudaEventRecord(e1, s->stream);
    rumd_thermo th;
    rumd_status st2 = rumd_get_thermo(s, &th);
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    if (st != RUMD_OK || st2 != RUMD_OK || !(ms > 0.f)) return 0.0;
    return 1000.0 * steps / ms;
}

// Coordinate descent over (method, tp, cell-build lanes, skin, persistent vs per-step kernels, block size).
// The paper's empirical claim that the time has a single minimum along each of pb, tp and skin is
// what makes this sound; the loop-breaking rules follow P:386-391 in spirit (stop a direction once it is
// worse than the best).  The B200 dimensions the paper does not have: lanes per particle of the cell build
// ("not been tried yet") and the persistent whole-run kernel vs per-step kernels in CUDA graphs.
namespace {
struct Tuner {
    rumd_system* s;
    int steps;
    rumd_tuning cur;
    double cur_tps = 0.0;
    int trials = 0;
    bool try_setting(const rumd_tuning& c)
    {
        ++trials;
        const double tps = trial(s, c, steps);
        if (tps > cur_tps) {
            cur = c;
            cur_tps = tps;
            return true;
        }
        return false;
    }
    // walk one parameter both ways with `next(c, dir)` (returns false when out of range) until no gain
    template <class Next> void descend(Next next)
    {
        for (int dir = -1; dir <= 1; dir += 2) {
            rumd_tuning c = cur;
            while (next(c, dir) && try_setting(c)) {}
        }
    }
};
} // namespace

extern "C" rumd_status rumd_autotune(rumd_system* s, rumd_tuning* out, int steps_per_trial, double* tps_out)
{
    SINGLE_ONLY(s);
    rumd_status st = ready(s, true);
    if (st != RUMD_OK) return st;
    if (s->integ == RUMD_INT_NPT_MTK) return fail(s, RUMD_ERR_INVALID_ARG, "autotune is not available for NPT (per-step kernels, n2 / none only)");
    if (steps_per_trial < 8) steps_per_trial = 8;
    const rumd_tuning saved = s->tune;
    st = rumd_snapshot(s);
    if (st != RUMD_OK) return st;
    const double rcm = rc_max_of(s);
    const double minL = std::min(s->box[0], std::min(s->box[1], s->box[2]));
    const float skin_max = (float)(0.5 * minL - rcm - 1e-4);
    rumd_tuning best = saved;
    double best_tps = 0.0;
    std::vector<int> methods;
    if (s->N <= 5000) methods.push_back(RUMD_NB_NONE); // "none" is not tried above 5000 particles
    if (s->N <= 20000) methods.push_back(RUMD_NB_N2); // n2 is not tried for large systems
    methods.push_back(RUMD_NB_CELL);
    if (s->N >= 4096) methods.push_back(RUMD_NB_TILE); // shared-memory staging needs tiles of >= 32 particles
    for (int method : methods) {
        rumd_tuning start;
        rumd_default_tuning(s, &start);
        start.method = method;
        if (method == RUMD_NB_TILE && start.tp > 8) {
            start.tp = 8;
            start.pb = 32;
        }
        start.skin = std::min(saved.skin, skin_max);
        if (!(start.skin > 0.f)) continue;
        Tuner T{s, steps_per_trial, start};
        if (!T.try_setting(start)) continue; // e.g. grid too coarse for the stencil (S18)
        for (int round = 0; round < 2; ++round) {
            const double before = T.cur_tps;
            T.descend([](rumd_tuning& c, int dir) { // threads per particle
                const int tp = dir < 0 ? c.tp / 2 : c.tp * 2;
                if (tp < 1 || tp > (c.method == RUMD_NB_TILE ? 8 : 32)) return false;
                const int threads = std::max(32, c.pb * c.tp);
                c.tp = tp;
                c.pb = std::max(1, threads / tp);
                return true;
            });
            T.descend([&](rumd_tuning& c, int dir) { // skin, +-15 % steps until the minimum is bracketed
                const float sk = c.skin * (dir < 0 ? 0.85f : 1.15f);
                if (sk < 0.05f || sk > skin_max) return false;
                c.skin = sk;
                return true;
            });
            if (method == RUMD_NB_CELL)
                T.descend([&](rumd_tuning& c, int dir) { // lanes per particle of the cell build
                    const int cur_b = c.build_tp > 0 ? c.build_tp : 1 << s->S.build_tp_shift;
                    const int b = dir < 0 ? cur_b / 2 : cur_b * 2;
                    if (b < 1 || b > 32) return false;
                    c.build_tp = b;
                    return true;
                });
            if (method == RUMD_NB_TILE)
                T.descend([&](rumd_tuning& c, int dir) { // tile edge in cells: halo overhead against blocks per SM
                    const int cur_t = c.tile > 0 ? c.tile : (s->N >= 500000 ? 6 : 4);
                    const int tl = cur_t + dir;
                    if (tl < 2 || tl > TILE_WMAX) return false;
                    c.tile = tl;
                    return true;
                });
            if (T.cur_tps < 1.02 * before) break;
        }
        if (method == RUMD_NB_N2 && s->N >= 1024) { // P:379 step 5: with n2, how often to re-sort the particles
            rumd_tuning c = T.cur;
            for (int si : {1, 4, 16}) {
                c.sort_interval = si;
                T.try_setting(c);
            }
        }
        if (method != RUMD_NB_TILE) { // per-step kernels in CUDA graphs instead of the persistent kernel; there the block size matters
            rumd_tuning c = T.cur;
            c.persistent = 0;
            c.use_graph = 1;
            if (T.try_setting(c))
                T.descend([](rumd_tuning& q, int dir) {
                    const int th = dir < 0 ? q.pb * q.tp / 2 : q.pb * q.tp * 2;
                    if (th < 32 || th > 1024 || th / q.tp < 1) return false;
                    q.pb = th / q.tp;
                    return true;
                });
        }
        if (T.cur_tps > best_tps) {
            best_tps = T.cur_tps;
            best = T.cur;
        }
    }
    rumd_status r1 = rumd_set_tuning(s, best_tps > 0.0 ? &best : &saved);
    rumd_status r2 = rumd_restore(s);
    if (r1 != RUMD_OK) return r1;
    if (r2 != RUMD_OK) return r2;
    CUDA_TRY(s, cudaStreamSynchronize(s->stream));
    if (best_tps <= 0.0) return fail(s, RUMD_ERR_NOT_READY, "autotune: no admissible setting");
    if (out) *out = best;
    if (tps_out) *tps_out = best_tps;
    return RUMD_OK;
}

// ---------------------------------------------------------------------------------------------- D10: tuning cache

// P:382 step 8: the tuned parameters are written to a file and reused by later runs with "the same user
// parameters" (system size, density, potential parameters, integrator, time step, temperature, GPU type).
// One JSON object per line; the key is a canonical string of exactly those inputs.
static std::string tuning_key(const rumd_system* s)
{
    char buf[256];
    std::string k;
    cudaDeviceProp prop;
    int dev = 0;
    cudaGetDevice(&dev);
    if (cudaGetDeviceProperties(&prop, dev) == cudaSuccess) k += prop.name;
    snprintf(buf, sizeof buf, "|N=%d|nt=%d|box=%.9g,%.9g,%.9g|int=%d|dt=%.9g|T=%.9g|tau=%.9g|rep=%d", s->N, s->ntypes,
             s->box[0], s->box[1], s->box[2], s->integ, s->dt, s->T0, s->tau, s->nrep);
    k += buf;
    for (int a = 0; a < s->ntypes; ++a)
        for (int b = a; b < s->ntypes; ++b) {
            const PotSlot& p = s->pot[a][b];
            snprintf(buf, sizeof buf, "|%d%d:lj=%d,%.9g,%.9g,%.9g,%d;x=%d,%d,%.9g,%.9g,%.9g,%.9g,%.9g,%d", a, b, (int)p.lj, p.eps,
                     p.sig, p.rc_lj, p.cut_lj, (int)p.coul, p.kind2, p.qq, p.b2, p.c2, p.d2, p.rc_c, p.cut_c);
            k += buf;
        }
    return k;
}

static bool cache_lookup(const char* path, const std::string& key, rumd_tuning* t, double* tps)
{
    FILE* f = fopen(path, "r");
    if (!f) return false;
    bool found = false;
    std::vector<char> line(8192);
    const std::string want = "{\"key\": \"" + key + "\", ";
    while (fgets(line.data(), (int)line.size(), f)) {
        if (strncmp(line.data(), want.c_str(), want.size()) != 0) continue;
        rumd_tuning c;
        double v = 0;
        if (sscanf(line.data() + want.size(),
                   "\"method\": %d, \"pb\": %d, \"tp\": %d, \"skin\": %f, \"sort_interval\": %d, \"use_graph\": %d, "
                   "\"steps_per_graph\": %d, \"persistent\": %d, \"build_tp\": %d, \"tile\": %d, \"timesteps_per_s\": %lf",
                   &c.method, &c.pb, &c.tp, &c.skin, &c.sort_interval, &c.use_graph, &c.steps_per_graph, &c.persistent,
                   &c.build_tp, &c.tile, &v) == 11) {
            *t = c; // the LAST matching line wins (a re-tune appends)
            *tps = v;
            found = true;
        }
    }
    fclose(f);
    return found;
}

// rumd_autotune with the paper's parameter file: a cached setting for the same inputs is applied without any
// trial run; otherwise the autotuner runs and its result is appended to the file.
extern "C" rumd_status rumd_autotune_cached(rumd_system* s, rumd_tuning* out, int steps_per_trial, double* tps_out,
                                            const char* cache_path, int* from_cache_out)
{
    if (!s) return RUMD_ERR_INVALID_ARG;
    if (from_cache_out) *from_cache_out = 0;
    if (!cache_path || !*cache_path) return rumd_autotune(s, out, steps_per_trial, tps_out);
    rumd_status st = ready(s, true);
    if (st != RUMD_OK) return st;
    const std::string key = tuning_key(s);
    rumd_tuning t;
    double tps = 0;
    if (cache_lookup(cache_path, key, &t, &tps) && rumd_set_tuning(s, &t) == RUMD_OK && refresh(s) == RUMD_OK) {
        if (out) *out = t;
        if (tps_out) *tps_out = tps;
        if (from_cache_out) *from_cache_out = 1;
        return RUMD_OK;
    }
    st = rumd_autotune(s, &t, steps_per_trial, &tps);
    if (st != RUMD_OK) return st;
    if (out) *out = t;
    if (tps_out) *tps_out = tps;
    FILE* f = fopen(cache_path, "a");
    if (!f) return fail(s, RUMD_ERR_INVALID_ARG, "cannot write the tuning cache %s", cache_path);
    fprintf(f,
            "{\"key\": \"%s\", \"method\": %d, \"pb\": %d, \"tp\": %d, \"skin\": %.9g, \"sort_interval\": %d, \"use_graph\": %d, "
            "\"steps_per_graph\": %d, \"persistent\": %d, \"build_tp\": %d, \"tile\": %d, \"timesteps_per_s\": %.6g}\n",
            key.c_str(), t.method, t.pb, t.tp, (double)t.skin, t.sort_interval, t.use_graph, t.steps_per_graph, t.persistent,
            t.build_tp, t.tile, tps);
    fclose(f);
    return RUMD_OK;
}
