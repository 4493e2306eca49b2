// rumd_types.cuh -- device-visible parameter blocks of librumd_b200 (sm_100a).  Product code: shares nothing
// with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define RUMD_MAXT 4
// Dzugutov potential, published constants (u = A (x^-16 - B) exp(c / (x - a)) [x < a] + B exp(d / (x - b)) [x < b])
#define DZ_A 5.82
#define DZ_B 1.28
#define DZ_a 1.87
#define DZ_b 1.94
#define DZ_c 1.1
#define DZ_d 0.27

// One record per ORDERED type pair; all derived constants are computed on the host in double precision
// from the user's fp32 parameters and rounded once.
//   LJ 12-6 (O3):  u = c12/r^12 - c6/r^6,  c12 = 4 eps sigma^12, c6 = 4 eps sigma^6
//   shifted force: u_SF = u(r) + fc*r - k0,  f_SF/r = f(r)/r - fc/r,  fc = f(rc), k0 = u(rc) + rc*fc
//   Coulomb (O4):  u = qq/r, same shift with fc = qq/rc^2, k0 = 2 qq/rc
struct __align__(16) PairParams {
    float c12x12, c6x6, rc2_lj, fc_lj; // float4 #0: force, LJ term
    float qq, rc2_c, fc_c, rc2_max;    // float4 #1: force, second term (qq = its prefactor a); rc2_max = max rc^2
    float c12, c6, k0_lj, k0_c;        // float4 #2: energies
    float rcl2, kind2, p1, p2;         // float4 #3: rcl2 = (rc_ab + skin)^2 list cutoff (S4); second term: kind
                                       // as int bits (0 Coulomb 1 IPL 2 Yukawa 3 Gaussian core 4 Buckingham), parameters
};

// Device scalars living in the workspace.
struct DevScalars {
    double xi, eta;       // Nose-Hoover variables (O7), at the time AFTER the last step
    double xi_t, eta_t;   // their values at the integer time t of the last step (for H(t), O10)
    double K, mv2;        // O10 kinetic energy at integer time; sum m v(t+dt/2)^2
    double U, W;          // filled by the thermo reduction
    long long n_steps;
    long long n_rebuilds;
    unsigned long long bar[2]; // persistent kernel: the two arrival counters of its grid barrier
    unsigned int flag;    // rebuild requested for the NEXT force evaluation (P:179 updateRequired)
    unsigned int pending; // set by the integrator's displacement check during a step
    unsigned int ticket;  // last-block-done counter of the integrator
    unsigned int overflow;
    int max_nbrs[2];      // largest list length of build number b in slot b & 1
    int nonfinite;        // 1: NaN/Inf energy; 2: grid barrier timed out
    int last_max;         // largest list length of the last COMPLETED build (written when its force evaluation starts)
    int build_queue;      // cell build inside the persistent kernel: next unit of 32 virtual threads (dynamic assignment)
    int pad_queue_;
    // NPT (rumd_npt.cuh): the box is a device quantity that changes every step
    double box[3];        // current box lengths (set from the handle's box at every reset)
    double box_next[3];   // box after the step in flight (k_npt_prepare -> k_integrate_npt)
    double box_build[3];  // box at the last list build
    double nu_o, nu_t;    // strain rate as the last step left it; strain rate at the integer time t of the last step
    double vol_t;         // volume at the integer time t of the last step
    double npt_a, npt_b, npt_s, npt_sh; // leap-frog factors of the step in flight
};

struct CellGrid {
    int n[3];        // cells per axis (S17)
    int ncell;       // n[0]*n[1]*n[2]
    float scale[3];  // n_k / L_k
};

// Everything a kernel needs, passed by value (lives in the constant bank).
struct Sys {
    int N, Npad, ntypes;
    int cap, cap_it;        // list capacity per particle (multiple of 32), cap / tp
    int tp_shift, ppw_shift;// log2(tp), log2(32/tp)
    float L[3], h[3], invL[3];
    float hin[3];           // h - (rc_max + 2 skin): inside this no listed neighbour is across a boundary
    float dt, half_skin2;   // (skin/2)^2
    double dt_d, T0, omega2, g;
    int sort_interval, method;
    int npt;                // 1: NPT integrator, box lengths live in DevScalars
    double P0, cP;          // NPT: target pressure; wP^2 / ((g + 3) T0)
    float rc_margin;        // rc_max + 2 skin + 1e-3 (hin = L/2 - rc_margin); rc_max + skin in rcl_max
    float rcl_max;
    float skin;
    CellGrid grid;
    // caller-owned state
    float4* r; float4* v; float4* f; float* w; int4* image; int* id;
    float4* r_out;          // where a fused force+integrate step writes r(t+dt): r itself or r_alt
    float4* r_alt;          // workspace: second position buffer (double buffering of the fused step)
    int build_tp_shift;     // log2(lanes per particle) of the cell-list build
    // workspace
    int* nbl; int* num_nbrs; float4* r_build;
    float4* tmp_r; float4* tmp_v; int4* tmp_image; int* tmp_id;
    int* cell_of; int* slot; int* perm;
    int* ccount; int* cstart_z; int* rowrank; int* blocksum; // cstart_z: ncell + 1 entries; rowrank: ny*nz
    // tile method (rumd_tile.cuh): the cell grid is cut into nt[0] x nt[1] x nt[2] tiles of <= TILE_WMAX cells per axis
    int nt[3], ntiles;
    int hcap;               // shared-memory halo slots per tile (slot hcap is the far-away dummy)
    int cap_it8;            // uint4 list chunks (8 entries) per lane: cap / (8 tp)
    int* halo_idx;          // [ntiles][hcap]: global particle index | ghost bits << 28 of every halo slot
    int* halo_cnt;          // [ntiles]: halo slots in use
    long long* prof;        // nullptr, or 8 cycle counters filled by block 0 of the persistent kernel (profiling run)
    double* partial;        // 2 sets x 2 doubles per block (kt, mv2) of the integrating kernel
    DevScalars* sc;
    PairParams pp[RUMD_MAXT * RUMD_MAXT];
};
