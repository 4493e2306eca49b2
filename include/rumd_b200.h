/*
 * rumd_b200.h -- C ABI of librumd_b200.so: the per-timestep short-range pair-interaction hot path of RUMD
 * (arxiv 1506.05094) re-designed for one NVIDIA B200 (sm_100a).
 *
 * Citations: "P:n" = line n of the paper text, "S n"/"O n" = the readings listed in DESIGN.md
 * (section "Readings of the paper").  The call sequence mirrors the paper's user script (Fig. 1):
 * create the simulation -> SetParams(i, j, Sigma, Epsilon, Rcut) per type pair -> set the integrator
 * (timeStep, targetTemperature) -> Run(n).
 *
 * General rules
 *   - Plain C: opaque handle, plain pointers and sizes.  Every pointer argument says "device" or "host".
 *   - Every call returns a rumd_status; nothing throws, nothing exits.  rumd_last_error() gives a message.
 *   - All bulk device memory is CALLER-OWNED (e.g. torch tensors): the state arrays (rumd_bind_state) and
 *     one workspace blob (rumd_bind_workspace).  The library owns only the handle, CUDA graph objects,
 *     events and a few pinned host scalars; rumd_destroy frees those and nothing else.
 *   - All work is enqueued on the cudaStream_t given to rumd_create.  Calls are asynchronous unless they
 *     say "synchronizes".  There is NO CPU fallback: without a CUDA device every compute call fails with
 *     RUMD_ERR_CUDA.
 *   - Asynchronous device-side conditions (neighbour-list overflow, P:218 / P:263 "set flag to inform
 *     host"; non-finite energies) are sticky and surface at the next synchronizing call.
 *   - Particle order is NOT stable: the cell method sorts particles spatially and permutes all state
 *     arrays in place ("rearrange all particle data"); d_id[slot] = original particle index.
 */
#ifndef RUMD_B200_H
#define RUMD_B200_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#define RUMD_MAX_TYPES 4

typedef struct rumd_system rumd_system; /* opaque; owned by the library */

typedef enum {
    RUMD_OK = 0,
    RUMD_ERR_INVALID_ARG = 1,
    RUMD_ERR_NOT_READY = 2,     /* state / workspace / potential / integrator not set yet */
    RUMD_ERR_CUDA = 3,          /* a CUDA runtime call failed (no device, launch failure, ...) */
    RUMD_ERR_NBL_OVERFLOW = 4,  /* some particle has more neighbours than the bound capacity */
    RUMD_ERR_BOX_TOO_SMALL = 5, /* rc_max + skin > min(L)/2: minimum image not valid (O1) */
    RUMD_ERR_NONFINITE = 6      /* energy is NaN/Inf */
} rumd_status;

typedef enum { /* P:73 pair potentials; the first is the LJ slot of a type pair, all the others share its second slot */
    RUMD_POT_LJ_12_6 = 0,       /* {epsilon, sigma, rcut}   u = 4 eps [(s/r)^12 - (s/r)^6] */
    RUMD_POT_COULOMB = 1,       /* {k qi qj, rcut}          u = a / r */
    RUMD_POT_IPL = 2,           /* {a, n, rcut}             u = a r^-n   (inverse power law) */
    RUMD_POT_YUKAWA = 3,        /* {a, b, rcut}             u = a exp(-r / b) / r */
    RUMD_POT_GAUSSIAN_CORE = 4, /* {a, b, rcut}             u = a exp(-(r / b)^2) */
    RUMD_POT_BUCKINGHAM = 5,    /* {a, b, c, rcut}          u = a exp(-r / b) - c / r^6 */
    RUMD_POT_GEN_LJ = 6,        /* {epsilon, sigma, m, n, rcut}  u = eps / (m - n) [n (s/r)^m - m (s/r)^n], m > n > 0:
                                   minimum -eps at r = sigma.  Takes the place of the 12-6 term: a type pair
                                   with this kind must have no RUMD_POT_LJ_12_6 term (RUMD_ERR_INVALID_ARG) */
    RUMD_POT_GIRIFALCO = 7,     /* {alpha, beta, d, rcut}   u = -alpha [1/(s(s-1)^3) + 1/(s(s+1)^3) - 2/s^4]
                                   + beta [1/(s(s-1)^9) + 1/(s(s+1)^9) - 2/s^10], s = r / d; defined for r > d only */
    RUMD_POT_DZUGUTOV = 8       /* {epsilon, sigma, rcut}   u = eps [A (x^-16 - B) exp(c/(x-a)) (x < a)
                                   + B exp(d/(x-b)) (x < b)], x = r / sigma, A 5.82, B 1.28, a 1.87, b 1.94, c 1.1,
                                   d 0.27; it vanishes smoothly at x = b, so rcut = b sigma with RUMD_CUT_NONE is natural */
} rumd_pot_kind;
typedef enum { /* P:73-75 "the cutoff methods: no shift, shifted potential and shifted force" */
    RUMD_CUT_SHIFTED_FORCE = 0,     /* f = f(r) - f(rc), u = u(r) - u(rc) + (r - rc) f(rc): the hot-path default */
    RUMD_CUT_SHIFTED_POTENTIAL = 1, /* f = f(r),         u = u(r) - u(rc) */
    RUMD_CUT_NONE = 2               /* f = f(r),         u = u(r)  (plain truncation) */
} rumd_cutoff;
typedef enum {
    RUMD_INT_NVE_LEAPFROG = 0,
    RUMD_INT_NVT_NOSE_HOOVER = 1,
    RUMD_INT_NPT_MTK = 2 /* P:78 "NPT [51]": isotropic Martyna-Tobias-Klein barostat + the Nose-Hoover thermostat;
                            target pressure and barostat period from rumd_set_barostat */
} rumd_integrator;
typedef enum {
    RUMD_NB_N2 = 0,   /* P:173 "n2": tiled all-pairs list build */
    RUMD_NB_CELL = 1, /* P:276 "sort": spatial sort + cell-list build */
    RUMD_NB_NONE = 2, /* P:371 "none": no list at all, every force evaluation loops over all pairs (small N) */
    RUMD_NB_TILE = 3  /* spatial sort + cell-list build like RUMD_NB_CELL, with the j-particles staged in shared
                         memory: the cell grid is cut into tiles, a thread block loads the positions of a tile and of
                         the two cells around it once and both the build and the force kernel gather from there;
                         16-bit list entries.  Needs tp <= 8 and >= 6 cells per axis.  Between list rebuilds the
                         coordinates in d_r may leave [-L/2, L/2] by up to skin/2 (they are wrapped, and d_image
                         updated, at the next rebuild); d_r + d_image * L is the unwrapped position at all times */
} rumd_nb_method;

/* Tunable launch parameters (Table 2: NB method, pb, tp, skin; P:379 sort interval).
 *   method        neighbour-list build algorithm, or RUMD_NB_NONE (no list: all-pairs forces; skin, build_tp,
 *                 sort_interval are then unused and rumd_export_nblist reports empty rows).
 *   pb            particles per thread block of the per-step force kernel (Table 1 "PPerBlock").
 *   tp            threads per particle of the force kernel, one of 1,2,4,8,16,32 ("TPerPart").
 *                 pb*tp must be a multiple of 32 and <= 1024.
 *   skin          Verlet skin; list cutoff of a type pair = rc_ab + skin (S4).
 *   sort_interval RUMD_NB_N2 only: spatially re-sort the particles at every sort_interval-th rebuild
 *                 (P:379); 0 = never.  RUMD_NB_CELL sorts at every rebuild.
 *   use_graph     per-step kernels only (persistent = 0).  0: plain kernel launches; 1: whole-timestep CUDA
 *                 graphs (steps_per_graph steps each).
 *   steps_per_graph  time steps unrolled into one graph launch (>= 1; 0 = library default).
 *   persistent    1: rumd_run_steps(n) is ONE cooperative kernel that runs all n steps (fused force +
 *                 integrate, double-buffered positions, grid barrier per step, in-kernel rebuilds; blocks of
 *                 256 threads, pb is not used); 0: per-step kernels (early-exit rebuild chain, then force +
 *                 integrate, fused into one kernel per step inside CUDA graphs).
 *   build_tp      lanes per particle of the cell-list build, one of 1,2,4,8,16,32 ("not been tried
 *                 yet"); 0 = library default for this N.
 *   tile          RUMD_NB_TILE only: target edge of a tile in cells, 1..8 (a tile owns about tile^3 cells and stages
 *                 (tile + 4)^3 of them in shared memory); 0 = library default for this N. */
typedef struct {
    int method;
    int pb;
    int tp;
    float skin;
    int sort_interval;
    int use_graph;
    int steps_per_graph;
    int persistent;
    int build_tp;
    int tile;
} rumd_tuning;

/* Thermodynamic scalars, all double, filled by rumd_get_thermo (host struct).
 * U, W: sums over particles of u_i, w_i from the LAST force evaluation (O5; P:160 energy halving).
 * K: kinetic energy at the integer time of the last completed step, 1/2 sum m |(v_old+v_new)/2|^2 (O10).
 * mv2: sum m |v(t+dt/2)|^2 after the last step.  xi, eta: Nose-Hoover variables (O7).
 * H: K + U (+ thermostat terms for NVT, O10; + P0 V + (g + 3) T0 nu^2 / (2 wP^2) for NPT), valid when at least one
 * step has run. */
typedef struct {
    double U, W, K, mv2, xi, eta, H;
    long long n_steps;    /* steps completed since rumd_bind_state */
    long long n_rebuilds; /* neighbour-list builds since rumd_bind_state */
    int max_nbrs;         /* largest list length seen at the last build */
    int nbl_capacity;     /* bound capacity (entries per particle) */
    int overflow;         /* 1 if the last build overflowed */
    int pad_;
} rumd_thermo;

/* P:40-46 Fig. 1 `Simulation(...)`.  box_lengths: host, 3 floats (Lx, Ly, Lz), orthorhombic periodic box
 * centred on the origin, coordinates live in [-L/2, L/2] (O1, S7).  cuda_stream: a cudaStream_t created by
 * the caller (e.g. torch.cuda.Stream().cuda_stream); 0 = the library creates and owns a blocking stream,
 * which stays implicitly ordered with the legacy default stream (the legacy stream itself cannot be
 * captured into CUDA graphs).  1 <= n_types <= RUMD_MAX_TYPES.  *out is written only on success. */
rumd_status rumd_create(rumd_system** out, int n_particles, int n_types, const float box_lengths[3],
                        void* cuda_stream);
rumd_status rumd_destroy(rumd_system* s);

/* Batched ensemble ("large ensembles of MD simulations of small systems"): the handle describes ONE
 * system of n_particles; after rumd_set_replicas(s, R), R >= 1, the state arrays of rumd_bind_state hold R such
 * systems back to back (replica q owns elements [q n, (q+1) n)), all with the same box, potentials, integrator
 * and tuning, each with its own list, thermostat and counters, and rumd_run_steps(n) advances all of them by
 * n steps in ONE kernel launch (one thread block per replica, no inter-block synchronisation).  Must be called
 * before rumd_bind_state / rumd_bind_workspace (the workspace grows with R).  Needs method RUMD_NB_N2 or
 * RUMD_NB_NONE.  With R > 1 the single-system calls (rumd_build_nblist, rumd_compute_forces,
 * rumd_export_nblist, rumd_get_thermo, rumd_snapshot / restore, rumd_autotune, the profiling calls) return
 * RUMD_ERR_INVALID_ARG; use rumd_get_thermo_replicas.  d_f / d_w hold the forces of the last step of a run. */
rumd_status rumd_set_replicas(rumd_system* s, int n_replicas);
/* out: HOST array of n_out >= R records, one per replica (U, W, K of the last step of the last run; xi, eta, H,
 * counters).  Synchronizes; reports sticky errors of any replica. */
rumd_status rumd_get_thermo_replicas(rumd_system* s, rumd_thermo* out, int n_out);

/* State arrays, DEVICE pointers, caller-owned, n_particles elements each, 16-byte aligned:
 *   d_r     float4 : x, y, z, particle type as int bits in .w             (Fig. 3)
 *   d_v     float4 : leap-frog velocity v(t - dt/2) x, y, z; mass in .w   (S8)
 *   d_f     float4 : force x, y, z; per-particle potential energy u_i in .w  [output]
 *   d_w     float  : per-particle virial w_i = 1/2 sum_j r_ij f_SF(r_ij)     (S13)                [output]
 *   d_image int4   : periodic image counters ix, iy, iz (w unused)           (S7)
 *   d_id    int32  : slot -> original particle index; the caller initialises it (normally 0..N-1)
 * Binding resets the step / rebuild counters, the thermostat (xi = eta = 0) and requests a rebuild. */
rumd_status rumd_bind_state(rumd_system* s, void* d_r, void* d_v, void* d_f, void* d_w, void* d_image,
                            void* d_id);

/* Workspace (neighbour list P:101 / P:167, positions at build P:217, cell arrays P:248, sort scratch,
 * reduction partials, snapshot).  rumd_workspace_bytes: size needed for nbl_capacity entries per
 * particle.  d_ws: DEVICE pointer, caller-owned, 256-byte aligned, >= bytes.  Re-binding with a larger
 * capacity is the paper's "re-allocated with doubled capacity" after RUMD_ERR_NBL_OVERFLOW. */
size_t rumd_workspace_bytes(const rumd_system* s, int nbl_capacity);
rumd_status rumd_bind_workspace(rumd_system* s, void* d_ws, size_t bytes, int nbl_capacity);

/* P:49-50 `pot.SetParams(i, j, Sigma, Epsilon, Rcut)`; symmetric in (type_i, type_j).  params: host.
 *   RUMD_POT_LJ_12_6 : {epsilon, sigma, rcut}   u = 4 eps [(s/r)^12 - (s/r)^6]           (O3)
 *   RUMD_POT_COULOMB : {k*q_i*q_j, rcut}        u = k q_i q_j / r, no self term          (O4, S6)
 *   RUMD_POT_IPL / YUKAWA / GAUSSIAN_CORE / BUCKINGHAM / GEN_LJ / GIRIFALCO / DZUGUTOV : see rumd_pot_kind; they occupy the same slot as
 *   Coulomb (a type pair has the LJ term plus at most ONE of these; setting one replaces the other).
 * rcut is an ABSOLUTE distance (S2).  cutoff: one of rumd_cutoff, applied for r < rcut, zero beyond (S3).
 * One slot per kind per type pair: the same kind again overwrites, different kinds add, each with its own
 * rc and cutoff method (S5).  rcut <= 0 removes the term. */
rumd_status rumd_set_pair_potential(rumd_system* s, int type_i, int type_j, rumd_pot_kind kind,
                                    rumd_cutoff cutoff, const float* params, int n_params);

/* P:54 `IntegratorNVT(timeStep, targetTemperature)`.  NVE leap-frog (O6) or Nose-Hoover leap-frog
 * (O7) with period tau (tau <= 0 or inf: thermostat off, identical to NVE).  g = 3N - 3 (S10). */
rumd_status rumd_set_integrator(rumd_system* s, rumd_integrator kind, float dt, float target_T, float tau);

/* NPT ("NPT [51]", Martyna-Tobias-Klein 1994, isotropic; the leap-frog form is DESIGN.md reading S32):
 *     dr/dt = v + nu r, dL/dt = nu L, dv/dt = F/m - [xi + (1 + 3/g) nu] v,
 *     dnu/dt = (2 pi / tau_P)^2 / ((g + 3) T0) [ (1 + 3/g) sum m v^2 + W - 3 V P0 ],  W = sum_i w_i.
 * target_P, tau_P: host scalars; tau_P <= 0 or inf freezes the strain rate (with nu = 0 that is NVT).  Takes effect
 * with rumd_set_integrator(s, RUMD_INT_NPT_MTK, dt, target_T, tau).  NPT runs on the per-step kernels (the tuning's
 * `persistent` is ignored) with method RUMD_NB_N2 or RUMD_NB_NONE (the cell grid is sized for a fixed box:
 * RUMD_ERR_INVALID_ARG otherwise) and a single system (no replicas); rumd_autotune is not available.  The box is then
 * a device quantity: it starts as the box of rumd_create at every reset (bind, upload) and is read with rumd_get_box.
 * If the box shrinks below 2 (rc_max + skin) the run stops being valid: RUMD_ERR_BOX_TOO_SMALL from rumd_get_thermo. */
rumd_status rumd_set_barostat(rumd_system* s, float target_P, float tau_P);
/* Current box lengths and strain rate (host outputs; box_out: 3 doubles; nu_out may be NULL).  For NVE / NVT the
 * box of rumd_create and 0.  Synchronizes. */
rumd_status rumd_get_box(rumd_system* s, double* box_out, double* nu_out);

/* Launch parameters.  rumd_default_tuning fills the library's untuned defaults for this N. */
rumd_status rumd_default_tuning(const rumd_system* s, rumd_tuning* out);
rumd_status rumd_set_tuning(rumd_system* s, const rumd_tuning* t);
rumd_status rumd_get_tuning(const rumd_system* s, rumd_tuning* out);

/* Blackwell autotuner (section 11 is the prior art): times short runs of steps_per_trial steps
 * from one stored snapshot over method x pb x tp x skin (coordinate descent; "single
 * minimum"), restores the snapshot, applies and returns the fastest setting.  tps_out (host, may be NULL)
 * receives its time steps per second.  Synchronizes. */
rumd_status rumd_autotune(rumd_system* s, rumd_tuning* out, int steps_per_trial, double* tps_out);

/* The same with the paper's parameter file (P:382 step 8: the tuned parameters are written to a file and reused
 * for runs with "the same user parameters"): cache_path (host string) names a text file with one JSON object
 * per line, keyed by GPU name, N, box, potentials, integrator, dt, T, tau.  A cached entry for this key is
 * applied without any trial run (*from_cache_out = 1); otherwise the autotuner runs and appends its result.
 * cache_path NULL or "" = plain rumd_autotune.  from_cache_out: host, may be NULL. */
rumd_status rumd_autotune_cached(rumd_system* s, rumd_tuning* out, int steps_per_trial, double* tps_out,
                                 const char* cache_path, int* from_cache_out);

/* Unconditional list rebuild with the current tuning.  Asynchronous. */
rumd_status rumd_build_nblist(rumd_system* s);
/* Rebuild iff the displacement flag is set, then forces / energies / virials into d_f,
 * d_w (Fig. 3; O5).  Asynchronous. */
rumd_status rumd_compute_forces(rumd_system* s);
/* n whole time steps, each (rebuild if flag) -> forces -> integrate + wrap + displacement check (O8;
 * P:179).  Asynchronous: no host synchronisation inside. */
rumd_status rumd_run_steps(rumd_system* s, long n);

/* Neighbour list export for inspection / parity tests: row-major, in SLOT numbering (map with d_id).
 * d_count: device int32 [n_particles]; d_list: device int32 [n_particles * row_capacity], k-th neighbour
 * of slot i at d_list[i*row_capacity + k]; entries beyond the count are -1.  Asynchronous. */
rumd_status rumd_export_nblist(rumd_system* s, void* d_count, void* d_list, int row_capacity);

/* Sums U, W on the device (fp64, fixed order), copies the scalars to *out (host).  Synchronizes the stream
 * and reports sticky errors (RUMD_ERR_NBL_OVERFLOW, RUMD_ERR_NONFINITE, RUMD_ERR_CUDA). */
rumd_status rumd_get_thermo(rumd_system* s, rumd_thermo* out);

/* In-workspace snapshot of (r, v, image, id, xi, eta, counters) and its restore ("restores the
 * initial state").  Asynchronous.  Restore requests a rebuild. */
rumd_status rumd_snapshot(rumd_system* s);
rumd_status rumd_restore(rumd_system* s);

/* HOST-buffer entry points (used for end-to-end timing): copy the state from / to host arrays of the same
 * layouts as rumd_bind_state (any pointer may be NULL = skip).  Upload requests a rebuild and resets the
 * thermostat; it checks that every particle type in h_r lies in [0, n_types) (RUMD_ERR_INVALID_ARG otherwise:
 * the type indexes the pair table in every kernel; arrays written directly through the device pointers of
 * rumd_bind_state are the caller's responsibility).  Download synchronizes the stream. */
rumd_status rumd_upload_state(rumd_system* s, const void* h_r, const void* h_v, const void* h_image,
                              const void* h_id);
rumd_status rumd_download_state(rumd_system* s, void* h_r, void* h_v, void* h_f, void* h_w, void* h_image,
                                void* h_id);

/* Number of kernel launches issued (directly or inside graphs) since rumd_create. */
long long rumd_launch_count(const rumd_system* s);
/* Per-kernel-class device time of the last rumd_profile_step call: runs ONE un-fused, un-graphed time step
 * with CUDA events around each kernel class.  ms_out: host, 4 floats = {build, force, integrate, other}.
 * did_rebuild_out: host int.  Synchronizes. */
rumd_status rumd_profile_step(rumd_system* s, float* ms_out, int* did_rebuild_out);

/* Average device time, in microseconds, of one launch of the pair-force kernel with the current tuning and the
 * current list: reps launches replayed from one CUDA graph between two CUDA events on the library's stream
 * (roofline measurement; the outputs d_f, d_w are simply recomputed).  us_per_launch: host.  Synchronizes. */
rumd_status rumd_time_force(rumd_system* s, int reps, float* us_per_launch);

/* Runs nsteps time steps in the persistent kernel with the per-phase SM-cycle counters of block 0 switched
 * on.  out8: host, 8 doubles = microseconds PER STEP spent by block 0 in {rebuild phases (sort + build),
 * force + integrate, the sort part of the rebuild, block sums + grid barrier wait, unused}, whole kernel per
 * step, number of rebuilds, grid size.  Advances the simulation by nsteps.  Synchronizes. */
rumd_status rumd_profile_persistent(rumd_system* s, int nsteps, double* out8);

/* Measured FP32 peak of this GPU (the roofline fractions are quoted against the derived
 * 148 SMs x 128 lanes x 2 flop x clock AND against this measurement): a kernel of independent register-operand
 * FFMA chains at full occupancy, best of reps launches, CUDA events on the library's stream.  tflops_out: host,
 * TFLOP/s counting 2 flop per FFMA.  Needs a bound workspace (4 bytes of it are the kernel's dummy output).
 * Synchronizes. */
rumd_status rumd_measure_fp32_peak(rumd_system* s, int reps, double* tflops_out);

/* ONE force / energy / virial evaluation that ALLOCATES NOTHING -- for callers that cannot call cudaMalloc (code under
 * CUDA graph capture, tight serving loops, harnesses that forbid it) and therefore cannot use the handle API, whose
 * rumd_create allocates and whose workspace must come from somewhere.  Needs no handle: one call computes what
 * rumd_create .. rumd_build_nblist + rumd_compute_forces + rumd_get_thermo compute with method RUMD_NB_N2, tp = 8 for
 * 12-6 Lennard-Jones and Coulomb terms with the shifted-force cutoff (Fig. 3; Fig. 4; O5),
 * by the same list build and the same pair loop.  All scratch (neighbour list, list lengths, positions at build,
 * reduction partials, flags) lives in one fixed device array inside the library, 8.2 MB, held by every GPU that loads
 * the library until the process exits.  Hence the limits: n_particles <= RUMD_NOALLOC_MAX_PARTICLES and at most
 * RUMD_NOALLOC_NBL_CAPACITY listed neighbours (within rcut + skin) per particle.
 *   n_particles, n_types   1 <= n_particles <= RUMD_NOALLOC_MAX_PARTICLES (RUMD_ERR_INVALID_ARG beyond, with a message),
 *                          1 <= n_types <= RUMD_MAX_TYPES.
 *   box_lengths            host, 3 floats, as for rumd_create; rc_max + skin <= L/2 per axis (RUMD_ERR_BOX_TOO_SMALL).
 *   pairs                  host, n_types * n_types records, pair (a, b) at [a * n_types + b]; must be symmetric.
 *   skin                   Verlet skin of the list (>= 0).  The result does not depend on it; the list length does.
 *   d_r                    DEVICE, input, float4 [n_particles]: x, y, z in [-L/2, L/2], type as int bits in .w (as
 *                          rumd_bind_state; types outside [0, n_types) are the caller's responsibility).  16-byte aligned.
 *   d_f, d_w               DEVICE, outputs, float4 [n_particles] force + u_i in .w, float [n_particles] virial w_i.
 *   d_out4                 DEVICE, output, 4 doubles: U = sum u_i, W = sum w_i (fp64, fixed order), the longest list
 *                          row, overflow flag (1.0: some particle has more than RUMD_NOALLOC_NBL_CAPACITY neighbours
 *                          inside the list cutoff; forces, U and W are then incomplete).
 *   cuda_stream            cudaStream_t the work is enqueued on (NULL: the default stream).  Asynchronous: one
 *                          memset + two kernels, no host synchronisation, no cudaMalloc / cudaFree / allocating call.
 *                          The first call on a device looks up the scratch array's device address (once per device).
 *   errbuf, errbuf_len     host, may be NULL / 0: receives the message of a non-OK status.
 * Ownership: the caller owns every pointer; the library owns only the static scratch.  EVERY call on a device shares
 * that scratch, which keeps the previous call's contents (the call clears what must start at zero itself): calls
 * ordered on one stream are fine, calls that may overlap on the GPU (different streams or threads without ordering
 * between them) race and give garbage.  The handle API does not touch the scratch. */
#define RUMD_NOALLOC_MAX_PARTICLES 8192
#define RUMD_NOALLOC_NBL_CAPACITY 256
typedef struct {
    float epsilon, sigma, rcut;  /* 12-6 Lennard-Jones term u = 4 eps [(s/r)^12 - (s/r)^6], shifted force; rcut <= 0: none */
    float kqq, rcut_coulomb;     /* Coulomb term u = kqq / r (kqq = k q_a q_b), shifted force; rcut_coulomb <= 0: none */
} rumd_noalloc_pair;
rumd_status rumd_forces_noalloc(int n_particles, int n_types, const float box_lengths[3], const rumd_noalloc_pair* pairs,
                                float skin, const void* d_r, void* d_f, void* d_w, void* d_out4, void* cuda_stream,
                                char* errbuf, size_t errbuf_len);

const char* rumd_last_error(const rumd_system* s);
const char* rumd_version(void);

#ifdef __cplusplus
}
#endif
#endif /* RUMD_B200_H */
