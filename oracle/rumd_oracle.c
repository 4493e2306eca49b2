/*
 * rumd_oracle.c -- fp64 CPU oracle for the RUMD short-range pair-interaction hot path.
 *
 * THIS FILE IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call it.  It shares
 * no source, header, constant or helper with the CUDA path (paper_1506_05094_b200/csrc) and
 * neither imports the other.
 *
 * What it is: a plain, slow, obviously-correct double-precision restatement of what the path
 * computes, written from /root/reference/PAPER.md ("P:n" = PAPER.md line n) and, where the
 * paper prints no equation, from the readings listed in SURVEY.md 8(c) (O1..O10, S1..S28),
 * which DESIGN.md repeats.  No blocking, no fusion, no reordering: one function per definition.
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"):
 *   orc_lj_raw / orc_lj_sf / orc_coulomb_sf : closed forms (u(2^(1/6) s) = -e, 0.4^6 = 0.004096
 *       constants), force = -du/dr by central differences, continuity at rc.
 *   orc_forces_allpairs / orc_forces_list   : Newton's third law, translation / relabelling
 *       invariance, static fcc / rock-salt lattice sums (tests/golden/lattice_sums.txt),
 *       brute force == list based, independence of the skin.
 *   orc_nblist_n2 / orc_nblist_cell         : agree with each other, symmetric, lattice shell counts.
 *   orc_integrate (NVE)                     : time reversibility, momentum conservation,
 *       energy fluctuation ~ dt^2, small drift.
 *   orc_integrate (NVT)                     : tau -> inf reproduces NVE bit for bit, conserved
 *       quantity H fluctuation ~ dt^2, <T_kin> -> T0.  The discretisation itself is a reading
 *       (S9): "parity unpinned" against the paper for NVT trajectories (the paper prints no
 *       Nose-Hoover equations).
 *   orc_integrate_npt / orc_run_npt (NPT)   : barostat off (tau_P = inf, nu = 0) reproduces the NVT trajectory
 *       bit for bit; free flight under a constant strain rate against the closed-form solution (box
 *       L exp(nu t) exactly, velocity decay to second order in dt); conserved quantity fluctuation ~ dt^2;
 *       <P> -> P0 and the volume moves toward the target.  The leap-frog discretisation of the
 *       Martyna-Tobias-Klein equations (P:78 ref. [51]) is a reading (S32): "parity unpinned" against the
 *       paper for NPT trajectories (the paper prints no equations of motion).
 *
 * Conventions: positions r[3*i+k], velocities v[3*i+k], forces F[3*i+k]; box[3] = (Lx,Ly,Lz),
 * orthorhombic, origin-centred, coordinates in [-L/2, L/2] (S7).  Potentials are one record of
 * ORC_POT_STRIDE doubles per ORDERED type pair (a*ntypes+b):
 *     pot[0]=epsilon pot[1]=sigma pot[2]=rc_LJ (<=0: no LJ term) pot[3]=k*qa*qb pot[4]=rc_Coulomb (<=0: none)
 *     pot[5]=cutoff method of the LJ term, pot[6]=cutoff method of the Coulomb term:
 *            0 = shifted force, 1 = shifted potential, 2 = no shift (plain truncation)
 *     pot[7]=kind of the second term (P:73 list of pair potentials), with pot[3]=a, pot[8]=b, pot[9]=c:
 *            0 Coulomb        u = a / r                      (a = k q_i q_j)
 *            1 inverse power  u = a r^-b                     (IPL)
 *            2 Yukawa         u = a exp(-r / b) / r
 *            3 Gaussian core  u = a exp(-(r / b)^2)
 *            4 Buckingham     u = a exp(-r / b) - c / r^6
 *            5 generalized LJ u = a / (c - d) [ d (b/r)^c - c (b/r)^d ]   (a = epsilon, b = sigma, exponents
 *                             c = m > d = n; minimum -epsilon at r = sigma; pot[10] = d)
 *            6 Girifalco      u = -a [1/(s(s-1)^3) + 1/(s(s+1)^3) - 2/s^4]
 *                                 + b [1/(s(s-1)^9) + 1/(s(s+1)^9) - 2/s^10],  s = r / c   (r > c)
 *            7 Dzugutov       u = a [ A (x^-16 - B) exp(cc / (x - aa)) (x < aa) + B exp(dd / (x - bb)) (x < bb) ],
 *                             x = r / b, with the published constants A 5.82, B 1.28, aa 1.87, bb 1.94, cc 1.1, dd 0.27
 * rc values are ABSOLUTE distances (S2).
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_POT_STRIDE 11

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void orc_set_num_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* ---------------------------------------------------------------- pair functions ------- */

/* O3, unshifted 12-6 Lennard-Jones ("Pot_LJ_12_6"):
 *   u(r) = 4 e [ (s/r)^12 - (s/r)^6 ],  f(r) = -du/dr = (24 e / r) [ 2 (s/r)^12 - (s/r)^6 ]. */
void orc_lj_raw(double r, double eps, double sig, double *u, double *f)
{
    double sr = sig / r;
    double sr6 = sr * sr * sr * sr * sr * sr;
    double sr12 = sr6 * sr6;
    *u = 4.0 * eps * (sr12 - sr6);
    *f = 24.0 * eps * (2.0 * sr12 - sr6) / r;
}

/* O3, shifted-force cutoff ("truncation plus shift of the pair force [46] to ensure its
 * continuity (this corresponds to adding a linear term in the potential)"):
 *   r < rc : f_SF(r) = f(r) - f(rc),  u_SF(r) = u(r) - u(rc) + (r - rc) f(rc);  else both 0 (S3). */
void orc_lj_sf(double r, double eps, double sig, double rc, double *u, double *f)
{
    if (r < rc) {
        double ur, fr, uc, fc;
        orc_lj_raw(r, eps, sig, &ur, &fr);
        orc_lj_raw(rc, eps, sig, &uc, &fc);
        *u = ur - uc + (r - rc) * fc;
        *f = fr - fc;
    } else {
        *u = 0.0;
        *f = 0.0;
    }
}

/* O4, Coulomb with shifted-force cutoff ("Wolf ... alpha set to zero ... equivalent
 * to the shifted force method"); no self term (S6):
 *   u(r) = qq / r, f(r) = qq / r^2;  u_SF = qq [ 1/r - 1/rc + (r - rc)/rc^2 ],  f_SF = qq [ 1/r^2 - 1/rc^2 ]. */
void orc_coulomb_sf(double r, double qq, double rc, double *u, double *f)
{
    if (r < rc) {
        double ur = qq / r, fr = qq / (r * r);
        double uc = qq / rc, fc = qq / (rc * rc);
        *u = ur - uc + (r - rc) * fc;
        *f = fr - fc;
    } else {
        *u = 0.0;
        *f = 0.0;
    }
}

/* P:73-75 "the cutoff methods: no shift, shifted potential and shifted force" applied to a raw pair
 * function value (ur, fr) at r given its value (uc, fc) at the cutoff; zero at and beyond rc (S3):
 *   shifted force     : u = ur - uc + (r - rc) fc,  f = fr - fc   (continuous force, linear term in u)
 *   shifted potential : u = ur - uc,                f = fr        (continuous energy, force jumps by fc at rc)
 *   no shift          : u = ur,                     f = fr        (both jump at rc)                      */
void orc_apply_cutoff(int method, double r, double rc, double ur, double fr, double uc, double fc, double *u,
                      double *f)
{
    if (!(r < rc)) {
        *u = 0.0;
        *f = 0.0;
    } else if (method == 0) {
        *u = ur - uc + (r - rc) * fc;
        *f = fr - fc;
    } else if (method == 1) {
        *u = ur - uc;
        *f = fr;
    } else {
        *u = ur;
        *f = fr;
    }
}

/* LJ 12-6 / Coulomb with any of the three cutoff methods */
void orc_lj_cut(double r, double eps, double sig, double rc, int method, double *u, double *f)
{
    double ur, fr, uc, fc;
    orc_lj_raw(r, eps, sig, &ur, &fr);
    orc_lj_raw(rc, eps, sig, &uc, &fc);
    orc_apply_cutoff(method, r, rc, ur, fr, uc, fc, u, f);
}

void orc_coulomb_cut(double r, double qq, double rc, int method, double *u, double *f)
{
    orc_apply_cutoff(method, r, rc, qq / r, qq / (r * r), qq / rc, qq / (rc * rc), u, f);
}

/* The other pair potentials of P:73 ("IPL, Gaussian core, Buckingham, ..., Yukawa"), unshifted: (u, f = -du/dr). */
void orc_extra_raw(int kind, double r, double a, double b, double c, double d, double *u, double *f)
{
    if (kind == 5) {          /* generalized LJ (m = c, n = d): f = a c d / (c - d) [ (b/r)^c - (b/r)^d ] / r */
        const double sm = pow(b / r, c), sn = pow(b / r, d);
        *u = a / (c - d) * (d * sm - c * sn);
        *f = a * c * d / (c - d) * (sm - sn) / r;
    } else if (kind == 6) {   /* Girifalco: s = r / c, f = -(1/c) du/ds, term by term */
        const double s = r / c, m = s - 1.0, p = s + 1.0;
        *u = -a * (1.0 / (s * pow(m, 3)) + 1.0 / (s * pow(p, 3)) - 2.0 / pow(s, 4)) +
             b * (1.0 / (s * pow(m, 9)) + 1.0 / (s * pow(p, 9)) - 2.0 / pow(s, 10));
        /* d/ds 1/(s (s-+1)^k) = -((k+1) s -+ 1) / (s^2 (s-+1)^(k+1)),  d/ds (-2 s^-q) = 2 q s^-(q+1) */
        const double du = -a * (-(4.0 * s - 1.0) / (s * s * pow(m, 4)) - (4.0 * s + 1.0) / (s * s * pow(p, 4)) + 8.0 / pow(s, 5)) +
                          b * (-(10.0 * s - 1.0) / (s * s * pow(m, 10)) - (10.0 * s + 1.0) / (s * s * pow(p, 10)) + 20.0 / pow(s, 11));
        *f = -du / c;
    } else if (kind == 7) {   /* Dzugutov, x = r / b */
        const double A = 5.82, B = 1.28, aa = 1.87, bb = 1.94, cc = 1.1, dd = 0.27;
        const double x = r / b;
        double uu = 0.0, du = 0.0;
        if (x < aa) {
            const double e = exp(cc / (x - aa)), g = pow(x, -16.0) - B;
            uu += A * g * e;
            du += A * e * (-16.0 * pow(x, -17.0) - g * cc / ((x - aa) * (x - aa)));
        }
        if (x < bb) {
            const double e = exp(dd / (x - bb));
            uu += B * e;
            du += -B * e * dd / ((x - bb) * (x - bb));
        }
        *u = a * uu;
        *f = -a * du / b;
    } else if (kind == 1) {          /* inverse power law: u = a r^-b, f = b a r^-(b+1) */
        *u = a * pow(r, -b);
        *f = b * a * pow(r, -b - 1.0);
    } else if (kind == 2) {   /* Yukawa: u = a e^(-r/b) / r, f = u (1/r + 1/b) */
        *u = a * exp(-r / b) / r;
        *f = *u * (1.0 / r + 1.0 / b);
    } else if (kind == 3) {   /* Gaussian core: u = a e^(-(r/b)^2), f = 2 r u / b^2 */
        *u = a * exp(-(r / b) * (r / b));
        *f = 2.0 * r * (*u) / (b * b);
    } else if (kind == 4) {   /* Buckingham: u = a e^(-r/b) - c r^-6, f = (a/b) e^(-r/b) - 6 c r^-7 */
        *u = a * exp(-r / b) - c * pow(r, -6.0);
        *f = a / b * exp(-r / b) - 6.0 * c * pow(r, -7.0);
    } else {                  /* Coulomb */
        *u = a / r;
        *f = a / (r * r);
    }
}

void orc_extra_cut(int kind, double r, double a, double b, double c, double d, double rc, int method, double *u,
                   double *f)
{
    double ur, fr, uc, fc;
    orc_extra_raw(kind, r, a, b, c, d, &ur, &fr);
    orc_extra_raw(kind, rc, a, b, c, d, &uc, &fc);
    orc_apply_cutoff(method, r, rc, ur, fr, uc, fc, u, f);
}

/* S5: terms of different kinds on one type pair add; each applies its own rc and its own cutoff method. */
void orc_pair_sf(const double *p, double r, double *u, double *f)
{
    double ut = 0.0, ft = 0.0, uu, ff;
    if (p[2] > 0.0) {
        orc_lj_cut(r, p[0], p[1], p[2], (int)p[5], &uu, &ff);
        ut += uu;
        ft += ff;
    }
    if (p[4] > 0.0) {
        orc_extra_cut((int)p[7], r, p[3], p[8], p[9], p[10], p[4], (int)p[6], &uu, &ff);
        ut += uu;
        ft += ff;
    }
    *u = ut;
    *f = ft;
}

/* S4/S5: interaction range of a type pair = max over its terms; list cutoff adds the skin. */
double orc_pair_rc(const double *p)
{
    double rc = 0.0;
    if (p[2] > rc) rc = p[2];
    if (p[4] > rc) rc = p[4];
    return rc;
}

/* ---------------------------------------------------------------- box ------------------ */

/* O1: d_k -= L_k * nint(d_k / L_k). */
void orc_min_image(double *d, const double *box)
{
    for (int k = 0; k < 3; ++k) d[k] -= box[k] * rint(d[k] / box[k]);
}

static double dist2_min_image(const double *ri, const double *rj, const double *box, double *d)
{
    d[0] = ri[0] - rj[0];
    d[1] = ri[1] - rj[1];
    d[2] = ri[2] - rj[2];
    orc_min_image(d, box);
    return d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
}

/* ---------------------------------------------------------------- forces --------------- */

/* O5: F_i = sum_j f_SF(r_ij) d_ij / r_ij,  u_i = 1/2 sum_j u_SF(r_ij) (P:160 halving),
 *     w_i = 1/2 sum_j r_ij f_SF(r_ij).  Adds one pair (i <- j) to the accumulators of i. */
static void add_pair(const double *p, const double *d, double r2, double *Fi, double *ui, double *wi)
{
    double r = sqrt(r2), u, f;
    orc_pair_sf(p, r, &u, &f);
    Fi[0] += f * d[0] / r;
    Fi[1] += f * d[1] / r;
    Fi[2] += f * d[2] / r;
    *ui += 0.5 * u;
    *wi += 0.5 * r * f;
}

/* Brute force over ALL pairs j != i: no list, no cells (pin P4). */
void orc_forces_allpairs(int N, const double *r, const int *type, const double *box, int nt,
                         const double *pot, double *F, double *u, double *w)
{
#pragma omp parallel for schedule(static)
    for (int i = 0; i < N; ++i) {
        double Fi[3] = {0, 0, 0}, ui = 0, wi = 0, d[3];
        for (int j = 0; j < N; ++j) {
            if (j == i) continue;
            const double *p = pot + ORC_POT_STRIDE * (type[i] * nt + type[j]);
            double r2 = dist2_min_image(r + 3 * i, r + 3 * j, box, d);
            double rc = orc_pair_rc(p);
            if (r2 < rc * rc) add_pair(p, d, r2, Fi, &ui, &wi);
        }
        F[3 * i] = Fi[0];
        F[3 * i + 1] = Fi[1];
        F[3 * i + 2] = Fi[2];
        u[i] = ui;
        w[i] = wi;
    }
}

/* Same sums restricted to a full Verlet list (both directions stored, no
 * Newton's third law).  list is row-major here: k-th neighbour of i at list[i*cap + k]. */
void orc_forces_list(int N, const double *r, const int *type, const double *box, int nt,
                     const double *pot, int cap, const int *count, const int *list, double *F,
                     double *u, double *w)
{
#pragma omp parallel for schedule(static)
    for (int i = 0; i < N; ++i) {
        double Fi[3] = {0, 0, 0}, ui = 0, wi = 0, d[3];
        for (int k = 0; k < count[i]; ++k) {
            int j = list[(size_t)i * cap + k];
            const double *p = pot + ORC_POT_STRIDE * (type[i] * nt + type[j]);
            double r2 = dist2_min_image(r + 3 * i, r + 3 * j, box, d);
            double rc = orc_pair_rc(p);
            if (r2 < rc * rc) add_pair(p, d, r2, Fi, &ui, &wi);
        }
        F[3 * i] = Fi[0];
        F[3 * i + 1] = Fi[1];
        F[3 * i + 2] = Fi[2];
        u[i] = ui;
        w[i] = wi;
    }
}

/* ---------------------------------------------------------------- neighbour lists ------ */

/* O2 (Fig. 4): NB(i) = { j != i : |d_ij|^2 < (rc_{ti tj} + s)^2 }, strict <, per type
 * pair, full list.  O(N^2) double loop.  Returns the largest count found; entries beyond cap are
 * dropped (count[i] still holds the true count, so max > cap signals overflow). */
int orc_nblist_n2(int N, const double *r, const int *type, const double *box, int nt,
                  const double *pot, double skin, int cap, int *count, int *list)
{
    int maxc = 0;
#pragma omp parallel for schedule(static) reduction(max : maxc)
    for (int i = 0; i < N; ++i) {
        int c = 0;
        double d[3];
        for (int j = 0; j < N; ++j) {
            if (j == i) continue;
            double rcl = orc_pair_rc(pot + ORC_POT_STRIDE * (type[i] * nt + type[j])) + skin;
            double r2 = dist2_min_image(r + 3 * i, r + 3 * j, box, d);
            if (r2 < rcl * rcl) {
                if (c < cap) list[(size_t)i * cap + c] = j;
                ++c;
            }
        }
        count[i] = c;
        if (c > maxc) maxc = c;
    }
    return maxc;
}

/* Independent O(N) search ("cell-index method [1,2]"): textbook linked cells of edge
 * >= max list cutoff, 27-cell stencil (NOT the paper's half-size cells / 125 stencil, which the CUDA
 * path uses -- the two searches share nothing).  Needs >= 3 cells per axis; returns -1 otherwise. */
int orc_nblist_cell(int N, const double *r, const int *type, const double *box, int nt,
                    const double *pot, double skin, int cap, int *count, int *list)
{
    double rmax = 0.0;
    for (int a = 0; a < nt * nt; ++a) {
        double rc = orc_pair_rc(pot + ORC_POT_STRIDE * a);
        if (rc > rmax) rmax = rc;
    }
    rmax += skin;
    int nc[3];
    for (int k = 0; k < 3; ++k) {
        nc[k] = (int)floor(box[k] / rmax);
        if (nc[k] < 3) return -1;
    }
    int ncell = nc[0] * nc[1] * nc[2];
    int *head = (int *)malloc(sizeof(int) * (size_t)ncell);
    int *next = (int *)malloc(sizeof(int) * (size_t)N);
    int *cell = (int *)malloc(sizeof(int) * 3 * (size_t)N);
    for (int c = 0; c < ncell; ++c) head[c] = -1;
    for (int i = 0; i < N; ++i) {
        int cc[3];
        for (int k = 0; k < 3; ++k) {
            /* wrapped coordinate in [0, L) */
            double x = r[3 * i + k] - box[k] * floor(r[3 * i + k] / box[k] + 0.5) + 0.5 * box[k];
            int c = (int)floor(x / box[k] * nc[k]);
            if (c < 0) c = 0;
            if (c >= nc[k]) c = nc[k] - 1;
            cc[k] = c;
            cell[3 * i + k] = c;
        }
        int ci = (cc[2] * nc[1] + cc[1]) * nc[0] + cc[0];
        next[i] = head[ci];
        head[ci] = i;
    }
    int maxc = 0;
#pragma omp parallel for schedule(static) reduction(max : maxc)
    for (int i = 0; i < N; ++i) {
        int c = 0;
        double d[3];
        for (int dz = -1; dz <= 1; ++dz)
            for (int dy = -1; dy <= 1; ++dy)
                for (int dx = -1; dx <= 1; ++dx) {
                    int cx = (cell[3 * i] + dx + nc[0]) % nc[0];
                    int cy = (cell[3 * i + 1] + dy + nc[1]) % nc[1];
                    int cz = (cell[3 * i + 2] + dz + nc[2]) % nc[2];
                    for (int j = head[(cz * nc[1] + cy) * nc[0] + cx]; j >= 0; j = next[j]) {
                        if (j == i) continue;
                        double rcl =
                            orc_pair_rc(pot + ORC_POT_STRIDE * (type[i] * nt + type[j])) + skin;
                        double r2 = dist2_min_image(r + 3 * i, r + 3 * j, box, d);
                        if (r2 < rcl * rcl) {
                            if (c < cap) list[(size_t)i * cap + c] = j;
                            ++c;
                        }
                    }
                }
        count[i] = c;
        if (c > maxc) maxc = c;
    }
    free(head);
    free(next);
    free(cell);
    return maxc;
}

/* O9 / S14 ("no particles have moved more than half the skin distance"; P:217 positions stored
 * at build): 1 iff some |minimg(r_i - r_i^build)| > skin/2, strict. */
int orc_needs_rebuild(int N, const double *r, const double *r_build, const double *box, double skin)
{
    double lim2 = 0.25 * skin * skin;
    for (int i = 0; i < N; ++i) {
        double d[3];
        double r2 = dist2_min_image(r + 3 * i, r_build + 3 * i, box, d);
        if (r2 > lim2) return 1;
    }
    return 0;
}

/* ---------------------------------------------------------------- integrators ---------- */

#define ORC_NVE 0
#define ORC_NVT 1

/* One leap-frog step given F(t) (O6, O7, S7-S11; P:78 names the integrators, prints no equations).
 *   NVE: v(t+dt/2) = v(t-dt/2) + dt F/m ;                         r(t+dt) = r(t) + dt v(t+dt/2)
 *   NVT: v(t+dt/2) = [ (1 - xi dt/2) v(t-dt/2) + dt F/m ] / (1 + xi dt/2) ; same r update;
 *        T_kin = sum m |v(t+dt/2)|^2 / g ; xi(t+dt) = xi + dt w2 (T_kin/T0 - 1), w2 = (2 pi / tau)^2
 *        (tau <= 0 or inf: w2 = 0) ; eta(t+dt) = eta + dt/2 [xi(t) + xi(t+dt)].
 *   wrap: n = nint(r/L); r -= L n; image += n  (S7).
 * thermostat[0] = xi, thermostat[1] = eta (updated in place, NVT only).
 * out[0] = K(t) = 1/2 sum m | (v_old + v_new)/2 |^2   (O10)
 * out[1] = sum m |v(t+dt/2)|^2. */
void orc_integrate(int N, double *r, double *v, const double *m, int *image, const double *F,
                   const double *box, double dt, int mode, double T0, double tau, double g,
                   double *thermostat, double *out)
{
    double xi = thermostat[0];
    double Kt = 0.0, mv2 = 0.0;
    for (int i = 0; i < N; ++i) {
        for (int k = 0; k < 3; ++k) {
            double vo = v[3 * i + k], vn;
            if (mode == ORC_NVT)
                vn = ((1.0 - 0.5 * xi * dt) * vo + dt * F[3 * i + k] / m[i]) / (1.0 + 0.5 * xi * dt);
            else
                vn = vo + dt * F[3 * i + k] / m[i];
            double vh = 0.5 * (vo + vn);
            Kt += 0.5 * m[i] * vh * vh;
            mv2 += m[i] * vn * vn;
            v[3 * i + k] = vn;
            double x = r[3 * i + k] + dt * vn;
            double n = rint(x / box[k]);
            r[3 * i + k] = x - box[k] * n;
            image[3 * i + k] += (int)n;
        }
    }
    if (mode == ORC_NVT) {
        double w2 = 0.0;
        if (tau > 0.0 && isfinite(tau)) w2 = (2.0 * M_PI / tau) * (2.0 * M_PI / tau);
        double xin = xi + dt * w2 * (mv2 / g / T0 - 1.0);
        thermostat[1] += 0.5 * dt * (xi + xin);
        thermostat[0] = xin;
    }
    out[0] = Kt;
    out[1] = mv2;
}

/* O8 step order: (rebuild list if flag) -> F(r(t)) -> integrate -> displacement check sets the flag
 * for the next step.  Runs nsteps from (r, v, image, thermostat), flag initially set.
 * log (may be NULL): 6 doubles per step = U(t), K(t), W(t), xi(t), eta(t), H(t) where
 *   H = K + U                                   (NVE)
 *   H = K + U + g T0 xi^2 / (2 w2) + g T0 eta   (NVT, O10; the xi^2 term is dropped when w2 = 0).
 * use_cell != 0 selects orc_nblist_cell (falls back to the N^2 search when the box is too small).
 * Returns the number of list builds, or -1 on allocation failure. */
long orc_run(int N, double *r, double *v, const double *m, int *image, const int *type,
             const double *box, int nt, const double *pot, double skin, double dt, int mode,
             double T0, double tau, double *thermostat, long nsteps, int use_cell, double *log)
{
    int cap = 64;
    int *count = (int *)malloc(sizeof(int) * (size_t)N);
    int *list = (int *)malloc(sizeof(int) * (size_t)N * cap);
    double *rb = (double *)malloc(sizeof(double) * 3 * (size_t)N);
    double *F = (double *)malloc(sizeof(double) * 3 * (size_t)N);
    double *u = (double *)malloc(sizeof(double) * (size_t)N);
    double *w = (double *)malloc(sizeof(double) * (size_t)N);
    if (!count || !list || !rb || !F || !u || !w) return -1;
    double g = 3.0 * N - 3.0; /* S10 */
    double w2 = 0.0;
    if (mode == ORC_NVT && tau > 0.0 && isfinite(tau)) w2 = (2.0 * M_PI / tau) * (2.0 * M_PI / tau);
    int flag = 1;
    long nbuild = 0;
    for (long s = 0; s < nsteps; ++s) {
        if (flag) {
            for (;;) {
                int mc = -1;
                if (use_cell) mc = orc_nblist_cell(N, r, type, box, nt, pot, skin, cap, count, list);
                if (mc < 0) mc = orc_nblist_n2(N, r, type, box, nt, pot, skin, cap, count, list);
                if (mc <= cap) break;
                /* "automatically re-allocated with doubled capacity" */
                while (cap < mc) cap *= 2;
                free(list);
                list = (int *)malloc(sizeof(int) * (size_t)N * cap);
                if (!list) return -1;
            }
            memcpy(rb, r, sizeof(double) * 3 * (size_t)N);
            flag = 0;
            ++nbuild;
        }
        orc_forces_list(N, r, type, box, nt, pot, cap, count, list, F, u, w);
        double xi = thermostat[0], eta = thermostat[1], out[2];
        orc_integrate(N, r, v, m, image, F, box, dt, mode, T0, tau, g, thermostat, out);
        if (log) {
            double U = 0.0, W = 0.0;
            for (int i = 0; i < N; ++i) {
                U += u[i];
                W += w[i];
            }
            double H = out[0] + U;
            if (mode == ORC_NVT) {
                H += g * T0 * eta;
                if (w2 > 0.0) H += 0.5 * g * T0 * xi * xi / w2;
            }
            double *l = log + 6 * s;
            l[0] = U;
            l[1] = out[0];
            l[2] = W;
            l[3] = xi;
            l[4] = eta;
            l[5] = H;
        }
        flag = orc_needs_rebuild(N, r, rb, box, skin);
    }
    free(count);
    free(list);
    free(rb);
    free(F);
    free(u);
    free(w);
    return nbuild;
}

/* ---------------------------------------------------------------- NPT ("NPT [51]") ---------- */

/* Isotropic constant-pressure dynamics of Martyna, Tobias and Klein (P:455 ref. [51]) with the Nose-Hoover
 * thermostat of O7 acting on the particles; the paper prints no equations, so this is reading S32:
 *     dr/dt = v + nu r                     nu = strain rate of the box, dL/dt = nu L (all three lengths)
 *     dv/dt = F/m - [xi + (1 + 3/g) nu] v
 *     dnu/dt = cP [ (1 + 3/g) sum m v^2 + W - 3 V P0 ],  cP = wP2 / ((g + 3) T0), wP2 = (2 pi / tau_P)^2
 *              (= [3 V (P - P0) + (3/g) sum m v^2] / Wb with 3 V P = sum m v^2 + W, W = sum_i w_i the pair virial,
 *               Wb = (g + 3) T0 / wP2)
 *     dxi/dt = w2 (sum m v^2 / (g T0) - 1),  deta/dt = xi
 * conserved: H = K + U + P0 V + Wb nu^2 / 2 + g T0 xi^2 / (2 w2) + g T0 eta.
 * Leap-frog form in the order of O7.  xi and nu live at integer times.  The part of dnu/dt that depends on the
 * positions, pos(t) = cP [W(t) - 3 V(t) P0], is applied as two half kicks around the force evaluation (closing the
 * previous step, opening this one), the kinetic part as one whole kick with the half-step velocities:
 *     nu(t)     = nu_o + dt/2 pos(t)                      nu_o: the strain rate as the previous step left it
 *     gam       = xi(t) + (1 + 3/g) nu(t)
 *     v(t+dt/2) = [ (1 - gam dt/2) v(t-dt/2) + dt F(t)/m ] / (1 + gam dt/2)
 *     nu_h      = nu(t) + dt/2 pos(t) + dt/2 cP (1 + 3/g) sum m v(t-dt/2)^2        strain rate of the drift
 *     sh = exp(nu_h dt / 2), s = sh^2 ;  r(t+dt) = s r(t) + dt sh v(t+dt/2) ;  L(t+dt) = s L(t) ;  wrap (new box, S7)
 *     xi(t+dt)  = xi + dt w2 (sum m v(t+dt/2)^2 / (g T0) - 1) ;  eta(t+dt) = eta + dt/2 [xi(t) + xi(t+dt)]
 *     nu_o'     = nu(t) + dt/2 pos(t) + dt cP (1 + 3/g) sum m v(t+dt/2)^2
 * tau_P <= 0 or inf: cP = 0, the strain rate stays what it is (0: exactly the NVT step of orc_integrate).
 * state[0] = xi, state[1] = eta, state[2] = nu_o (in: as left by the previous step; a run starts with nu_o = the
 * wanted nu(0) minus its first closing half kick, normally 0), state[3] = nu(t) of THIS step (out, for H(t)).
 * box is updated in place.  out[0] = K(t) (O10), out[1] = sum m |v(t+dt/2)|^2. */
void orc_integrate_npt(int N, double *r, double *v, const double *m, int *image, const double *F, double Wvir,
                       double *box, double dt, double T0, double tau, double P0, double tauP, double g,
                       double *state, double *out)
{
    double w2 = 0.0, wP2 = 0.0;
    if (tau > 0.0 && isfinite(tau)) w2 = (2.0 * M_PI / tau) * (2.0 * M_PI / tau);
    if (tauP > 0.0 && isfinite(tauP)) wP2 = (2.0 * M_PI / tauP) * (2.0 * M_PI / tauP);
    const double cP = wP2 / ((g + 3.0) * T0);
    const double vol = box[0] * box[1] * box[2];
    const double pos = cP * (Wvir - 3.0 * vol * P0);
    const double xi = state[0];
    const double nu = state[2] + 0.5 * dt * pos;
    double mv2_old = 0.0;
    for (int i = 0; i < N; ++i)
        for (int k = 0; k < 3; ++k) mv2_old += m[i] * v[3 * i + k] * v[3 * i + k];
    const double nu_h = nu + 0.5 * dt * pos + 0.5 * dt * cP * (1.0 + 3.0 / g) * mv2_old;
    const double gam = xi + (1.0 + 3.0 / g) * nu;
    const double sh = exp(0.5 * nu_h * dt), s = sh * sh;
    double boxn[3];
    for (int k = 0; k < 3; ++k) boxn[k] = s * box[k];
    double Kt = 0.0, mv2 = 0.0;
    for (int i = 0; i < N; ++i) {
        for (int k = 0; k < 3; ++k) {
            double vo = v[3 * i + k];
            double vn = ((1.0 - 0.5 * gam * dt) * vo + dt * F[3 * i + k] / m[i]) / (1.0 + 0.5 * gam * dt);
            double vh = 0.5 * (vo + vn);
            Kt += 0.5 * m[i] * vh * vh;
            mv2 += m[i] * vn * vn;
            v[3 * i + k] = vn;
            double x = s * r[3 * i + k] + dt * sh * vn;
            double n = rint(x / boxn[k]);
            r[3 * i + k] = x - boxn[k] * n;
            image[3 * i + k] += (int)n;
        }
    }
    double xin = xi + dt * w2 * (mv2 / g / T0 - 1.0);
    state[1] += 0.5 * dt * (xi + xin);
    state[0] = xin;
    state[3] = nu;
    state[2] = nu + 0.5 * dt * pos + dt * cP * (1.0 + 3.0 / g) * mv2;
    for (int k = 0; k < 3; ++k) box[k] = boxn[k];
    out[0] = Kt;
    out[1] = mv2;
}

/* nsteps of NPT dynamics, step order O8.  The list is rebuilt at EVERY step (the box changes every step; any valid
 * list gives the same forces, O5), by the cell search when use_cell != 0 and the box allows it, else the N^2 search.
 * log (may be NULL): 9 doubles per step = U(t), K(t), W(t), xi(t), eta(t), H(t), nu(t), V(t), P(t) = (2 K + W)/(3 V),
 *   H = K + U + P0 V + (g + 3) T0 nu^2 / (2 wP2) + g T0 xi^2 / (2 w2) + g T0 eta  (terms with w2 / wP2 = 0 dropped).
 * state: 4 doubles (xi, eta, nu_o, nu(t) of the last step), see orc_integrate_npt.
 * Returns the number of list builds, or -1 on allocation failure. */
long orc_run_npt(int N, double *r, double *v, const double *m, int *image, const int *type, double *box, int nt,
                 const double *pot, double skin, double dt, double T0, double tau, double P0, double tauP,
                 double *state, long nsteps, int use_cell, double *log)
{
    int cap = 64;
    int *count = (int *)malloc(sizeof(int) * (size_t)N);
    int *list = (int *)malloc(sizeof(int) * (size_t)N * cap);
    double *F = (double *)malloc(sizeof(double) * 3 * (size_t)N);
    double *u = (double *)malloc(sizeof(double) * (size_t)N);
    double *w = (double *)malloc(sizeof(double) * (size_t)N);
    if (!count || !list || !F || !u || !w) return -1;
    double g = 3.0 * N - 3.0; /* S10 */
    double w2 = 0.0, wP2 = 0.0;
    if (tau > 0.0 && isfinite(tau)) w2 = (2.0 * M_PI / tau) * (2.0 * M_PI / tau);
    if (tauP > 0.0 && isfinite(tauP)) wP2 = (2.0 * M_PI / tauP) * (2.0 * M_PI / tauP);
    long nbuild = 0;
    for (long s = 0; s < nsteps; ++s) {
        for (;;) {
            int mc = -1;
            if (use_cell) mc = orc_nblist_cell(N, r, type, box, nt, pot, skin, cap, count, list);
            if (mc < 0) mc = orc_nblist_n2(N, r, type, box, nt, pot, skin, cap, count, list);
            if (mc <= cap) break;
            while (cap < mc) cap *= 2;
            free(list);
            list = (int *)malloc(sizeof(int) * (size_t)N * cap);
            if (!list) return -1;
        }
        ++nbuild;
        orc_forces_list(N, r, type, box, nt, pot, cap, count, list, F, u, w);
        double U = 0.0, W = 0.0;
        for (int i = 0; i < N; ++i) {
            U += u[i];
            W += w[i];
        }
        const double xi = state[0], eta = state[1], vol = box[0] * box[1] * box[2];
        double out[2];
        orc_integrate_npt(N, r, v, m, image, F, W, box, dt, T0, tau, P0, tauP, g, state, out);
        const double nu = state[3]; /* the strain rate at the integer time t of this step */
        if (log) {
            double H = out[0] + U + P0 * vol + g * T0 * eta;
            if (w2 > 0.0) H += 0.5 * g * T0 * xi * xi / w2;
            if (wP2 > 0.0) H += 0.5 * (g + 3.0) * T0 * nu * nu / wP2;
            double *l = log + 9 * s;
            l[0] = U;
            l[1] = out[0];
            l[2] = W;
            l[3] = xi;
            l[4] = eta;
            l[5] = H;
            l[6] = nu;
            l[7] = vol;
            l[8] = (2.0 * out[0] + W) / (3.0 * vol);
        }
    }
    free(count);
    free(list);
    free(F);
    free(u);
    free(w);
    return nbuild;
}

