"""Pins for the fp64 oracle (oracle/rumd_oracle.c): closed forms, invariants, lattice sums, brute force.

The paper prints no worked numerical example, so every pin comes from what the
mathematics fixes.  Each test names the SURVEY.md 8(c) pin (P1..P12) it implements.  CPU only.
"""
import itertools
import math
import os

import numpy as np
import pytest

import oracle
from paper_1506_05094_b200 import workloads as W

GOLD = {}
with open(os.path.join(os.path.dirname(__file__), "golden", "lattice_sums.txt")) as fh:
    for line in fh:
        line = line.split("#")[0].split()
        if len(line) == 2:
            GOLD[line[0]] = float(line[1])

KA = W.kob_andersen()
CH = W.charged_lj()
LJ = W.lj_single()


def test_golden_file_is_reproduced_by_its_generator():
    """tests/golden/lattice_sums.txt is written by a committed pure-Python script that imports nothing from oracle/
    (closed-form pair functions over integer lattice vectors): the stored pins are reproducible and independent."""
    import importlib.util

    path = os.path.join(os.path.dirname(__file__), "golden", "make_lattice_sums.py")
    src = open(path).read()
    import re

    assert not re.search(r"^\s*(import|from)\s+(oracle|paper_1506_05094_b200)", src, flags=re.M)
    spec = importlib.util.spec_from_file_location("make_lattice_sums", path)
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    assert mod.check() == []
    assert len(mod.table()) >= 23


# ------------------------------------------------------------------ P1 / P2: pair functions, closed forms


def test_P1_lj_minimum_is_minus_epsilon():
    for eps, sig in ((1.0, 1.0), (1.5, 0.8), (0.5, 0.88), (3.0, 2.0)):
        u, f = oracle.lj_raw(2.0 ** (1.0 / 6.0) * sig, eps, sig)
        assert u == pytest.approx(-eps, rel=1e-14)
        assert abs(f) < 1e-12 * eps / sig
        u0, f0 = oracle.lj_raw(sig, eps, sig)           # u(sigma) = 0, f(sigma) = 24 eps / sigma
        assert abs(u0) < 1e-14 * eps
        assert f0 == pytest.approx(24.0 * eps / sig, rel=1e-14)


def test_P1_lj_decimal_closed_forms():
    # r = 10 sigma: (s/r)^6 = 1e-6 exactly in decimal
    u, f = oracle.lj_raw(10.0, 1.0, 1.0)
    assert u == pytest.approx(4.0 * (1e-12 - 1e-6), rel=1e-13)
    assert f == pytest.approx(24.0 * (2e-12 - 1e-6) / 10.0, rel=1e-13)
    # r = 0.5 sigma: (s/r)^6 = 64
    u, f = oracle.lj_raw(0.5, 1.0, 1.0)
    assert u == pytest.approx(4.0 * (4096.0 - 64.0), rel=1e-14)
    assert f == pytest.approx(24.0 * (8192.0 - 64.0) / 0.5, rel=1e-14)
    # homogeneity: u(r; eps, sig) = eps * u(r/sig; 1, 1), f = eps/sig * f(r/sig; 1, 1)
    u1, f1 = oracle.lj_raw(1.3 / 0.8, 1.0, 1.0)
    u2, f2 = oracle.lj_raw(1.3, 1.5, 0.8)
    assert u2 == pytest.approx(1.5 * u1, rel=1e-13)
    assert f2 == pytest.approx(1.5 / 0.8 * f1, rel=1e-13)


def test_P2_shifted_force_constants():
    uc, fc = oracle.lj_raw(2.5, 1.0, 1.0)
    assert uc == pytest.approx(GOLD["sf_lj_u_rc"], rel=1e-12)      # 0.4^6 = 0.004096 closed form
    assert fc == pytest.approx(GOLD["sf_lj_f_rc"], rel=1e-12)
    assert uc == pytest.approx(4 * (0.004096 ** 2 - 0.004096), rel=1e-13)
    u, f = oracle.lj_sf(2.0 ** (1.0 / 6.0), 1.0, 1.0, 2.5)
    assert u == pytest.approx(GOLD["sf_lj_u_at_2p16"], rel=1e-11)
    assert f == pytest.approx(-GOLD["sf_lj_f_rc"], rel=1e-11)       # f(2^(1/6)) = 0 -> f_SF = -f(rc)
    # minimum of the SF potential: root of f_SF by bisection
    lo, hi = 1.0, 1.3
    for _ in range(200):
        mid = 0.5 * (lo + hi)
        if oracle.lj_sf(mid, 1, 1, 2.5)[1] > 0:
            lo = mid
        else:
            hi = mid
    assert lo == pytest.approx(GOLD["sf_lj_rmin"], rel=1e-11)
    assert oracle.lj_sf(lo, 1, 1, 2.5)[0] == pytest.approx(GOLD["sf_lj_umin"], rel=1e-11)


def test_P2_shifted_force_is_continuous_and_zero_outside():
    for rec in (KA[0, 0], KA[0, 1], KA[1, 1], CH[0, 1], CH[0, 0]):
        rc = max(rec[2], rec[4])
        for r in (rc, rc * (1 + 1e-12), rc + 0.1, 10 * rc):
            assert oracle.pair_sf(rec, r) == (0.0, 0.0)
        d = 1e-5
        u, f = oracle.pair_sf(rec, rc - d)
        # u_SF ~ (1/2) u''(rc) d^2, f_SF ~ -f'(rc) d near rc; a term with a smaller rc jumps only at its own rc
        assert abs(u) < 50 * d * d and abs(f) < 50 * d
    # LJ term of the charged system is continuous at ITS rc = 2.5 while Coulomb (rc 4.0) is still on (S5)
    ua, fa = oracle.pair_sf(CH[0, 1], 2.5 - 1e-7)
    ub, fb = oracle.pair_sf(CH[0, 1], 2.5 + 1e-7)
    assert abs(ua - ub) < 1e-6 and abs(fa - fb) < 1e-6
    uc, fc = oracle.coulomb_sf(2.5 + 1e-7, -1.0, 4.0)
    assert (ub, fb) == pytest.approx((uc, fc), rel=1e-14)


def test_O4_coulomb_closed_forms():
    # qq = 1, rc = 4: u_SF(2) = 1/2 - 1/4 + (2-4)/16 = 1/8 ; f_SF(2) = 1/4 - 1/16 = 3/16
    assert oracle.coulomb_sf(2.0, 1.0, 4.0) == pytest.approx((0.125, 0.1875), rel=1e-15)
    assert oracle.coulomb_sf(1.0, 1.0, 4.0) == pytest.approx((0.5625, 0.9375), rel=1e-15)
    assert oracle.coulomb_sf(1.0, -1.0, 4.0) == pytest.approx((-0.5625, -0.9375), rel=1e-15)
    assert oracle.coulomb_sf(2.0, 3.0, 4.0) == pytest.approx((0.375, 0.5625), rel=1e-15)


@pytest.mark.parametrize("rec", [KA[0, 0], KA[0, 1], KA[1, 1], CH[0, 0], CH[0, 1], LJ[0, 0]])
def test_P3_force_is_minus_gradient(rec):
    rc = max(rec[2], rec[4])
    h = 1e-6
    for r in np.linspace(0.85 * max(rec[1], 0.8), rc - 1e-3, 41):
        if abs(r - rec[2]) < 2 * h:     # skip the inner (LJ) cutoff of a two-term pair
            continue
        up, _ = oracle.pair_sf(rec, r + h)
        um, _ = oracle.pair_sf(rec, r - h)
        _, f = oracle.pair_sf(rec, r)
        assert f == pytest.approx(-(up - um) / (2 * h), rel=2e-8, abs=2e-8)


# ------------------------------------------------------------------ two-particle worked examples (O1, O5)


def test_O5_two_particles_through_the_periodic_boundary():
    L = 10.0
    box = np.array([L, 12.0, 14.0])
    r = np.array([[-L / 2 + 0.5, 1.0, -2.0], [L / 2 - 0.5, 1.0, -2.0]])   # distance 1.0 through the x face
    F, u, w = oracle.forces_allpairs(r, [0, 0], box, LJ)
    fsf = 24.0 - GOLD["sf_lj_f_rc"]                                        # f(1) - f(rc), f(1) = 24
    usf = 0.0 - GOLD["sf_lj_u_rc"] + (1.0 - 2.5) * GOLD["sf_lj_f_rc"]
    # minimum image of r0 - r1 = -9 is +1: particle 0 is pushed in +x (repulsion, r < 2^(1/6))
    assert F[0] == pytest.approx([fsf, 0, 0], rel=1e-12, abs=1e-12)
    assert F[1] == pytest.approx([-fsf, 0, 0], rel=1e-12, abs=1e-12)
    assert u == pytest.approx([0.5 * usf, 0.5 * usf], rel=1e-12)          # P:160 halving
    assert w == pytest.approx([0.5 * fsf, 0.5 * fsf], rel=1e-12)          # r f / 2, r = 1
    # oblique displacement: F parallel to d, |F| = f_SF(|d|)
    r = np.array([[0.1, 0.2, 0.3], [0.1 + 0.6, 0.2 - 0.8, 0.3 + 1.2]])    # |d| = sqrt(.36+.64+1.44) = 1.5620499
    F, u, w = oracle.forces_allpairs(r, [0, 0], box, LJ)
    d = r[0] - r[1]
    rr = np.linalg.norm(d)
    us, fs = oracle.lj_sf(rr, 1, 1, 2.5)
    assert F[0] == pytest.approx(fs * d / rr, rel=1e-12)
    assert fs < 0 and np.dot(F[0], d) < 0                                  # attraction beyond the minimum
    assert w[0] == pytest.approx(0.5 * rr * fs, rel=1e-12)


def test_O1_min_image():
    box = np.array([10.0, 20.0, 5.0])
    assert oracle.min_image([9.0, -11.0, 2.4], box) == pytest.approx([-1.0, 9.0, 2.4])
    assert oracle.min_image([4.9, 10.1, -2.6], box) == pytest.approx([4.9, -9.9, 2.4])


# ------------------------------------------------------------------ P4 / P5 / P12: brute force, invariances


def _gas(N, pot, box, seed):
    r, t = W.random_gas(N, pot.shape[0], box, seed)
    return r.astype(np.float64), t, np.asarray(box, dtype=np.float64)


CASES = [(200, KA, (7.0, 6.5, 8.0), 1), (512, KA, (8.0, 8.0, 8.0), 2), (300, CH, (9.0, 10.0, 11.0), 3),
         (256, LJ, (7.0, 7.0, 7.0), 4)]


@pytest.mark.parametrize("N,pot,box,seed", CASES)
def test_P4_list_forces_equal_brute_force_for_any_skin(N, pot, box, seed):
    r, t, box = _gas(N, pot, box, seed)
    F0, u0, w0 = oracle.forces_allpairs(r, t, box, pot)
    assert np.abs(F0).max() > 1.0            # a real, non-degenerate configuration
    for skin in (0.0, 0.3, 0.6):
        if max(pot[..., 2].max(), pot[..., 4].max()) + skin > box.min() / 2:
            continue
        for method in ("n2", "cell"):
            try:
                cnt, lst = oracle.nblist(r, t, box, pot, skin, method=method)
            except ValueError:
                continue
            F, u, w = oracle.forces_list(r, t, box, pot, cnt, lst)
            scale = np.abs(F0).max()
            assert np.abs(F - F0).max() <= 1e-12 * scale
            assert abs(u.sum() - u0.sum()) <= 1e-12 * np.abs(u0).sum()
            assert abs(w.sum() - w0.sum()) <= 1e-12 * np.abs(w0).sum()


@pytest.mark.parametrize("N,pot,box,seed", CASES)
def test_P5_newton_third_law_and_invariances(N, pot, box, seed):
    r, t, box = _gas(N, pot, box, seed)
    F, u, w = oracle.forces_allpairs(r, t, box, pot)
    assert np.abs(F.sum(axis=0)).max() <= 1e-10 * np.abs(F).sum()
    # rigid translation + re-wrap
    shift = np.array([0.37, -2.9, 5.21])
    r2 = r + shift
    r2 -= box * np.rint(r2 / box)
    F2, u2, w2 = oracle.forces_allpairs(r2, t, box, pot)
    assert np.abs(F2 - F).max() <= 1e-9 * np.abs(F).max()
    assert np.abs(u2 - u).max() <= 1e-9 * np.abs(u).max()
    # relabelling
    perm = np.random.default_rng(seed).permutation(N)
    F3, u3, w3 = oracle.forces_allpairs(r[perm], t[perm], box, pot)
    assert np.abs(F3 - F[perm]).max() <= 1e-10 * np.abs(F).max()
    assert np.abs(w3 - w[perm]).max() <= 1e-10 * np.abs(w).max()
    # virial by definition: W = -(1/2) sum_i sum_j d_ij . grad -> check via uniform dilation of the box:
    # dU/dlnV = -W/3 * ... ; finite difference U(lambda) with r -> lambda r, L -> lambda L: dU/dlambda = -2W... see below
    lam = 1e-6
    Up = oracle.forces_allpairs(r * (1 + lam), t, box * (1 + lam), pot)[1].sum()
    Um = oracle.forces_allpairs(r * (1 - lam), t, box * (1 - lam), pot)[1].sum()
    # U = sum_pairs u(lambda r_ij) -> dU/dlambda = sum_pairs r u' = -sum_pairs r f = -W_total (W = sum_i w_i = sum_pairs r f)
    assert (Up - Um) / (2 * lam) == pytest.approx(-w.sum(), rel=1e-6)


# ------------------------------------------------------------------ P6 / P7 / P8: static lattices


def _shell_sum(vectors_iter, a, rc_list, pair):
    """Lattice sum over integer-derived vectors: returns (sum u, sum r f, count inside each radius).  Knows
    nothing about particles, boxes or minimum images."""
    U = WW = 0.0
    counts = [0] * len(rc_list)
    for vec, rec in vectors_iter:
        d = a * math.sqrt(vec)
        for k, rc in enumerate(rc_list):
            if d < rc:
                counts[k] += 1
        u, f = pair(rec, d)
        U += u
        WW += d * f
    return U, WW, counts


def test_P6_fcc_lattice_sum():
    a = (4.0 / 0.8442) ** (1.0 / 3.0)
    assert a == pytest.approx(GOLD["fcc_a"], rel=1e-9)
    # fcc = all (i,j,k)/2 with i+j+k even; squared length (i^2+j^2+k^2)/4
    def vecs():
        for i, j, k in itertools.product(range(-8, 9), repeat=3):
            if (i + j + k) % 2 == 0 and (i, j, k) != (0, 0, 0):
                yield (i * i + j * j + k * k) / 4.0, LJ[0, 0]
    U, WW, (n_rc, n_list) = _shell_sum(vecs(), a, [2.5, 2.8], oracle.pair_sf)
    assert (n_rc, n_list) == (GOLD["fcc_n_inside_rc"], GOLD["fcc_n_list"])
    assert 0.5 * U == pytest.approx(GOLD["fcc_u_per_n"], rel=1e-11)
    assert 0.5 * WW == pytest.approx(GOLD["fcc_w_per_n"], rel=1e-11)
    # particle code on the same lattice in fp64 (6x6x6 cells, P12)
    r, box = W.fcc_lattice(6, 6, 6, 0.8442)
    t = np.zeros(len(r), np.int32)
    F, u, w = oracle.forces_allpairs(r, t, box, LJ)
    assert u.sum() / len(r) == pytest.approx(GOLD["fcc_u_per_n"], rel=1e-11)
    assert w.sum() / len(r) == pytest.approx(GOLD["fcc_w_per_n"], rel=1e-11)
    assert np.allclose(u, u[0], rtol=1e-11) and np.abs(F).max() < 1e-10
    cnt, lst = oracle.nblist(r, t, box, LJ, 0.3)
    assert cnt.min() == cnt.max() == GOLD["fcc_n_list"]
    cnt0, _ = oracle.nblist(r, t, box, LJ, 0.0)
    assert cnt0.min() == cnt0.max() == GOLD["fcc_n_inside_rc"]
    # the fp32-rounded workload (what the GPU sees) is the same lattice to rounding
    wl = W.lj_fcc(6)
    F, u, w = oracle.forces_allpairs(wl.r, wl.types, wl.box, wl.pot)
    assert u.sum() / wl.N == pytest.approx(GOLD["fcc_u_per_n"], rel=1e-6)


def test_P7_rocksalt_lattice_sum():
    a = 0.5 ** (-1.0 / 3.0)
    assert a == pytest.approx(GOLD["rocksalt_a"], rel=1e-9)

    def vecs(pot):
        for i, j, k in itertools.product(range(-5, 6), repeat=3):
            if (i, j, k) != (0, 0, 0):
                yield float(i * i + j * j + k * k), pot[0, (i + j + k) % 2]   # seen from a + ion
    U, WW, counts = _shell_sum(vecs(CH), a, [2.5, 4.0, 4.3], oracle.pair_sf)
    assert counts == [GOLD["rocksalt_n_inside_2p5"], GOLD["rocksalt_n_inside_4p0"], GOLD["rocksalt_n_list"]]
    assert 0.5 * U == pytest.approx(GOLD["rocksalt_u_per_n"], rel=1e-11)
    assert 0.5 * WW == pytest.approx(GOLD["rocksalt_w_per_n"], rel=1e-11)
    only_lj = CH.copy(); only_lj[..., 4] = 0.0
    only_cl = CH.copy(); only_cl[..., 2] = 0.0
    assert 0.5 * _shell_sum(vecs(only_lj), a, [], oracle.pair_sf)[0] == pytest.approx(GOLD["rocksalt_u_lj_per_n"], rel=1e-11)
    assert 0.5 * _shell_sum(vecs(only_cl), a, [], oracle.pair_sf)[0] == pytest.approx(GOLD["rocksalt_u_coul_per_n"], rel=1e-11)
    # particle code, 8^3 ions (L/2 = 5.04 >= 4.3)
    r, box, ijk = W.sc_lattice(8, 8, 8, 0.5)
    t = (ijk.sum(axis=1) % 2).astype(np.int32)
    F, u, w = oracle.forces_allpairs(r, t, box, CH)
    assert u.sum() / len(r) == pytest.approx(GOLD["rocksalt_u_per_n"], rel=1e-11)
    assert w.sum() / len(r) == pytest.approx(GOLD["rocksalt_w_per_n"], rel=1e-11)
    assert np.abs(F).max() < 1e-10
    cnt, _ = oracle.nblist(r, t, box, CH, 0.3)
    assert cnt.min() == cnt.max() == GOLD["rocksalt_n_list"]
    assert oracle.forces_allpairs(r, t, box, only_cl)[1].sum() / len(r) == pytest.approx(GOLD["rocksalt_u_coul_per_n"], rel=1e-11)


def test_P8_ka_simple_cubic_counts():
    a = 1.2 ** (-1.0 / 3.0)
    sites = {}
    for name, R in (("aa", 2.8), ("ab", 2.3), ("bb", 2.5)):
        sites[name] = sum(1 for v in itertools.product(range(-4, 5), repeat=3)
                          if v != (0, 0, 0) and a * a * (v[0] ** 2 + v[1] ** 2 + v[2] ** 2) < R * R)
    assert (sites["aa"], sites["ab"], sites["bb"]) == (GOLD["ka_sc_sites_aa"], GOLD["ka_sc_sites_ab"], GOLD["ka_sc_sites_bb"])
    # per-particle list length on the N=512 lattice by integer site arithmetic vs the oracle's search
    wl = W.ka_lattice(512)
    nx, ny, nz = wl.meta["dims"]
    tgrid = wl.types.reshape(nx, ny, nz)
    R2 = {(0, 0): 2.8 ** 2, (0, 1): 2.3 ** 2, (1, 0): 2.3 ** 2, (1, 1): 2.5 ** 2}
    expect = np.zeros((nx, ny, nz), dtype=int)
    for v in itertools.product(range(-3, 4), repeat=3):
        if v == (0, 0, 0):
            continue
        d2 = a * a * (v[0] ** 2 + v[1] ** 2 + v[2] ** 2)
        tj = np.roll(tgrid, shift=(-v[0], -v[1], -v[2]), axis=(0, 1, 2))
        for (ti, tjv), rr in R2.items():
            if d2 < rr:
                expect += ((tgrid == ti) & (tj == tjv)).astype(int)
    cnt, _ = oracle.nblist(wl.r, wl.types, wl.box, wl.pot, wl.skin)
    assert np.array_equal(cnt, expect.ravel())
    # weak statistical pin on U/N of the random-type lattice
    w8 = W.ka_lattice(8000)
    cnt, lst = oracle.nblist(w8.r, w8.types, w8.box, w8.pot, 0.0, method="cell")
    u = oracle.forces_list(w8.r, w8.types, w8.box, w8.pot, cnt, lst)[1]
    assert u.sum() / w8.N == pytest.approx(GOLD["ka_sc_u_per_n_mean"], abs=0.03)


# ------------------------------------------------------------------ P9: neighbour lists


def _as_sets(cnt, lst):
    return [frozenset(lst[i, :cnt[i]].tolist()) for i in range(len(cnt))]


@pytest.mark.parametrize("N,pot,box,seed", [(600, KA, (9.0, 9.5, 10.0), 11), (1500, CH, (13.5, 14.0, 15.0), 12)])
def test_P9_two_independent_searches_agree(N, pot, box, seed):
    r, t, box = _gas(N, pot, box, seed)
    c1, l1 = oracle.nblist(r, t, box, pot, 0.3, method="n2")
    c2, l2 = oracle.nblist(r, t, box, pot, 0.3, method="cell")
    s1, s2 = _as_sets(c1, l1), _as_sets(c2, l2)
    assert s1 == s2
    assert all(len(s) == c for s, c in zip(s1, c1))             # no duplicates
    assert all(i not in s for i, s in enumerate(s1))            # self excluded
    for i, s in enumerate(s1):                                  # symmetric (full list)
        for j in s:
            assert i in s1[j]
    # brute-force definition on a sample of particles, per type pair, strict <
    rng = np.random.default_rng(seed)
    for i in rng.choice(N, 25, replace=False):
        d = r[i] - r
        d -= box * np.rint(d / box)
        rcl = np.maximum(pot[t[i], t, 2], pot[t[i], t, 4]) + 0.3
        expect = set(np.nonzero((d * d).sum(axis=1) < rcl * rcl)[0].tolist()) - {int(i)}
        assert expect == set(s1[i])


def test_P9_mean_list_length_estimates():
    # uniform-density estimate 4/3 pi (rc+s)^3 rho; the paper's own figure: rc=6, rho=0.3677 -> "~330"
    assert 4.0 / 3.0 * math.pi * 6.0 ** 3 * 0.3677 == pytest.approx(332.7, abs=0.1)
    r, t, box = _gas(4000, LJ, (17.0, 17.0, 17.0), 5)
    cnt, _ = oracle.nblist(r, t, box, LJ, 0.3, method="cell")
    rho = 4000 / 17.0 ** 3
    assert cnt.mean() == pytest.approx(4.0 / 3.0 * math.pi * 2.8 ** 3 * rho, rel=0.03)


def test_P9_list_stays_valid_until_rebuild_flag():
    """Skin/2 rule: while no particle moved more than skin/2 the list built earlier still contains
    every interacting pair, i.e. list forces == brute-force forces."""
    wl = W.lj_fcc(4)
    r = wl.r.astype(np.float64); v = 1.5 * wl.v.astype(np.float64); m = wl.m.astype(np.float64)
    img = np.zeros((wl.N, 3), np.int32)
    cnt, lst = oracle.nblist(r, wl.types, wl.box, wl.pot, wl.skin)
    rb = r.copy()
    checked = rebuilt = 0
    for step in range(120):
        if oracle.needs_rebuild(r, rb, wl.box, wl.skin):
            cnt, lst = oracle.nblist(r, wl.types, wl.box, wl.pot, wl.skin)
            rb = r.copy()
            rebuilt += 1
        F, u, w = oracle.forces_list(r, wl.types, wl.box, wl.pot, cnt, lst)
        if step % 6 == 0:
            F0, u0, _ = oracle.forces_allpairs(r, wl.types, wl.box, wl.pot)
            assert np.abs(F - F0).max() <= 1e-11 * max(1.0, np.abs(F0).max())
            assert abs(u.sum() - u0.sum()) <= 1e-11 * abs(u0.sum())
            checked += 1
        r, v, img, *_ = oracle.integrate(r, v, m, img, F, wl.box, wl.dt)
    assert rebuilt >= 2 and checked >= 10


def test_O9_rebuild_criterion_is_strict_and_periodic():
    box = np.array([10.0, 10.0, 10.0])
    rb = np.array([[4.9, 0.0, 0.0], [0.0, 0.0, 0.0]])
    r = rb.copy()
    r[0, 0] = -4.96                         # moved +0.14 through the face
    assert not oracle.needs_rebuild(r, rb, box, 0.3)
    r[0, 0] = -4.94                         # moved 0.16 > 0.15
    assert oracle.needs_rebuild(r, rb, box, 0.3)
    r = rb.copy(); r[1] = [0.0, 0.09, 0.12]  # exactly 0.15: not "more than" (S14)
    assert not oracle.needs_rebuild(r, rb, box, 0.3)


# ------------------------------------------------------------------ integrator worked examples (O6, O7, S7)


def test_O6_free_flight_wrap_and_image():
    box = np.array([10.0, 8.0, 6.0])
    r = np.array([[4.999, -3.9995, 1.0], [0.0, 0.0, 0.0]])
    v = np.array([[1.0, -2.0, 0.5], [0.0, 0.0, 0.0]])
    m = np.array([2.0, 1.0])
    F = np.array([[4.0, 0.0, 0.0], [0.0, 0.0, 0.0]])
    rn, vn, img, xi, eta, Kt, mv2 = oracle.integrate(r, v, m, np.zeros((2, 3), np.int32), F, box, 0.01)
    assert vn[0] == pytest.approx([1.0 + 0.01 * 4.0 / 2.0, -2.0, 0.5], rel=1e-15)
    assert rn[0] == pytest.approx([4.999 + 0.01 * 1.02 - 10.0, -3.9995 - 0.02 + 8.0, 1.005], rel=1e-13)
    assert img[0].tolist() == [1, -1, 0] and img[1].tolist() == [0, 0, 0]
    assert mv2 == pytest.approx(2.0 * (1.02 ** 2 + 4.0 + 0.25), rel=1e-14)
    assert Kt == pytest.approx(0.5 * 2.0 * (1.01 ** 2 + 4.0 + 0.25), rel=1e-14)   # O10: mean of half-step velocities


def test_O7_nose_hoover_single_step_worked_example():
    # N=2, g=3, m=2, v=+-1, F=+-2, xi=1/2, dt=1/10, tau=2pi (w2=1), T0=1
    box = np.array([100.0, 100.0, 100.0])
    r = np.array([[1.0, 0, 0], [-1.0, 0, 0]])
    v = np.array([[1.0, 0, 0], [-1.0, 0, 0]])
    F = np.array([[2.0, 0, 0], [-2.0, 0, 0]])
    m = np.array([2.0, 2.0])
    rn, vn, img, xi, eta, Kt, mv2 = oracle.integrate(r, v, m, np.zeros((2, 3), np.int32), F, box, 0.1,
                                                     mode=oracle.NVT, T0=1.0, tau=2 * math.pi, xi=0.5, eta=0.25)
    vx = (0.975 * 1.0 + 0.1 * 2.0 / 2.0) / 1.025          # = 43/41
    assert vn[0, 0] == pytest.approx(43.0 / 41.0, rel=1e-15) and vn[1, 0] == pytest.approx(-43.0 / 41.0, rel=1e-15)
    assert rn[0, 0] == pytest.approx(1.0 + 0.1 * vx, rel=1e-15)
    assert mv2 == pytest.approx(4.0 * vx * vx, rel=1e-14)
    xin = 0.5 + 0.1 * 1.0 * (4.0 * vx * vx / 3.0 - 1.0)
    assert xi == pytest.approx(xin, rel=1e-13)
    assert eta == pytest.approx(0.25 + 0.05 * (0.5 + xin), rel=1e-13)
    assert Kt == pytest.approx(0.5 * 4.0 * (0.5 * (1.0 + vx)) ** 2, rel=1e-14)


# ------------------------------------------------------------------ P10: NVE trajectories


def _lj(ncell=3, scale_v=1.0):
    wl = W.lj_fcc(ncell)
    return wl, wl.r.astype(np.float64), scale_v * wl.v.astype(np.float64), wl.m.astype(np.float64)


def test_P10_nve_time_reversibility_and_momentum():
    wl, r0, v0, m = _lj(4)
    img0 = np.zeros((wl.N, 3), np.int32)
    n = 60
    a = oracle.run(r0, v0, m, img0, wl.types, wl.box, wl.pot, wl.skin, wl.dt, n)
    p0 = (m[:, None] * v0).sum(axis=0)
    p1 = (m[:, None] * a["v"]).sum(axis=0)
    assert np.abs(p1 - p0).max() < 1e-11
    assert np.abs(a["r"] - r0).max() > 0.05                     # it really moved
    # one more kick with F(r(n)) puts v at n+1/2 relative to r(n); negate and run n steps back
    F, _, _ = oracle.forces_allpairs(a["r"], wl.types, wl.box, wl.pot)
    vk = a["v"] + wl.dt * F / m[:, None]
    b = oracle.run(a["r"], -vk, m, a["image"], wl.types, wl.box, wl.pot, wl.skin, wl.dt, n)
    d = b["r"] - r0
    d -= wl.box * np.rint(d / wl.box)
    assert np.abs(d).max() < 1e-9
    assert np.array_equal(b["image"], img0)


def test_P10_nve_energy_fluctuation_scales_as_dt2_and_no_drift():
    wl, r0, v0, m = _lj(4)
    img0 = np.zeros((wl.N, 3), np.int32)
    T = 2.0                                                      # time units
    sd = []
    for dt in (0.008, 0.004):
        out = oracle.run(r0, v0, m, img0, wl.types, wl.box, wl.pot, wl.skin, dt, int(round(T / dt)))
        E = out["log"][:, 5] / wl.N
        assert np.array_equal(out["log"][:, 5], out["log"][:, 0] + out["log"][:, 1])
        sd.append(E[len(E) // 4:].std())
        slope = np.polyfit(np.arange(len(E)) * dt, E, 1)[0]
        assert abs(slope) * T < 3 * sd[-1]                       # no drift beyond the fluctuation
    assert sd[0] / sd[1] == pytest.approx(4.0, rel=0.35)         # ~ dt^2
    assert sd[1] < 2e-4


def test_S26_nve_drift_of_config0_in_fp64():
    """configs[0] for 10^4 steps: least-squares slope of E/N times 10^4 steps stays far below the 1e-4
    budget that the fp32 CUDA path is allowed (BASELINE.json north_star)."""
    wl = W.lj_fcc(6)
    out = oracle.run(wl.r, wl.v, wl.m, np.zeros((wl.N, 3), np.int32), wl.types, wl.box, wl.pot, wl.skin, wl.dt, 10000)
    E = out["log"][:, 5] / wl.N
    slope = np.polyfit(np.arange(len(E)), E, 1)[0]
    assert abs(slope) * 1e4 < 2e-5
    assert np.abs(E - E[0]).max() < 1e-3                           # leap-frog O(dt^2) fluctuation, not drift
    assert out["n_builds"] > 100
    K = out["log"][2000:, 1]
    assert 2.0 * K.mean() / (3 * wl.N - 3) == pytest.approx(0.722 / 2, rel=0.15)   # equipartition from the lattice: T ~ T(0)/2


# ------------------------------------------------------------------ P11: NVT


def test_P11_nvt_with_infinite_tau_is_nve_bit_for_bit():
    wl, r0, v0, m = _lj(3)
    img0 = np.zeros((wl.N, 3), np.int32)
    a = oracle.run(r0, v0, m, img0, wl.types, wl.box, wl.pot, wl.skin, wl.dt, 200, mode=oracle.NVE)
    b = oracle.run(r0, v0, m, img0, wl.types, wl.box, wl.pot, wl.skin, wl.dt, 200, mode=oracle.NVT, T0=0.7, tau=float("inf"))
    assert np.array_equal(a["r"], b["r"]) and np.array_equal(a["v"], b["v"])
    assert b["xi"] == 0.0 and b["eta"] == 0.0


def test_P11_nvt_conserved_quantity_and_temperature():
    wl, r0, v0, m = _lj(4, scale_v=math.sqrt(1.5 / 0.722))      # T(0) = 1.5 -> T0 = 1
    img0 = np.zeros((wl.N, 3), np.int32)
    T = 4.0
    sd = []
    for dt in (0.004, 0.002):
        out = oracle.run(r0, v0, m, img0, wl.types, wl.box, wl.pot, wl.skin, dt, int(round(T / dt)),
                         mode=oracle.NVT, T0=1.0, tau=0.2)
        H = out["log"][:, 5] / wl.N
        sd.append(H.std())
        slope = np.polyfit(np.arange(len(H)) * dt, H, 1)[0]
        assert abs(slope) * T < 4 * sd[-1]
        assert np.abs(out["log"][:, 3]).max() > 0.1             # the thermostat is doing something
    assert sd[0] / sd[1] == pytest.approx(4.0, rel=0.4)
    assert sd[1] < 1e-3
    # <T_kin> -> T0 after equilibration
    out = oracle.run(r0, v0, m, img0, wl.types, wl.box, wl.pot, wl.skin, 0.004, 3000, mode=oracle.NVT, T0=1.0, tau=0.2)
    Tk = 2.0 * out["log"][1000:, 1] / (3 * wl.N - 3)
    assert Tk.mean() == pytest.approx(1.0, abs=0.03)


def test_run_is_independent_of_the_search_method_and_skin():
    wl = W.ka_lattice(512)
    img0 = np.zeros((wl.N, 3), np.int32)
    kw = dict(mode=oracle.NVT, T0=wl.T0, tau=wl.tau)
    a = oracle.run(wl.r, wl.v, wl.m, img0, wl.types, wl.box, wl.pot, 0.3, wl.dt, 50, **kw)
    b = oracle.run(wl.r, wl.v, wl.m, img0, wl.types, wl.box, wl.pot, 0.6, wl.dt, 50, **kw)
    assert np.abs(a["r"] - b["r"]).max() < 1e-9 and a["n_builds"] >= b["n_builds"]
    assert np.abs(a["log"][:, 0] - b["log"][:, 0]).max() < 1e-8 * np.abs(a["log"][:, 0]).max()


# ------------------------------------------------------------------ the three cutoff methods


def test_cutoff_methods_closed_forms():
    """shifted force / shifted potential / no shift against the raw pair function they are built from."""
    eps, sig, rc = 1.5, 0.8, 2.0
    uc, fc = oracle.lj_raw(rc, eps, sig)
    for r in (0.75, 0.9, 1.3, 1.99):
        ur, fr = oracle.lj_raw(r, eps, sig)
        assert oracle.lj_cut(r, eps, sig, rc, 0) == pytest.approx((ur - uc + (r - rc) * fc, fr - fc), rel=1e-13)
        assert oracle.lj_cut(r, eps, sig, rc, 0) == pytest.approx(oracle.lj_sf(r, eps, sig, rc), rel=1e-15)
        assert oracle.lj_cut(r, eps, sig, rc, 1) == pytest.approx((ur - uc, fr), rel=1e-13)
        assert oracle.lj_cut(r, eps, sig, rc, 2) == pytest.approx((ur, fr), rel=1e-15)
        qq, rcc = -1.0, 4.0
        assert oracle.coulomb_cut(r, qq, rcc, 0) == pytest.approx(oracle.coulomb_sf(r, qq, rcc), rel=1e-15)
        assert oracle.coulomb_cut(r, qq, rcc, 1) == pytest.approx((qq / r - qq / rcc, qq / r ** 2), rel=1e-13)
        assert oracle.coulomb_cut(r, qq, rcc, 2) == pytest.approx((qq / r, qq / r ** 2), rel=1e-15)
    for m in (0, 1, 2):
        assert oracle.lj_cut(rc, eps, sig, rc, m) == (0.0, 0.0) and oracle.lj_cut(rc + 0.3, eps, sig, rc, m) == (0.0, 0.0)
    # what is continuous at the cutoff: SF both, SP the energy only (the force jumps by f(rc)), none neither
    below = rc * (1 - 1e-12)
    assert oracle.lj_cut(below, eps, sig, rc, 0) == pytest.approx((0.0, 0.0), abs=1e-10)
    u1, f1 = oracle.lj_cut(below, eps, sig, rc, 1)
    assert abs(u1) < 1e-10 and f1 == pytest.approx(fc, rel=1e-9)
    assert oracle.lj_cut(below, eps, sig, rc, 2) == pytest.approx((uc, fc), rel=1e-9)


@pytest.mark.parametrize("method", [0, 1, 2])
def test_cutoff_methods_force_is_minus_gradient(method):
    rec = np.array([1.5, 0.8, 2.0, -1.0, 3.0, method, method, 0, 0, 0, 0])
    h = 1e-6
    for r in (0.8, 1.1, 1.7, 1.95, 2.5, 2.9):
        up, _ = oracle.pair_sf(rec, r + h)
        um, _ = oracle.pair_sf(rec, r - h)
        _, f = oracle.pair_sf(rec, r)
        assert f == pytest.approx(-(up - um) / (2 * h), rel=2e-7)


def test_cutoff_methods_fcc_lattice_sums():
    """Static fcc lattice energies for plain truncation and the shifted potential, by the
    integer-shell lattice sum and by the particle code; and the exact relations between the three methods:
    U_SP = U_none - (54/2) u(rc),  U_SF = U_SP + 1/2 sum (r - rc) f(rc)."""
    a = (4.0 / 0.8442) ** (1.0 / 3.0)
    r, box = W.fcc_lattice(6, 6, 6, 0.8442)
    t = np.zeros(len(r), np.int32)
    res = {}
    for method, key in ((2, "fcc_u_per_n_noshift"), (1, "fcc_u_per_n_shiftedpot"), (0, "fcc_u_per_n")):
        pot = W.pot_table(1)
        W.set_lj(pot, 0, 0, 1.0, 1.0, 2.5, cut=method)

        def vecs():
            for i, j, k in itertools.product(range(-8, 9), repeat=3):
                if (i + j + k) % 2 == 0 and (i, j, k) != (0, 0, 0):
                    yield (i * i + j * j + k * k) / 4.0, pot[0, 0]
        U, WW, _ = _shell_sum(vecs(), a, [2.5], oracle.pair_sf)
        assert 0.5 * U == pytest.approx(GOLD[key], rel=2e-10)
        F, u, w = oracle.forces_allpairs(r, t, box, pot)
        assert u.sum() / len(r) == pytest.approx(GOLD[key], rel=2e-10)
        assert np.abs(F).max() < 1e-10
        res[method] = (u.sum() / len(r), w.sum() / len(r))
    uc, fc = oracle.lj_raw(2.5, 1.0, 1.0)
    assert res[1][0] == pytest.approx(res[2][0] - 27 * uc, rel=1e-12)          # 54 neighbours inside rc
    assert res[1][1] == pytest.approx(res[2][1], rel=1e-12)                    # same forces -> same virial
    # SF adds (r - rc) f(rc) per pair to u and subtracts r f(rc) from r f
    shells = [(math.sqrt(0.5) * a, 12), (a, 6), (math.sqrt(1.5) * a, 24), (math.sqrt(2.0) * a, 12)]
    assert res[0][0] == pytest.approx(res[1][0] + 0.5 * sum(n * (d - 2.5) * fc for d, n in shells), rel=1e-12)
    assert res[0][1] == pytest.approx(res[1][1] - 0.5 * sum(n * d * fc for d, n in shells), rel=1e-12)


def test_cutoff_methods_list_forces_equal_brute_force():
    pot = W.pot_table(2)
    W.set_lj(pot, 0, 0, 1.0, 1.0, 2.5, cut=1)
    W.set_lj(pot, 0, 1, 1.5, 0.8, 2.0, cut=2)
    W.set_lj(pot, 1, 1, 0.5, 0.88, 2.2, cut=0)
    W.set_coulomb(pot, 0, 1, -1.0, 3.0, cut=1)
    r, t = W.random_gas(200, 2, (8.0, 9.0, 10.0), 5)
    box = np.array([8.0, 9.0, 10.0])
    F, u, w = oracle.forces_allpairs(r.astype(np.float64), t, box, pot)
    cnt, lst = oracle.nblist(r.astype(np.float64), t, box, pot, 0.4)
    F2, u2, w2 = oracle.forces_list(r.astype(np.float64), t, box, pot, cnt, lst)
    assert np.allclose(F, F2, rtol=1e-12, atol=1e-12) and np.allclose(u, u2, rtol=1e-12) and np.allclose(w, w2, rtol=1e-12)
    assert np.abs(F.sum(0)).max() < 1e-10 * np.abs(F).sum()


# ------------------------------------------------------------------ the other pair potentials


def test_extra_potentials_closed_forms():
    """IPL, Yukawa, Gaussian core, Buckingham at points where the value is known in closed form."""
    # IPL a r^-n: r = 2, n = 12 -> a / 4096; f = n u / r
    u, f = oracle.extra_raw(1, 2.0, 3.0, 12.0)
    assert u == pytest.approx(3.0 / 4096.0, rel=1e-14) and f == pytest.approx(12.0 * u / 2.0, rel=1e-14)
    # IPL with n = 1 is Coulomb
    assert oracle.extra_raw(1, 1.7, -2.0, 1.0) == pytest.approx(oracle.extra_raw(0, 1.7, -2.0), rel=1e-14)
    # LJ 12-6 = IPL(4 eps s^12, 12) - IPL(4 eps s^6, 6)
    eps, sig, r = 1.5, 0.8, 1.1
    u12, f12 = oracle.extra_raw(1, r, 4 * eps * sig ** 12, 12.0)
    u6, f6 = oracle.extra_raw(1, r, 4 * eps * sig ** 6, 6.0)
    assert (u12 - u6, f12 - f6) == pytest.approx(oracle.lj_raw(r, eps, sig), rel=1e-12)
    # Yukawa at r = b: u = a / (e b), f = 2 u / b; b -> infinity is Coulomb
    u, f = oracle.extra_raw(2, 0.7, 2.0, 0.7)
    assert u == pytest.approx(2.0 / (math.e * 0.7), rel=1e-14) and f == pytest.approx(2.0 * u / 0.7, rel=1e-14)
    assert oracle.extra_raw(2, 1.3, 2.0, 1e12) == pytest.approx(oracle.extra_raw(0, 1.3, 2.0), rel=1e-10)
    # Gaussian core at r = b: u = a / e, f = 2 u / b; at r = 0+ the force vanishes
    u, f = oracle.extra_raw(3, 1.5, 4.0, 1.5)
    assert u == pytest.approx(4.0 / math.e, rel=1e-14) and f == pytest.approx(2.0 * u / 1.5, rel=1e-14)
    assert oracle.extra_raw(3, 1e-9, 4.0, 1.5)[1] == pytest.approx(0.0, abs=1e-7)
    # Buckingham = exponential repulsion - dispersion: with a = 0 it is -c r^-6 (an IPL), with c = 0 a pure exponential
    assert oracle.extra_raw(4, 1.4, 0.0, 0.3, 2.0) == pytest.approx(tuple(-x for x in oracle.extra_raw(1, 1.4, 2.0, 6.0)), rel=1e-13)
    u, f = oracle.extra_raw(4, 0.6, 50.0, 0.3, 0.0)
    assert u == pytest.approx(50.0 * math.exp(-2.0), rel=1e-14) and f == pytest.approx(u / 0.3, rel=1e-14)


@pytest.mark.parametrize("kind,a,b,c", [(1, 1.3, 9.0, 0.0), (1, 2.0, 18.0, 0.0), (2, -1.5, 0.9, 0.0), (3, 3.0, 1.2, 0.0),
                                        (4, 800.0, 0.27, 1.9)])
@pytest.mark.parametrize("method", [0, 1, 2])
def test_extra_potentials_force_is_minus_gradient_and_cutoffs(kind, a, b, c, method):
    rc, h = 2.4, 1e-6
    rec = np.array([0.0, 0.0, 0.0, a, rc, 0, method, kind, b, c, 0.0])
    for r in (0.85, 1.2, 1.9, 2.39):
        up, _ = oracle.pair_sf(rec, r + h)
        um, _ = oracle.pair_sf(rec, r - h)
        _, f = oracle.pair_sf(rec, r)
        assert f == pytest.approx(-(up - um) / (2 * h), rel=3e-7, abs=1e-9)
    assert oracle.pair_sf(rec, rc) == (0.0, 0.0) and oracle.pair_sf(rec, 3.0) == (0.0, 0.0)
    ur, fr = oracle.extra_raw(kind, 1.3, a, b, c)
    uc, fc = oracle.extra_raw(kind, rc, a, b, c)
    want = {0: (ur - uc + (1.3 - rc) * fc, fr - fc), 1: (ur - uc, fr), 2: (ur, fr)}[method]
    assert oracle.pair_sf(rec, 1.3) == pytest.approx(want, rel=1e-13)


def test_generalized_lj_girifalco_dzugutov_pins():
    """The remaining pair potentials of P:73, pinned to what does not depend on this code: generalized LJ to the 12-6
    potential and to its defining properties; Girifalco to the C60 figures of Girifalco, J. Phys. Chem. 96, 858 (1992)
    (alpha 74.94e-15 erg, beta 135.95e-18 erg, 2a = 7.1 A: well depth 0.2773 eV = 3218 K at 10.056 A) and to its
    van der Waals limit; Dzugutov to the extrema of Dzugutov, Phys. Rev. A 46, R2984 (1992) (minimum -0.581 at 1.13,
    maximum 0.460 at 1.63, zero from 1.94)."""
    from scipy.optimize import minimize_scalar
    # generalized LJ: (m, n) = (12, 6) is 12-6 LJ with sigma_LJ = sigma / 2^(1/6); minimum -eps at r = sigma for any (m, n)
    eps, sig = 1.7, 1.1
    for r in (0.95, 1.1, 1.6, 2.3):
        assert oracle.extra_raw(5, r, eps, sig, 12.0, 6.0) == pytest.approx(oracle.lj_raw(r, eps, sig / 2 ** (1 / 6)), rel=1e-12, abs=1e-14)
    for m, n in ((12.0, 6.0), (9.0, 6.0), (18.0, 4.0), (7.5, 3.5)):
        u, f = oracle.extra_raw(5, sig, eps, sig, m, n)
        assert u == pytest.approx(-eps, rel=1e-14) and abs(f) < 1e-13
        # r -> large: -eps m / (m - n) (sig / r)^n dominates
        u, _ = oracle.extra_raw(5, 40.0 * sig, eps, sig, m, n)
        assert u == pytest.approx(-eps * m / (m - n) * 40.0 ** -n, rel=1e-4)
    # Girifalco, C60 (energies in eV, lengths in Angstrom)
    al, be, d = 74.94e-15 / 1.602177e-12, 135.95e-18 / 1.602177e-12, 7.1
    res = minimize_scalar(lambda r: oracle.extra_raw(6, r, al, be, d)[0], bounds=(9.0, 12.0), method="bounded", options={"xatol": 1e-10})
    assert res.x == pytest.approx(10.056, abs=2e-3) and res.fun == pytest.approx(-0.2773, abs=2e-4)
    assert res.fun * 11604.5 == pytest.approx(-3218.0, abs=2.0)
    assert abs(oracle.extra_raw(6, res.x, al, be, d)[1]) < 1e-7
    u, _ = oracle.extra_raw(6, 60.0 * d, al, be, d)  # s -> infinity: -12 alpha / s^6
    assert u == pytest.approx(-12.0 * al / 60.0 ** 6, rel=2e-3)
    # Dzugutov (eps = sigma = 1), then scaled
    res = minimize_scalar(lambda r: oracle.extra_raw(7, r, 1.0, 1.0)[0], bounds=(1.0, 1.4), method="bounded", options={"xatol": 1e-10})
    assert res.x == pytest.approx(1.13, abs=2e-3) and res.fun == pytest.approx(-0.581, abs=1e-3)
    res = minimize_scalar(lambda r: -oracle.extra_raw(7, r, 1.0, 1.0)[0], bounds=(1.4, 1.9), method="bounded", options={"xatol": 1e-10})
    assert res.x == pytest.approx(1.63, abs=3e-3) and -res.fun == pytest.approx(0.460, abs=1e-3)
    assert oracle.extra_raw(7, 1.94, 1.0, 1.0) == (0.0, 0.0) and oracle.extra_raw(7, 2.5, 1.0, 1.0) == (0.0, 0.0)
    u1, f1 = oracle.extra_raw(7, 1.2, 1.0, 1.0)
    u2, f2 = oracle.extra_raw(7, 1.2 * 1.5, 2.5, 1.5)
    assert (u2, f2) == pytest.approx((2.5 * u1, 2.5 * f1 / 1.5), rel=1e-13)


@pytest.mark.parametrize("kind,a,b,c,d", [(5, 1.3, 1.05, 12.0, 6.0), (5, 0.8, 1.2, 9.5, 4.0), (6, 3.0, 0.004, 0.75, 0.0),
                                          (7, 1.4, 1.1, 0.0, 0.0)])
@pytest.mark.parametrize("method", [0, 1, 2])
def test_more_potentials_force_is_minus_gradient_and_cutoffs(kind, a, b, c, d, method):
    rc, h = 2.05, 1e-6
    rec = np.array([0.0, 0.0, 0.0, a, rc, 0, method, kind, b, c, d])
    for r in (0.98, 1.2, 1.45, 1.9, 2.04):
        up, _ = oracle.pair_sf(rec, r + h)
        um, _ = oracle.pair_sf(rec, r - h)
        _, f = oracle.pair_sf(rec, r)
        assert f == pytest.approx(-(up - um) / (2 * h), rel=1e-6, abs=1e-8)
    assert oracle.pair_sf(rec, rc) == (0.0, 0.0) and oracle.pair_sf(rec, 3.0) == (0.0, 0.0)
    ur, fr = oracle.extra_raw(kind, 1.3, a, b, c, d)
    uc, fc = oracle.extra_raw(kind, rc, a, b, c, d)
    want = {0: (ur - uc + (1.3 - rc) * fc, fr - fc), 1: (ur - uc, fr), 2: (ur, fr)}[method]
    assert oracle.pair_sf(rec, 1.3) == pytest.approx(want, rel=1e-13)


def test_extra_potentials_list_forces_equal_brute_force_and_newton():
    pot = W.pot_table(2)
    W.set_lj(pot, 0, 0, 1.0, 1.0, 2.5)
    W.set_second_term(pot, 0, 0, W.KIND_YUKAWA, 1.2, 0.8, 0.0, 3.0)
    W.set_second_term(pot, 0, 1, W.KIND_BUCKINGHAM, 900.0, 0.28, 1.5, 2.6, cut=W.CUT_SHIFTED_POTENTIAL)
    W.set_second_term(pot, 1, 1, W.KIND_IPL, 1.0, 12.0, 0.0, 2.0)
    r, t = W.random_gas(216, 2, (8.5, 8.5, 9.5), 3)
    box = np.array([8.5, 8.5, 9.5])
    r64 = r.astype(np.float64)
    F, u, w = oracle.forces_allpairs(r64, t, box, pot)
    cnt, lst = oracle.nblist(r64, t, box, pot, 0.35)
    F2, u2, w2 = oracle.forces_list(r64, t, box, pot, cnt, lst)
    assert np.allclose(F, F2, rtol=1e-12, atol=1e-12) and np.allclose(u, u2, rtol=1e-12) and np.allclose(w, w2, rtol=1e-12)
    assert np.abs(F.sum(0)).max() < 1e-10 * np.abs(F).sum()
    # virial = -dU/d(ln scale): uniform dilation (as in P5)
    lam = 1e-6
    Up = oracle.forces_allpairs(r64 * (1 + lam), t, box * (1 + lam), pot)[1].sum()
    Um = oracle.forces_allpairs(r64 * (1 - lam), t, box * (1 - lam), pot)[1].sum()
    # only valid for continuous energies: the shifted-potential AB term is continuous in u, fine
    assert (Up - Um) / (2 * lam) == pytest.approx(-w.sum(), rel=2e-5)


# ------------------------------------------------------------------ P13: NPT ("NPT [51]"; reading S32)


def _lj_fluid(ncell=3, density=0.7, T=1.5, seed=11):
    r, box = W.fcc_lattice(ncell, ncell, ncell, density)
    rng = np.random.default_rng(seed)
    N = r.shape[0]
    m = np.ones(N)
    v = W.maxwell_boltzmann(rng, m, T)
    return r, v, m, np.zeros((N, 3), np.int32), np.zeros(N, np.int32), box, LJ


def test_P13_npt_with_the_barostat_off_is_nvt_bit_for_bit():
    """tau_P = inf and nu(0) = 0: the strain rate stays 0, exp(0) = 1, and every expression of the NPT step reduces
    to the NVT step of O7 -- positions, velocities, thermostat and box identical bit for bit over 60 steps."""
    r, v, m, im, t, box, pot = _lj_fluid()
    a = oracle.run(r, v, m, im, t, box, pot, 0.3, 0.004, 60, mode=oracle.NVT, T0=1.2, tau=0.2)
    b = oracle.run_npt(r, v, m, im, t, box, pot, 0.3, 0.004, 60, T0=1.2, tau=0.2, P0=3.0, tauP=float("inf"))
    assert np.array_equal(a["r"], b["r"]) and np.array_equal(a["v"], b["v"]) and np.array_equal(a["image"], b["image"])
    assert a["xi"] == b["xi"] and a["eta"] == b["eta"] and b["nu"] == 0.0 and np.array_equal(b["box"], box)
    assert np.array_equal(a["log"][:, :5], b["log"][:, :5])
    # ... and with P0 = 0 the conserved quantities coincide too (H_NPT = H_NVT + P0 V)
    c = oracle.run_npt(r, v, m, im, t, box, pot, 0.3, 0.004, 60, T0=1.2, tau=0.2, P0=0.0, tauP=0.0)
    assert np.array_equal(a["log"][:, 5], c["log"][:, 5])


def test_P13_npt_free_flight_under_constant_strain_rate_closed_form():
    """No forces (rc far below every distance is not needed: an empty potential table), thermostat off, barostat
    frozen at nu = nu0 (tau_P = inf): the continuous equations integrate in closed form,
        L(t) = L0 exp(nu0 t),   v(t) = v0 exp(-(1 + 3/g) nu0 t),   unwrapped r(t) = e^{nu0 t} [ r0 + v0 (1 - e^{-k t}) / k ],
    k = (2 + 3/g) nu0.  The discrete box follows L0 exp(nu0 n dt) EXACTLY; velocities and positions converge to the
    closed form with the second order of a leap-frog scheme (error ratio 4 when dt is halved)."""
    N, L0, nu0, T = 5, 9.0, 0.37, 0.8
    rng = np.random.default_rng(3)
    r0 = rng.uniform(-1.0, 1.0, (N, 3))
    v0 = rng.standard_normal((N, 3))
    m = np.ones(N)
    g = 3.0 * N - 3.0
    pot = W.pot_table(1)                         # no potential terms at all: F = 0, W = 0
    k = (2.0 + 3.0 / g) * nu0
    errs = []
    for n in (40, 80, 160):
        dt = T / n
        # leap-frog input velocities are v(-dt/2): the closed form evaluated there
        vm = v0 * math.exp((1.0 + 3.0 / g) * nu0 * 0.5 * dt)
        o = oracle.run_npt(r0, vm, m, np.zeros((N, 3), np.int32), np.zeros(N, np.int32), np.full(3, L0), pot, 0.3, dt, n,
                           T0=1.0, tau=0.0, P0=0.0, tauP=float("inf"), nu=nu0)
        assert np.allclose(o["box"], L0 * math.exp(nu0 * T), rtol=1e-13)        # product of exp(nu0 dt): exact
        assert o["nu"] == nu0 and o["xi"] == 0.0
        v_exact = v0 * math.exp(-(1.0 + 3.0 / g) * nu0 * (T - 0.5 * dt))         # v(T - dt/2)
        r_exact = math.exp(nu0 * T) * (r0 + v0 * (1.0 - math.exp(-k * T)) / k)
        r_unwrapped = o["r"] + o["image"] * o["box"]
        errs.append((np.abs(o["v"] - v_exact).max(), np.abs(r_unwrapped - r_exact).max()))
    for col in (0, 1):
        assert errs[0][col] / errs[1][col] == pytest.approx(4.0, rel=0.15)
        assert errs[1][col] / errs[2][col] == pytest.approx(4.0, rel=0.15)
    assert errs[2][0] < 1e-5 and errs[2][1] < 1e-4


def test_P13_npt_single_step_worked_example():
    """One step with numbers chosen so the scale factors are powers of two: N = 2 (g = 3), xi = 0, barostat frozen
    (tau_P = 0) at nu with nu dt / 2 = ln 2 -> sh = 2, s = 4, gam dt / 2 = (1 + 3/3) nu dt / 2 = 2 ln 2.  F = 0:
        v' = (1 - 2 ln 2)/(1 + 2 ln 2) v,   r' = 4 r + dt * 2 * v',   L' = 4 L.
    Then the strain-rate update with the barostat on (W = 7, P0 = 0.2, tau_P = 2): two half kicks of the position part
    pos = cP (W - 3 V P0) around nu(t), one whole kick of the kinetic part (1 + 3/g) cP sum m v'^2."""
    dt, ln2 = 0.5, math.log(2.0)
    nu = 2.0 * ln2 / dt
    r = np.array([[0.25, -0.5, 0.125], [-0.75, 0.5, 0.375]])
    v = np.array([[1.0, -2.0, 0.5], [-1.0, 2.0, -0.5]])
    m = np.array([1.0, 2.0])
    box = np.array([4.0, 5.0, 6.0])
    T0 = 1.5
    rn, vn, im, boxn, xi, eta, nun, Kt, mv2 = oracle.integrate_npt(r, v, m, np.zeros((2, 3), np.int32), np.zeros((2, 3)), 0.0,
                                                                   box, dt, T0, 0.0, 0.2, 0.0, nu=nu)
    fac = (1.0 - 2.0 * ln2) / (1.0 + 2.0 * ln2)
    assert np.allclose(vn, fac * v, rtol=1e-14)
    assert np.allclose(boxn, 4.0 * box, rtol=1e-14)
    x = 4.0 * r + dt * 2.0 * fac * v
    assert np.allclose(rn + im * boxn, x, rtol=1e-13, atol=1e-14)
    assert np.all(np.abs(rn) <= 0.5 * boxn + 1e-12)
    assert mv2 == pytest.approx((m[:, None] * (fac * v) ** 2).sum(), rel=1e-14)
    assert nun == nu and xi == 0.0 and eta == 0.0
    assert Kt == pytest.approx(0.5 * (m[:, None] * (0.5 * (1.0 + fac) * v) ** 2).sum(), rel=1e-14)
    # barostat on: V = 120, g = 3, cP = pi^2 / (6 T0) for tau_P = 2
    Wv, P0 = 7.0, 0.2
    cP = math.pi ** 2 / (6.0 * T0)
    pos = cP * (Wv - 3.0 * 120.0 * P0)
    nu_t = nu + 0.5 * dt * pos
    gam = 2.0 * nu_t
    v2 = (1.0 - 0.5 * gam * dt) / (1.0 + 0.5 * gam * dt) * v
    smv2_old, smv2_new = (m[:, None] * v * v).sum(), (m[:, None] * v2 * v2).sum()
    out = oracle.integrate_npt(r, v, m, np.zeros((2, 3), np.int32), np.zeros((2, 3)), Wv, box, dt, T0, 0.0, P0, 2.0, nu=nu)
    assert np.allclose(out[1], v2, rtol=1e-13)
    assert out[6] == pytest.approx(nu_t + 0.5 * dt * pos + dt * cP * 2.0 * smv2_new, rel=1e-13)
    nu_h = nu_t + 0.5 * dt * pos + 0.5 * dt * cP * 2.0 * smv2_old
    assert np.allclose(out[3], box * math.exp(nu_h * dt), rtol=1e-13)


def test_P13_npt_conserved_quantity_and_target_pressure():
    """LJ fluid, N = 500: (a) the conserved quantity H_NPT fluctuates ~ dt^2 with no drift; (b) started at a pressure
    well below P0 the volume shrinks, and the time-averaged pressure settles at P0 (and <T_kin> at T0)."""
    r, v, m, im, t, box, pot = _lj_fluid(ncell=5, density=0.5, T=2.0, seed=5)
    N = r.shape[0]
    T0, P0, tauP = 2.0, 2.0, 2.0
    eq = oracle.run_npt(r, v, m, im, t, box, pot, 0.3, 0.004, 1500, T0=T0, tau=0.2, P0=P0, tauP=tauP)
    assert eq["log"][0, 8] < 0.5 * P0                        # the start is far below the target pressure ...
    assert np.prod(eq["box"]) < 0.95 * np.prod(box)          # ... so the box has shrunk
    amp = []
    for dt, n in ((0.004, 1000), (0.002, 2000)):
        o = oracle.run_npt(eq["r"], eq["v"], m, eq["image"], t, eq["box"], pot, 0.3, dt, n, T0=T0, tau=0.2, P0=P0, tauP=tauP,
                           xi=eq["xi"], eta=eq["eta"], nu=eq["nu"])
        H = o["log"][:, 5] / N
        tt = np.arange(n) * dt
        fit = np.polyfit(tt, H, 1)
        amp.append(np.std(H - np.polyval(fit, tt)))
        assert abs(fit[0]) * n * dt < 2e-3                   # no drift over the run
    assert amp[0] / amp[1] == pytest.approx(4.0, rel=0.4)    # fluctuation ~ dt^2
    long = oracle.run_npt(eq["r"], eq["v"], m, eq["image"], t, eq["box"], pot, 0.3, 0.004, 6000, T0=T0, tau=0.2, P0=P0,
                          tauP=tauP, xi=eq["xi"], eta=eq["eta"], nu=eq["nu"])
    P = long["log"][:, 8]
    Tk = 2.0 * long["log"][:, 1] / (3.0 * N - 3.0)
    assert P.mean() == pytest.approx(P0, abs=0.08)
    assert Tk.mean() == pytest.approx(T0, rel=0.02)
