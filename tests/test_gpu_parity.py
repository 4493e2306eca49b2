"""GPU parity tests: the CUDA path (through the C ABI, via the ctypes binding) against the fp64 oracle,
element by element, on the same seeded fp32-representable inputs.  Run with ``-m gpu`` on a B200.

Bars (BASELINE.json north_star; norms per DESIGN.md S25):
  * neighbour lists identical as pair sets, apart from pairs within 1e-6 sigma of the list cutoff;
  * per-particle fp32 forces: max_i |F_i - F_i^oracle| <= 1e-4 * rms_i |F_i^oracle|;
  * potential energy (and virial) to 1e-5 relative after one step from identical inputs.
"""
import numpy as np
import pytest

import oracle
from paper_1506_05094_b200 import workloads as W

pytestmark = pytest.mark.gpu

FORCE_TOL = 1e-4
ENERGY_TOL = 1e-5
BAND = 1e-6


@pytest.fixture(scope="module")
def rumd():
    from paper_1506_05094_b200 import rumd as R

    return R


def perturbed(wl, amp=0.05, seed=7):
    a = amp * wl.meta.get("a", 1.0)
    wl.r = W.perturb(wl.r, wl.box, a, seed)
    return wl


def lattice_spacing(wl):
    return (1.0 / wl.meta["density"]) ** (1.0 / 3.0) if wl.meta["lattice"] != "fcc" else (4.0 / wl.meta["density"]) ** (1.0 / 3.0)


def make(kind, **kw):
    wl = {"lj": W.lj_fcc, "ka": W.ka_lattice, "ch": W.charged_sc}[kind](**kw)
    wl.meta["a"] = lattice_spacing(wl)
    return wl


def pair_keys(count, lst, ids=None):
    """Set of directed pairs i*N+j (original numbering when ids is given)."""
    N = count.shape[0]
    rows = np.repeat(np.arange(N), count)
    mask = np.arange(lst.shape[1])[None, :] < count[:, None]
    cols = lst[mask]
    if ids is not None:
        rows = ids[rows]
        cols = ids[cols]
    return rows.astype(np.int64) * N + cols.astype(np.int64)


def check_nblist(sys_, r64, types, box, pot, skin):
    """GPU list == oracle O2 set, except pairs within BAND of the list cutoff."""
    cnt, lst = sys_.export_nblist()
    ids = sys_.d_id.cpu().numpy().astype(np.int64)
    assert cnt.max() <= sys_.capacity
    gpu = pair_keys(cnt, lst, ids)
    assert np.unique(gpu).size == gpu.size, "duplicate neighbours"
    oc, ol = oracle.nblist(r64, types, box, pot, skin, method="n2" if r64.shape[0] <= 20000 else "cell")
    ora = pair_keys(oc, ol)
    diff = np.setxor1d(gpu, ora)
    N = r64.shape[0]
    if diff.size:
        i, j = diff // N, diff % N
        d = r64[i] - r64[j]
        d -= box * np.rint(d / box)
        dist = np.sqrt((d * d).sum(1))
        rc = np.maximum(pot[types[i], types[j], 2], pot[types[i], types[j], 4]) + skin
        assert np.all(np.abs(dist - rc) <= BAND), "pair sets differ outside the 1e-6 band: %d pairs, worst %g" % (
            diff.size, np.abs(dist - rc).max())
    return cnt, gpu.size, diff.size


def check_forces(sys_, r64, types, box, pot, cancelling=False):
    """Forces (S25 norm), U and W (1e-5 relative, north_star) and per-particle u_i, w_i against the oracle.
    cancelling=True ONLY for the simple-cubic Kob-Andersen lattice start, where U = sum u_i nearly cancels
    (U/N ~ -0.01 with |u_i| ~ 5): there the scale of the 1e-5 bar is sum |u_i| (S29); everywhere else
    it is |U| itself."""
    st = sys_.state()
    F, u, w = oracle.forces_allpairs(r64, types, box, pot) if r64.shape[0] <= 20000 else \
        oracle.forces_list(r64, types, box, pot, *oracle.nblist(r64, types, box, pot, 0.0, method="cell"))
    rms = np.sqrt((F * F).sum(1).mean())
    err = np.sqrt(((st["F"].astype(np.float64) - F) ** 2).sum(1)).max()
    assert err <= FORCE_TOL * rms, "max|dF| = %g > 1e-4 * rms|F| = %g" % (err, FORCE_TOL * rms)
    th = sys_.get_thermo()
    uscale = np.abs(u).sum() if cancelling else abs(u.sum())
    wscale = np.abs(w).sum() if cancelling else abs(w.sum())
    assert abs(th["U"] - u.sum()) <= ENERGY_TOL * uscale, (th["U"], u.sum())
    assert abs(th["W"] - w.sum()) <= ENERGY_TOL * wscale, (th["W"], w.sum())
    # per-particle energies and virials (absolute tolerance scaled by their rms)
    assert np.abs(st["u"] - u).max() <= 1e-5 * max(1.0, np.abs(u).max())
    assert np.abs(st["w"] - w).max() <= 1e-5 * max(1.0, np.abs(w).max())
    return err / rms


def check_nblist_rows(sys_, r64, types, box, pot, skin):
    """check_nblist for sizes where 10^8 pair keys are too many to sort: both lists as (N, width) arrays of
    ORIGINAL neighbour indices, every row sorted; rows that differ are then compared as sets, and every
    disagreement must lie within BAND of the pair's list cutoff.  Covers ALL rows."""
    N = r64.shape[0]
    cnt, lst = sys_.export_nblist()
    ids = sys_.d_id.cpu().numpy().astype(np.int64)
    assert cnt.max() <= sys_.capacity
    oc, ol = oracle.nblist(r64, types, box, pot, skin, method="cell")
    width = max(int(cnt.max()), int(oc.max()))
    BIG = np.int32(2 ** 31 - 1)

    def rows(count, table, idmap):
        t = table[:, :width] if table.shape[1] >= width else np.pad(table, ((0, 0), (0, width - table.shape[1])), constant_values=-1)
        valid = np.arange(width)[None, :] < count[:, None]
        out = np.where(valid, idmap[np.maximum(t, 0)].astype(np.int32) if idmap is not None else t, BIG)
        out.sort(axis=1)
        return out

    G = np.empty((N, width), np.int32)
    G[ids] = rows(cnt, lst, ids)          # row of slot s belongs to original particle ids[s]
    del lst
    O = rows(oc, ol, None)
    gcnt = np.empty(N, np.int64)
    gcnt[ids] = cnt
    assert ((G[:, 1:] != G[:, :-1]) | (G[:, 1:] == BIG)).all(), "duplicate neighbours"
    bad = np.flatnonzero((G != O).any(1))
    nband = 0
    for i in bad:
        g = set(G[i][G[i] != BIG].tolist())
        o = set(O[i][O[i] != BIG].tolist())
        for j in g ^ o:
            d = r64[j] - r64[i]
            d -= box * np.rint(d / box)
            rcl = max(pot[types[i], types[j], 2], pot[types[i], types[j], 4]) + skin
            assert abs(np.sqrt((d * d).sum()) - rcl) <= BAND, "pair (%d, %d) differs outside the 1e-6 band" % (i, j)
            nband += 1
    return gcnt, int(oc.sum()), nband


CASES = [
    ("lj", dict(ncell=6), "n2", 32),          # configs[0], N = 864
    ("lj", dict(ncell=6), "cell", 4),
    ("lj", dict(ncell=10), "cell", 1),        # N = 4000, several tiles + ragged tail
    ("ka", dict(N=1000), "n2", 16),
    ("ka", dict(N=4096), "cell", 8),
    ("ka", dict(N=8000), "cell", 2),          # configs[1]
    ("ka", dict(N=2048), "n2", 1),            # orthorhombic box 16x16x8
    ("ch", dict(n=12), "cell", 8),            # charged, N = 1728, rc 4.0 + LJ 2.5
    ("ch", dict(n=10), "n2", 4),
    # tile method (j-particles staged in shared memory, 16-bit slot lists)
    ("lj", dict(ncell=10), "tile", 1),        # 12 cells per axis -> 3x3x3 tiles, every tile touches a face
    ("lj", dict(ncell=16), "tile", 2),        # N = 16384, 19 cells per axis: interior and boundary tiles
    ("ka", dict(N=8000), "tile", 8),          # configs[1]
    ("ka", dict(N=4096), "tile", 4),
    ("ka", dict(N=16384), "tile", 1),         # orthorhombic 32x32x16 lattice
    ("ch", dict(n=16), "tile", 2),            # charged, rc 4.0: 9 cells per axis
]

METHODS = {"n2": 0, "cell": 1, "none": 2, "tile": 3}


def test_one_lane_build_wide_box_matches_oracle(rumd):
    """A4 with one thread per particle (the paper's P:278 configuration) in a wide box: N = 42592 (22^3 fcc
    cells, 26 cells per axis, interior fast path of the minimum image in play), whole list and all forces
    against the oracle's cell search."""
    wl = perturbed(make("lj", ncell=22))
    s = rumd.from_workload(wl)
    s.set_tuning(method=rumd.NB_CELL, tp=1, pb=256, build_tp=1)
    s.compute_forces()
    r64 = wl.r.astype(np.float64)
    box = wl.box.astype(np.float64)
    cnt, npairs, nband = check_nblist(s, r64, wl.types, box, wl.pot, float(wl.skin))
    assert npairs > 3e6
    check_forces(s, r64, wl.types, box, wl.pot)
    # the same list as the several-lanes-per-particle build (as sets; row order differs)
    keys_g1 = np.sort(pair_keys(*s.export_nblist(), s.d_id.cpu().numpy().astype(np.int64)))
    s.set_tuning(build_tp=8)
    s.build_nblist()
    keys_g8 = np.sort(pair_keys(*s.export_nblist(), s.d_id.cpu().numpy().astype(np.int64)))
    assert np.array_equal(keys_g1, keys_g8)
    s.close()


def _sampled_check(rumd, s, wl, nsample, seed):
    """List rows, forces and energies of sampled particles against the oracle run on the cluster of all particles
    within rc_max + skin + 0.2 of the sample (it contains every interaction partner of the sample)."""
    N = wl.N
    r64 = wl.r.astype(np.float64)
    box = wl.box.astype(np.float64)
    cnt, lst = s.export_nblist()
    ids = s.d_id.cpu().numpy().astype(np.int64)
    slot_of = np.empty(N, np.int64)
    slot_of[ids] = np.arange(N)
    st = s.state()
    skin = float(s.get_tuning().skin)
    rcm = wl.rc_max()
    rmsF = np.sqrt((st["F"].astype(np.float64) ** 2).sum(1).mean())
    for i in np.random.default_rng(seed).choice(N, nsample, replace=False):
        d = r64 - r64[i]
        d -= box * np.rint(d / box)
        near = np.flatnonzero((d * d).sum(1) < (rcm + skin + 0.2) ** 2)
        sub = np.concatenate(([i], near[near != i]))
        F, u, w = oracle.forces_allpairs(r64[sub], wl.types[sub], box, wl.pot)
        oc, ol = oracle.nblist(r64[sub], wl.types[sub], box, wl.pot, skin, method="n2")
        want = set(sub[ol[0, :oc[0]]].tolist())
        row = slot_of[i]
        got = set(ids[lst[row, :cnt[row]]].tolist())
        for j in want ^ got:
            dj = r64[j] - r64[i]
            dj -= box * np.rint(dj / box)
            rcl = max(wl.pot[wl.types[i], wl.types[j], 2], wl.pot[wl.types[i], wl.types[j], 4]) + skin
            assert abs(np.sqrt((dj * dj).sum()) - rcl) <= BAND
        assert np.sqrt(((st["F"][i] - F[0]) ** 2).sum()) <= FORCE_TOL * rmsF
        assert abs(st["u"][i] - u[0]) <= 1e-5 * max(1.0, abs(u[0]))
        assert abs(st["w"][i] - w[0]) <= 1e-5 * max(1.0, abs(w[0]))
    return cnt, st


@pytest.mark.parametrize("kind,kw", [("ch", dict(n=32)), ("ka", dict(N=131072))])
def test_full_size_configs_sampled_against_oracle(rumd, kind, kw):
    """configs[4] (charged, N = 32768, ~170 list entries) and the largest configs[2] entry (KA N = 131072) at full
    size with the library's default tuning for that N, after 40 time steps from the perturbed lattice (so the
    list has been rebuilt and the particles re-sorted in flight): sampled rows against the oracle."""
    wl = perturbed(make(kind, **kw))
    s = rumd.from_workload(wl)
    s.run_steps(40)
    s.build_nblist()                      # list of the CURRENT positions (the one in flight is a few steps old)
    s.compute_forces()
    st0 = s.state()
    wl.r = st0["r"]                       # the oracle sees the positions the GPU now holds (fp32 values)
    cnt, st = _sampled_check(rumd, s, wl, 48, 11)
    assert s.get_thermo()["n_rebuilds"] >= 2 and cnt.sum() % 2 == 0
    Fsum = st["F"].astype(np.float64).sum(0)
    assert np.abs(Fsum).max() <= 1e-3 * np.abs(st["F"]).sum()
    s.close()


def test_full_size_million_particles_whole_system_against_oracle(rumd):
    """configs[3] at full size (N = 1 048 576) in the configuration bench.py times (library defaults for this N:
    cell build with spatial sort, one lane per particle), WHOLE system: every row of the list against the
    oracle's cell search as a set (1e-6 band), every force, u_i and w_i against orc_forces_list, total U and W
    at 1e-5 of |U|, |W|.  Then the unperturbed 64^3 lattice: 78 entries in every row and the P6 lattice sum."""
    wl = perturbed(make("lj", ncell=64))
    s = rumd.from_workload(wl)
    s.compute_forces()
    N = wl.N
    r64 = wl.r.astype(np.float64)
    box = wl.box.astype(np.float64)
    skin = float(wl.skin)
    gcnt, npairs, nband = check_nblist_rows(s, r64, wl.types, box, wl.pot, skin)
    assert npairs > 7e7 and int(gcnt.sum()) in range(npairs - nband, npairs + nband + 1)
    # particles whose list reaches across a face of the box (exact-shift minimum image at L = 107): all covered
    assert (np.abs(r64) > 0.5 * box - (2.5 + skin)).any(1).sum() > 1e5
    err = check_forces(s, r64, wl.types, box, wl.pot)      # all rows; U, W at the |U|, |W| scale
    assert err < 1e-4
    th = s.get_thermo()
    assert th["overflow"] == 0 and th["max_nbrs"] == gcnt.max()
    s.close()
    # perfect lattice (P6): 78 list entries per particle, U/N = -5.693278275711, W/N = -20.165268242841
    wl0 = make("lj", ncell=64)
    s = rumd.from_workload(wl0)
    s.compute_forces()
    cnt, _ = s.export_nblist()
    assert cnt.min() == 78 and cnt.max() == 78
    th = s.get_thermo()
    assert th["U"] / N == pytest.approx(-5.693278275711, rel=ENERGY_TOL)
    assert th["W"] / N == pytest.approx(-20.165268242841, rel=ENERGY_TOL)
    s.close()


def _fresh_from_state(rumd, wl, st):
    """A new System (thermostat and counters at zero) holding the fp32 state `st` in ORIGINAL particle order."""
    wl.r, wl.v = st["r"].copy(), st["v"].copy()
    return rumd.from_workload(wl)


@pytest.mark.parametrize("name,kind,kw,equil,tuning", [
    # configs[1] with the tuning bench.py's autotuner picks for it (profiles/r01_bench_sweep.md)
    ("C1", "ka", dict(N=8000), 2000, dict(method=1, tp=8, pb=32, build_tp=8, skin=0.388, persistent=1)),
    ("C4", "ch", dict(n=32), 200, dict()),
    ("C3", "lj", dict(ncell=64), 60, dict()),
])
def test_one_step_at_bench_sizes_matches_oracle(rumd, name, kind, kw, equil, tuning):
    """north_star: "potential energy must agree to 1e-5 relative after one step from identical inputs", at the
    sizes and tunings the bench times.  The state is first relaxed on the GPU (the lattice starts are a hot
    transient; on the KA one U nearly cancels, S29), read back, and handed as fp32 values to BOTH sides:
    one whole step (build -> forces -> integrate) on each, then U, K, xi, positions and velocities, and U, W,
    forces of the NEW configuration at the |U| scale."""
    wl = make(kind, **kw)
    if kind != "ka":
        wl = perturbed(wl)
    s0 = rumd.from_workload(wl)
    if tuning:
        s0.set_tuning(**tuning)
    s0.run_steps(equil)
    st0 = s0.state()
    assert s0.get_thermo()["overflow"] == 0
    s0.close()
    s = _fresh_from_state(rumd, wl, st0)
    if tuning:
        s.set_tuning(**tuning)
    N = wl.N
    r64, v64, m64 = wl.r.astype(np.float64), wl.v.astype(np.float64), wl.m.astype(np.float64)
    box = wl.box.astype(np.float64)
    skin = float(s.get_tuning().skin)
    o = oracle.run(r64, v64, m64, np.zeros((N, 3), np.int32), wl.types, box, wl.pot, skin, float(wl.dt), 1,
                   mode=wl.integrator, T0=wl.T0, tau=wl.tau, use_cell=N >= 4096)
    s.run_steps(1)
    th1 = s.get_thermo()
    st = s.state()
    d = st["r"].astype(np.float64) + st["image"] * box - (o["r"] + o["image"] * box)
    assert np.abs(d).max() < max(2e-6, 6e-8 * box.max())   # half an fp32 ulp of the largest coordinate
    assert np.abs(st["v"] - o["v"]).max() < 1e-5 * max(1.0, np.abs(o["v"]).max())
    U0, K0 = o["log"][0, 0], o["log"][0, 1]
    assert th1["U"] == pytest.approx(U0, rel=ENERGY_TOL)
    assert th1["K"] == pytest.approx(K0, rel=ENERGY_TOL)
    if wl.integrator == W.NVT:
        assert th1["xi"] == pytest.approx(o["xi"], rel=1e-4, abs=1e-7)
        assert th1["eta"] == pytest.approx(o["eta"], rel=1e-4, abs=1e-9)
    # forces / energies of the NEW configuration: the oracle evaluates the positions the GPU now holds
    s.compute_forces()
    r1 = s.state()["r"].astype(np.float64)
    check_forces(s, r1, wl.types, box, wl.pot)
    s.close()


def test_c1_nvt_conserved_quantity_drift(rumd):
    """S26 on configs[1]: Nose-Hoover conserved quantity H_NH (O10) over 1e4 steps after equilibration, least-squares
    slope of H/N times the run length <= 1e-4 per particle.  (The Nose-Hoover discretisation and tau = 0.2 are
    readings: this checks the GPU integrator against its own invariant.)"""
    wl = make("ka", N=8000)
    s = rumd.from_workload(wl)
    s.set_tuning(method=rumd.NB_CELL, tp=8, pb=32, build_tp=8, skin=0.388)
    s.run_steps(2000)
    H = []
    for _ in range(100):
        s.run_steps(100)
        H.append(s.get_thermo()["H"] / wl.N)
    H = np.array(H)
    slope = np.polyfit(np.arange(H.size) * 100.0, H, 1)[0]
    assert abs(slope * 1e4) <= 1e-4, "H_NH drift %g per particle over 1e4 steps" % (slope * 1e4)
    assert np.abs(H - H[0]).max() < 5e-3
    s.close()


def test_c3_nve_energy_drift(rumd):
    """S26 on configs[3] (N = 1 048 576, cell build + re-sorting in flight, the unit queue of the build): the FULL 1e4
    NVE steps of the north_star bar, slope of E/N times the run length <= 1e-4 per particle."""
    wl = make("lj", ncell=64)
    s = rumd.from_workload(wl)
    s.run_steps(200)                # melt off the lattice
    E = []
    for _ in range(100):
        s.run_steps(100)
        th = s.get_thermo()
        E.append((th["K"] + th["U"]) / wl.N)
    E = np.array(E)
    slope = np.polyfit(np.arange(E.size) * 100.0, E, 1)[0]
    assert abs(slope * 1e4) <= 1e-4, "drift %g per particle per 1e4 steps" % (slope * 1e4)
    assert np.abs(E - E[0]).max() < 5e-3
    assert s.get_thermo()["n_rebuilds"] >= 500
    s.close()


@pytest.mark.parametrize("kind,kw,tuning", [
    ("ch", dict(n=32), dict(method=1, tp=2, pb=128, build_tp=2, skin=0.345)),       # configs[4] with its bench tuning
    ("ka", dict(N=131072), dict(method=1, tp=2, pb=128, build_tp=4, skin=0.30)),    # largest configs[2] entry
    ("ka", dict(N=8000), dict(method=1, tp=8, pb=32, build_tp=8, skin=0.397)),      # configs[1] run as NVE
])
def test_nve_energy_drift_at_the_other_bench_sizes(rumd, kind, kw, tuning):
    """S26 / north_star drift bar at the remaining bench sizes, run as NVE (two particle types: the register-select
    force loop; C4: the Coulomb term): 1e4 steps after 2000 steps of equilibration under the workload's thermostat,
    slope of E/N times the run length <= 1e-4 per particle."""
    wl = make(kind, **kw)
    s = rumd.from_workload(wl)
    s.set_tuning(**tuning)
    s.run_steps(2000)               # off the lattice and to temperature (NVT)
    s.set_integrator(W.NVE, wl.dt, wl.T0, wl.tau)
    s.run_steps(100)
    E = []
    for _ in range(100):
        s.run_steps(100)
        th = s.get_thermo()
        E.append((th["K"] + th["U"]) / wl.N)
    E = np.array(E)
    slope = np.polyfit(np.arange(E.size) * 100.0, E, 1)[0]
    assert abs(slope * 1e4) <= 1e-4, "drift %g per particle per 1e4 steps" % (slope * 1e4)
    assert np.abs(E - E[0]).max() < 5e-3
    s.close()


@pytest.mark.parametrize("kind,kw,method,tp", CASES)
def test_nblist_and_forces_match_oracle(rumd, kind, kw, method, tp):
    wl = perturbed(make(kind, **kw))
    s = rumd.from_workload(wl)
    s.set_tuning(method=METHODS[method], tp=tp, pb=max(32 // tp, 128 // tp))
    s.compute_forces()
    r64 = wl.r.astype(np.float64)
    box = wl.box.astype(np.float64)
    cnt, npairs, nband = check_nblist(s, r64, wl.types, box, wl.pot, float(wl.skin))
    assert npairs > 0
    check_forces(s, r64, wl.types, box, wl.pot, cancelling=(kind == "ka"))
    th = s.get_thermo()
    assert th["n_rebuilds"] == 1 and th["max_nbrs"] == cnt.max()
    s.close()


def test_perfect_lattice_energy_and_counts(rumd):
    """P6: static fcc lattice, every particle has 78 list entries; U/N = lattice sum; F = 0."""
    wl = make("lj", ncell=6)
    s = rumd.from_workload(wl)
    s.compute_forces()
    cnt, _ = s.export_nblist()
    assert np.all(cnt == 78)
    th = s.get_thermo()
    F, u, w = oracle.forces_allpairs(wl.r.astype(np.float64), wl.types, wl.box.astype(np.float64), wl.pot)
    assert th["U"] == pytest.approx(u.sum(), rel=ENERGY_TOL)          # 1e-5 of |U| (north_star)
    assert th["W"] == pytest.approx(w.sum(), rel=ENERGY_TOL)
    assert th["U"] / wl.N == pytest.approx(-5.693278275711, rel=ENERGY_TOL)   # SURVEY 8(c) P6 lattice sum
    assert np.abs(s.state()["F"]).max() < 1e-3
    s.close()


@pytest.mark.parametrize("tp", [1, 2, 4, 8, 16, 32])
def test_all_tp_layouts_give_the_same_list_and_forces(rumd, tp):
    wl = perturbed(make("ka", N=1000))
    ref = None
    for method in (rumd.NB_N2, rumd.NB_CELL):
        s = rumd.from_workload(wl)
        s.set_tuning(method=method, tp=tp, pb=max(32 // tp, 64 // tp))
        s.compute_forces()
        cnt, lst = s.export_nblist()
        keys = np.sort(pair_keys(cnt, lst, s.d_id.cpu().numpy().astype(np.int64)))
        F = s.state()["F"]
        if ref is None:
            ref = (keys, F)
        else:
            assert np.array_equal(keys, ref[0])
            assert np.abs(F - ref[1]).max() <= 1e-4 * np.sqrt((ref[1] ** 2).sum(1).mean())
        s.close()


def test_bitwise_reproducible(rumd):
    wl = perturbed(make("ka", N=4096))
    out = []
    for _ in range(2):
        s = rumd.from_workload(wl)
        s.set_tuning(method=rumd.NB_CELL, tp=4, pb=32)
        s.run_steps(50)
        st = s.state()
        out.append((st["r"], st["v"], st["F"]))
        s.close()
    for a, b in zip(*out):
        assert np.array_equal(a, b)


@pytest.mark.parametrize("kind,kw,nvt", [("lj", dict(ncell=6), False), ("ka", dict(N=1000), True)])
def test_one_step_matches_oracle(rumd, kind, kw, nvt):
    """From identical inputs: one full step (build -> forces -> integrate), then the forces/energies of the
    NEW configuration; positions modulo L, velocities, thermostat, energies."""
    wl = perturbed(make(kind, **kw))
    s = rumd.from_workload(wl)
    r64, v64, m64 = wl.r.astype(np.float64), wl.v.astype(np.float64), wl.m.astype(np.float64)
    box = wl.box.astype(np.float64)
    o = oracle.run(r64, v64, m64, np.zeros((wl.N, 3), np.int32), wl.types, box, wl.pot, float(wl.skin), float(wl.dt),
                   1, mode=wl.integrator, T0=wl.T0, tau=wl.tau)
    s.run_steps(1)
    th1 = s.get_thermo()
    st = s.state()
    d = st["r"].astype(np.float64) + st["image"] * box - (o["r"] + o["image"] * box)
    assert np.abs(d).max() < 2e-6
    assert np.abs(st["v"] - o["v"]).max() < 1e-5 * max(1.0, np.abs(o["v"]).max())
    U0, K0 = o["log"][0, 0], o["log"][0, 1]
    assert th1["U"] == pytest.approx(U0, rel=ENERGY_TOL)
    assert th1["K"] == pytest.approx(K0, rel=ENERGY_TOL)
    if nvt:
        assert th1["xi"] == pytest.approx(o["xi"], rel=1e-4, abs=1e-7)
        assert th1["eta"] == pytest.approx(o["eta"], rel=1e-4, abs=1e-9)
    # potential energy after one step (north_star): forces of the new configuration on both sides
    s.compute_forces()
    th2 = s.get_thermo()
    F, u, w = oracle.forces_allpairs(o["r"], wl.types, box, wl.pot)
    assert th2["U"] == pytest.approx(u.sum(), rel=ENERGY_TOL)
    s.close()


def test_lockstep_spot_checks_and_list_validity(rumd):
    """Protocol (3): every k steps copy the GPU state into the oracle and repeat the list / force checks; the
    list in use must contain every pair inside the interaction range (skin/2 invariant)."""
    wl = perturbed(make("ka", N=1000))
    s = rumd.from_workload(wl)
    s.set_tuning(method=rumd.NB_N2, tp=16, pb=8)
    box = wl.box.astype(np.float64)
    for _ in range(4):
        s.run_steps(37)
        s.compute_forces()   # forces of the current positions with the list in use (rebuilt iff flagged)
        st = s.state()
        r64 = st["r"].astype(np.float64)
        cnt, lst = s.export_nblist()
        ids = s.d_id.cpu().numpy().astype(np.int64)
        have = np.unique(pair_keys(cnt, lst, ids))
        oc, ol = oracle.nblist(r64, wl.types, box, wl.pot, 0.0)
        need = pair_keys(oc, ol)
        assert np.isin(need, have).all(), "list in use misses interacting pairs"
        check_forces(s, r64, wl.types, box, wl.pot, cancelling=True)
    th = s.get_thermo()
    assert th["n_rebuilds"] >= 2
    s.close()


def test_nve_energy_drift(rumd):
    """north_star: over 1e4 NVE steps, total-energy drift <= 1e-4 per particle (S26: least-squares slope of
    E/N times the run length).  configs[0] extended to 1e4 steps."""
    wl = make("lj", ncell=6)
    s = rumd.from_workload(wl)
    E = []
    s.run_steps(1)
    for _ in range(100):
        s.run_steps(100)
        th = s.get_thermo()
        E.append((th["K"] + th["U"]) / wl.N)
    E = np.array(E)
    t = np.arange(E.size) * 100.0
    slope = np.polyfit(t, E, 1)[0]
    assert abs(slope * 1e4) <= 1e-4, "drift %g per particle over 1e4 steps" % (slope * 1e4)
    assert np.abs(E - E[0]).max() < 5e-3
    s.close()


def test_nvt_short_trajectory_tracks_oracle(rumd):
    """20 NVT steps from identical inputs: thermostat variables and energies follow the oracle closely
    (before chaos separates the trajectories)."""
    wl = perturbed(make("ka", N=1000), amp=0.02)
    s = rumd.from_workload(wl)
    n = 20
    o = oracle.run(wl.r.astype(np.float64), wl.v.astype(np.float64), wl.m.astype(np.float64),
                   np.zeros((wl.N, 3), np.int32), wl.types, wl.box.astype(np.float64), wl.pot, float(wl.skin),
                   float(wl.dt), n, mode=W.NVT, T0=wl.T0, tau=wl.tau)
    s.run_steps(n)
    th = s.get_thermo()
    assert th["xi"] == pytest.approx(o["xi"], rel=1e-3, abs=1e-6)
    assert th["eta"] == pytest.approx(o["eta"], rel=1e-3, abs=1e-8)
    assert th["U"] == pytest.approx(o["log"][-1, 0], rel=1e-4)
    assert th["K"] == pytest.approx(o["log"][-1, 1], rel=1e-4)
    assert th["H"] == pytest.approx(o["log"][-1, 5], rel=1e-4)
    s.close()


def test_overflow_is_reported_and_capacity_doubles(rumd):
    wl = perturbed(make("lj", ncell=6))
    s = rumd.System(wl.r, wl.v, wl.m, wl.types, wl.box, wl.pot, capacity=32)
    s.set_integrator(wl.integrator, wl.dt, wl.T0, wl.tau)
    s.set_tuning(skin=float(wl.skin))
    s.compute_forces()
    with pytest.raises(rumd.RumdError) as e:
        s.get_thermo()
    assert e.value.status == rumd.ERR_NBL_OVERFLOW
    assert s.get_thermo(grow=True) is None     # re-binds a larger workspace
    s.compute_forces()
    th = s.get_thermo()
    assert th["overflow"] == 0 and th["max_nbrs"] <= th["nbl_capacity"]
    check_forces(s, wl.r.astype(np.float64), wl.types, wl.box.astype(np.float64), wl.pot)
    s.close()


@pytest.mark.parametrize("kind,kw,tp,persistent", [("lj", dict(ncell=4), 32, 1), ("ka", dict(N=512), 16, 1),
                                                   ("ch", dict(n=8), 8, 0), ("ka", dict(N=1000), 4, 1)])
def test_none_method_all_pairs_forces(rumd, kind, kw, tp, persistent):
    """P:371 "none": no neighbour list, every force evaluation visits all pairs.  Forces / energies / virials
    against the oracle's brute force, and the same trajectory as the list-based path (to fp32 summation order)."""
    wl = perturbed(make(kind, **kw))
    s = rumd.from_workload(wl)
    s.set_tuning(method=rumd.NB_NONE, tp=tp, pb=max(1, 128 // tp), persistent=persistent, use_graph=0)
    s.compute_forces()
    check_forces(s, wl.r.astype(np.float64), wl.types, wl.box.astype(np.float64), wl.pot, cancelling=(kind == "ka"))
    cnt, _ = s.export_nblist()
    assert cnt.sum() == 0
    s.run_steps(25)
    a = s.state()
    th = s.get_thermo()
    assert th["n_steps"] == 25 and th["n_rebuilds"] == 0
    s.close()
    s2 = rumd.from_workload(wl)
    s2.set_tuning(method=rumd.NB_N2, tp=tp, pb=max(1, 128 // tp), persistent=persistent, use_graph=0)
    s2.run_steps(25)
    b = s2.state()
    s2.close()
    d = a["r"].astype(np.float64) - b["r"]
    box = wl.box.astype(np.float64)
    d -= box * np.rint(d / box)
    assert np.abs(d).max() < 1e-4 and np.abs(a["v"] - b["v"]).max() < 2e-3


def _with_cutoffs(pot, cut_lj, cut_c):
    pot = pot.copy()
    pot[..., 5] = cut_lj
    pot[..., 6] = cut_c
    return pot


@pytest.mark.parametrize("kind,kw,cut_lj,cut_c,method,tp", [
    ("ka", dict(N=1000), W.CUT_SHIFTED_POTENTIAL, 0, "n2", 16),
    ("ka", dict(N=2048), W.CUT_NONE, 0, "cell", 4),
    ("ch", dict(n=10), W.CUT_SHIFTED_POTENTIAL, W.CUT_NONE, "cell", 8),
    ("ch", dict(n=12), W.CUT_NONE, W.CUT_SHIFTED_POTENTIAL, "cell", 1),
    ("lj", dict(ncell=6), W.CUT_SHIFTED_POTENTIAL, 0, "none", 32),
])
def test_other_cutoff_methods_match_oracle(rumd, kind, kw, cut_lj, cut_c, method, tp):
    """shifted potential and plain truncation (next to the hot path's shifted force) on the same
    kernels.  With these methods the pair force JUMPS at rc (by f(rc) ~ 0.04), so a pair within fp32 rounding
    of a cutoff may be counted on one side only: particles owning a pair within 1e-6 of one of its cutoffs are
    left out of the force comparison (S30) -- the analogue of the 1e-6 band of the list."""
    wl = perturbed(make(kind, **kw))
    wl.pot = _with_cutoffs(wl.pot, cut_lj, cut_c)
    s = rumd.from_workload(wl)
    m = {"n2": rumd.NB_N2, "cell": rumd.NB_CELL, "none": rumd.NB_NONE}[method]
    s.set_tuning(method=m, tp=tp, pb=max(1, 128 // tp))
    s.compute_forces()
    r64, box = wl.r.astype(np.float64), wl.box.astype(np.float64)
    F, u, w = oracle.forces_allpairs(r64, wl.types, box, wl.pot)
    d = r64[:, None, :] - r64[None, :, :]
    d -= box * np.rint(d / box)
    dist = np.sqrt((d * d).sum(-1))
    ti, tj = wl.types[:, None], wl.types[None, :]
    near = np.zeros(dist.shape, bool)
    for col in (2, 4):
        rc = wl.pot[ti, tj, col]
        near |= (rc > 0) & (np.abs(dist - rc) <= BAND)
    keep = ~near.any(1)
    assert keep.sum() >= 0.99 * wl.N
    st = s.state()
    rms = np.sqrt((F * F).sum(1).mean())
    err = np.sqrt(((st["F"].astype(np.float64) - F) ** 2).sum(1))
    assert err[keep].max() <= FORCE_TOL * rms
    assert np.abs(st["u"] - u)[keep].max() <= 1e-5 * max(1.0, np.abs(u).max())
    assert np.abs(st["w"] - w)[keep].max() <= 1e-5 * max(1.0, np.abs(w).max())
    if keep.all():
        th = s.get_thermo()
        cancelling = kind == "ka"      # the sc-lattice KA start only (S29)
        assert abs(th["U"] - u.sum()) <= ENERGY_TOL * (np.abs(u).sum() if cancelling else abs(u.sum()))
        assert abs(th["W"] - w.sum()) <= ENERGY_TOL * (np.abs(w).sum() if cancelling else abs(w.sum()))
    # the three methods really differ: the energy is not the shifted-force one
    F0, u0, w0 = oracle.forces_allpairs(r64, wl.types, box, _with_cutoffs(wl.pot, 0, 0))
    assert abs(u.sum() - u0.sum()) > 1e-3 * np.abs(u0).sum()
    s.run_steps(20)
    assert np.isfinite(s.get_thermo()["H"])
    s.close()


def _extra_pot(which):
    pot = W.pot_table(2)
    if which == "ipl":          # purely repulsive IPL-12 mixture (no LJ term at all)
        for (a, b), (amp, rc) in {(0, 0): (1.0, 2.0), (0, 1): (1.3, 1.8), (1, 1): (0.7, 1.9)}.items():
            W.set_second_term(pot, a, b, W.KIND_IPL, amp, 12.0, 0.0, rc)
    elif which == "yukawa":     # LJ + screened charges
        pot = W.kob_andersen()
        for (a, b), q in {(0, 0): 1.0, (0, 1): -1.0, (1, 1): 1.0}.items():
            W.set_second_term(pot, a, b, W.KIND_YUKAWA, q, 1.2, 0.0, 3.2)
    elif which == "gauss":      # Gaussian core, shifted potential
        for (a, b) in ((0, 0), (0, 1), (1, 1)):
            W.set_second_term(pot, a, b, W.KIND_GAUSSIAN_CORE, 3.0 + a + b, 0.9, 0.0, 2.6, cut=W.CUT_SHIFTED_POTENTIAL)
    elif which == "buck":       # Buckingham on unlike pairs, LJ on like pairs
        W.set_lj(pot, 0, 0, 1.0, 1.0, 2.5)
        W.set_lj(pot, 1, 1, 0.5, 0.88, 2.2)
        W.set_second_term(pot, 0, 1, W.KIND_BUCKINGHAM, 2500.0, 0.2, 1.6, 2.4)
    elif which == "glj":        # generalized LJ with three different exponent pairs (no 12-6 term)
        for (a, b), (eps, sig, m, n) in {(0, 0): (1.0, 1.02, 12.0, 6.0), (0, 1): (1.5, 0.9, 9.0, 6.0), (1, 1): (0.5, 0.95, 10.0, 5.0)}.items():
            W.set_second_term(pot, a, b, W.KIND_GEN_LJ, eps, sig, m, 2.3 * sig, pd=n)
    elif which == "girifalco":  # C60-like ratio beta / alpha, diameters well below the nearest-neighbour distance
        for (a, b), (al, d) in {(0, 0): (0.17, 0.6), (0, 1): (0.25, 0.55), (1, 1): (0.1, 0.5)}.items():
            W.set_second_term(pot, a, b, W.KIND_GIRIFALCO, al, 1.814e-3 * al, d, 3.5 * d)
    elif which == "dzugutov":   # vanishes smoothly at 1.94 sigma: plain truncation there
        for (a, b), (eps, sig) in {(0, 0): (0.5, 0.92), (0, 1): (0.7, 0.85), (1, 1): (0.3, 0.88)}.items():
            W.set_second_term(pot, a, b, W.KIND_DZUGUTOV, eps, sig, 0.0, 1.94 * sig, cut=W.CUT_NONE)
    return pot


@pytest.mark.parametrize("which,method,tp,persistent", [("ipl", "cell", 8, 1), ("yukawa", "cell", 4, 1), ("gauss", "n2", 16, 0),
                                                        ("buck", "cell", 2, 1), ("yukawa", "none", 32, 1),
                                                        ("glj", "cell", 8, 1), ("girifalco", "cell", 4, 1),
                                                        ("dzugutov", "n2", 16, 0), ("dzugutov", "none", 32, 1),
                                                        ("glj", "n2", 1, 0)])
def test_other_pair_potentials_match_oracle(rumd, which, method, tp, persistent):
    """inverse power law, Yukawa, Gaussian core, Buckingham, generalized LJ, Girifalco and Dzugutov as the
    second term of a type pair, on the same kernels: list, forces, energies and virials against the oracle, then a short trajectory."""
    wl = perturbed(make("ka", N=4096 if method != "none" else 512))
    wl.pot = _extra_pot(which)
    s = rumd.from_workload(wl)
    m = {"n2": rumd.NB_N2, "cell": rumd.NB_CELL, "none": rumd.NB_NONE}[method]
    s.set_tuning(method=m, tp=tp, pb=max(1, 128 // tp), persistent=persistent, use_graph=0)
    s.compute_forces()
    r64, box = wl.r.astype(np.float64), wl.box.astype(np.float64)
    if method != "none":
        check_nblist(s, r64, wl.types, box, wl.pot, float(wl.skin))
    if which == "gauss":        # shifted potential: discontinuous force at rc (S30)
        F, u, w = oracle.forces_allpairs(r64, wl.types, box, wl.pot)
        st = s.state()
        rms = np.sqrt((F * F).sum(1).mean())
        err = np.sqrt(((st["F"].astype(np.float64) - F) ** 2).sum(1))
        assert np.sort(err)[-8] <= FORCE_TOL * rms and np.median(err) <= 0.1 * FORCE_TOL * rms
    else:
        check_forces(s, r64, wl.types, box, wl.pot, cancelling=True)
    s.run_steps(25)
    th = s.get_thermo()
    o = oracle.run(r64, wl.v.astype(np.float64), wl.m.astype(np.float64), np.zeros((wl.N, 3), np.int32), wl.types, box,
                   wl.pot, float(wl.skin), float(wl.dt), 25, mode=wl.integrator, T0=wl.T0, tau=wl.tau)
    st = s.state()
    d = st["r"].astype(np.float64) - o["r"]
    d -= box * np.rint(d / box)
    assert np.abs(d).max() < 3e-4 and np.isfinite(th["H"])
    s.close()


def _gas(N, ntypes, box, seed, pot):
    r, types = W.random_gas(N, ntypes, box, seed)
    rng = np.random.default_rng(seed + 1)
    m = np.ones(N, np.float32)
    v = (0.5 * rng.standard_normal((N, 3))).astype(np.float32)
    return r, v, m, types, np.asarray(box, np.float32), pot


@pytest.mark.parametrize("N,box,method,tp,persistent", [
    (1, (12.0, 12.0, 12.0), "n2", 32, 1),        # a single particle: empty list, zero force
    (5, (30.0, 30.0, 30.0), "cell", 1, 1),       # dilute: almost every cell empty, most rows empty
    (33, (9.0, 9.0, 9.0), "n2", 4, 0),           # one particle past a warp boundary
    (33, (9.0, 9.0, 9.0), "cell", 8, 1),
    (257, (8.0, 11.0, 14.0), "cell", 2, 1),      # orthorhombic, ragged last block, 4 types
    (257, (8.0, 11.0, 14.0), "n2", 16, 0),
])
def test_degenerate_and_ragged_inputs(rumd, N, box, method, tp, persistent):
    """Edge cases of every kernel path: empty and nearly empty lists, sizes that are not multiples of the warp,
    block or tile sizes, four particle types with all six pair potentials different, anisotropic boxes."""
    nt = 4 if N > 33 else 1
    pot = W.pot_table(nt)
    for a in range(nt):
        for b in range(a, nt):
            W.set_lj(pot, a, b, 1.0 + 0.1 * (a + b), 1.0 - 0.04 * (a + b), 2.5 * (1.0 - 0.04 * (a + b)))
    r, v, m, types, boxf, pot = _gas(N, nt, box, 77 + N, pot)
    s = rumd.System(r, v, m, types, boxf, pot)
    s.set_integrator(rumd.INT_NVE_LEAPFROG, 0.004)
    s.set_tuning(method=rumd.NB_CELL if method == "cell" else rumd.NB_N2, tp=tp, pb=max(1, 64 // tp), skin=0.3,
                 persistent=persistent, use_graph=0)
    s.compute_forces()
    r64, b64 = r.astype(np.float64), boxf.astype(np.float64)
    cnt, lst = s.export_nblist()
    ids = s.d_id.cpu().numpy().astype(np.int64)
    oc, ol = oracle.nblist(r64, types, b64, pot, 0.3, method="n2")
    assert np.array_equal(np.sort(pair_keys(cnt, lst, ids)), np.sort(pair_keys(oc, ol)))
    F, u, w = oracle.forces_allpairs(r64, types, b64, pot)
    st = s.state()
    scale = max(1e-3, np.sqrt((F * F).sum(1).mean()))
    assert np.sqrt(((st["F"] - F) ** 2).sum(1)).max() <= FORCE_TOL * scale
    assert np.abs(st["u"] - u).max() <= 1e-5 * max(1.0, np.abs(u).max())
    # 37 steps (odd: ends in the alternate position buffer) against the oracle's trajectory: short, so fp32
    # and fp64 have not separated yet
    s.run_steps(37)
    th = s.get_thermo()
    assert th["n_steps"] == 37 and np.isfinite(th["H"])
    o = oracle.run(r64, v.astype(np.float64), m.astype(np.float64), np.zeros((N, 3), np.int32), types, b64, pot, 0.3,
                   0.004, 37)
    st = s.state()
    d = st["r"].astype(np.float64) - o["r"]
    d -= b64 * np.rint(d / b64)                     # positions compared modulo L (S7)
    assert np.abs(d).max() < 2e-4
    assert s.run_steps(0) is None                   # zero steps is a no-op
    assert s.get_thermo()["n_steps"] == 37
    s.close()


@pytest.mark.parametrize("nvt", [False, True])
def test_graph_and_plain_launch_agree(rumd, nvt):
    """Per-step path: CUDA graphs of fused force + integrate step pairs (double-buffered positions) against plain
    launches of the un-fused force and integrate kernels.  NVE: bit-identical (same arithmetic, same order).
    NVT: the fp64 sums of m v^2 are grouped by different block sizes, so xi agrees to rounding only."""
    wl = perturbed(make("ka", N=1000))
    if not nvt:
        wl.integrator = W.NVE
    res = []
    for g in (0, 1):
        s = rumd.from_workload(wl)
        s.set_tuning(persistent=0, use_graph=g, steps_per_graph=8, method=rumd.NB_N2)
        s.run_steps(43)     # 5 graphs of 8 fused steps + 3 single steps
        st = s.state()
        th = s.get_thermo()
        res.append((st, th))
        assert th["n_steps"] == 43
        s.close()
    (a, ta), (b, tb) = res
    assert ta["n_rebuilds"] == tb["n_rebuilds"] >= 2
    if nvt:
        assert np.abs(a["r"] - b["r"]).max() < 1e-4 and np.abs(a["v"] - b["v"]).max() < 1e-3
        assert ta["xi"] == pytest.approx(tb["xi"], rel=1e-7)
    else:
        for key in ("r", "v", "F", "u", "w", "image"):
            assert np.array_equal(a[key], b[key]), key
        assert ta["U"] == tb["U"]


@pytest.mark.parametrize("kind,kw,method,tp,nsteps", [
    ("lj", dict(ncell=6), "n2", 16, 61),        # odd step count: positions end in the alternate buffer
    ("lj", dict(ncell=8), "cell", 4, 80),       # N = 2048
    ("ch", dict(n=10), "cell", 8, 40),
])
def test_persistent_kernel_equals_per_step_kernels_bitwise_nve(rumd, kind, kw, method, tp, nsteps):
    """A7: the one-launch cooperative kernel (fused force + integrate, grid barriers, in-kernel rebuilds) and
    the per-step kernel chain run the same arithmetic in the same order: NVE trajectories are bit-identical,
    including across list rebuilds and spatial sorts."""
    wl = perturbed(make(kind, **kw))
    wl.integrator = W.NVE
    res = []
    for persistent in (1, 0):
        s = rumd.from_workload(wl)
        s.set_tuning(method=rumd.NB_CELL if method == "cell" else rumd.NB_N2, tp=tp, pb=256 // tp,
                     persistent=persistent, use_graph=0)
        s.run_steps(nsteps)
        s.run_steps(7)
        th = s.get_thermo()
        st = s.state()
        res.append((st, th))
        assert th["n_steps"] == nsteps + 7
        s.close()
    (a, ta), (b, tb) = res
    assert ta["n_rebuilds"] == tb["n_rebuilds"] and ta["n_rebuilds"] >= 2
    for key in ("r", "v", "F", "u", "w", "image"):
        assert np.array_equal(a[key], b[key]), key
    assert ta["U"] == tb["U"] and ta["max_nbrs"] == tb["max_nbrs"]
    assert ta["K"] == pytest.approx(tb["K"], rel=1e-12)


def test_persistent_kernel_nvt_tracks_per_step_kernels(rumd):
    """NVT: both paths add the same per-particle fp64 terms but group them by different block sizes, so xi
    agrees to rounding, not bitwise."""
    wl = perturbed(make("ka", N=4096))
    res = []
    for persistent in (1, 0):
        s = rumd.from_workload(wl)
        s.set_tuning(method=rumd.NB_CELL, tp=8, pb=32, persistent=persistent)
        s.run_steps(30)
        th = s.get_thermo()
        res.append((s.state(), th))
        s.close()
    (a, ta), (b, tb) = res
    assert ta["xi"] == pytest.approx(tb["xi"], rel=1e-9)
    assert ta["H"] == pytest.approx(tb["H"], rel=1e-7)
    assert np.abs(a["r"] - b["r"]).max() < 1e-4


def test_snapshot_restore_and_host_buffers(rumd):
    wl = perturbed(make("ka", N=1000))
    s = rumd.from_workload(wl)
    s.snapshot()
    s.run_steps(25)
    a = s.state()
    s.restore()
    s.run_steps(25)
    b = s.state()
    assert np.array_equal(a["r"], b["r"]) and np.array_equal(a["v"], b["v"])
    # host-buffer entry points: upload the pinned initial state again, run, download
    s.upload_state()
    s.run_steps(25)
    import torch

    h_r = torch.empty((wl.N, 4), dtype=torch.float32).pin_memory()
    h_id = torch.empty((wl.N,), dtype=torch.int32).pin_memory()
    s.download_state(h_r=h_r, h_id=h_id)
    inv = np.empty(wl.N, np.int64)
    inv[h_id.numpy().astype(np.int64)] = np.arange(wl.N)
    assert np.array_equal(h_r.numpy()[inv][:, :3], a["r"])
    s.close()


def test_autotune_returns_valid_setting_and_preserves_state(rumd):
    wl = perturbed(make("ka", N=1000))
    s = rumd.from_workload(wl)
    s.run_steps(10)
    before = s.state()
    t, tps = s.autotune(steps_per_trial=40)
    assert tps > 0 and t.tp in (1, 2, 4, 8, 16, 32) and (t.pb * t.tp) % 32 == 0 and t.skin > 0
    after = s.state()
    assert np.array_equal(before["r"], after["r"]) and np.array_equal(before["v"], after["v"])
    s.compute_forces()
    st = s.state()
    check_forces(s, st["r"].astype(np.float64), wl.types, wl.box.astype(np.float64), wl.pot, cancelling=True)
    s.close()


def test_invalid_arguments_are_rejected(rumd):
    wl = make("lj", ncell=6)
    s = rumd.from_workload(wl)
    with pytest.raises(rumd.RumdError):
        s.set_tuning(tp=3)
    with pytest.raises(rumd.RumdError):
        s.set_tuning(pb=3, tp=1)
    with pytest.raises(rumd.RumdError):
        s.set_integrator(0, -1.0)
    s.set_tuning(skin=4.0)      # rc + skin > L/2 -> lazily at the next compute call
    with pytest.raises(rumd.RumdError) as e:
        s.compute_forces()
    assert e.value.status == rumd.ERR_BOX_TOO_SMALL
    s.set_tuning(skin=0.3)
    with pytest.raises(rumd.RumdError):     # generalized LJ needs m > n > 0
        s.set_pair_potential(0, 0, rumd.POT_GEN_LJ, [1.0, 1.0, 6.0, 12.0, 2.5], 0)
    with pytest.raises(rumd.RumdError):     # Girifalco: rcut must exceed the diameter
        s.set_pair_potential(0, 0, rumd.POT_GIRIFALCO, [1.0, 0.002, 1.0, 0.9], 0)
    with pytest.raises(rumd.RumdError):     # wrong parameter count
        s.set_pair_potential(0, 0, rumd.POT_DZUGUTOV, [1.0, 1.0], 0)
    s.set_pair_potential(0, 0, rumd.POT_GEN_LJ, [1.0, 1.0, 12.0, 6.0, 2.5], 0)
    with pytest.raises(rumd.RumdError):     # ... and it replaces the 12-6 term, which this pair still has
        s.compute_forces()
    s.close()


# ------------------------------------------------------------------ batched ensembles


def _ensemble_inputs(kind, kw, R, seed0=100):
    wls = []
    for q in range(R):
        wl = perturbed(make(kind, **kw), seed=seed0 + q)
        rng = np.random.default_rng(seed0 + 50 + q)
        wl.v = W.maxwell_boltzmann(rng, wl.m.astype(np.float64), float(wl.T0)).astype(np.float32)
        wls.append(wl)
    return wls


@pytest.mark.parametrize("kind,kw,tp,method,nvt", [("lj", dict(ncell=4), 16, "n2", False), ("ka", dict(N=512), 32, "n2", True),
                                                   ("ka", dict(N=1000), 8, "n2", True), ("lj", dict(ncell=4), 32, "none", False)])
def test_batched_ensemble_replicas_match_oracle_and_single_runs(rumd, kind, kw, tp, method, nvt):
    """R independent replicas (different positions and velocities) advanced by ONE launch, one block each:
    every replica's forces / energy against the oracle, its trajectory against the oracle's and -- in NVE --
    bit for bit against the same system run alone through the single-system path."""
    R, nsteps = 5, 31
    wls = _ensemble_inputs(kind, kw, R)
    wl0 = wls[0]
    integ = W.NVT if nvt else W.NVE
    s = rumd.System(np.stack([w.r for w in wls]), np.stack([w.v for w in wls]), wl0.m, wl0.types if kind != "ka" else
                    np.stack([w.types for w in wls]), wl0.box, wl0.pot)
    assert s.replicas == R
    s.set_integrator(integ, wl0.dt, wl0.T0, wl0.tau)
    m = rumd.NB_N2 if method == "n2" else rumd.NB_NONE
    s.set_tuning(method=m, tp=tp, pb=256 // tp, skin=0.3)
    s.run_steps(1)
    th = s.get_thermo_replicas()
    box = wl0.box.astype(np.float64)
    for q, wl in enumerate(wls):
        F, u, w = oracle.forces_allpairs(wl.r.astype(np.float64), wl.types, box, wl.pot)
        cancelling = kind == "ka"      # the sc-lattice KA start only (S29)
        assert abs(th[q]["U"] - u.sum()) <= ENERGY_TOL * (np.abs(u).sum() if cancelling else abs(u.sum()))
        assert abs(th[q]["W"] - w.sum()) <= ENERGY_TOL * (np.abs(w).sum() if cancelling else abs(w.sum()))
        assert th[q]["n_steps"] == 1 and (th[q]["n_rebuilds"] == (1 if method == "n2" else 0))
    st1 = s.state()
    for q, wl in enumerate(wls):
        F, u, w = oracle.forces_allpairs(wl.r.astype(np.float64), wl.types, box, wl.pot)
        rms = np.sqrt((F * F).sum(1).mean())
        assert np.sqrt(((st1["F"][q] - F) ** 2).sum(1)).max() <= FORCE_TOL * rms
    s.run_steps(nsteps - 1)
    st = s.state()
    th = s.get_thermo_replicas()
    for q, wl in enumerate(wls):
        o = oracle.run(wl.r.astype(np.float64), wl.v.astype(np.float64), wl.m.astype(np.float64), np.zeros((wl.N, 3), np.int32),
                       wl.types, box, wl.pot, 0.3, float(wl.dt), nsteps, mode=integ, T0=wl.T0, tau=wl.tau)
        d = st["r"][q].astype(np.float64) - o["r"]
        d -= box * np.rint(d / box)
        assert np.abs(d).max() < 2e-4
        assert th[q]["n_steps"] == nsteps
        assert th[q]["U"] == pytest.approx(o["log"][-1, 0], rel=1e-4, abs=1e-3)
        if nvt:
            assert th[q]["xi"] == pytest.approx(o["xi"], rel=1e-3, abs=1e-6)
    s.close()
    if not nvt:   # the same replica alone, single-system persistent path: bit-identical
        for q in (0, R - 1):
            wl = wls[q]
            s1 = rumd.System(wl.r, wl.v, wl.m, wl.types, wl.box, wl.pot)
            s1.set_integrator(integ, wl.dt, wl.T0, wl.tau)
            s1.set_tuning(method=m, tp=tp, pb=256 // tp, skin=0.3, persistent=1)
            s1.run_steps(1)
            s1.run_steps(nsteps - 1)
            a = s1.state()
            assert np.array_equal(a["r"], st["r"][q]) and np.array_equal(a["v"], st["v"][q])
            assert np.array_equal(a["F"], st["F"][q])
            s1.close()


def test_batched_ensemble_rejects_single_system_calls(rumd):
    wls = _ensemble_inputs("lj", dict(ncell=4), 3)
    s = rumd.System(np.stack([w.r for w in wls]), np.stack([w.v for w in wls]), wls[0].m, wls[0].types, wls[0].box, wls[0].pot)
    s.set_integrator(W.NVE, 0.005)
    for call in (s.compute_forces, s.build_nblist, s.get_thermo, s.snapshot):
        with pytest.raises(rumd.RumdError):
            call()
    s.set_tuning(method=rumd.NB_CELL)
    with pytest.raises(rumd.RumdError):
        s.run_steps(1)
    s.close()


def test_long_run_crosses_launch_chunks_and_conserves_energy(rumd):
    """70 000 NVE steps of configs[0] in one rumd_run_steps call: more than one cooperative launch (a launch
    runs at most 2^16 steps), thousands of in-kernel rebuilds; step count exact, energy conserved (S26 bar)."""
    wl = make("lj", ncell=6)
    s = rumd.from_workload(wl)
    s.run_steps(2000)
    th0 = s.get_thermo()
    s.run_steps(70000)
    th1 = s.get_thermo()
    assert th1["n_steps"] - th0["n_steps"] == 70000
    assert th1["n_rebuilds"] - th0["n_rebuilds"] > 2000
    assert abs(th1["H"] - th0["H"]) / wl.N < 1e-4 * 7      # 1e-4 per particle per 10^4 steps
    assert np.isfinite(th1["U"]) and th1["overflow"] == 0
    s.close()


def test_autotune_cache_file_is_written_and_reused(rumd, tmp_path):
    """D10 / P:382 step 8: the tuned parameters go to a file keyed by the user's parameters; a second system
    with the same parameters takes them from the file without a trial run, a different one does not."""
    path = str(tmp_path / "tuning.jsonl")
    wl = perturbed(make("ka", N=1000))
    s = rumd.from_workload(wl)
    s.run_steps(20)
    t1, tps1 = s.autotune(steps_per_trial=40, cache_path=path)
    assert not s.tuning_from_cache and tps1 > 0
    lines = open(path).read().strip().splitlines()
    assert len(lines) == 1
    import json as _json
    rec = _json.loads(lines[0])
    assert rec["tp"] == t1.tp and rec["method"] == t1.method and "N=1000" in rec["key"] and "B200" in rec["key"]
    s.close()
    s2 = rumd.from_workload(wl)
    n0 = s2.launch_count()
    t2, tps2 = s2.autotune(steps_per_trial=40, cache_path=path)
    assert s2.tuning_from_cache and t2.as_dict() == t1.as_dict() and tps2 == pytest.approx(tps1, rel=1e-5)
    assert s2.launch_count() - n0 <= 3                      # no trial runs
    assert s2.get_tuning().as_dict() == t1.as_dict()
    s2.run_steps(10)
    s2.close()
    wl3 = perturbed(make("ka", N=512))
    s3 = rumd.from_workload(wl3)
    s3.autotune(steps_per_trial=40, cache_path=path)
    assert not s3.tuning_from_cache and len(open(path).read().strip().splitlines()) == 2
    s3.close()


@pytest.mark.parametrize("persistent", [1, 0])
def test_n2_method_with_periodic_sort(rumd, persistent):
    """P:379 step 5 (K13): with the N^2 build the particles are spatially re-sorted at every sort_interval-th
    rebuild.  The permutation must be transparent: same trajectory (to fp32 summation order) as without sorting,
    list and forces against the oracle in the sorted order."""
    wl = perturbed(make("ka", N=2048))
    res = []
    for si in (0, 2):
        s = rumd.from_workload(wl)
        s.set_tuning(method=rumd.NB_N2, tp=16, pb=16, sort_interval=si, persistent=persistent, use_graph=0, skin=0.3)
        s.run_steps(60)
        th = s.get_thermo()
        assert th["n_rebuilds"] >= 3
        ids = s.d_id.cpu().numpy()
        assert sorted(ids.tolist()) == list(range(wl.N))
        assert (ids != np.arange(wl.N)).any() == (si > 0)
        st = s.state()
        res.append(st)
        if si:
            s.build_nblist()
            s.compute_forces()
            st2 = s.state()
            r64 = st2["r"].astype(np.float64)
            check_nblist(s, r64, wl.types, wl.box.astype(np.float64), wl.pot, 0.3)
            check_forces(s, r64, wl.types, wl.box.astype(np.float64), wl.pot, cancelling=True)
        s.close()
    d = res[0]["r"].astype(np.float64) - res[1]["r"]
    box = wl.box.astype(np.float64)
    d -= box * np.rint(d / box)
    assert np.abs(d).max() < 2e-4


def test_cell_grid_finer_than_the_bound_workspace_is_refused(rumd):
    """The cell arrays of the workspace are sized from the potentials in force at rumd_bind_workspace.  A shorter
    rc_max set afterwards needs a finer grid than was carved: the library must refuse (RUMD_ERR_NOT_READY) instead
    of writing past the cell arrays, and work again after a re-bind."""
    wl = perturbed(make("ka", N=8000))
    s = rumd.from_workload(wl)                     # carved for rc_max = 2.5
    s.set_tuning(method=rumd.NB_CELL)
    s.compute_forces()
    for a, b in ((0, 0), (0, 1), (1, 1)):          # rc 1.12 at L = 18.8: 17576 cells against 3375 carved
        s.set_pair_potential(a, b, rumd.POT_LJ_12_6, [1.0, 1.0, 1.12], rumd.CUT_SHIFTED_FORCE)
    with pytest.raises(rumd.RumdError) as e:
        s.compute_forces()
    assert e.value.status == rumd.ERR_NOT_READY and "re-bind" in str(e.value)
    s.bind_workspace(s.capacity)
    s.compute_forces()
    pot = wl.pot.copy()
    pot[..., 0], pot[..., 1], pot[..., 2] = 1.0, 1.0, np.float32(1.12)
    check_nblist(s, wl.r.astype(np.float64), wl.types, wl.box.astype(np.float64), pot, float(wl.skin))
    s.close()


@pytest.mark.parametrize("method,sort_interval,kind,kw", [("cell", 0, "lj", dict(ncell=8)), ("n2", 1, "ka", dict(N=2048)),
                                                         ("cell", 0, "ka", dict(N=4096))])
def test_fused_step_graphs_with_sorting_equal_plain_launches_bitwise(rumd, method, sort_interval, kind, kw):
    """Per-step path inside CUDA graphs of fused step PAIRS (r -> r_alt -> r; the second step's rebuild chain
    assigns cells, permutes and builds on the alternate buffer) with a spatial sort at every rebuild, against plain
    launches of the un-fused kernels: NVE, bit-identical.  Step counts are chosen so that rebuilds land on both
    the even and the odd step of a pair."""
    wl = perturbed(make(kind, **kw))
    wl.integrator = W.NVE
    res = []
    for g in (1, 0):
        s = rumd.from_workload(wl)
        s.set_tuning(persistent=0, use_graph=g, steps_per_graph=8, sort_interval=sort_interval, tp=4, pb=32,
                     method=rumd.NB_CELL if method == "cell" else rumd.NB_N2, skin=0.25)
        nreb = []
        for n in (8, 8, 16, 24, 41):            # 97 steps: graphs of 8 fused steps + a single-step tail
            s.run_steps(n)
            nreb.append(s.get_thermo()["n_rebuilds"])
        res.append((s.state(), s.get_thermo(), nreb))
        ids = s.d_id.cpu().numpy()
        assert (ids != np.arange(wl.N)).any()     # the particles really were re-sorted
        s.close()
    (a, ta, na), (b, tb, nb) = res
    assert na == nb and ta["n_rebuilds"] >= 5
    for key in ("r", "v", "F", "u", "w", "image"):
        assert np.array_equal(a[key], b[key]), key
    assert ta["U"] == tb["U"] and ta["max_nbrs"] == tb["max_nbrs"] > 0


def test_particle_types_are_validated_on_the_host(rumd):
    wl = make("ka", N=1000)
    bad = wl.types.copy()
    bad[17] = 2                                    # two types only
    with pytest.raises(rumd.RumdError) as e:
        rumd.System(wl.r, wl.v, wl.m, bad, wl.box, wl.pot)
    assert e.value.status == rumd.ERR_INVALID_ARG
    s = rumd.from_workload(wl)
    import torch

    s.h_r.view(torch.int32)[5, 3] = -1
    with pytest.raises(rumd.RumdError) as e:
        s.upload_state()
    assert e.value.status == rumd.ERR_INVALID_ARG
    s.close()


def test_max_nbrs_survives_a_pending_rebuild_flag(rumd):
    """rumd_get_thermo reports the longest row of the last COMPLETED build also when the last step's displacement
    check has already raised the flag for the next one (its slot is then zeroed)."""
    wl = perturbed(make("ka", N=1000))
    for persistent in (1, 0):
        s = rumd.from_workload(wl)
        s.set_tuning(method=rumd.NB_N2, tp=16, pb=8, persistent=persistent, use_graph=0, skin=0.2)
        seen = 0
        for _ in range(60):
            s.run_steps(1)
            th = s.get_thermo()
            assert 60 <= th["max_nbrs"] <= th["nbl_capacity"], th
            seen = max(seen, th["n_rebuilds"])
        assert seen >= 3                           # several runs ended with the flag raised
        s.close()


# ------------------------------------------------------------------ tile method (shared-memory j staging)


def fold(r, box):
    """Positions folded into [-L/2, L/2): the tile method wraps coordinates only at list rebuilds (between them
    they may leave the box by up to skin/2; r + image L is the unwrapped position at all times)."""
    r = np.asarray(r, np.float64)
    return r - box * np.rint(r / box)


@pytest.mark.parametrize("kind,kw,tp,tile,nsteps", [
    ("lj", dict(ncell=10), 1, 0, 75),
    ("ka", dict(N=8000), 8, 3, 60),
    ("ka", dict(N=16384), 2, 4, 41),          # odd: positions end in the alternate buffer
    ("ch", dict(n=16), 4, 0, 40),
])
def test_tile_method_persistent_equals_per_step_bitwise_and_tracks_the_cell_method(rumd, kind, kw, tp, tile, nsteps):
    """RUMD_NB_TILE: the persistent kernel and the per-step kernels (k_build_tile, k_force_tile, k_integrate) run
    the same arithmetic in the same order -> NVE bit-identical across rebuilds, sorts and lazily wrapped
    coordinates; and the trajectory stays with the cell method's (same displacements, other summation order)."""
    wl = perturbed(make(kind, **kw))
    wl.integrator = W.NVE
    box = wl.box.astype(np.float64)
    res = []
    for method, persistent in ((rumd.NB_TILE, 1), (rumd.NB_TILE, 0), (rumd.NB_CELL, 1)):
        s = rumd.from_workload(wl)
        s.set_tuning(method=method, tp=tp, pb=256 // tp, tile=tile, persistent=persistent, use_graph=0, skin=0.25)
        s.run_steps(nsteps)
        s.run_steps(7)
        th = s.get_thermo()
        st = s.state()
        assert th["n_steps"] == nsteps + 7 and th["n_rebuilds"] >= 3 and th["overflow"] == 0
        res.append((st, th))
        s.close()
    (a, ta), (b, tb), (c, tc) = res
    assert ta["n_rebuilds"] == tb["n_rebuilds"]
    for key in ("r", "v", "F", "u", "w", "image"):
        assert np.array_equal(a[key], b[key]), key
    assert ta["U"] == tb["U"] and ta["max_nbrs"] == tb["max_nbrs"]
    d = (a["r"].astype(np.float64) + a["image"] * box) - (c["r"].astype(np.float64) + c["image"] * box)
    assert np.abs(d).max() < 2e-4
    assert ta["U"] == pytest.approx(tc["U"], rel=1e-4)


def test_tile_method_lockstep_with_particles_crossing_the_faces(rumd):
    """Protocol (3) for the tile method over several rebuilds: at every stop the list in use (halo slots mapped back
    to particles) contains every interacting pair, forces match the oracle, coordinates that left the box are within
    skin/2 of it and r + image L is continuous; some particles do cross faces during the run."""
    wl = perturbed(make("lj", ncell=10))
    wl.integrator = W.NVE
    s = rumd.from_workload(wl)
    s.set_tuning(method=rumd.NB_TILE, tp=2, pb=128, skin=0.3)
    box = wl.box.astype(np.float64)
    crossed = 0
    for _ in range(6):
        s.run_steps(53)
        s.compute_forces()
        st = s.state()
        out = np.abs(st["r"].astype(np.float64)) - 0.5 * box
        assert out.max() <= 0.5 * 0.3 + 1e-5
        crossed += int((np.abs(st["image"]).sum(1) > 0).sum())
        r64 = fold(st["r"], box)
        cnt, lst = s.export_nblist()
        ids = s.d_id.cpu().numpy().astype(np.int64)
        have = np.unique(pair_keys(cnt, lst, ids))
        assert have.size == cnt.sum()
        oc, ol = oracle.nblist(r64, wl.types, box, wl.pot, 0.0)
        assert np.isin(pair_keys(oc, ol), have).all(), "list in use misses interacting pairs"
        check_forces(s, r64, wl.types, box, wl.pot)
    assert crossed > 0 and s.get_thermo()["n_rebuilds"] >= 8
    s.close()


def test_tile_method_full_size_million_particles_whole_system(rumd):
    """configs[3] with the tile method at its default tile size: the whole list (every row, as sets, 1e-6 band), every
    force, U and W against the oracle; then one whole step and a short run (rebuilds with the sort in flight)."""
    wl = perturbed(make("lj", ncell=64))
    s = rumd.from_workload(wl)
    s.set_tuning(method=rumd.NB_TILE, tp=1, pb=256)
    s.compute_forces()
    r64 = wl.r.astype(np.float64)
    box = wl.box.astype(np.float64)
    gcnt, npairs, nband = check_nblist_rows(s, r64, wl.types, box, wl.pot, float(wl.skin))
    assert npairs > 7e7
    check_forces(s, r64, wl.types, box, wl.pot)
    th = s.get_thermo()
    assert th["overflow"] == 0 and th["max_nbrs"] == gcnt.max()
    s.run_steps(50)
    s.compute_forces()
    st = s.state()
    assert s.get_thermo()["n_rebuilds"] >= 3
    check_forces(s, fold(st["r"], box), wl.types, box, wl.pot)
    s.close()


@pytest.mark.parametrize("kind,kw,tuning", [
    ("ka", dict(N=8000), dict(method=3, tp=8, pb=32, tile=3, skin=0.35)),
    ("ch", dict(n=32), dict(method=3, tp=2, pb=128)),
    ("ka", dict(N=65536), dict(method=3, tp=1, pb=256, tile=4)),
])
def test_tile_method_one_step_matches_oracle(rumd, kind, kw, tuning):
    """One whole step (build -> forces -> integrate) of the tile method from identical inputs: U, K, xi, positions and
    velocities against the oracle, then U, W, forces of the new configuration."""
    wl = make(kind, **kw)
    wl = perturbed(wl) if kind != "ka" else wl
    s0 = rumd.from_workload(wl)
    s0.set_tuning(**tuning)
    s0.run_steps(300)
    st0 = s0.state()
    s0.close()
    box = wl.box.astype(np.float64)
    wl.r = fold(st0["r"], box).astype(np.float32)
    wl.r = np.where(wl.r >= 0.5 * wl.box, wl.r - wl.box, wl.r).astype(np.float32)
    wl.v = st0["v"].copy()
    s = rumd.from_workload(wl)
    s.set_tuning(**tuning)
    N = wl.N
    skin = float(s.get_tuning().skin)
    o = oracle.run(wl.r.astype(np.float64), wl.v.astype(np.float64), wl.m.astype(np.float64), np.zeros((N, 3), np.int32),
                   wl.types, box, wl.pot, skin, float(wl.dt), 1, mode=wl.integrator, T0=wl.T0, tau=wl.tau, use_cell=N >= 4096)
    s.run_steps(1)
    th1 = s.get_thermo()
    st = s.state()
    d = st["r"].astype(np.float64) + st["image"] * box - (o["r"] + o["image"] * box)
    assert np.abs(d).max() < max(2e-6, 6e-8 * box.max())
    assert np.abs(st["v"] - o["v"]).max() < 1e-5 * max(1.0, np.abs(o["v"]).max())
    assert th1["U"] == pytest.approx(o["log"][0, 0], rel=ENERGY_TOL)
    assert th1["K"] == pytest.approx(o["log"][0, 1], rel=ENERGY_TOL)
    if wl.integrator == W.NVT:
        assert th1["xi"] == pytest.approx(o["xi"], rel=1e-4, abs=1e-7)
    s.compute_forces()
    check_forces(s, fold(s.state()["r"], box), wl.types, box, wl.pot)
    s.close()


def test_tile_method_refuses_what_it_cannot_do(rumd):
    wl = make("lj", ncell=6)                       # 7 cells per axis: fine (6 is the minimum)
    s = rumd.from_workload(wl)
    with pytest.raises(rumd.RumdError):
        s.set_tuning(method=rumd.NB_TILE, tp=16, pb=16)
    s.set_tuning(method=rumd.NB_TILE, tp=8, pb=32, skin=1.0)   # rc + skin = 3.5 -> 5 cells per axis
    with pytest.raises(rumd.RumdError) as e:
        s.compute_forces()
    assert e.value.status == rumd.ERR_BOX_TOO_SMALL
    s.close()


# ------------------------------------------------------------------ NPT ("NPT [51]"; reading S32)


def _npt_system(rumd, N=1000, tp=8, method=None, P0=2.0, tauP=2.0, T0=2.0, density=0.5, seed=5):
    ncell = {500: 5, 864: 6, 2048: 8}.get(N)
    if ncell:
        r, box = W.fcc_lattice(ncell, ncell, ncell, density)
    else:
        n = round(N ** (1.0 / 3.0))
        r, box, _ = W.sc_lattice(n, n, n, density)
    N = r.shape[0]
    rng = np.random.default_rng(seed)
    m = np.ones(N)
    v = W.maxwell_boltzmann(rng, m, T0)
    wl = W.Workload(name="npt", r=W._fold32(r, box), v=v.astype(np.float32), m=m.astype(np.float32),
                    types=np.zeros(N, np.int32), box=box.astype(np.float32), pot=W.lj_single(), skin=W.f32(0.3),
                    dt=W.f32(0.004), integrator=rumd.INT_NPT_MTK, T0=W.f32(T0), tau=W.f32(0.2))
    wl.r = W.perturb(wl.r, wl.box, 0.05, 3)
    s = rumd.System(wl.r, wl.v, wl.m, wl.types, wl.box, wl.pot)
    s.set_barostat(P0, tauP)
    s.set_integrator(rumd.INT_NPT_MTK, wl.dt, wl.T0, wl.tau)
    s.set_tuning(method=rumd.NB_N2 if method is None else method, tp=tp, pb=256 // tp, skin=float(wl.skin), persistent=0,
                 use_graph=0)
    return s, wl


@pytest.mark.parametrize("N,method,use_graph", [(500, 0, 0), (1000, 0, 1), (864, 2, 0)])
def test_npt_steps_match_oracle(rumd, N, method, use_graph):
    """NPT (Martyna-Tobias-Klein barostat + Nose-Hoover thermostat, reading S32) on the per-step kernels against the
    oracle from identical inputs: after 1 step positions, velocities, box, thermostat and strain rate; after 25 more
    the box, nu, xi, U, K, H still track (before chaos separates the trajectories)."""
    s, wl = _npt_system(rumd, N=N, method=method)
    s.set_tuning(use_graph=use_graph, steps_per_graph=4)
    P0, tauP = 2.0, 2.0
    N = wl.N
    r64, v64, m64 = wl.r.astype(np.float64), wl.v.astype(np.float64), wl.m.astype(np.float64)
    box = wl.box.astype(np.float64)
    args = dict(T0=float(wl.T0), tau=float(wl.tau), P0=P0, tauP=tauP)
    o = oracle.run_npt(r64, v64, m64, np.zeros((N, 3), np.int32), wl.types, box, wl.pot, 0.3, float(wl.dt), 1, **args)
    s.run_steps(1)
    th = s.get_thermo()
    st = s.state()
    gbox, gnu = s.get_box()
    assert np.allclose(gbox, o["box"], rtol=1e-7)
    # nu = dt cP [ (1 + 3/g) sum m v^2 + W - 3 V P0 ]: the three terms nearly cancel, so the 1e-5 relative accuracy of
    # the fp32 virial sum W (north_star) is the scale of the tolerance, not nu itself
    g = 3.0 * N - 3.0
    cP = (2.0 * np.pi / tauP) ** 2 / ((g + 3.0) * float(wl.T0))
    # (in this fluid the per-particle virials w_i have both signs and W = sum w_i nearly cancels: as for U on the KA
    # lattice start, S29, the scale of the fp32 sum's 1e-5 is sum |w_i|)
    w_scale = np.abs(oracle.forces_allpairs(r64, wl.types, box, wl.pot)[2]).sum()
    nu_tol = float(wl.dt) * cP * ENERGY_TOL * w_scale
    assert gnu == pytest.approx(o["nu"], abs=nu_tol)
    d = st["r"].astype(np.float64) + st["image"] * gbox - (o["r"] + o["image"] * o["box"])
    assert np.abs(d).max() < 3e-6
    assert np.abs(st["v"] - o["v"]).max() < 1e-5 * max(1.0, np.abs(o["v"]).max())
    assert th["U"] == pytest.approx(o["log"][0, 0], rel=ENERGY_TOL)
    assert abs(th["W"] - o["log"][0, 2]) <= ENERGY_TOL * w_scale
    assert th["K"] == pytest.approx(o["log"][0, 1], rel=ENERGY_TOL)
    assert th["H"] == pytest.approx(o["log"][0, 5], rel=ENERGY_TOL)
    # xi = dt w^2 (T_kin / T0 - 1) with T_kin within 1e-3 of T0 here: the fp32 velocities' 1e-7 sets the absolute scale
    assert th["xi"] == pytest.approx(o["xi"], rel=1e-4, abs=float(wl.dt) * (2.0 * np.pi / float(wl.tau)) ** 2 * 3e-7)
    # 25 more steps
    o2 = oracle.run_npt(r64, v64, m64, np.zeros((N, 3), np.int32), wl.types, box, wl.pot, 0.3, float(wl.dt), 26, **args)
    s.run_steps(25)
    th = s.get_thermo()
    gbox, gnu = s.get_box()
    assert np.allclose(gbox, o2["box"], rtol=1e-6)
    assert gnu == pytest.approx(o2["nu"], rel=1e-3, abs=30.0 * nu_tol)
    assert th["xi"] == pytest.approx(o2["xi"], rel=1e-3, abs=1e-6)
    assert th["U"] == pytest.approx(o2["log"][-1, 0], rel=1e-4)
    assert th["K"] == pytest.approx(o2["log"][-1, 1], rel=1e-4)
    assert th["H"] == pytest.approx(o2["log"][-1, 5], rel=1e-4)
    assert th["n_steps"] == 26
    # forces of the configuration the GPU now holds, in ITS box
    s.compute_forces()
    st = s.state()
    F, u, w = oracle.forces_allpairs(st["r"].astype(np.float64), wl.types, gbox, wl.pot)
    rms = np.sqrt((F * F).sum(1).mean())
    assert np.sqrt(((st["F"] - F) ** 2).sum(1)).max() <= FORCE_TOL * rms
    s.close()


def test_npt_with_the_barostat_off_equals_the_nvt_kernels_bitwise(rumd):
    """tau_P = 0 freezes the strain rate at 0: every factor of the NPT step reduces to the NVT step (reading S32), and
    with 8 lanes per particle both paths add the pair forces in the same order -> bit-identical while the two lists
    are the same (the NPT list is rebuilt at 0.4 skin instead of skin/2, so only up to the first rebuild)."""
    s, wl = _npt_system(rumd, N=1000, tauP=0.0)
    s.run_steps(6)
    a, ta = s.state(), s.get_thermo()
    s.close()
    s2 = rumd.System(wl.r, wl.v, wl.m, wl.types, wl.box, wl.pot)
    s2.set_integrator(rumd.INT_NVT_NOSE_HOOVER, wl.dt, wl.T0, wl.tau)
    s2.set_tuning(method=rumd.NB_N2, tp=8, pb=32, skin=float(wl.skin), persistent=0, use_graph=0)
    s2.run_steps(6)
    b, tb = s2.state(), s2.get_thermo()
    s2.close()
    assert ta["n_rebuilds"] == tb["n_rebuilds"] == 1
    for key in ("r", "v", "image"):
        assert np.array_equal(a[key], b[key]), key
    assert ta["xi"] == tb["xi"] and ta["K"] == pytest.approx(tb["K"], rel=1e-12)


def test_npt_reaches_the_target_pressure_and_conserves_its_invariant(rumd):
    """LJ fluid started well below the target pressure: the box shrinks, <P> settles at P0, <T_kin> at T0, and the
    conserved quantity of the extended system does not drift (slope of H/N over 1e4 steps <= 1e-3; fp32 positions
    and forces, no 1e-4 bar is claimed for NPT: the paper only requires NVE to be drift-free-ish)."""
    s, wl = _npt_system(rumd, N=2048, density=0.5, P0=2.0, tauP=2.0)
    N = wl.N
    V0 = float(np.prod(wl.box.astype(np.float64)))
    s.run_steps(3000)
    gbox, _ = s.get_box()
    assert np.prod(gbox) < 0.95 * V0
    P, T, H = [], [], []
    for _ in range(100):
        s.run_steps(100)
        th = s.get_thermo()
        gbox, _ = s.get_box()
        P.append((2.0 * th["K"] + th["W"]) / (3.0 * np.prod(gbox)))
        T.append(2.0 * th["K"] / (3.0 * N - 3.0))
        H.append(th["H"] / N)
    assert np.mean(P) == pytest.approx(2.0, abs=0.1)
    assert np.mean(T) == pytest.approx(2.0, rel=0.03)
    slope = np.polyfit(np.arange(100) * 100.0, np.array(H), 1)[0]
    assert abs(slope * 1e4) <= 1e-3
    assert s.get_thermo()["n_rebuilds"] > 100
    s.close()


def test_npt_refuses_cell_methods_and_autotune(rumd):
    s, wl = _npt_system(rumd, N=1000)
    s.set_tuning(method=rumd.NB_CELL)
    with pytest.raises(rumd.RumdError) as e:
        s.run_steps(1)
    assert e.value.status == rumd.ERR_INVALID_ARG
    s.set_tuning(method=rumd.NB_N2)
    with pytest.raises(rumd.RumdError):
        s.autotune(steps_per_trial=10)
    s.run_steps(3)
    assert s.get_thermo()["n_steps"] == 3
    s.close()


def test_tile_method_ragged_gas_four_types_and_halo_overflow(rumd):
    """Tile method away from lattices: a jittered gas of N = 4099 particles (not a multiple of anything) of four types
    with six different pair potentials in an orthorhombic box -- list as a set, forces, a 37-step trajectory against
    the oracle; then a configuration squeezed into one corner of the box, whose halo cannot fit the shared-memory
    slots sized for a uniform density: the sticky overflow error must come back, not a wrong list."""
    nt = 4
    pot = W.pot_table(nt)
    for a in range(nt):
        for b in range(a, nt):
            W.set_lj(pot, a, b, 1.0 + 0.1 * (a + b), 1.0 - 0.04 * (a + b), 2.5 * (1.0 - 0.04 * (a + b)))
    box = (15.0, 19.0, 23.0)
    r, v, m, types, boxf, pot = _gas(4099, nt, box, 4242, pot)
    s = rumd.System(r, v, m, types, boxf, pot)
    s.set_integrator(rumd.INT_NVE_LEAPFROG, 0.004)
    s.set_tuning(method=rumd.NB_TILE, tp=2, pb=128, skin=0.3, tile=3)
    s.compute_forces()
    r64, b64 = r.astype(np.float64), boxf.astype(np.float64)
    check_nblist(s, r64, types, b64, pot, 0.3)
    F, u, w = oracle.forces_allpairs(r64, types, b64, pot)
    st = s.state()
    scale = max(1e-3, np.sqrt((F * F).sum(1).mean()))
    assert np.sqrt(((st["F"] - F) ** 2).sum(1)).max() <= FORCE_TOL * scale
    assert np.abs(st["u"] - u).max() <= 1e-5 * max(1.0, np.abs(u).max())
    s.run_steps(37)
    th = s.get_thermo()
    assert th["n_steps"] == 37 and th["overflow"] == 0
    o = oracle.run(r64, v.astype(np.float64), m.astype(np.float64), np.zeros((4099, 3), np.int32), types, b64, pot, 0.3,
                   0.004, 37)
    st = s.state()
    d = st["r"].astype(np.float64) + st["image"] * b64 - (o["r"] + o["image"] * b64)
    assert np.abs(d).max() < 2e-4
    s.close()
    # everything in one octant: eight times the mean density there
    rc = (0.5 * r - 0.25 * boxf).astype(np.float32)
    s = rumd.System(rc, v, m, types, boxf, pot)
    s.set_integrator(rumd.INT_NVE_LEAPFROG, 0.001)
    s.set_tuning(method=rumd.NB_TILE, tp=2, pb=128, skin=0.3, tile=3)
    s.compute_forces()
    with pytest.raises(rumd.RumdError) as e:
        s.get_thermo()
    assert e.value.status == rumd.ERR_NBL_OVERFLOW
    s.close()


@pytest.mark.parametrize("kind,kw,tp", [("ka", dict(N=4096), 8), ("ka", dict(N=16384), 2), ("ch", dict(n=16), 4)])
def test_two_type_register_select_equals_the_table_lookup_bitwise(rumd, kind, kw, tp):
    """A5, two-type systems: force_loop keeps both parameter records of a lane in registers and selects per pair (TWO).
    The same system declared with a THIRD, unused particle type goes through the generic shared-memory table instead;
    the arithmetic is the same, so forces, energies, virials and a short NVE trajectory agree bit for bit -- through the
    stand-alone force kernel, the persistent kernel and the per-step kernels."""
    wl2 = perturbed(make(kind, **kw))
    wl2.integrator = W.NVE
    wl3 = perturbed(make(kind, **kw))
    wl3.integrator = W.NVE
    pot3 = W.pot_table(3)
    pot3[:2, :2] = wl2.pot
    W.set_lj(pot3, 0, 2, 1.0, 1.0, 2.0)   # a type nobody has; cutoffs below rc_max, so the cell grid is the same
    W.set_lj(pot3, 1, 2, 1.0, 1.0, 2.0)
    W.set_lj(pot3, 2, 2, 1.0, 1.0, 2.0)
    wl3.pot = pot3
    assert wl3.ntypes == 3 and wl2.ntypes == 2 and wl3.rc_max() == wl2.rc_max()
    for persistent in (1, 0):
        res = []
        for wl in (wl2, wl3):
            s = rumd.from_workload(wl)
            s.set_tuning(method=rumd.NB_CELL, tp=tp, pb=256 // tp, persistent=persistent, use_graph=0)
            s.compute_forces()
            st0 = s.state()
            s.run_steps(25)
            res.append((st0, s.state(), s.get_thermo()))
            s.close()
        (a0, a1, ta), (b0, b1, tb) = res
        for key in ("F", "u", "w"):
            assert np.array_equal(a0[key], b0[key]), key
        for key in ("r", "v", "F", "u", "w", "image"):
            assert np.array_equal(a1[key], b1[key]), (key, persistent)
        assert ta["U"] == tb["U"] and ta["W"] == tb["W"] and ta["n_rebuilds"] == tb["n_rebuilds"]
    # and the two-type path against the oracle, on the same state
    s = rumd.from_workload(wl2)
    s.set_tuning(method=rumd.NB_CELL, tp=tp, pb=256 // tp)
    s.compute_forces()
    check_forces(s, wl2.r.astype(np.float64), wl2.types, wl2.box.astype(np.float64), wl2.pot, cancelling=kind == "ka")
    s.close()


@pytest.mark.parametrize("kind,kw,tp,build_tp", [("ka", dict(N=131072), 2, 4), ("lj", dict(ncell=64), 1, 1)])
def test_list_built_inside_the_persistent_kernel_from_the_unit_queue(rumd, kind, kw, tp, build_tp):
    """A4 inside A7 at sizes where a warp has several units to build: k_persist hands them out from a device counter
    (DevScalars::build_queue).  The list the first step builds -- at the initial positions, after the spatial sort --
    is compared with the oracle's as a set, ALL rows (1e-6 band), and the forces of that step's evaluation with it."""
    wl = perturbed(make(kind, **kw))
    wl.integrator = W.NVE
    s = rumd.from_workload(wl)
    s.set_tuning(method=rumd.NB_CELL, tp=tp, pb=256 // tp, build_tp=build_tp, persistent=1)
    s.run_steps(1)
    th = s.get_thermo()
    assert th["n_rebuilds"] == 1 and th["overflow"] == 0
    r64 = wl.r.astype(np.float64)
    box = wl.box.astype(np.float64)
    gcnt, npairs, nband = check_nblist_rows(s, r64, wl.types, box, wl.pot, float(wl.skin))
    assert int(gcnt.sum()) in range(npairs - nband, npairs + nband + 1) and th["max_nbrs"] == gcnt.max()
    # forces of the step's (only) force evaluation belong to the initial positions too
    st = s.state()
    F, u, w = oracle.forces_list(r64, wl.types, box, wl.pot, *oracle.nblist(r64, wl.types, box, wl.pot, 0.0, method="cell"))
    rms = np.sqrt((F * F).sum(1).mean())
    assert np.sqrt(((st["F"].astype(np.float64) - F) ** 2).sum(1)).max() <= FORCE_TOL * rms
    s.close()
