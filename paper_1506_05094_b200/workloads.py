"""Seeded synthetic inputs shaped like the paper's benchmarks.

This module serves BOTH the CUDA path and the fp64 oracle and therefore holds none of the method's
arithmetic: no pair function, no minimum image, no neighbour criterion, no integrator -- only
lattices, random numbers and parameter tables.  Everything is generated in float64 from
``numpy.random.default_rng(seed)`` and then ROUNDED TO float32; both sides receive the same
fp32-representable values.  It imports neither ``oracle`` nor the CUDA binding.

The workloads stand in for the LAMMPS "Lennard-Jones" melting-fcc benchmark and the paper's
molten-salt benchmark, whose input decks are not available; shapes, densities and cutoffs
come from BASELINE.json ``configs``.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

SEED0 = 150605094  # + 1000*config + index-in-sweep

NVE, NVT = 0, 1
POT_STRIDE = 11  # (epsilon, sigma, rc_LJ, a, rc_2, cut_LJ, cut_2, kind_2, b, c, d); rc <= 0 disables the term
KIND_COULOMB, KIND_IPL, KIND_YUKAWA, KIND_GAUSSIAN_CORE, KIND_BUCKINGHAM = 0, 1, 2, 3, 4  # second term
KIND_GEN_LJ, KIND_GIRIFALCO, KIND_DZUGUTOV = 5, 6, 7
KIND_NPARAMS = (1, 2, 2, 2, 3, 4, 3, 2)  # how many of (a, b, c, d) each kind takes
CUT_SHIFTED_FORCE, CUT_SHIFTED_POTENTIAL, CUT_NONE = 0, 1, 2


@dataclass
class Workload:
    name: str
    r: np.ndarray          # (N,3) float32, origin-centred box, coordinates in [-L/2, L/2)
    v: np.ndarray          # (N,3) float32, leap-frog velocities v(-dt/2)
    m: np.ndarray          # (N,)  float32
    types: np.ndarray      # (N,)  int32
    box: np.ndarray        # (3,)  float32
    pot: np.ndarray        # (nt,nt,5) float64 holding fp32-representable values
    skin: float
    dt: float
    integrator: int        # NVE / NVT
    T0: float
    tau: float = 0.2       # Nose-Hoover period (S9); unused for NVE
    steps: int = 1000
    meta: dict = field(default_factory=dict)

    @property
    def N(self) -> int:
        return int(self.r.shape[0])

    @property
    def ntypes(self) -> int:
        return int(self.pot.shape[0])

    def rc_max(self) -> float:
        return float(max(self.pot[..., 2].max(), self.pot[..., 4].max()))


def f32(x):
    """Round to float32 and return as python float / float64 array (the shared fp32-representable value)."""
    a = np.asarray(x, dtype=np.float64).astype(np.float32)
    return float(a) if a.ndim == 0 else a.astype(np.float64)


# ----------------------------------------------------------------------------- lattices


def fcc_lattice(nx: int, ny: int, nz: int, density: float):
    """4*nx*ny*nz sites of an fcc lattice at the given number density; returns (r float64 (N,3), box (3,))."""
    a = (4.0 / density) ** (1.0 / 3.0)
    basis = np.array([[0, 0, 0], [0.5, 0.5, 0], [0.5, 0, 0.5], [0, 0.5, 0.5]], dtype=np.float64)
    ii, jj, kk = np.meshgrid(np.arange(nx), np.arange(ny), np.arange(nz), indexing="ij")
    cells = np.stack([ii.ravel(), jj.ravel(), kk.ravel()], axis=1).astype(np.float64)
    r = (cells[:, None, :] + basis[None, :, :] + 0.25).reshape(-1, 3) * a
    box = np.array([nx, ny, nz], dtype=np.float64) * a
    return r - 0.5 * box, box


def sc_lattice(nx: int, ny: int, nz: int, density: float):
    """nx*ny*nz sites of a simple-cubic lattice; site (i,j,k) at ((i,j,k)+1/2) a - L/2, index = (i*ny+j)*nz+k."""
    a = (1.0 / density) ** (1.0 / 3.0)
    ii, jj, kk = np.meshgrid(np.arange(nx), np.arange(ny), np.arange(nz), indexing="ij")
    ijk = np.stack([ii.ravel(), jj.ravel(), kk.ravel()], axis=1)
    r = (ijk.astype(np.float64) + 0.5) * a
    box = np.array([nx, ny, nz], dtype=np.float64) * a
    return r - 0.5 * box, box, ijk


def maxwell_boltzmann(rng, m: np.ndarray, T: float) -> np.ndarray:
    """N(0, T/m) per component, centre-of-mass velocity removed, rescaled so sum m v^2/(3N-3) = T."""
    N = m.shape[0]
    v = rng.standard_normal((N, 3)) * np.sqrt(T / m)[:, None]
    v -= (m[:, None] * v).sum(axis=0) / m.sum()
    tk = (m[:, None] * v * v).sum() / (3.0 * N - 3.0)
    return v * np.sqrt(T / tk)


def perturb(r: np.ndarray, box: np.ndarray, amplitude: float, seed: int) -> np.ndarray:
    """Seeded uniform displacement in [-amplitude, amplitude] per coordinate, folded back into the box,
    rounded to float32 (S24: force parity is measured on a perturbed state, F = 0 on the perfect lattice)."""
    rng = np.random.default_rng(seed)
    x = np.asarray(r, dtype=np.float64) + rng.uniform(-amplitude, amplitude, size=r.shape)
    b = np.asarray(box, dtype=np.float64)
    x = x - b * np.floor(x / b + 0.5)
    return _fold32(x, b)


def _fold32(x: np.ndarray, box: np.ndarray) -> np.ndarray:
    """float32 positions guaranteed inside [-L/2, L/2) after rounding."""
    b32 = box.astype(np.float32)
    x32 = x.astype(np.float32)
    half = (0.5 * b32).astype(np.float32)
    x32 = np.where(x32 >= half, x32 - b32, x32)
    x32 = np.where(x32 < -half, x32 + b32, x32)
    return x32.astype(np.float32)


# ----------------------------------------------------------------------------- potentials


def pot_table(ntypes: int) -> np.ndarray:
    return np.zeros((ntypes, ntypes, POT_STRIDE), dtype=np.float64)


def set_lj(pot, a, b, eps, sig, rc, cut=CUT_SHIFTED_FORCE):
    for i, j in ((a, b), (b, a)):
        pot[i, j, 0], pot[i, j, 1], pot[i, j, 2], pot[i, j, 5] = f32(eps), f32(sig), f32(rc), float(cut)


def set_coulomb(pot, a, b, qq, rc, cut=CUT_SHIFTED_FORCE):
    set_second_term(pot, a, b, KIND_COULOMB, qq, 0.0, 0.0, rc, cut)


def set_second_term(pot, a, b, kind, pa, pb, pc, rc, cut=CUT_SHIFTED_FORCE, pd=0.0):
    """The pair's second term: Coulomb pa/r, IPL pa r^-pb, Yukawa pa exp(-r/pb)/r, Gaussian core pa exp(-(r/pb)^2),
    Buckingham pa exp(-r/pb) - pc/r^6, generalized LJ (epsilon pa, sigma pb, exponents pc > pd), Girifalco (alpha pa,
    beta pb, diameter pc), Dzugutov (epsilon pa, sigma pb) (formulas in include/rumd_b200.h)."""
    for i, j in ((a, b), (b, a)):
        pot[i, j, 3], pot[i, j, 4], pot[i, j, 6] = f32(pa), f32(rc), float(cut)
        pot[i, j, 7], pot[i, j, 8], pot[i, j, 9], pot[i, j, 10] = float(kind), f32(pb), f32(pc), f32(pd)


def lj_single() -> np.ndarray:
    pot = pot_table(1)
    set_lj(pot, 0, 0, 1.0, 1.0, 2.5)
    return pot


def kob_andersen() -> np.ndarray:
    """eps AA/AB/BB = 1/1.5/0.5, sigma = 1/0.8/0.88, rc = 2.5 sigma_ab (BASELINE.json configs[1])."""
    pot = pot_table(2)
    set_lj(pot, 0, 0, 1.0, 1.0, 2.5)
    set_lj(pot, 0, 1, 1.5, 0.8, 2.5 * 0.8)
    set_lj(pot, 1, 1, 0.5, 0.88, 2.5 * 0.88)
    return pot


def charged_lj() -> np.ndarray:
    """LJ eps = sigma = 1, rc 2.5 on all pairs + SF Coulomb q = +-1, rc 4.0, prefactor 1 (configs[4])."""
    pot = pot_table(2)
    for a, b in ((0, 0), (0, 1), (1, 1)):
        set_lj(pot, a, b, 1.0, 1.0, 2.5)
    q = (+1.0, -1.0)
    for a, b in ((0, 0), (0, 1), (1, 1)):
        set_coulomb(pot, a, b, q[a] * q[b], 4.0)
    return pot


# ----------------------------------------------------------------------------- configs


def _finish(name, r, box, types, pot, T, seed, **kw) -> Workload:
    rng = np.random.default_rng(seed)
    N = r.shape[0]
    m = np.ones(N, dtype=np.float64)
    v = maxwell_boltzmann(rng, m, T)
    return Workload(name=name, r=_fold32(r, box), v=v.astype(np.float32), m=m.astype(np.float32),
                    types=np.ascontiguousarray(types, dtype=np.int32), box=box.astype(np.float32), pot=pot,
                    T0=f32(T), **kw)


def lj_fcc(ncell: int = 6, seed: int = SEED0, steps: int = 1000) -> Workload:
    """configs[0] (ncell=6, N=864) and configs[3] (ncell=64, N=1 048 576): single-component LJ on fcc,
    density 0.8442, T=0.722, NVE dt=0.005, rc=2.5 SF, skin 0.3."""
    r, box = fcc_lattice(ncell, ncell, ncell, 0.8442)
    N = r.shape[0]
    return _finish("lj_fcc_N%d" % N, r, box, np.zeros(N, np.int32), lj_single(), 0.722, seed,
                   skin=f32(0.3), dt=f32(0.005), integrator=NVE, steps=steps,
                   meta=dict(config=0 if ncell == 6 else 3, lattice="fcc", density=0.8442))


KA_DIMS = {512: (8, 8, 8), 1000: (10, 10, 10), 2048: (16, 16, 8), 4096: (16, 16, 16), 8000: (20, 20, 20),
           8192: (32, 16, 16), 16384: (32, 32, 16), 32768: (32, 32, 32), 65536: (64, 32, 32),
           131072: (64, 64, 32)}
KA_SWEEP = (512, 1000, 2048, 4096, 8192, 16384, 32768, 65536, 131072)


def ka_lattice(N: int = 8000, seed: int | None = None, steps: int = 10000) -> Workload:
    """configs[1] (N=8000) and configs[2] (the sweep): Kob-Andersen 80:20 on a simple-cubic lattice at
    density 1.2 (S23 for the non-cubic sizes), 20 % B chosen by rng.choice, T=0.8, NVT dt=0.0025."""
    dims = KA_DIMS[N]
    if seed is None:
        seed = SEED0 + (1000 if N == 8000 else 2000 + KA_SWEEP.index(N))
    r, box, _ = sc_lattice(*dims, 1.2)
    rng = np.random.default_rng(seed)
    types = np.zeros(N, np.int32)
    types[rng.choice(N, int(round(0.2 * N)), replace=False)] = 1
    return _finish("ka_N%d" % N, r, box, types, kob_andersen(), 0.8, seed + 1,
                   skin=f32(0.3), dt=f32(0.0025), integrator=NVT, tau=f32(0.2), steps=steps,
                   meta=dict(config=1 if N == 8000 else 2, lattice="sc", density=1.2, dims=dims))


def charged_sc(n: int = 32, seed: int = SEED0 + 4000, steps: int = 5000) -> Workload:
    """configs[4]: N = n^3 ions on a simple-cubic lattice with alternating charge (rock salt), density 0.5,
    LJ rc 2.5 + SF Coulomb rc 4.0, T=1.0, NVT dt=0.002.  Type 0 = +1, type 1 = -1."""
    r, box, ijk = sc_lattice(n, n, n, 0.5)
    types = (ijk.sum(axis=1) % 2).astype(np.int32)
    return _finish("charged_N%d" % (n ** 3), r, box, types, charged_lj(), 1.0, seed,
                   skin=f32(0.3), dt=f32(0.002), integrator=NVT, tau=f32(0.2), steps=steps,
                   meta=dict(config=4, lattice="rocksalt", density=0.5))


def random_gas(N: int, ntypes: int, box, seed: int, min_dist: float = 0.85) -> tuple[np.ndarray, np.ndarray]:
    """Small random configurations for brute-force pins: a jittered lattice so no two particles overlap
    (pure uniform positions give r -> 0 pairs whose r^-12 forces swamp every tolerance)."""
    rng = np.random.default_rng(seed)
    box = np.asarray(box, dtype=np.float64)
    n = np.maximum(1, np.floor(box / min_dist)).astype(int)
    while n.prod() < N:
        raise ValueError("box too small for N at this min_dist")
    sites = rng.choice(int(n.prod()), N, replace=False)
    k = np.stack(np.unravel_index(sites, tuple(n)), axis=1).astype(np.float64)
    a = box / n
    jitter = 0.5 * (a - min_dist * 0.98)
    x = (k + 0.5) * a + rng.uniform(-1, 1, size=(N, 3)) * jitter - 0.5 * box
    types = rng.integers(0, ntypes, size=N).astype(np.int32)
    return _fold32(x, box), types
