"""fp64 CPU oracle for the RUMD hot path -- TEST INFRASTRUCTURE, not the product.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It shares no code with the CUDA path
(``paper_1506_05094_b200``) and neither imports the other.  The arithmetic lives in
``rumd_oracle.c`` (plain C, double precision, one function per definition, each citing
PAPER.md); this module only compiles it with gcc, loads it with ctypes and marshals numpy
arrays.  See the header of ``rumd_oracle.c`` for the list of pins.

Array conventions: positions / velocities / forces are float64 ``(N, 3)``; types int32 ``(N,)``;
box float64 ``(3,)``; potentials float64 ``(ntypes, ntypes, 5)`` with records
``(epsilon, sigma, rc_LJ, a, rc_2, cut_LJ, cut_2, kind_2, b, c)`` (an rc <= 0 disables that term;
cut = 0 shifted force, 1 shifted potential, 2 no shift; kind_2 = 0 Coulomb a/r, 1 IPL a r^-b,
2 Yukawa a exp(-r/b)/r, 3 Gaussian core a exp(-(r/b)^2), 4 Buckingham a exp(-r/b) - c/r^6).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "rumd_oracle.c")
_LIB = os.path.join(_HERE, "librumd_oracle.so")

NVE, NVT, NPT = 0, 1, 2
POT_STRIDE = 11


def build(force: bool = False) -> str:
    """Compile rumd_oracle.c -> librumd_oracle.so (gcc -O2 -fopenmp, no fast-math)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp%d" % os.getpid()
        subprocess.check_call(
            ["gcc", "-O2", "-std=c99", "-D_GNU_SOURCE", "-fopenmp", "-fPIC", "-shared", "-o", tmp, _SRC, "-lm"]
        )
        os.replace(tmp, _LIB)
    return _LIB


_lib = None
_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int)


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.orc_num_threads.restype = C.c_int
        L.orc_set_num_threads.argtypes = [C.c_int]
        L.orc_lj_raw.argtypes = [C.c_double] * 3 + [_dp, _dp]
        L.orc_lj_sf.argtypes = [C.c_double] * 4 + [_dp, _dp]
        L.orc_coulomb_sf.argtypes = [C.c_double] * 3 + [_dp, _dp]
        L.orc_lj_cut.argtypes = [C.c_double] * 4 + [C.c_int, _dp, _dp]
        L.orc_coulomb_cut.argtypes = [C.c_double] * 3 + [C.c_int, _dp, _dp]
        L.orc_extra_raw.argtypes = [C.c_int] + [C.c_double] * 5 + [_dp, _dp]
        L.orc_extra_cut.argtypes = [C.c_int] + [C.c_double] * 6 + [C.c_int, _dp, _dp]
        L.orc_pair_sf.argtypes = [_dp, C.c_double, _dp, _dp]
        L.orc_pair_rc.argtypes = [_dp]
        L.orc_pair_rc.restype = C.c_double
        L.orc_min_image.argtypes = [_dp, _dp]
        L.orc_forces_allpairs.argtypes = [C.c_int, _dp, _ip, _dp, C.c_int, _dp, _dp, _dp, _dp]
        L.orc_forces_list.argtypes = [C.c_int, _dp, _ip, _dp, C.c_int, _dp, C.c_int, _ip, _ip, _dp, _dp, _dp]
        for f in (L.orc_nblist_n2, L.orc_nblist_cell):
            f.argtypes = [C.c_int, _dp, _ip, _dp, C.c_int, _dp, C.c_double, C.c_int, _ip, _ip]
            f.restype = C.c_int
        L.orc_needs_rebuild.argtypes = [C.c_int, _dp, _dp, _dp, C.c_double]
        L.orc_needs_rebuild.restype = C.c_int
        L.orc_integrate.argtypes = [C.c_int, _dp, _dp, _dp, _ip, _dp, _dp, C.c_double, C.c_int,
                                    C.c_double, C.c_double, C.c_double, _dp, _dp]
        L.orc_run.argtypes = [C.c_int, _dp, _dp, _dp, _ip, _ip, _dp, C.c_int, _dp, C.c_double, C.c_double,
                              C.c_int, C.c_double, C.c_double, _dp, C.c_long, C.c_int, _dp]
        L.orc_run.restype = C.c_long
        L.orc_integrate_npt.argtypes = [C.c_int, _dp, _dp, _dp, _ip, _dp, C.c_double, _dp, C.c_double, C.c_double,
                                        C.c_double, C.c_double, C.c_double, C.c_double, _dp, _dp]
        L.orc_run_npt.argtypes = [C.c_int, _dp, _dp, _dp, _ip, _ip, _dp, C.c_int, _dp, C.c_double, C.c_double,
                                  C.c_double, C.c_double, C.c_double, C.c_double, _dp, C.c_long, C.c_int, _dp]
        L.orc_run_npt.restype = C.c_long
        _lib = L
    return _lib


def _d(a):
    return a.ctypes.data_as(_dp)


def _i(a):
    return a.ctypes.data_as(_ip)


def _f64(a, shape=None):
    a = np.ascontiguousarray(a, dtype=np.float64)
    if shape is not None:
        assert a.shape == shape, (a.shape, shape)
    return a


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def num_threads() -> int:
    return int(lib().orc_num_threads())


def set_num_threads(n: int) -> None:
    lib().orc_set_num_threads(int(n))


def _pair(fn, *args):
    u, f = C.c_double(), C.c_double()
    fn(*args, C.byref(u), C.byref(f))
    return u.value, f.value


def lj_raw(r, eps, sig):
    """(u, f=-du/dr) of the unshifted 12-6 LJ potential."""
    return _pair(lib().orc_lj_raw, float(r), float(eps), float(sig))


def lj_sf(r, eps, sig, rc):
    return _pair(lib().orc_lj_sf, float(r), float(eps), float(sig), float(rc))


def coulomb_sf(r, qq, rc):
    return _pair(lib().orc_coulomb_sf, float(r), float(qq), float(rc))


def lj_cut(r, eps, sig, rc, method):
    """(u, f) of LJ 12-6 with cutoff method 0 = shifted force, 1 = shifted potential, 2 = no shift."""
    return _pair(lib().orc_lj_cut, float(r), float(eps), float(sig), float(rc), int(method))


def coulomb_cut(r, qq, rc, method):
    return _pair(lib().orc_coulomb_cut, float(r), float(qq), float(rc), int(method))


def extra_raw(kind, r, a, b=0.0, c=0.0, d=0.0):
    """(u, f) of the unshifted second-term potentials: 0 Coulomb, 1 IPL, 2 Yukawa, 3 Gaussian core, 4 Buckingham,
    5 generalized LJ, 6 Girifalco, 7 Dzugutov."""
    return _pair(lib().orc_extra_raw, int(kind), float(r), float(a), float(b), float(c), float(d))


def extra_cut(kind, r, a, b, c, rc, method, d=0.0):
    return _pair(lib().orc_extra_cut, int(kind), float(r), float(a), float(b), float(c), float(d), float(rc), int(method))


def pair_sf(rec, r):
    rec = _f64(rec, (POT_STRIDE,))
    return _pair(lib().orc_pair_sf, _d(rec), float(r))


def min_image(d, box):
    d = _f64(d).copy()
    lib().orc_min_image(_d(d), _d(_f64(box, (3,))))
    return d


def _prep(r, types, box, pot):
    r = _f64(r)
    N = r.shape[0]
    assert r.shape == (N, 3)
    types = _i32(types)
    assert types.shape == (N,)
    box = _f64(box, (3,))
    pot = _f64(pot)
    nt = pot.shape[0]
    assert pot.shape == (nt, nt, POT_STRIDE)
    assert types.min(initial=0) >= 0 and types.max(initial=0) < nt
    return r, N, types, box, pot, nt


def forces_allpairs(r, types, box, pot):
    """Brute force over all pairs -> (F (N,3), u (N,), w (N,))."""
    r, N, types, box, pot, nt = _prep(r, types, box, pot)
    F = np.zeros((N, 3))
    u = np.zeros(N)
    w = np.zeros(N)
    lib().orc_forces_allpairs(N, _d(r), _i(types), _d(box), nt, _d(pot), _d(F), _d(u), _d(w))
    return F, u, w


def nblist(r, types, box, pot, skin, method="n2", cap=None):
    """Full Verlet list -> (count (N,), list (N, cap)).  method 'n2' or 'cell'.  Capacity doubles
    until everything fits."""
    r, N, types, box, pot, nt = _prep(r, types, box, pot)
    fn = {"n2": lib().orc_nblist_n2, "cell": lib().orc_nblist_cell}[method]
    cap = int(cap or 128)
    while True:
        count = np.zeros(N, dtype=np.int32)
        lst = np.full((N, cap), -1, dtype=np.int32)
        mc = fn(N, _d(r), _i(types), _d(box), nt, _d(pot), float(skin), cap, _i(count), _i(lst))
        if mc < 0:
            raise ValueError("box too small for the cell search (needs >= 3 cells per axis)")
        if mc <= cap:
            return count, lst
        while cap < mc:
            cap *= 2


def forces_list(r, types, box, pot, count, lst):
    r, N, types, box, pot, nt = _prep(r, types, box, pot)
    count = _i32(count)
    lst = _i32(lst)
    cap = lst.shape[1]
    F = np.zeros((N, 3))
    u = np.zeros(N)
    w = np.zeros(N)
    lib().orc_forces_list(N, _d(r), _i(types), _d(box), nt, _d(pot), cap, _i(count), _i(lst), _d(F), _d(u), _d(w))
    return F, u, w


def needs_rebuild(r, r_build, box, skin) -> bool:
    r = _f64(r)
    rb = _f64(r_build)
    return bool(lib().orc_needs_rebuild(r.shape[0], _d(r), _d(rb), _d(_f64(box, (3,))), float(skin)))


def integrate(r, v, m, image, F, box, dt, mode=NVE, T0=1.0, tau=0.2, xi=0.0, eta=0.0):
    """One leap-frog step given F.  Returns new (r, v, image, xi, eta, K_t, sum_m_v2)."""
    r = _f64(r).copy()
    v = _f64(v).copy()
    N = r.shape[0]
    m = _f64(m, (N,))
    image = _i32(image).copy()
    F = _f64(F, (N, 3))
    th = np.array([xi, eta], dtype=np.float64)
    out = np.zeros(2)
    g = 3.0 * N - 3.0
    lib().orc_integrate(N, _d(r), _d(v), _d(m), _i(image), _d(F), _d(_f64(box, (3,))), float(dt), int(mode),
                        float(T0), float(tau), g, _d(th), _d(out))
    return r, v, image, float(th[0]), float(th[1]), float(out[0]), float(out[1])


def run(r, v, m, image, types, box, pot, skin, dt, nsteps, mode=NVE, T0=1.0, tau=0.2, xi=0.0, eta=0.0,
        use_cell=False, want_log=True):
    """nsteps of the whole path (O8 order).  Returns dict(r, v, image, xi, eta, n_builds, log) where
    log[s] = (U, K, W, xi, eta, H) at integer time t_s (before the step's update)."""
    r, N, types, box, pot, nt = _prep(r, types, box, pot)
    r = r.copy()
    v = _f64(v).copy()
    m = _f64(m, (N,))
    image = _i32(image).copy()
    th = np.array([xi, eta], dtype=np.float64)
    log = np.zeros((int(nsteps), 6)) if want_log else None
    nb = lib().orc_run(N, _d(r), _d(v), _d(m), _i(image), _i(types), _d(box), nt, _d(pot), float(skin), float(dt),
                       int(mode), float(T0), float(tau), _d(th), int(nsteps), int(bool(use_cell)),
                       _d(log) if want_log else None)
    if nb < 0:
        raise MemoryError("orc_run")
    return dict(r=r, v=v, image=image, xi=float(th[0]), eta=float(th[1]), n_builds=int(nb), log=log)


def integrate_npt(r, v, m, image, F, Wvir, box, dt, T0, tau, P0, tauP, xi=0.0, eta=0.0, nu=0.0):
    """One NPT leap-frog step (reading S32) given F and the pair virial W; nu is the strain rate as the previous step
    left it (nu_o of orc_integrate_npt).  Returns new (r, v, image, box, xi, eta, nu_o, K_t, sum_m_v2)."""
    r = _f64(r).copy()
    v = _f64(v).copy()
    N = r.shape[0]
    m = _f64(m, (N,))
    image = _i32(image).copy()
    F = _f64(F, (N, 3))
    box = _f64(box, (3,)).copy()
    st = np.array([xi, eta, nu, nu], dtype=np.float64)
    out = np.zeros(2)
    g = 3.0 * N - 3.0
    lib().orc_integrate_npt(N, _d(r), _d(v), _d(m), _i(image), _d(F), float(Wvir), _d(box), float(dt), float(T0),
                            float(tau), float(P0), float(tauP), g, _d(st), _d(out))
    return r, v, image, box, float(st[0]), float(st[1]), float(st[2]), float(out[0]), float(out[1])


def run_npt(r, v, m, image, types, box, pot, skin, dt, nsteps, T0, tau, P0, tauP, xi=0.0, eta=0.0, nu=0.0,
            use_cell=False, want_log=True):
    """nsteps of NPT dynamics.  Returns dict(r, v, image, box, xi, eta, nu, n_builds, log) with
    log[s] = (U, K, W, xi, eta, H, nu, V, P) at integer time t_s (before the step's update)."""
    r, N, types, box, pot, nt = _prep(r, types, box, pot)
    r = r.copy()
    box = box.copy()
    v = _f64(v).copy()
    m = _f64(m, (N,))
    image = _i32(image).copy()
    st = np.array([xi, eta, nu, nu], dtype=np.float64)
    log = np.zeros((int(nsteps), 9)) if want_log else None
    nb = lib().orc_run_npt(N, _d(r), _d(v), _d(m), _i(image), _i(types), _d(box), nt, _d(pot), float(skin), float(dt),
                           float(T0), float(tau), float(P0), float(tauP), _d(st), int(nsteps), int(bool(use_cell)),
                           _d(log) if want_log else None)
    if nb < 0:
        raise MemoryError("orc_run_npt")
    return dict(r=r, v=v, image=image, box=box, xi=float(st[0]), eta=float(st[1]), nu=float(st[2]), n_builds=int(nb),
                log=log)

