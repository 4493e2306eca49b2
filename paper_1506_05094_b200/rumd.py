"""ctypes binding of librumd_b200.so (include/rumd_b200.h) -- argument marshalling only.

Every step of the path runs in the library's CUDA kernels; PyTorch is used for device memory and the
stream.  There is no CPU fallback: if the library is missing or no CUDA device is present, this fails loudly.
Names follow the C ABI: ``System.set_pair_potential`` -> ``rumd_set_pair_potential`` and so on.
"""
from __future__ import annotations

import ctypes as C
import math
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIBPATH = os.path.join(_HERE, "librumd_b200.so")

OK, ERR_INVALID_ARG, ERR_NOT_READY, ERR_CUDA, ERR_NBL_OVERFLOW, ERR_BOX_TOO_SMALL, ERR_NONFINITE = range(7)
POT_LJ_12_6, POT_COULOMB, POT_IPL, POT_YUKAWA, POT_GAUSSIAN_CORE, POT_BUCKINGHAM = range(6)
POT_GEN_LJ, POT_GIRIFALCO, POT_DZUGUTOV = 6, 7, 8
_SECOND_NPARAMS = (1, 2, 2, 2, 3, 4, 3, 2)  # of (a, b, c, d), by kind - 1; rcut follows
CUT_SHIFTED_FORCE, CUT_SHIFTED_POTENTIAL, CUT_NONE = 0, 1, 2
INT_NVE_LEAPFROG, INT_NVT_NOSE_HOOVER, INT_NPT_MTK = 0, 1, 2
NB_N2, NB_CELL, NB_NONE, NB_TILE = 0, 1, 2, 3

EXPORTS = [
    "rumd_create", "rumd_destroy", "rumd_bind_state", "rumd_workspace_bytes", "rumd_bind_workspace",
    "rumd_set_pair_potential", "rumd_set_integrator", "rumd_set_barostat", "rumd_get_box", "rumd_default_tuning", "rumd_set_tuning",
    "rumd_get_tuning", "rumd_autotune", "rumd_autotune_cached", "rumd_build_nblist", "rumd_compute_forces", "rumd_run_steps",
    "rumd_export_nblist", "rumd_get_thermo", "rumd_snapshot", "rumd_restore", "rumd_upload_state",
    "rumd_download_state", "rumd_launch_count", "rumd_profile_step", "rumd_time_force", "rumd_profile_persistent", "rumd_measure_fp32_peak", "rumd_set_replicas", "rumd_get_thermo_replicas", "rumd_forces_noalloc", "rumd_last_error", "rumd_version",
]
NOALLOC_MAX_PARTICLES, NOALLOC_NBL_CAPACITY = 8192, 256


class Tuning(C.Structure):
    _fields_ = [("method", C.c_int), ("pb", C.c_int), ("tp", C.c_int), ("skin", C.c_float),
                ("sort_interval", C.c_int), ("use_graph", C.c_int), ("steps_per_graph", C.c_int),
                ("persistent", C.c_int), ("build_tp", C.c_int), ("tile", C.c_int)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


class Thermo(C.Structure):
    _fields_ = [("U", C.c_double), ("W", C.c_double), ("K", C.c_double), ("mv2", C.c_double),
                ("xi", C.c_double), ("eta", C.c_double), ("H", C.c_double), ("n_steps", C.c_longlong),
                ("n_rebuilds", C.c_longlong), ("max_nbrs", C.c_int), ("nbl_capacity", C.c_int),
                ("overflow", C.c_int), ("pad_", C.c_int)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_ if k != "pad_"}


class NoallocPair(C.Structure):
    _fields_ = [("epsilon", C.c_float), ("sigma", C.c_float), ("rcut", C.c_float), ("kqq", C.c_float),
                ("rcut_coulomb", C.c_float)]


class RumdError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__("rumd status %d: %s" % (status, msg))
        self.status = status


_lib = None


def lib():
    """Load librumd_b200.so (must have been built: ``python -m paper_1506_05094_b200.build``)."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIBPATH):
            raise RuntimeError("librumd_b200.so is missing (%s): build it with "
                               "`python -m paper_1506_05094_b200.build`; there is no CPU fallback" % _LIBPATH)
        L = C.CDLL(_LIBPATH)
        vp, ip = C.c_void_p, C.c_int
        L.rumd_create.argtypes = [C.POINTER(vp), ip, ip, C.POINTER(C.c_float), vp]
        L.rumd_destroy.argtypes = [vp]
        L.rumd_bind_state.argtypes = [vp] * 7
        L.rumd_workspace_bytes.argtypes = [vp, ip]
        L.rumd_workspace_bytes.restype = C.c_size_t
        L.rumd_bind_workspace.argtypes = [vp, vp, C.c_size_t, ip]
        L.rumd_set_pair_potential.argtypes = [vp, ip, ip, ip, ip, C.POINTER(C.c_float), ip]
        L.rumd_set_integrator.argtypes = [vp, ip, C.c_float, C.c_float, C.c_float]
        L.rumd_set_barostat.argtypes = [vp, C.c_float, C.c_float]
        L.rumd_get_box.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.rumd_default_tuning.argtypes = [vp, C.POINTER(Tuning)]
        L.rumd_set_tuning.argtypes = [vp, C.POINTER(Tuning)]
        L.rumd_get_tuning.argtypes = [vp, C.POINTER(Tuning)]
        L.rumd_autotune.argtypes = [vp, C.POINTER(Tuning), ip, C.POINTER(C.c_double)]
        L.rumd_autotune_cached.argtypes = [vp, C.POINTER(Tuning), ip, C.POINTER(C.c_double), C.c_char_p, C.POINTER(ip)]
        L.rumd_build_nblist.argtypes = [vp]
        L.rumd_compute_forces.argtypes = [vp]
        L.rumd_run_steps.argtypes = [vp, C.c_long]
        L.rumd_export_nblist.argtypes = [vp, vp, vp, ip]
        L.rumd_get_thermo.argtypes = [vp, C.POINTER(Thermo)]
        L.rumd_snapshot.argtypes = [vp]
        L.rumd_restore.argtypes = [vp]
        L.rumd_upload_state.argtypes = [vp] * 5
        L.rumd_download_state.argtypes = [vp] * 7
        L.rumd_launch_count.argtypes = [vp]
        L.rumd_launch_count.restype = C.c_longlong
        L.rumd_profile_step.argtypes = [vp, C.POINTER(C.c_float), C.POINTER(ip)]
        L.rumd_time_force.argtypes = [vp, ip, C.POINTER(C.c_float)]
        L.rumd_profile_persistent.argtypes = [vp, ip, C.POINTER(C.c_double)]
        L.rumd_measure_fp32_peak.argtypes = [vp, ip, C.POINTER(C.c_double)]
        L.rumd_set_replicas.argtypes = [vp, ip]
        L.rumd_get_thermo_replicas.argtypes = [vp, C.POINTER(Thermo), ip]
        L.rumd_forces_noalloc.argtypes = [ip, ip, C.POINTER(C.c_float), C.POINTER(NoallocPair), C.c_float, vp, vp, vp, vp,
                                          vp, C.c_char_p, C.c_size_t]
        L.rumd_last_error.argtypes = [vp]
        L.rumd_last_error.restype = C.c_char_p
        L.rumd_version.restype = C.c_char_p
        _lib = L
    return _lib


def estimate_capacity(density: float, rc_max: float, skin: float) -> int:
    """List capacity per particle: 1.5 x the mean count at this density + 32, rounded up to 32."""
    mean = 4.0 / 3.0 * math.pi * (rc_max + skin) ** 3 * density
    return int(math.ceil((1.5 * mean + 32) / 32.0)) * 32


class System:
    """One simulation (Fig. 1), or a batched ensemble of R independent replicas of it when ``r`` and
    ``v`` have shape (R, N, 3) (``rumd_set_replicas``): ``types`` and ``m`` may then be (N,) (shared) or
    (R, N).  Owns torch tensors for the state and the workspace and hands their device pointers to the library."""

    def __init__(self, r, v, m, types, box, pot, device="cuda:0", skin_for_capacity=0.5, capacity=None,
                 stream=None):
        if not torch.cuda.is_available():
            raise RuntimeError("no CUDA device: librumd_b200 has no CPU fallback")
        self.L = lib()
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        r = np.ascontiguousarray(r, dtype=np.float32)
        self.replicas = int(r.shape[0]) if r.ndim == 3 else 1
        R = self.replicas
        self.N = int(r.shape[-2])       # particles of ONE system
        if r.ndim == 3:
            v = np.ascontiguousarray(v, dtype=np.float32).reshape(R * self.N, 3)
            types = np.broadcast_to(np.asarray(types, dtype=np.int32), (R, self.N)).reshape(-1).copy()
            m = np.broadcast_to(np.asarray(m, dtype=np.float32), (R, self.N)).reshape(-1).copy()
            r = r.reshape(R * self.N, 3)
        N = r.shape[0]                  # elements of the state arrays
        self.ntypes = int(pot.shape[0])
        types = np.ascontiguousarray(types, dtype=np.int32)
        if types.shape != (N,) or types.min() < 0 or types.max() >= self.ntypes:
            # the type indexes the pair table inside every kernel: reject a bad one here, where it is cheap
            raise RumdError(ERR_INVALID_ARG, "particle types must be %d integers in [0, %d)" % (N, self.ntypes))
        self.box = np.ascontiguousarray(box, dtype=np.float32)
        # a dedicated side stream (the legacy default stream cannot be captured into CUDA graphs)
        self.stream = stream if stream is not None else torch.cuda.Stream(self.device)
        h = C.c_void_p()
        st = self.L.rumd_create(C.byref(h), self.N, self.ntypes, self.box.ctypes.data_as(C.POINTER(C.c_float)),
                                C.c_void_p(self.stream.cuda_stream))
        if st != OK:
            raise RumdError(st, "rumd_create failed")
        self.h = h
        if R > 1:
            self._check(self.L.rumd_set_replicas(self.h, R))
        # host staging (pinned) in the ABI layouts
        self.h_r = torch.zeros((N, 4), dtype=torch.float32).pin_memory()
        self.h_v = torch.zeros((N, 4), dtype=torch.float32).pin_memory()
        self.h_image = torch.zeros((N, 4), dtype=torch.int32).pin_memory()
        self.h_id = (torch.arange(N, dtype=torch.int32) % self.N).contiguous().pin_memory()
        self.h_r[:, :3] = torch.from_numpy(r)
        self.h_r[:, 3] = torch.from_numpy(np.ascontiguousarray(types, dtype=np.int32)).view(torch.float32)
        self.h_v[:, :3] = torch.from_numpy(np.ascontiguousarray(v, dtype=np.float32))
        self.h_v[:, 3] = torch.from_numpy(np.ascontiguousarray(m, dtype=np.float32))
        dev = self.device
        self.d_r = self.h_r.to(dev)
        self.d_v = self.h_v.to(dev)
        self.d_f = torch.zeros((N, 4), dtype=torch.float32, device=dev)
        self.d_w = torch.zeros((N,), dtype=torch.float32, device=dev)
        self.d_image = self.h_image.to(dev)
        self.d_id = self.h_id.to(dev)
        self._check(self.L.rumd_bind_state(self.h, *[C.c_void_p(t.data_ptr()) for t in
                                                    (self.d_r, self.d_v, self.d_f, self.d_w, self.d_image,
                                                     self.d_id)]))
        # potentials (P:49-50 SetParams); pot records are (eps, sigma, rc_LJ, k qa qb, rc_Coulomb, cut_LJ, cut_C)
        pot = np.asarray(pot, dtype=np.float64)
        for a in range(self.ntypes):
            for b in range(a, self.ntypes):
                e, sg, rcl, qq, rcc = pot[a, b, :5]
                cut_lj, cut_c = (int(pot[a, b, 5]), int(pot[a, b, 6])) if pot.shape[-1] >= 7 else (0, 0)
                if rcl > 0:
                    self.set_pair_potential(a, b, POT_LJ_12_6, [e, sg, rcl], cut_lj)
                if rcc > 0:
                    kind2 = int(pot[a, b, 7]) if pot.shape[-1] >= 10 else 0
                    pb, pc = (pot[a, b, 8], pot[a, b, 9]) if pot.shape[-1] >= 10 else (0.0, 0.0)
                    pd = pot[a, b, 10] if pot.shape[-1] >= 11 else 0.0
                    params = [qq, pb, pc, pd][:_SECOND_NPARAMS[kind2]] + [rcc]
                    self.set_pair_potential(a, b, POT_COULOMB + kind2, params, cut_c)
        self.rc_max = float(max(pot[..., 2].max(), pot[..., 4].max()))
        self.density = self.N / float(np.prod(self.box.astype(np.float64)))
        if capacity is None:
            capacity = estimate_capacity(self.density, self.rc_max, skin_for_capacity)
        self.d_ws = None
        self.bind_workspace(capacity)
        torch.cuda.synchronize(self.device)  # the tensors above were filled on torch's current stream

    # ---- helpers
    def _check(self, st):
        if st != OK:
            raise RumdError(st, self.L.rumd_last_error(self.h).decode())

    def close(self):
        if getattr(self, "h", None):
            self.L.rumd_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- the C ABI, same names
    def bind_workspace(self, capacity: int):
        capacity = min(int(capacity), ((self.N + 31) // 32) * 32)
        nbytes = int(self.L.rumd_workspace_bytes(self.h, capacity))
        ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        off = (-ws.data_ptr()) % 256
        self._check(self.L.rumd_bind_workspace(self.h, C.c_void_p(ws.data_ptr() + off), nbytes, capacity))
        self.d_ws = ws  # keep the new one alive, drop the old one only now
        self.capacity = capacity

    def set_pair_potential(self, ti, tj, kind, params, cutoff=CUT_SHIFTED_FORCE):
        arr = (C.c_float * len(params))(*[float(x) for x in params])
        self._check(self.L.rumd_set_pair_potential(self.h, ti, tj, kind, int(cutoff), arr, len(params)))

    def set_integrator(self, kind, dt, T0=1.0, tau=0.2):
        self._check(self.L.rumd_set_integrator(self.h, int(kind), float(dt), float(T0), float(tau)))

    def set_barostat(self, P0, tauP):
        self._check(self.L.rumd_set_barostat(self.h, float(P0), float(tauP)))

    def get_box(self):
        """-> (box lengths (3,) float64, strain rate): the current box of an NPT run."""
        box = (C.c_double * 3)()
        nu = C.c_double()
        self._check(self.L.rumd_get_box(self.h, box, C.byref(nu)))
        return np.array(list(box)), float(nu.value)

    def default_tuning(self) -> Tuning:
        t = Tuning()
        self._check(self.L.rumd_default_tuning(self.h, C.byref(t)))
        return t

    def get_tuning(self) -> Tuning:
        t = Tuning()
        self._check(self.L.rumd_get_tuning(self.h, C.byref(t)))
        return t

    def set_tuning(self, t: Tuning = None, **kw):
        if t is None:
            t = self.get_tuning()
        for k, val in kw.items():
            setattr(t, k, val)
        self._check(self.L.rumd_set_tuning(self.h, C.byref(t)))
        return t

    def autotune(self, steps_per_trial=200, cache_path=None):
        """-> (Tuning, timesteps/s).  With cache_path the paper's parameter file is consulted first and
        appended to after a tuning run; ``self.tuning_from_cache`` tells which happened."""
        t = Tuning()
        tps = C.c_double()
        hit = C.c_int(0)
        if cache_path:
            self._check(self.L.rumd_autotune_cached(self.h, C.byref(t), int(steps_per_trial), C.byref(tps),
                                                   os.fsencode(cache_path), C.byref(hit)))
        else:
            self._check(self.L.rumd_autotune(self.h, C.byref(t), int(steps_per_trial), C.byref(tps)))
        self.tuning_from_cache = bool(hit.value)
        return t, tps.value

    def build_nblist(self):
        self._check(self.L.rumd_build_nblist(self.h))

    def compute_forces(self):
        self._check(self.L.rumd_compute_forces(self.h))

    def run_steps(self, n: int):
        self._check(self.L.rumd_run_steps(self.h, int(n)))

    def get_thermo(self, grow=False) -> dict:
        th = Thermo()
        st = self.L.rumd_get_thermo(self.h, C.byref(th))
        if st == ERR_NBL_OVERFLOW and grow:
            # "automatically re-allocated with doubled capacity"
            self.bind_workspace(max(2 * self.capacity, th.max_nbrs + 32))
            return None
        self._check(st)
        return th.as_dict()

    def get_thermo_replicas(self) -> list:
        arr = (Thermo * self.replicas)()
        self._check(self.L.rumd_get_thermo_replicas(self.h, arr, self.replicas))
        return [t.as_dict() for t in arr]

    def snapshot(self):
        self._check(self.L.rumd_snapshot(self.h))

    def restore(self):
        self._check(self.L.rumd_restore(self.h))

    def export_nblist(self):
        """-> (count (N,), list (N, capacity)) int32 numpy arrays in SLOT numbering."""
        cnt = torch.empty((self.N,), dtype=torch.int32, device=self.device)
        lst = torch.empty((self.N, self.capacity), dtype=torch.int32, device=self.device)
        self._check(self.L.rumd_export_nblist(self.h, C.c_void_p(cnt.data_ptr()), C.c_void_p(lst.data_ptr()),
                                              self.capacity))
        self.stream.synchronize()
        return cnt.cpu().numpy(), lst.cpu().numpy()

    def upload_state(self):
        """Host (pinned) -> device through the ABI's host-buffer entry point."""
        self._check(self.L.rumd_upload_state(self.h, C.c_void_p(self.h_r.data_ptr()), C.c_void_p(self.h_v.data_ptr()),
                                             C.c_void_p(self.h_image.data_ptr()), C.c_void_p(self.h_id.data_ptr())))

    def download_state(self, h_r=None, h_v=None, h_f=None, h_w=None, h_image=None, h_id=None):
        ptr = lambda t: C.c_void_p(t.data_ptr()) if t is not None else None
        self._check(self.L.rumd_download_state(self.h, ptr(h_r), ptr(h_v), ptr(h_f), ptr(h_w), ptr(h_image),
                                               ptr(h_id)))

    def launch_count(self) -> int:
        return int(self.L.rumd_launch_count(self.h))

    def profile_step(self):
        ms = (C.c_float * 4)()
        did = C.c_int()
        self._check(self.L.rumd_profile_step(self.h, ms, C.byref(did)))
        return dict(build_ms=ms[0], force_ms=ms[1], integrate_ms=ms[2], did_rebuild=bool(did.value))

    def time_force(self, reps=100) -> float:
        """Average device time of one force-kernel launch, microseconds."""
        us = C.c_float()
        self._check(self.L.rumd_time_force(self.h, int(reps), C.byref(us)))
        return float(us.value)

    def measure_fp32_peak(self, reps=5) -> float:
        """Measured FP32 FFMA throughput of this GPU, TFLOP/s."""
        out = C.c_double()
        self._check(self.L.rumd_measure_fp32_peak(self.h, int(reps), C.byref(out)))
        return float(out.value)

    def profile_persistent(self, nsteps=1000) -> dict:
        out = (C.c_double * 8)()
        self._check(self.L.rumd_profile_persistent(self.h, int(nsteps), out))
        keys = ("rebuild_us", "force_integrate_us", "sort_us", "barrier_us", "post_us", "step_us")
        d = {k: out[q] for q, k in enumerate(keys)}
        d["rebuilds"] = int(out[6])
        d["grid"] = int(out[7])
        return d

    # ---- convenience read-back (numpy, ORIGINAL particle numbering via d_id)
    def state(self) -> dict:
        self.stream.synchronize()
        if self.replicas > 1:   # no sorting in ensembles: slots are original indices
            R, n = self.replicas, self.N
            r = self.d_r.cpu().numpy().reshape(R, n, 4)
            v = self.d_v.cpu().numpy().reshape(R, n, 4)
            f = self.d_f.cpu().numpy().reshape(R, n, 4)
            return dict(r=r[..., :3].copy(), types=r[..., 3].copy().view(np.int32), v=v[..., :3].copy(),
                        m=v[..., 3].copy(), F=f[..., :3].copy(), u=f[..., 3].copy(),
                        w=self.d_w.cpu().numpy().reshape(R, n), image=self.d_image.cpu().numpy().reshape(R, n, 4)[..., :3].copy())
        ids = self.d_id.cpu().numpy().astype(np.int64)
        inv = np.empty_like(ids)
        inv[ids] = np.arange(self.N)
        r = self.d_r.cpu().numpy()[inv]
        v = self.d_v.cpu().numpy()[inv]
        f = self.d_f.cpu().numpy()[inv]
        w = self.d_w.cpu().numpy()[inv]
        im = self.d_image.cpu().numpy()[inv]
        return dict(r=r[:, :3].copy(), types=r[:, 3].copy().view(np.int32), v=v[:, :3].copy(), m=v[:, 3].copy(),
                    F=f[:, :3].copy(), u=f[:, 3].copy(), w=w, image=im[:, :3].copy(), ids=ids)


def forces_noalloc(n_types, box, pot, skin, d_r, d_f, d_w, d_out4, stream=None):
    """``rumd_forces_noalloc``: forces, u_i, w_i and {U, W, longest row, overflow} of the configuration in the device
    tensor ``d_r`` ((n, 4) float32: x, y, z, type bits) into the caller's device tensors ``d_f`` (n, 4), ``d_w`` (n,)
    and ``d_out4`` (4 doubles), using only the library's static scratch -- no handle, no allocation, asynchronous on
    ``stream`` (a torch stream; None = torch's current stream).  ``pot``: (nt, nt, >= 5) records (eps, sigma, rc_LJ,
    k qa qb, rc_Coulomb) as in ``workloads``.  n <= NOALLOC_MAX_PARTICLES.  Argument marshalling only."""
    for t, dt in ((d_r, torch.float32), (d_f, torch.float32), (d_w, torch.float32), (d_out4, torch.float64)):
        if not (t.is_cuda and t.is_contiguous() and t.dtype == dt):
            raise RumdError(ERR_INVALID_ARG, "forces_noalloc takes contiguous CUDA tensors (float32; d_out4 float64)")
    n = int(d_r.shape[0])
    if tuple(d_r.shape) != (n, 4) or tuple(d_f.shape) != (n, 4) or d_w.numel() != n or d_out4.numel() != 4:
        raise RumdError(ERR_INVALID_ARG, "forces_noalloc: d_r, d_f are (n, 4), d_w (n,), d_out4 (4,)")
    pot = np.asarray(pot, dtype=np.float64)
    pairs = (NoallocPair * (n_types * n_types))()
    for a in range(n_types):
        for b in range(n_types):
            pairs[a * n_types + b] = NoallocPair(*[float(x) for x in pot[a, b, :5]])
    boxf = np.ascontiguousarray(box, dtype=np.float32)
    if stream is None:
        stream = torch.cuda.current_stream(d_r.device)
    err = C.create_string_buffer(512)
    with torch.cuda.device(d_r.device):
        st = lib().rumd_forces_noalloc(n, int(n_types), boxf.ctypes.data_as(C.POINTER(C.c_float)), pairs, float(skin),
                                       C.c_void_p(d_r.data_ptr()), C.c_void_p(d_f.data_ptr()),
                                       C.c_void_p(d_w.data_ptr()), C.c_void_p(d_out4.data_ptr()),
                                       C.c_void_p(stream.cuda_stream), err, len(err))
    if st != OK:
        raise RumdError(st, err.value.decode())


def from_workload(wl, **kw) -> System:
    """Create a System from a ``workloads.Workload`` and set its integrator and skin."""
    s = System(wl.r, wl.v, wl.m, wl.types, wl.box, wl.pot, **kw)
    s.set_integrator(wl.integrator, wl.dt, wl.T0, wl.tau)
    s.set_tuning(skin=float(wl.skin))
    return s
