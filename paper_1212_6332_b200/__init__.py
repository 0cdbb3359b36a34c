"""paper_1212_6332_b200 — B200-native (sm_100a) EAM / TB-SMA molecular-dynamics hot path.

Thin Python binding of the C ABI in include/md.h (libmd_b200.so).  Argument marshalling only:
every step of the path (binning, re-ordering, neighbour list, density, force, integrator) runs in the
hand-written CUDA kernels under csrc/.  PyTorch is used for device memory (the workspace and any
device-side arrays the caller passes) and for the CUDA stream.  There is no CPU fallback: if the
library cannot be loaded, importing `lib()` raises, and on a box without a GPU `MDSystem` raises.

Method: Hou et al., arxiv 1212.6332 (eq.(1)-(3); sections 3.2-3.3, Figs. 3, 5, 6).
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from .build import LIB, build as build_library

MD_OK, MD_EINVAL, MD_EBOX, MD_EOVERFLOW, MD_ENONFINITE, MD_ECUDA, MD_ESTATE = 0, -1, -2, -3, -4, -5, -6
MD_FLAG_OVERFLOW, MD_FLAG_NONFINITE = 1, 2
MD_POT_TBSMA, MD_POT_EAM_TABLE = 0, 1
MD_OPT_STEP_OBSERVABLES, MD_OPT_PROFILE, MD_OPT_FORCE_VARIANT, MD_OPT_GRAPH, MD_OPT_HALF_LIST = 1, 2, 3, 4, 5
MD_INT_VERLET, MD_INT_GEAR5 = 0, 1
KERNEL_CLASSES = ("bin", "scan", "sort", "reorder", "list", "density", "force", "integrate", "reduce", "force_chained")

_D = C.POINTER(C.c_double)
_I = C.POINTER(C.c_int)


class MdDesc(C.Structure):
    _fields_ = [("n_atoms", C.c_int), ("n_boxes", C.c_int), ("n_types", C.c_int), ("box", C.c_double * 3),
                ("cutoff", C.c_double), ("skin", C.c_double), ("positions", C.c_void_p), ("velocities", C.c_void_p),
                ("types", C.c_void_p), ("mass", C.c_void_p), ("pot_kind", C.c_int), ("A", C.c_void_p),
                ("xi", C.c_void_p), ("p", C.c_void_p), ("q", C.c_void_p), ("r0", C.c_void_p), ("taper_on", C.c_double),
                ("nr", C.c_int), ("dr", C.c_double), ("f_val", C.c_void_p), ("f_der", C.c_void_p),
                ("phi_val", C.c_void_p), ("phi_der", C.c_void_p), ("nrho", C.c_int), ("drho", C.c_double),
                ("F_val", C.c_void_p), ("F_der", C.c_void_p), ("max_neighbors", C.c_int), ("stream", C.c_void_p),
                ("pair_cutoff", C.c_void_p), ("pair_taper_on", C.c_void_p)]


class MdStats(C.Structure):
    _fields_ = [("steps", C.c_long), ("rebuilds", C.c_long), ("max_neighbors", C.c_int), ("error_flags", C.c_int),
                ("last_max_disp2", C.c_double), ("neighbor_capacity", C.c_int), ("kernel_launches", C.c_long), ("list_entries", C.c_long),
                ("graph_active", C.c_int), ("graph_error", C.c_int)]


class MDError(RuntimeError):
    def __init__(self, code: int, text: str):
        super().__init__(f"md error {code}: {text}")
        self.code = code


_lib = None


def lib() -> C.CDLL:
    """Load libmd_b200.so (building it in-tree with nvcc if it is missing or stale).  Raises if that fails."""
    global _lib
    if _lib is None:
        path = LIB
        if not os.path.exists(path) or os.environ.get("MD_B200_REBUILD"):
            path = build_library()
        L = C.CDLL(path)
        L.md_strerror.restype = C.c_char_p
        L.md_version.restype = C.c_char_p
        L.md_kernel_name.restype = C.c_char_p
        L.md_workspace_bytes.argtypes = [C.POINTER(MdDesc), C.POINTER(C.c_size_t)]
        L.md_create.argtypes = [C.POINTER(MdDesc), C.c_void_p, C.c_size_t, C.POINTER(C.c_void_p)]
        for name in ("md_destroy", "md_build_neighbors", "md_profile_reset"):
            getattr(L, name).argtypes = [C.c_void_p]
        L.md_compute_forces.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.md_step.argtypes = [C.c_void_p, C.c_int, C.c_double]
        L.md_prepare_step.argtypes = [C.c_void_p, C.c_int, C.c_double]
        for name in ("md_get_positions", "md_get_velocities", "md_set_positions", "md_set_velocities"):
            getattr(L, name).argtypes = [C.c_void_p, C.c_void_p]
        for name in ("md_set_state", "md_get_state"):
            getattr(L, name).argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.md_step_get_state.argtypes = [C.c_void_p, C.c_int, C.c_double, C.c_void_p, C.c_void_p]
        L.md_get_neighbors.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int]
        L.md_get_densities.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.md_get_energies.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.md_get_stats.argtypes = [C.c_void_p, C.POINTER(MdStats)]
        L.md_set_option.argtypes = [C.c_void_p, C.c_int, C.c_int]
        L.md_set_integrator.argtypes = [C.c_void_p, C.c_int]
        L.md_set_thermostat.argtypes = [C.c_void_p, C.c_double, C.c_double]
        L.md_set_barostat.argtypes = [C.c_void_p, C.c_double, C.c_double]
        L.md_get_box.argtypes = [C.c_void_p, C.POINTER(C.c_double)]
        L.md_get_pressure.argtypes = [C.c_void_p, C.POINTER(C.c_double)]
        L.md_profile_read.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_long), C.POINTER(C.c_double)]
        L.md_fp64_dfma_rate.argtypes = [C.c_void_p, _D, _D]
        L.md_kinetic_energy_noalloc.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, _D, C.c_int, C.c_int, C.c_void_p,
                                                C.c_char_p, C.c_int]
        _lib = L
    return _lib


def check(rc: int):
    if rc != MD_OK:
        raise MDError(rc, lib().md_strerror(rc).decode())


def _ptr(a):
    """Raw address of a numpy array (host) or a torch tensor (host or device); None -> NULL."""
    if a is None:
        return None
    if isinstance(a, np.ndarray):
        assert a.flags["C_CONTIGUOUS"]
        return a.ctypes.data
    assert a.is_contiguous()
    return a.data_ptr()


def _host(a, dtype):
    """numpy / torch-CPU inputs become contiguous numpy of `dtype`; torch CUDA tensors pass through."""
    if a is None:
        return None
    if isinstance(a, np.ndarray) or not hasattr(a, "data_ptr"):
        return np.ascontiguousarray(a, dtype=dtype)
    return a.contiguous()


def fp64_dfma_rate():
    """(DFMA thread-instructions per second, SM clock in MHz) measured on the current device."""
    import torch
    rate, mhz = C.c_double(), C.c_double()
    check(lib().md_fp64_dfma_rate(C.c_void_p(torch.cuda.current_stream().cuda_stream), C.byref(rate), C.byref(mhz)))
    return rate.value, mhz.value


def probe_table_gather():
    """ns per warp-wide gather of 32-byte table records: (global random, shared random, global sorted, shared sorted)."""
    import torch
    out = (C.c_double * 4)()
    check(lib().md_probe_table_gather(C.c_void_p(torch.cuda.current_stream().cuda_stream), out))
    return tuple(out)


MD_NOALLOC_MAX_ATOMS = 4194304


def kinetic_energy_noalloc(v, types, mass, out):
    """E_kin (eV) of velocities `v` [n, 3] (torch CUDA float64) into `out` (torch CUDA float64, 1 element) without any
    allocation on the device: the scratch is a fixed array inside the library (n <= MD_NOALLOC_MAX_ATOMS).  `types`: torch
    CUDA int32 [n] or None for one species; `mass`: amu per type (host).  Enqueued on torch's current stream; returns `out`."""
    import torch
    assert v.is_cuda and v.dtype == torch.float64 and v.is_contiguous() and v.dim() == 2 and v.shape[1] == 3
    assert out.is_cuda and out.dtype == torch.float64 and out.numel() >= 1
    assert types is None or (types.is_cuda and types.dtype == torch.int32 and types.is_contiguous() and types.numel() == v.shape[0])
    m = (C.c_double * len(mass))(*[float(x) for x in mass])
    err = C.create_string_buffer(256)
    with torch.cuda.device(v.device):
        rc = lib().md_kinetic_energy_noalloc(C.c_void_p(torch.cuda.current_stream().cuda_stream), C.c_void_p(v.data_ptr()),
                                             C.c_void_p(types.data_ptr()) if types is not None else None, m, len(mass),
                                             int(v.shape[0]), C.c_void_p(out.data_ptr()), err, len(err))
    if rc != MD_OK:
        raise MDError(rc, err.value.decode() or lib().md_strerror(rc).decode())
    return out


class MDSystem:
    """One system on the current CUDA device.  `w` is a workloads.Workload (or pass the same fields by keyword).
    Array arguments may be numpy arrays (host) or torch CUDA tensors (device)."""

    def __init__(self, w=None, max_neighbors: int = 0, device=None, **kw):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1212_6332_b200 needs a CUDA device (no CPU fallback)")
        self._torch = torch
        self.device = torch.device(device if device is not None else f"cuda:{torch.cuda.current_device()}")
        g = (lambda k, default=None: kw.get(k, getattr(w, k, default) if w is not None else default))
        keep = []
        d = MdDesc()
        pos = _host(g("positions"), np.float64)
        self.n_atoms = d.n_atoms = int(pos.shape[0])
        self.n_boxes = d.n_boxes = int(g("n_boxes", 1))
        mass = np.ascontiguousarray(g("mass"), dtype=np.float64)
        d.n_types = int(mass.shape[0])
        d.box = (C.c_double * 3)(*[float(v) for v in g("box")])
        d.cutoff, d.skin = float(g("cutoff")), float(g("skin"))
        vel, types = _host(g("velocities"), np.float64), _host(g("types"), np.int32)
        d.positions, d.velocities, d.types, d.mass = _ptr(pos), _ptr(vel), _ptr(types), _ptr(mass)
        keep += [pos, vel, types, mass]
        d.pot_kind = int(g("pot_kind", 0))
        tb, tab = g("tbsma"), g("tables")
        if d.pot_kind == MD_POT_TBSMA:
            for k in ("A", "xi", "p", "q", "r0"):
                a = np.ascontiguousarray(np.atleast_1d(tb[k]), dtype=np.float64)
                keep.append(a)
                setattr(d, k, _ptr(a))
            d.taper_on = float(tb["taper_on"])
        else:
            d.nr, d.dr, d.nrho, d.drho = int(tab["nr"]), float(tab["dr"]), int(tab["nrho"]), float(tab["drho"])
            for k in ("f_val", "f_der", "phi_val", "phi_der", "F_val", "F_der"):
                a = _host(tab[k], np.float64)
                keep.append(a)
                setattr(d, k, _ptr(a))
        for k in ("pair_cutoff", "pair_taper_on"):                # optional per-pair cut-offs (RCUT(ity,jty))
            v = g(k)
            if v is not None:
                a = np.ascontiguousarray(v, dtype=np.float64)
                keep.append(a)
                setattr(d, k, _ptr(a))
        d.max_neighbors = int(max_neighbors)
        with torch.cuda.device(self.device):
            self.stream = torch.cuda.current_stream()
            d.stream = self.stream.cuda_stream
            nbytes = C.c_size_t()
            check(lib().md_workspace_bytes(C.byref(d), C.byref(nbytes)))
            self.workspace_bytes = nbytes.value
            self._ws = torch.empty(nbytes.value + 256, dtype=torch.uint8, device=self.device)
            if os.environ.get("MD_POISON_WORKSPACE"):            # test hook: the library must never read what it has not written
                self._ws.fill_(0xAB)
            base = (self._ws.data_ptr() + 255) & ~255
            self._h = C.c_void_p()
            check(lib().md_create(C.byref(d), C.c_void_p(base), nbytes.value, C.byref(self._h)))

    # -- lifetime
    def close(self):
        if getattr(self, "_h", None) and _lib is not None:
            _lib.md_destroy(self._h)
            self._h = None
            self._ws = None

    __del__ = close

    def _out(self, shape, dtype, device_out):
        if device_out:
            t = self._torch
            return t.empty(shape, dtype=t.float64 if dtype == np.float64 else t.int32, device=self.device)
        return np.empty(shape, dtype=dtype)

    # -- the calls of include/md.h
    def build_neighbors(self):
        check(lib().md_build_neighbors(self._h))

    def compute_forces(self, device_out: bool = False, forces=True, e_atom=True, virial=True):
        f = self._out((self.n_atoms, 3), np.float64, device_out) if forces else None
        e = self._out((self.n_atoms,), np.float64, device_out) if e_atom else None
        w = self._out((self.n_boxes, 6), np.float64, device_out) if virial else None
        check(lib().md_compute_forces(self._h, _ptr(f), _ptr(e), _ptr(w)))
        return f, e, w

    def step(self, n: int, dt: float):
        check(lib().md_step(self._h, int(n), float(dt)))

    def prepare_step(self, n: int, dt: float):
        """Build the CUDA graphs step(n, dt) will replay (set-up work, no time step)."""
        check(lib().md_prepare_step(self._h, int(n), float(dt)))

    def positions(self, device_out: bool = False, out=None):
        x = out if out is not None else self._out((self.n_atoms, 3), np.float64, device_out)
        check(lib().md_get_positions(self._h, _ptr(x)))
        return x

    def velocities(self, device_out: bool = False, out=None):
        v = out if out is not None else self._out((self.n_atoms, 3), np.float64, device_out)
        check(lib().md_get_velocities(self._h, _ptr(v)))
        return v

    def set_positions(self, x):
        x = _host(x, np.float64)
        check(lib().md_set_positions(self._h, _ptr(x)))

    def set_velocities(self, v):
        v = _host(v, np.float64)
        check(lib().md_set_velocities(self._h, _ptr(v)))

    def set_state(self, x=None, v=None):
        x, v = _host(x, np.float64), _host(v, np.float64)
        check(lib().md_set_state(self._h, _ptr(x), _ptr(v)))

    def get_state(self, device_out: bool = False, out=None):
        x, v = out if out is not None else (self._out((self.n_atoms, 3), np.float64, device_out),
                                            self._out((self.n_atoms, 3), np.float64, device_out))
        check(lib().md_get_state(self._h, _ptr(x), _ptr(v)))
        return x, v

    def step_get_state(self, n: int, dt: float, device_out: bool = False, out=None):
        x, v = out if out is not None else (self._out((self.n_atoms, 3), np.float64, device_out),
                                            self._out((self.n_atoms, 3), np.float64, device_out))
        check(lib().md_step_get_state(self._h, int(n), float(dt), _ptr(x), _ptr(v)))
        return x, v

    def neighbors(self, stride: int = 256, device_out: bool = False):
        cnt = self._out((self.n_atoms,), np.int32, device_out)
        lst = self._out((self.n_atoms, stride), np.int32, device_out)
        if device_out:
            lst.fill_(-1)
        else:
            lst.fill(-1)
        check(lib().md_get_neighbors(self._h, _ptr(cnt), _ptr(lst), int(stride)))
        return cnt, lst

    def densities(self, device_out: bool = False):
        rho = self._out((self.n_atoms,), np.float64, device_out)
        fp = self._out((self.n_atoms,), np.float64, device_out)
        check(lib().md_get_densities(self._h, _ptr(rho), _ptr(fp)))
        return rho, fp

    def energies(self, out=None):
        ep, ek = out if out is not None else (np.empty(self.n_boxes), np.empty(self.n_boxes))
        check(lib().md_get_energies(self._h, _ptr(ep), _ptr(ek)))
        return ep, ek

    def stats(self) -> dict:
        st = MdStats()
        check(lib().md_get_stats(self._h, C.byref(st)))
        return {k: getattr(st, k) for k, _ in MdStats._fields_}

    def set_integrator(self, integrator: int):
        """MD_INT_VERLET (default) or MD_INT_GEAR5, the paper's predictor-corrector scheme."""
        check(lib().md_set_integrator(self._h, int(integrator)))

    def set_thermostat(self, T_e: float, tau: float):
        """eq.(4) electron-bath thermostat (K, fs); tau <= 0 switches it off."""
        check(lib().md_set_thermostat(self._h, float(T_e), float(tau)))

    def set_barostat(self, P0: float, tau_p: float):
        """eq.(5)-(6) Berendsen barostat (eV/A^3, fs eV/A^3); tau_p <= 0 switches it off."""
        check(lib().md_set_barostat(self._h, float(P0), float(tau_p)))

    def box(self):
        b = (C.c_double * 3)()
        check(lib().md_get_box(self._h, b))
        return np.array(list(b))

    def pressure(self) -> float:
        p = C.c_double()
        check(lib().md_get_pressure(self._h, C.byref(p)))
        return p.value

    def set_option(self, option: int, value: int):
        check(lib().md_set_option(self._h, int(option), int(value)))

    def profile_reset(self):
        check(lib().md_profile_reset(self._h))

    def profile(self) -> dict:
        """{kernel class: (launches, total ms)} since the last reset (needs MD_OPT_PROFILE)."""
        out = {}
        for k, name in enumerate(KERNEL_CLASSES):
            n, ms = C.c_long(), C.c_double()
            check(lib().md_profile_read(self._h, k, C.byref(n), C.byref(ms)))
            out[name] = (n.value, ms.value)
        return out
