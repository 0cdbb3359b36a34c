"""ctypes binding of the CPU oracle (oracle/eam_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and the
cpu_baseline / --impl reference legs of bench.py import this package.  It imports nothing
from paper_1212_6332_b200 and that package imports nothing from here.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from .build import build as build_library

_D = C.POINTER(C.c_double)
_I = C.POINTER(C.c_int)


class _Desc(C.Structure):
    _fields_ = [("n_atoms", C.c_int), ("n_boxes", C.c_int), ("n_types", C.c_int), ("box", C.c_double * 3),
                ("cutoff", C.c_double), ("skin", C.c_double), ("positions", _D), ("velocities", _D), ("types", _I),
                ("mass", _D), ("pot_kind", C.c_int), ("A", _D), ("xi", _D), ("p", _D), ("q", _D), ("r0", _D),
                ("taper_on", C.c_double), ("nr", C.c_int), ("dr", C.c_double), ("f_val", _D), ("f_der", _D),
                ("phi_val", _D), ("phi_der", _D), ("nrho", C.c_int), ("drho", C.c_double), ("F_val", _D),
                ("F_der", _D), ("max_neighbors", C.c_int), ("pair_cutoff", _D), ("pair_taper_on", _D)]


class _Stats(C.Structure):
    _fields_ = [("steps", C.c_long), ("rebuilds", C.c_long), ("max_neighbors", C.c_int), ("error_flags", C.c_int),
                ("last_max_disp2", C.c_double)]


class OracleError(RuntimeError):
    def __init__(self, code: int, text: str):
        super().__init__(f"oracle error {code}: {text}")
        self.code = code


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build_library())
        _lib.oracle_strerror.restype = C.c_char_p
        _lib.oracle_hermite_eval.argtypes = [_D, _D, C.c_int, C.c_double, C.c_double, _D, _D]
        _lib.oracle_tbsma_eval.argtypes = [C.c_double] * 8 + [_D]
        _lib.oracle_min_image.argtypes = [_D, _D, _D, _D, _D]
        _lib.oracle_step.argtypes = [C.c_void_p, C.c_int, C.c_double]
        _lib.oracle_set_thermostat.argtypes = [C.c_void_p, C.c_double, C.c_double]
        _lib.oracle_set_integrator.argtypes = [C.c_void_p, C.c_int]
        _lib.oracle_set_barostat.argtypes = [C.c_void_p, C.c_double, C.c_double]
        _lib.oracle_get_box.argtypes = [C.c_void_p, _D]
        _lib.oracle_get_pressure.argtypes = [C.c_void_p, _D]
    return _lib


def _dp(a):
    return None if a is None else a.ctypes.data_as(_D)


def _f64(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float64)


def set_threads(n: int) -> int:
    return int(lib().oracle_set_threads(C.c_int(n)))


def tbsma_eval(r, A, xi, p, q, r0, r_on, r_c):
    """(f, f', V, V', S, S') of the TB-SMA radial functions at distance r."""
    out = np.zeros(6)
    lib().oracle_tbsma_eval(r, A, xi, p, q, r0, r_on, r_c, _dp(out))
    return out


def hermite_eval(val, der, h, x):
    val, der = _f64(val), _f64(der)
    H, dH = C.c_double(), C.c_double()
    lib().oracle_hermite_eval(_dp(val), _dp(der), len(val), h, x, C.byref(H), C.byref(dH))
    return H.value, dH.value


def min_image(xi, xj, box):
    xi, xj, box = _f64(xi), _f64(xj), _f64(box)
    d, r2 = np.zeros(3), C.c_double()
    lib().oracle_min_image(_dp(xi), _dp(xj), _dp(box), _dp(d), C.byref(r2))
    return d, r2.value


class Oracle:
    """One oracle system built from a `workloads.Workload` (or the same fields given by keyword)."""

    def __init__(self, w=None, max_neighbors: int = 0, **kw):
        g = (lambda k, default=None: kw.get(k, getattr(w, k, default) if w is not None else default))
        self._keep = []
        d = _Desc()
        pos = _f64(g("positions"))
        self.n_atoms = d.n_atoms = int(pos.shape[0])
        self.n_boxes = d.n_boxes = int(g("n_boxes", 1))
        mass = _f64(g("mass"))
        d.n_types = int(mass.shape[0])
        d.box = (C.c_double * 3)(*[float(v) for v in g("box")])
        d.cutoff, d.skin = float(g("cutoff")), float(g("skin"))
        vel = _f64(g("velocities"))
        types = np.ascontiguousarray(g("types"), dtype=np.int32)
        d.positions, d.velocities, d.mass = _dp(pos), _dp(vel), _dp(mass)
        d.types = types.ctypes.data_as(_I)
        d.pot_kind = int(g("pot_kind", 0))
        self._keep += [pos, vel, types, mass]
        tb, tab = g("tbsma"), g("tables")
        if d.pot_kind == 0:
            for k in ("A", "xi", "p", "q", "r0"):
                a = _f64(np.atleast_1d(tb[k]))
                self._keep.append(a)
                setattr(d, k, _dp(a))
            d.taper_on = float(tb["taper_on"])
        else:
            d.nr, d.dr, d.nrho, d.drho = int(tab["nr"]), float(tab["dr"]), int(tab["nrho"]), float(tab["drho"])
            for k in ("f_val", "f_der", "phi_val", "phi_der", "F_val", "F_der"):
                a = _f64(tab[k])
                self._keep.append(a)
                setattr(d, k, _dp(a))
        for k in ("pair_cutoff", "pair_taper_on"):
            v = g(k)
            if v is not None:
                a = _f64(v)
                self._keep.append(a)
                setattr(d, k, _dp(a))
        d.max_neighbors = int(max_neighbors)
        self._h = C.c_void_p()
        self._check(lib().oracle_create(C.byref(d), C.byref(self._h)))

    def _check(self, rc):
        if rc != 0:
            raise OracleError(rc, lib().oracle_strerror(rc).decode())

    def close(self):
        if getattr(self, "_h", None):
            lib().oracle_destroy(self._h)
            self._h = None

    __del__ = close

    def build_neighbors(self, brute_force: bool = False):
        self._check(lib().oracle_build_neighbors(self._h, 1 if brute_force else 0))

    def compute_forces(self):
        """-> (forces (N,3), e_atom (N,), virial (n_boxes,6))"""
        f, e, w = np.zeros((self.n_atoms, 3)), np.zeros(self.n_atoms), np.zeros((self.n_boxes, 6))
        self._check(lib().oracle_compute_forces(self._h, _dp(f), _dp(e), _dp(w)))
        return f, e, w

    def step(self, n: int, dt: float):
        self._check(lib().oracle_step(self._h, int(n), float(dt)))

    def set_integrator(self, kind: int):
        """0: velocity-Verlet (default); 1: five-value Gear predictor-corrector."""
        self._check(lib().oracle_set_integrator(self._h, int(kind)))

    def set_thermostat(self, T_e: float, tau: float):
        """eq.(4): electron-bath thermostat (K, fs); tau <= 0 switches it off."""
        self._check(lib().oracle_set_thermostat(self._h, float(T_e), float(tau)))

    def set_barostat(self, P0: float, tau_p: float):
        """eq.(5)-(6): Berendsen barostat (eV/A^3, fs eV/A^3); tau_p <= 0 switches it off."""
        self._check(lib().oracle_set_barostat(self._h, float(P0), float(tau_p)))

    def box(self):
        b = np.zeros(3)
        self._check(lib().oracle_get_box(self._h, _dp(b)))
        return b

    def pressure(self) -> float:
        p = C.c_double()
        self._check(lib().oracle_get_pressure(self._h, C.byref(p)))
        return p.value

    def positions(self):
        x = np.zeros((self.n_atoms, 3))
        self._check(lib().oracle_get_positions(self._h, _dp(x)))
        return x

    def velocities(self):
        v = np.zeros((self.n_atoms, 3))
        self._check(lib().oracle_get_velocities(self._h, _dp(v)))
        return v

    def set_positions(self, x):
        x = _f64(x)
        self._check(lib().oracle_set_positions(self._h, _dp(x)))

    def set_velocities(self, v):
        v = _f64(v)
        self._check(lib().oracle_set_velocities(self._h, _dp(v)))

    def neighbors(self, stride: int = 256):
        """-> (count (N,), list (N,stride)) with ascending original ids per atom"""
        cnt = np.zeros(self.n_atoms, dtype=np.int32)
        lst = np.full((self.n_atoms, stride), -1, dtype=np.int32)
        self._check(lib().oracle_get_neighbors(self._h, cnt.ctypes.data_as(_I), lst.ctypes.data_as(_I), stride))
        return cnt, lst

    def densities(self):
        rho, fp = np.zeros(self.n_atoms), np.zeros(self.n_atoms)
        self._check(lib().oracle_get_densities(self._h, _dp(rho), _dp(fp)))
        return rho, fp

    def energies(self):
        ep, ek = np.zeros(self.n_boxes), np.zeros(self.n_boxes)
        self._check(lib().oracle_get_energies(self._h, _dp(ep), _dp(ek)))
        return ep, ek

    def stats(self) -> dict:
        st = _Stats()
        self._check(lib().oracle_get_stats(self._h, C.byref(st)))
        return {k: getattr(st, k) for k, _ in _Stats._fields_}

    def list_covers_cutoff(self) -> bool:
        rc = lib().oracle_list_covers_cutoff(self._h)
        if rc < 0:
            self._check(rc)
        return bool(rc)
