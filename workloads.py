"""Seeded synthetic inputs for the EAM / TB-SMA hot path (shared by tests, bench and smoke).

This module holds NO arithmetic of the method (no distances, densities, forces,
integrator): it only emits the *inputs* — crystal sites, thermal jitter, Maxwell-Boltzmann
velocities, a primary knock-on atom, potential parameters and the node data of the
look-up tables — as plain numpy arrays that are handed identically to the CPU oracle
(`oracle/`) and to the CUDA library (`paper_1212_6332_b200/`).  Neither of those two
imports the other; both may be fed from here.

The inputs stand in for the paper's own workloads, which are perfect bcc-W crystals of
2*n^3 atoms, 2000 ... 2 000 000 (section 4) and 100 small boxes of 2000 atoms
run as one system (section 4.4).  The paper's W potential (Ackland-Thetford,
PAPER.md:173) is not printed in the paper, so BASELINE.json's `configs` name synthetic
stand-ins: Cu TB-SMA (F = -sqrt(rho), the same embedding form the paper uses) and an
analytic EAM tabulated on 5000 points (look-up tables built once on the
CPU).  The recipe (seed, draw order, conventions) is the one stated in DESIGN.md section 4.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

BASE_SEED = 12126332                     # arXiv id of the paper
AMU_TO_EV_FS2_PER_A2 = 103.642696526805  # 1 amu * (1 A/fs)^2 in eV
KB_EV_PER_K = 8.617333262e-5

MASS_AMU = {"Cu": 63.546, "Fe": 55.845, "W": 183.84}

FCC_BASIS = np.array([[0, 0, 0], [0, .5, .5], [.5, 0, .5], [.5, .5, 0]], dtype=np.float64)
BCC_BASIS = np.array([[0, 0, 0], [.5, .5, .5]], dtype=np.float64)

# TB-SMA (second-moment tight binding, Cleri-Rosato form) Cu, BASELINE.json configs[0]
CU_TBSMA = dict(A=0.0855, xi=1.224, p=10.96, q=2.278, r0=2.5562)


@dataclass
class Workload:
    """One synthetic system: everything `md_create` / `oracle_create` needs."""
    name: str
    box: np.ndarray                 # (3,) orthorhombic edges, Angstrom (same for every box)
    positions: np.ndarray           # (N,3) float64, Angstrom
    velocities: np.ndarray          # (N,3) float64, Angstrom/fs
    types: np.ndarray               # (N,) int32
    mass: np.ndarray                # (n_types,) amu
    cutoff: float
    skin: float
    n_boxes: int = 1
    pot_kind: int = 0               # 0 = TB-SMA analytic, 1 = EAM cubic-Hermite tables
    tbsma: dict | None = None       # A, xi, p, q, r0: (n_types*n_types,) arrays; taper_on: float
    tables: dict | None = None      # nr, dr, f_val, f_der, phi_val, phi_der, nrho, drho, F_val, F_der
    pair_cutoff: np.ndarray | None = None    # (n_types*n_types,) per-pair cut-offs <= cutoff (paper's RCUT(ity,jty)), or None
    pair_taper_on: np.ndarray | None = None  # (n_types*n_types,) TB-SMA: start of each pair's switch, or None
    dt: float = 1.0                 # fs
    steps: int = 100
    meta: dict = field(default_factory=dict)

    @property
    def n_atoms(self) -> int:
        return int(self.positions.shape[0])

    @property
    def n_types(self) -> int:
        return int(self.mass.shape[0])


# --------------------------------------------------------------------------------------
# crystals, jitter, velocities
# --------------------------------------------------------------------------------------
def lattice_sites(kind: str, a: float, n: tuple[int, int, int]) -> np.ndarray:
    """Perfect crystal sites, emitted unit cell by unit cell with x slowest, z fastest,
    basis atoms innermost (deliberately NOT the library's internal cell order)."""
    basis = FCC_BASIS if kind == "fcc" else BCC_BASIS
    ix, iy, iz = np.meshgrid(np.arange(n[0]), np.arange(n[1]), np.arange(n[2]), indexing="ij")
    cells = np.stack([ix.ravel(), iy.ravel(), iz.ravel()], axis=1).astype(np.float64)
    sites = (cells[:, None, :] + basis[None, :, :]).reshape(-1, 3) * a
    return np.ascontiguousarray(sites)


def maxwell_boltzmann(rng: np.random.Generator, n: int, mass_amu: float, temperature: float) -> np.ndarray:
    """N(0, kT/m) per Cartesian component, centre-of-mass velocity removed, then rescaled
    so that the kinetic temperature with 3N-3 degrees of freedom is exactly `temperature`."""
    m = mass_amu * AMU_TO_EV_FS2_PER_A2
    v = rng.standard_normal((n, 3)) * np.sqrt(KB_EV_PER_K * temperature / m)
    if temperature <= 0.0 or n < 2:
        return np.zeros((n, 3))
    v -= v.mean(axis=0, keepdims=True)
    t_now = m * float((v * v).sum()) / ((3 * n - 3) * KB_EV_PER_K)
    v *= np.sqrt(temperature / t_now)
    return v


def _jitter_and_velocities(rng, sites, sigma, mass_amu, temperature):
    # draw order fixed by the recipe: jitter first, velocities second
    pos = sites + sigma * rng.standard_normal(sites.shape)
    vel = maxwell_boltzmann(rng, sites.shape[0], mass_amu, temperature)
    return pos, vel


# --------------------------------------------------------------------------------------
# potentials (parameters and table *node data* only; evaluation lives in oracle/ and csrc/)
# --------------------------------------------------------------------------------------
def cu_tbsma_params(cutoff: float, taper_width: float = 0.5) -> dict:
    d = {k: np.array([v], dtype=np.float64) for k, v in CU_TBSMA.items()}
    d["taper_on"] = float(cutoff - taper_width)
    return d


def eam_tables(re: float, cutoff: float, nr: int = 5000, nrho: int = 5000, rho_max: float = 100.0,
               fe: float = 1.0, beta: float = 6.0, A: float = 0.4, B: float = 0.6, alpha: float = 8.0,
               kappa: float = 4.0, F0: float = 2.5, rhoe: float = 20.0, taper_width: float = 0.0) -> dict:
    """Node values and analytic node slopes of the analytic EAM of BASELINE.json configs[1]:
    f(r) = fe exp(-beta (r/re-1)); phi(r) = A exp(-alpha (r/re-1)) - B exp(-kappa (r/re-1));
    F(rho) = -F0 sqrt(rho/rhoe), on r_k = k*cutoff/(nr-1) and rho_k = k*rho_max/(nrho-1).
    The slope of F at node 0 (analytically -inf) is the secant to node 1 (reading A8).
    `taper_width` > 0 multiplies f and phi by the quintic switch over the last `taper_width`
    Angstrom: used only by the energy-conservation pin of the table path (reading A9)."""
    r = np.arange(nr, dtype=np.float64) * (cutoff / (nr - 1))
    x = r / re - 1.0
    f = fe * np.exp(-beta * x)
    df = -(beta / re) * f
    e1, e2 = A * np.exp(-alpha * x), B * np.exp(-kappa * x)
    phi = e1 - e2
    dphi = -(alpha / re) * e1 + (kappa / re) * e2
    if taper_width > 0.0:
        t = np.clip((r - (cutoff - taper_width)) / taper_width, 0.0, 1.0)
        s = 1.0 - t ** 3 * (10.0 - 15.0 * t + 6.0 * t * t)
        ds = -30.0 * t * t * (1.0 - t) ** 2 / taper_width
        df, f = df * s + f * ds, f * s
        dphi, phi = dphi * s + phi * ds, phi * s
    rho = np.arange(nrho, dtype=np.float64) * (rho_max / (nrho - 1))
    Fv = -F0 * np.sqrt(rho / rhoe)
    with np.errstate(divide="ignore"):
        Fd = -F0 / (2.0 * np.sqrt(rho * rhoe))
    Fd[0] = (Fv[1] - Fv[0]) / (rho[1] - rho[0])
    return dict(nr=nr, dr=float(cutoff / (nr - 1)), f_val=f, f_der=df, phi_val=phi, phi_der=dphi,
                nrho=nrho, drho=float(rho_max / (nrho - 1)), F_val=Fv, F_der=Fd)


# --------------------------------------------------------------------------------------
# generic builders
# --------------------------------------------------------------------------------------
def cu_fcc(ncell: int, cutoff: float = 4.9, skin: float = 0.3, sigma: float = 0.05, temperature: float = 300.0,
           seed: int = BASE_SEED, a: float = 3.615, n_boxes: int = 1, steps: int = 100, name: str | None = None,
           box_seeds: list[int] | None = None) -> Workload:
    """Cu fcc ncell^3 unit cells with the TB-SMA potential; `n_boxes` > 1 packs independent
    boxes (paper's multiple-box-in-one-run scheme), each seeded separately."""
    sites = lattice_sites("fcc", a, (ncell,) * 3)
    pos, vel = [], []
    for b in range(n_boxes):
        s = seed if n_boxes == 1 else (box_seeds[b] if box_seeds is not None else seed + 1000 * (b + 1))
        rng = np.random.Generator(np.random.PCG64(s))
        p, v = _jitter_and_velocities(rng, sites, sigma, MASS_AMU["Cu"], temperature)
        pos.append(p)
        vel.append(v)
    n = sites.shape[0] * n_boxes
    return Workload(name=name or f"cu_fcc_{ncell}^3_rc{cutoff}" + (f"_x{n_boxes}" if n_boxes > 1 else ""),
                    box=np.full(3, a * ncell), positions=np.concatenate(pos), velocities=np.concatenate(vel),
                    types=np.zeros(n, dtype=np.int32), mass=np.array([MASS_AMU["Cu"]]), cutoff=cutoff, skin=skin,
                    n_boxes=n_boxes, pot_kind=0, tbsma=cu_tbsma_params(cutoff), dt=1.0, steps=steps,
                    meta=dict(lattice="fcc", a=a, ncell=ncell, sigma=sigma, temperature=temperature, seed=seed))


def bcc_eam(ncell: int, a: float, re: float, cutoff: float, element: str, skin: float = 0.3, sigma: float = 0.05,
            temperature: float = 600.0, seed: int = BASE_SEED, dt: float = 1.0, steps: int = 1000,
            pka_ev: float = 0.0, taper_width: float = 0.0, name: str | None = None, rho_max: float = 100.0) -> Workload:
    """bcc crystal with the tabulated analytic EAM; optional primary knock-on atom (PKA):
    the atom nearest the box centre (lowest index on ties) has its velocity REPLACED by
    sqrt(2 E/m) along a seeded isotropic direction, after the centre-of-mass step."""
    sites = lattice_sites("bcc", a, (ncell,) * 3)
    rng = np.random.Generator(np.random.PCG64(seed))
    pos, vel = _jitter_and_velocities(rng, sites, sigma, MASS_AMU[element], temperature)
    meta = dict(lattice="bcc", a=a, ncell=ncell, sigma=sigma, temperature=temperature, seed=seed, re=re)
    if pka_ev > 0.0:
        u = rng.standard_normal(3)
        u /= np.sqrt((u * u).sum())
        centre = 0.5 * a * ncell
        d2 = ((sites - centre) ** 2).sum(axis=1)
        ipka = int(np.argmin(d2))           # argmin returns the lowest index on ties
        m = MASS_AMU[element] * AMU_TO_EV_FS2_PER_A2
        vel[ipka] = np.sqrt(2.0 * pka_ev / m) * u
        meta.update(pka_index=ipka, pka_ev=pka_ev)
    n = sites.shape[0]
    return Workload(name=name or f"{element}_bcc_{ncell}^3_rc{cutoff}", box=np.full(3, a * ncell), positions=pos,
                    velocities=vel, types=np.zeros(n, dtype=np.int32), mass=np.array([MASS_AMU[element]]),
                    cutoff=cutoff, skin=skin, n_boxes=1, pot_kind=1,
                    tables=eam_tables(re, cutoff, taper_width=taper_width, rho_max=rho_max), dt=dt, steps=steps, meta=meta)


# --------------------------------------------------------------------------------------
# BASELINE.json configs
# --------------------------------------------------------------------------------------
def config(k: int | str, scale: int | None = None, replica: int = 0) -> Workload:
    """BASELINE.json `configs[k]`; k = '3a' / '3b' select the two cut-offs of configs[3].
    `scale` overrides the number of unit cells per edge (boxes for config 2) for reduced
    parity-test sizes; None gives the full size.  `replica` > 0 draws an independent copy of
    the same system (seed + 100003 * replica): bench.py gives one replica to every GPU."""
    k = str(k)
    if replica:
        global BASE_SEED
        saved, BASE_SEED = BASE_SEED, BASE_SEED + 100003 * int(replica)
        try:
            return config(k, scale)
        finally:
            BASE_SEED = saved
    if k == "0":
        return cu_fcc(scale or 6, 4.9, seed=BASE_SEED + 0, steps=100, name="cfg0_cu_fcc6_tbsma")
    if k == "1":
        return bcc_eam(scale or 32, 2.855, 2.4725, 5.0, "Fe", temperature=600.0, seed=BASE_SEED + 1, steps=1000,
                       name="cfg1_fe_bcc32_eam")
    if k == "2":
        nb = scale or 2048
        return cu_fcc(5, 4.9, seed=BASE_SEED + 2, n_boxes=nb, steps=500, name=f"cfg2_cu_fcc5_x{nb}_tbsma",
                      box_seeds=[BASE_SEED + 2 + 1000 * (b + 1) for b in range(nb)])
    if k in ("3", "3a"):
        return cu_fcc(scale or 64, 4.9, seed=BASE_SEED + 3, steps=200, name="cfg3a_cu_fcc64_rc4.9")
    if k == "3b":
        return cu_fcc(scale or 64, 6.5, seed=BASE_SEED + 3, steps=200, name="cfg3b_cu_fcc64_rc6.5")
    if k == "4":
        return bcc_eam(scale or 128, 3.165, 2.741, 5.5, "W", temperature=1500.0, seed=BASE_SEED + 4, dt=0.2,
                       steps=200, pka_ev=2000.0, name="cfg4_w_bcc128_eam_pka")
    raise ValueError(f"unknown config {k!r}")


def _tbsma_type_set(a: dict, s: float) -> dict:
    """synthetic TB-SMA parameter set of a type at fraction s in [0, 1] between the base element (s = 0) and the
    larger, stiffer synthetic element of the binary alloy (s = 1)"""
    return dict(A=(1 + 0.2 * s) * a["A"], xi=(1 - 0.04 * s) * a["xi"], p=(1 - 0.003 * s) * a["p"], q=(1 + 0.38 * s) * a["q"],
                r0=(1 + 0.06 * s) * a["r0"])


def alloy(w: Workload, seed: int, fraction: float = 0.5, pair_cutoffs: bool = False, n_types: int = 2) -> Workload:
    """Alloy on the sites of `w` (the paper's rho^(ab), V^(ab)).
    n_types = 2: a seeded `fraction` of the atoms becomes type 1.  TB-SMA: type 1 gets a second, synthetic parameter
    set (larger atom, different stiffness) and the cross pair (0,1) = (1,0) its own set, so that every entry of the 2x2
    parameter arrays differs; tables: the three pair tables are the analytic EAM with different (re, beta, A, B) and the
    two embedding tables differ in F0.  n_types = 3, 4 (MD_MAX_TYPES): equal seeded fractions; type t sits at
    s_t = t/(n_types-1) between the two elements of the binary alloy, a cross pair (s,t) takes the mean of its two types
    times a factor that is symmetric in (s,t) and different for every unordered pair, so every one of the
    n_types(n_types+1)/2 parameter sets / tables differs; masses 1, 1.7, 1.3, 2.1 x the base mass.
    Parameter arrays are indexed [ti * n_types + tj].  `pair_cutoffs`: every unordered pair also gets its own cut-off
    in [0.93 r_c, r_c] (pair (0,0) keeps r_c; TB-SMA: each switch over its last 0.5 A)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    u = rng.random(w.n_atoms)
    nt = int(n_types)
    types = (u < fraction).astype(np.int32) if nt == 2 else np.minimum((u * nt).astype(np.int32), nt - 1)
    w2 = Workload(**{**w.__dict__})
    w2.types = types
    w2.mass = w.mass[0] * np.array([1.0, 1.7, 1.3, 2.1][:nt])
    w2.name = w.name + ("_alloy" if nt == 2 else f"_alloy{nt}")
    pairs = [(s, t) for s in range(nt) for t in range(nt)]
    cross = lambda s, t: 1.0 + 0.011 * (s + t) + 0.006 * s * t                 # symmetric, distinct per unordered pair
    if w.pot_kind == 0:
        a = {k: float(w.tbsma[k][0]) for k in ("A", "xi", "p", "q", "r0")}
        if nt == 2:
            b = dict(A=1.2 * a["A"], xi=0.96 * a["xi"], p=0.997 * a["p"], q=1.38 * a["q"], r0=1.06 * a["r0"])     # type 1
            c = dict(A=1.09 * a["A"], xi=0.985 * a["xi"], p=1.01 * a["p"], q=1.17 * a["q"], r0=1.03 * a["r0"])    # cross
            w2.tbsma = {k: np.array([a[k], c[k], c[k], b[k]]) for k in a}
        else:
            sets = [_tbsma_type_set(a, t / (nt - 1)) for t in range(nt)]

            def entry(k, s, t):
                if s == t:
                    return sets[s][k]
                mean = 0.5 * (sets[s][k] + sets[t][k])
                return mean * cross(s, t) if k in ("A", "q") else mean / cross(s, t) if k == "xi" else mean
            w2.tbsma = {k: np.array([entry(k, s, t) for s, t in pairs]) for k in a}
        w2.tbsma["taper_on"] = w.tbsma["taper_on"]
    else:
        t0 = w.tables
        re = w.meta.get("re", 2.4725)
        rc = t0["dr"] * (t0["nr"] - 1)
        rho_max = t0["drho"] * (t0["nrho"] - 1)

        def mk(re, **kw):
            return eam_tables(re, rc, nr=t0["nr"], nrho=t0["nrho"], rho_max=rho_max, **kw)
        if nt == 2:
            t11 = mk(re=1.05 * re, beta=5.5, A=0.45, B=0.62, F0=2.9)
            t01 = mk(re=1.02 * re, beta=5.8, A=0.42, B=0.61)
            tabs = {(0, 0): t0, (0, 1): t01, (1, 0): t01, (1, 1): t11}
        else:
            par = lambda s: dict(re=(1 + 0.05 * s) * re, beta=6.0 - 0.5 * s, A=0.4 + 0.05 * s, B=0.6 + 0.02 * s, F0=2.5 + 0.4 * s)
            tabs = {}
            for s, t in pairs:
                if (t, s) in tabs:
                    tabs[(s, t)] = tabs[(t, s)]
                elif s == t:
                    tabs[(s, t)] = t0 if s == 0 else mk(**par(s / (nt - 1)))
                else:
                    ps, pt = par(s / (nt - 1)), par(t / (nt - 1))
                    m = {k: 0.5 * (ps[k] + pt[k]) for k in ps}
                    tabs[(s, t)] = mk(re=m["re"], beta=m["beta"] / cross(s, t), A=m["A"] * cross(s, t), B=m["B"])
        pair = lambda k: np.concatenate([tabs[st][k] for st in pairs])
        w2.tables = dict(nr=t0["nr"], dr=t0["dr"], nrho=t0["nrho"], drho=t0["drho"],
                         f_val=pair("f_val"), f_der=pair("f_der"), phi_val=pair("phi_val"), phi_der=pair("phi_der"),
                         F_val=np.concatenate([tabs[(t, t)]["F_val"] for t in range(nt)]),
                         F_der=np.concatenate([tabs[(t, t)]["F_der"] for t in range(nt)]))
    if pair_cutoffs:
        rc = w.cutoff
        if nt == 2:
            w2.pair_cutoff = np.array([rc, 0.93 * rc, 0.93 * rc, 0.97 * rc])
        else:
            # unordered pair number u = 0 .. n(n+1)/2 - 1 in the order (0,0), (0,1), ...: cut-offs spread over [0.93 r_c, r_c]
            order = {st: k for k, st in enumerate((s, t) for s in range(nt) for t in range(s, nt))}
            npair = len(order)
            w2.pair_cutoff = np.array([rc * (1.0 - 0.07 * ((order[(min(s, t), max(s, t))] * 7) % npair) / (npair - 1)) for s, t in pairs])
        if w.pot_kind == 0:
            w2.pair_taper_on = w2.pair_cutoff - 0.5
        w2.name += "_rcut"
    return w2


def permuted(w: Workload, seed: int) -> tuple[Workload, np.ndarray]:
    """Same system with atoms listed in a seeded random order (within each box); returns the
    workload and `perm` with new[i] = old[perm[i]].  Exercises reorder / un-permute."""
    rng = np.random.Generator(np.random.PCG64(seed))
    npb = w.n_atoms // w.n_boxes
    perm = np.concatenate([b * npb + rng.permutation(npb) for b in range(w.n_boxes)])
    w2 = Workload(**{**w.__dict__})
    w2.positions = np.ascontiguousarray(w.positions[perm])
    w2.velocities = np.ascontiguousarray(w.velocities[perm])
    w2.types = np.ascontiguousarray(w.types[perm])
    return w2, perm
