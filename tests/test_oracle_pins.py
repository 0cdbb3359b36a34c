"""Pins of the CPU oracle against things that are NOT the oracle: closed-form lattice sums
(mpmath, tests/golden/make_lattice_pins.py), a live 40-digit evaluation of eq.(1) on small
clusters, finite differences of the energy, brute force, symmetries and conservation laws.
No GPU.  Each test names the plausible mistake it is there to catch."""
import numpy as np
import pytest

import oracle
import workloads
from oracle import Oracle, OracleError

CU = workloads.CU_TBSMA


def perfect_cu(ncell=6, cutoff=4.9, a=3.615, **kw):
    return workloads.cu_fcc(ncell, cutoff, sigma=0.0, temperature=0.0, a=a, **kw)


def big_box_cluster(pos, cutoff=4.9, pot="cu", box=40.0):
    """A free cluster: atoms near the centre of a box so large that no periodic image is in range."""
    n = len(pos)
    kw = dict(box=np.full(3, box), positions=np.asarray(pos, float) + box / 2, velocities=np.zeros((n, 3)),
              types=np.zeros(n, np.int32), cutoff=cutoff, skin=0.3, n_boxes=1)
    if pot == "cu":
        return Oracle(pot_kind=0, mass=np.array([63.546]), tbsma=workloads.cu_tbsma_params(cutoff), **kw)
    return Oracle(pot_kind=1, mass=np.array([55.845]), tables=workloads.eam_tables(2.4725, cutoff), **kw)


# ---------------------------------------------------------------- closed forms on perfect crystals
@pytest.mark.parametrize("tag,cutoff", [("cu49", 4.9), ("cu65", 6.5)])
def test_cu_lattice_sums(pins, tag, cutoff):
    """dropped term / wrong factor 2 in V / taper misplaced / wrong shell count."""
    w = perfect_cu(6, cutoff)
    o = Oracle(w)
    f, e, vir = o.compute_forces()
    rho, fp = o.densities()
    cnt, _ = o.neighbors()
    assert np.all(cnt == int(pins[f"{tag}.n_in_list"]))
    assert np.abs(e - pins[f"{tag}.E"]).max() < 1e-13
    assert np.abs(rho - pins[f"{tag}.rho"]).max() < 2e-13
    assert np.abs(fp - pins[f"{tag}.Fp"]).max() < 1e-14
    assert abs(vir[0, :3].sum() / w.n_atoms - pins[f"{tag}.W"]) < 1e-12        # radial derivatives, exact
    assert np.abs(vir[0, :3] / w.n_atoms - pins[f"{tag}.W"] / 3).max() < 1e-12  # cubic symmetry
    assert np.abs(vir[0, 3:]).max() / w.n_atoms < 1e-13
    assert np.abs(f).max() < 1e-12                                              # inversion symmetry


@pytest.mark.parametrize("tag,a,re,cutoff,el,ncell", [("fe", 2.855, 2.4725, 5.0, "Fe", 6), ("w", 3.165, 2.741, 5.5, "W", 6)])
def test_eam_table_lattice_sums(pins, tag, a, re, cutoff, el, ncell):
    """table path: wrong node spacing / index / Hermite coefficient; 5000-point tables add <~1e-12."""
    w = workloads.bcc_eam(ncell, a, re, cutoff, el, sigma=0.0, temperature=0.0)
    o = Oracle(w)
    f, e, vir = o.compute_forces()
    rho, fp = o.densities()
    cnt, _ = o.neighbors()
    assert np.all(cnt == int(pins[f"{tag}.n_in_list"]))
    assert np.abs(e - pins[f"{tag}.E"]).max() < 1e-11
    assert np.abs(rho - pins[f"{tag}.rho"]).max() < 1e-11
    assert np.abs(fp - pins[f"{tag}.Fp"]).max() < 1e-11
    assert abs(vir[0, :3].sum() / w.n_atoms - pins[f"{tag}.W"]) < 2e-8     # interpolant slope error O(h^3)
    assert np.abs(f).max() < 1e-12


def test_cu_equilibrium_lattice_constant(pins):
    """analytic cohesive energy and lattice constant of the truncated potential (north_star)."""
    from scipy.optimize import minimize_scalar

    def e_of_a(a):
        return Oracle(perfect_cu(5, 4.9, a=a)).compute_forces()[1][0]
    res = minimize_scalar(e_of_a, bracket=(3.60, 3.62, 3.64), tol=1e-12)
    assert abs(res.x - pins["cu49.a_eq"]) < 2e-7
    assert abs(res.fun - pins["cu49.E_eq"]) < 1e-12
    assert abs(res.x - 3.615) / 3.615 < 2e-3 and abs(res.fun + 3.54) < 0.05    # textbook Cu: 3.615 A, 3.54 eV


@pytest.mark.parametrize("tag,r", [("dimer25", 2.5), ("dimer46", 4.6)])
def test_cu_dimer_closed_form(pins, tag, r):
    """(F'_i + F'_j) written as F'_i only / sign of the force / taper derivative (r=4.6 is inside the taper)."""
    o = big_box_cluster([[0, 0, 0], [r * 0.6, 0.0, r * 0.8]])
    f, e, vir = o.compute_forces()
    assert abs(e.sum() - pins[f"{tag}.E"]) < 1e-14
    u = np.array([0.6, 0.0, 0.8])                       # (r_2 - r_1)/r
    # pins F = -dE/dr is the force on atom 1 along (r_1 - r_2)/r; negative = attraction
    assert abs(f[0] @ (-u) - pins[f"{tag}.F"]) < 1e-13
    assert np.abs(f[0] + f[1]).max() < 1e-15
    assert np.abs(f[0] - (f[0] @ u) * u).max() < 1e-15  # central force
    assert abs(vir[0, :3].sum() - pins[f"{tag}.F"] * r) < 1e-13     # W = sum_pairs r_ij . f_ij = r * F_radial


def test_pair_term_in_isolation_born_mayer():
    """xi = 0 kills the many-body term: f_i = -sum_j V'(r) r_hat, a Born-Mayer pair potential."""
    rng = np.random.default_rng(5)
    pos = rng.uniform(-1.25, 1.25, (9, 3))              # diameter < 4.4: every pair below the taper
    n = len(pos)
    tb = workloads.cu_tbsma_params(4.9)
    tb["xi"] = np.array([0.0])
    o = Oracle(pot_kind=0, mass=np.array([63.546]), tbsma=tb, box=np.full(3, 40.0), positions=pos + 20, cutoff=4.9,
               skin=0.3, velocities=np.zeros((n, 3)), types=np.zeros(n, np.int32), n_boxes=1)
    f, e, _ = o.compute_forces()
    A, p, r0 = CU["A"], CU["p"], CU["r0"]
    fref, eref = np.zeros((n, 3)), 0.0
    for i in range(n):
        for j in range(n):
            d = pos[i] - pos[j]
            r = np.sqrt(d @ d)
            if i != j and r < 4.4:                      # stay below the taper: pure exponential
                eref += 0.5 * 2 * A * np.exp(-p * (r / r0 - 1))
                fref[i] += (p / r0) * 2 * A * np.exp(-p * (r / r0 - 1)) * d / r
    rr = np.sqrt(((pos[:, None] - pos[None]) ** 2).sum(-1))
    assert not np.any((rr > 4.4) & (rr < 4.9)), "test geometry must avoid the taper window"
    assert abs(e.sum() - eref) < 1e-13 * abs(eref) and np.abs(f - fref).max() < 1e-13 * np.abs(fref).max()


# ---------------------------------------------------------------- 40-digit evaluation of eq.(1)
def _mp_energy(pos, cutoff, ron):
    from mpmath import exp, mpf, sqrt
    A, xi, p, q, r0 = (mpf(str(CU[k])) for k in ("A", "xi", "p", "q", "r0"))
    rc, ron = mpf(str(cutoff)), mpf(str(ron))
    etot = mpf(0)
    for i in range(len(pos)):
        rho = pair = mpf(0)
        for j in range(len(pos)):
            if i == j:
                continue
            r = sqrt(sum((pos[i][a] - pos[j][a]) ** 2 for a in range(3)))
            if r >= rc:
                continue
            s = mpf(1)
            if r > ron:
                t = (r - ron) / (rc - ron)
                s = 1 - t ** 3 * (10 - 15 * t + 6 * t * t)
            x = r / r0 - 1
            rho += xi * xi * exp(-2 * q * x) * s
            pair += 2 * A * exp(-p * x) * s
        etot += (-sqrt(rho) if rho > 0 else 0) + pair / 2
    return etot


def test_cluster_against_mpmath():
    """whole energy AND force expression, independent arithmetic: eq.(1) summed at 40 digits and its
    gradient by a 40-digit central difference (step 1e-15 A => truncation error ~1e-30)."""
    from mpmath import mp, mpf
    mp.dps = 40
    rng = np.random.default_rng(11)
    a = 3.615
    sites = np.array([[0, 0, 0]] + [[sx * a / 2 * u, sy * a / 2 * v, sz * a / 2 * w] for (u, v, w) in
                     ((1, 1, 0), (1, 0, 1), (0, 1, 1)) for sx in (1, -1) for sy in (1, -1) for sz in (1,)][:12]
                     + [[a, 0, 0], [0, -a, 0], [a, a, 0.0]])
    sites = np.unique(np.round(sites, 9), axis=0)
    pos = sites + 0.08 * rng.standard_normal(sites.shape)
    o = big_box_cluster(pos)
    f, e, _ = o.compute_forces()
    shifted = pos + 20.0                                    # the doubles the oracle actually saw
    mpos = [[mpf(float(c)) for c in row] for row in shifted]
    eref = _mp_energy(mpos, 4.9, 4.4)
    assert abs(mpf(float(e.sum())) - eref) < mpf("1e-13")
    h = mpf("1e-15")
    for i in (0, 3, len(pos) - 1):
        for c in range(3):
            mpos[i][c] += h
            ep = _mp_energy(mpos, 4.9, 4.4)
            mpos[i][c] -= 2 * h
            em = _mp_energy(mpos, 4.9, 4.4)
            mpos[i][c] += h
            assert abs(mpf(float(f[i, c])) + (ep - em) / (2 * h)) < mpf("1e-12"), (i, c)


# ---------------------------------------------------------------- force = -grad E (finite differences)
@pytest.mark.parametrize("cfg", ["cu", "eam"])
def test_forces_are_minus_gradient_fd(cfg):
    """sign / missing F'_j term / derivative of a different interpolant than the energy's."""
    w = workloads.config(0, scale=5) if cfg == "cu" else workloads.config(1, scale=6)
    o = Oracle(w)
    f, _, _ = o.compute_forces()
    x0 = o.positions()

    def etot(x):
        o.set_positions(x)
        return o.energies()[0][0]
    rng = np.random.default_rng(3)
    for i in rng.choice(w.n_atoms, 5, replace=False):
        for c in range(3):
            d = []
            for h in (1e-4, 2e-4):
                xp, xm = x0.copy(), x0.copy()
                xp[i, c] += h
                xm[i, c] -= h
                d.append((etot(xp) - etot(xm)) / (2 * h))
            fd = (4 * d[0] - d[1]) / 3                     # Richardson
            assert abs(f[i, c] + fd) < 2e-8, (i, c, f[i, c], fd)


@pytest.mark.parametrize("cfg", ["cu", "eam"])
def test_virial_is_strain_derivative(cfg):
    """W^{aa} = -L_a dE/dL_a under affine scaling of one axis: pins each diagonal virial component."""
    w = workloads.config(0, scale=5) if cfg == "cu" else workloads.config(1, scale=6)
    _, _, vir = Oracle(w).compute_forces()

    def e_scaled(axis, s):
        box, pos = w.box.copy(), w.positions.copy()
        box[axis] *= s
        pos[:, axis] *= s
        kw = {k: getattr(w, k) for k in ("velocities", "types", "mass", "cutoff", "skin", "n_boxes", "pot_kind", "tbsma", "tables")}
        return Oracle(box=box, positions=pos, **kw).energies()[0][0]
    for axis in range(3):
        d = [(e_scaled(axis, 1 + h) - e_scaled(axis, 1 - h)) / (2 * h) for h in (1e-5, 2e-5)]
        fd = (4 * d[0] - d[1]) / 3
        assert abs(vir[0, axis] + fd) < 2e-6 * max(1.0, abs(fd)), (axis, vir[0, axis], -fd)


def test_virial_offdiagonal_by_rotation():
    """W transforms as a tensor: rotate a free cluster by 45 deg about z; pins xy (and, by relabelling, xz, yz)."""
    rng = np.random.default_rng(9)
    pos = rng.uniform(-3.2, 3.2, (20, 3))
    c, s = np.cos(0.7), np.sin(0.7)
    for R in (np.array([[c, -s, 0], [s, c, 0], [0, 0, 1.0]]), np.array([[c, 0, -s], [0, 1.0, 0], [s, 0, c]]),
              np.array([[1.0, 0, 0], [0, c, -s], [0, s, c]])):
        _, _, v0 = big_box_cluster(pos).compute_forces()
        _, _, v1 = big_box_cluster(pos @ R.T).compute_forces()
        full = lambda v: np.array([[v[0], v[3], v[4]], [v[3], v[1], v[5]], [v[4], v[5], v[2]]])
        assert np.abs(full(v1[0]) - R @ full(v0[0]) @ R.T).max() < 1e-13 * np.abs(v0).max()


# ---------------------------------------------------------------- neighbour lists
@pytest.mark.parametrize("make", [lambda: workloads.config(0), lambda: workloads.config(0, scale=5),
                                  lambda: workloads.config(2, scale=3), lambda: workloads.config(1, scale=6),
                                  lambda: workloads.cu_fcc(8, 6.5, seed=77)])
def test_cell_list_equals_brute_force(make):
    """stencil / wrap / box offset errors: the cell list must give the same pair SETS as all-pairs."""
    w = make()
    a, b = Oracle(w), Oracle(w)
    a.build_neighbors(brute_force=False)
    b.build_neighbors(brute_force=True)
    ca, la = a.neighbors()
    cb, lb = b.neighbors()
    assert np.array_equal(ca, cb) and np.array_equal(la, lb)
    assert np.abs(a.compute_forces()[0] - b.compute_forces()[0]).max() == 0.0
    # directed pairs come in symmetric couples
    pairs = {(i, j) for i in range(w.n_atoms) for j in la[i, :ca[i]]}
    assert all((j, i) in pairs for (i, j) in pairs)


def test_noncubic_box_and_positions_outside_box():
    w = workloads.config(0, scale=5)
    kw = {k: getattr(w, k) for k in ("velocities", "types", "mass", "cutoff", "skin", "n_boxes", "pot_kind", "tbsma")}
    box = w.box * np.array([1.0, 1.1, 1.3])
    pos = w.positions * np.array([1.0, 1.1, 1.3])
    shift = np.array([3.7, -55.1, 1234.5])                 # far outside [0,L): the build wraps
    a, b = Oracle(box=box, positions=pos, **kw), Oracle(box=box, positions=pos + shift, **kw)
    a.build_neighbors(True)
    b.build_neighbors(False)
    assert np.array_equal(a.neighbors()[1], b.neighbors()[1])
    assert np.abs(a.compute_forces()[0] - b.compute_forces()[0]).max() < 1e-11
    x = b.positions()
    assert np.all(x >= 0) and np.all(x <= box)


def test_min_image_canonical_form():
    d, r2 = oracle.min_image([0.5, 9.6, 5.0], [9.75, 0.25, 5.0], [10.0, 10.0, 10.0])
    assert np.array_equal(d, [9.75 - 0.5 - 10.0, 0.25 - 9.6 + 10.0, 0.0])
    assert r2 == (d[0] * d[0] + d[1] * d[1]) + d[2] * d[2]


# ---------------------------------------------------------------- symmetries
def test_invariants_sum_permutation_translation():
    w = workloads.config(0)
    o = Oracle(w)
    f, e, vir = o.compute_forces()
    assert np.abs(f.sum(0)).max() < 1e-10 * np.sqrt(w.n_atoms)      # Newton's third law, summed
    w2, perm = workloads.permuted(w, 123)
    f2, e2, vir2 = Oracle(w2).compute_forces()
    assert np.abs(f2 - f[perm]).max() < 1e-12 and np.abs(e2 - e[perm]).max() < 1e-12
    assert np.abs(vir2 - vir).max() < 1e-9
    for shift in ([0.123, -4.56, 7.89], [w.box[0] * 0.5, w.box[1] * 3, -w.box[2] * 0.75]):
        o3 = Oracle(w, positions=w.positions + np.array(shift))
        f3, e3, vir3 = o3.compute_forces()
        assert np.abs(f3 - f).max() < 1e-11 and abs(e3.sum() - e.sum()) < 1e-9 and np.abs(vir3 - vir).max() < 1e-8


def test_batched_boxes_are_independent():
    """box id / cell offset leaks: a batch must equal each box run alone."""
    w = workloads.config(2, scale=3)
    fb, eb, vb = Oracle(w).compute_forces()
    npb = w.n_atoms // 3
    for b in range(3):
        sl = slice(b * npb, (b + 1) * npb)
        o = Oracle(w, positions=w.positions[sl], velocities=w.velocities[sl], types=w.types[sl], n_boxes=1)
        f1, e1, v1 = o.compute_forces()
        assert np.array_equal(f1, fb[sl]) and np.array_equal(e1, eb[sl]) and np.array_equal(v1[0], vb[b])
    assert not np.array_equal(fb[:npb], fb[npb:2 * npb])            # boxes really are seeded separately


# ---------------------------------------------------------------- radial functions
def test_taper_and_tbsma_functions():
    args = (CU["A"], CU["xi"], CU["p"], CU["q"], CU["r0"], 4.4, 4.9)
    f, df, V, dV, S, dS = oracle.tbsma_eval(2.5562, *args)
    assert S == 1.0 and dS == 0.0 and abs(f - CU["xi"] ** 2) < 1e-15 and abs(V - 2 * CU["A"]) < 1e-16   # x = 0
    assert oracle.tbsma_eval(4.4, *args)[4] == 1.0 and oracle.tbsma_eval(4.9, *args)[4] == 0.0
    assert abs(oracle.tbsma_eval(4.65, *args)[4] - 0.5) < 1e-15     # the quintic switch is odd about its midpoint
    for r in (2.3, 3.3, 4.45, 4.7, 4.89):
        h = 1e-5
        lo, hi, mid = oracle.tbsma_eval(r - h, *args), oracle.tbsma_eval(r + h, *args), oracle.tbsma_eval(r, *args)
        for val, der in ((0, 1), (2, 3), (4, 5)):
            assert abs((hi[val] - lo[val]) / (2 * h) - mid[der]) < 1e-8 * max(1.0, abs(mid[der]))
    # C2 at both ends: S' and (numerically) S'' vanish
    assert abs(oracle.tbsma_eval(4.4 + 1e-7, *args)[5]) < 1e-11 and abs(oracle.tbsma_eval(4.9 - 1e-7, *args)[5]) < 1e-11


def test_hermite_reproduces_cubics_exactly():
    """a cubic Hermite interpolant of a cubic is that cubic: pins node indexing, t and both coefficient formulas."""
    h, n = 0.37, 12
    xk = np.arange(n) * h
    poly = np.polynomial.Polynomial([0.3, -1.1, 0.45, 0.07])
    val, der = poly(xk), poly.deriv()(xk)
    for x in (0.0, 0.1, 0.37, 1.0, 2.2222, xk[-1] - 1e-9, xk[-2]):
        H, dH = oracle.hermite_eval(val, der, h, x)
        assert abs(H - poly(x)) < 1e-13 and abs(dH - poly.deriv()(x)) < 1e-13


def test_table_matches_analytic_functions():
    t = workloads.eam_tables(2.4725, 5.0)
    for r in (1.9, 2.4725, 3.3333, 4.9995):
        x = r / 2.4725 - 1
        H, dH = oracle.hermite_eval(t["f_val"], t["f_der"], t["dr"], r)
        assert abs(H - np.exp(-6 * x)) < 1e-12 and abs(dH + 6 / 2.4725 * np.exp(-6 * x)) < 1e-9
        H, dH = oracle.hermite_eval(t["phi_val"], t["phi_der"], t["dr"], r)
        assert abs(H - (0.4 * np.exp(-8 * x) - 0.6 * np.exp(-4 * x))) < 1e-12
    H, dH = oracle.hermite_eval(t["F_val"], t["F_der"], t["drho"], 10.76)
    assert abs(H + 2.5 * np.sqrt(10.76 / 20)) < 1e-9


# ---------------------------------------------------------------- integrator
def _total_energy_trace(w, dt, nsteps, every=1):
    o = Oracle(w)
    tr = []
    for _ in range(nsteps // every):
        ep, ek = o.energies()
        tr.append(ep.sum() + ek.sum())
        o.step(every, dt)
    ep, ek = o.energies()
    tr.append(ep.sum() + ek.sum())
    return np.array(tr), o


def test_nve_energy_conservation_and_dt2_scaling():
    """integrator order and rebuild logic: the error is bounded, ~dt^2, and a missed pair would show as a jump."""
    w = workloads.config(0)
    tr1, o1 = _total_energy_trace(w, 1.0, 100)
    tr2, _ = _total_energy_trace(w, 0.5, 200, every=2)
    e1, e2 = np.abs(tr1 - tr1[0]).max() / w.n_atoms, np.abs(tr2 - tr2[0]).max() / w.n_atoms
    assert e1 < 5e-6 and 3.5 < e1 / e2 < 4.5, (e1, e2)
    st = o1.stats()
    assert st["steps"] == 100 and 3 <= st["rebuilds"] - 1 <= 8        # about every 20 steps at 300 K


def test_nve_tapered_table_path():
    """reading A9: the untapered configs 1/4 cannot conserve energy; the table path is pinned with tapered tables."""
    w = workloads.bcc_eam(6, 2.855, 2.4725, 5.0, "Fe", temperature=600.0, seed=4, taper_width=0.5)
    tr1, _ = _total_energy_trace(w, 1.0, 100)
    tr2, _ = _total_energy_trace(w, 0.5, 200, every=2)
    e1, e2 = np.abs(tr1 - tr1[0]).max() / w.n_atoms, np.abs(tr2 - tr2[0]).max() / w.n_atoms
    assert e1 < 5e-5 and 3.0 < e1 / e2 < 5.0, (e1, e2)


def test_time_reversibility_and_momentum():
    w = workloads.config(0, scale=5)
    o = Oracle(w)
    x0, v0 = o.positions(), o.velocities()
    o.step(40, 1.0)
    p = (o.velocities() * 63.546).sum(0)
    assert np.abs(p).max() < 1e-9                                     # sum m v stays 0
    o.set_velocities(-o.velocities())
    o.step(40, 1.0)
    d = o.positions() - x0
    d -= np.round(d / w.box) * w.box
    assert np.abs(d).max() < 1e-9 and np.abs(o.velocities() + v0).max() < 1e-10


def test_list_always_covers_cutoff_between_rebuilds():
    """skin logic: at every step all pairs inside r_c must be in the list then in use."""
    w = workloads.config(0, scale=5)
    w.velocities *= 2.0                                               # ~1200 K: frequent rebuilds
    o = Oracle(w)
    o.build_neighbors()
    for _ in range(60):
        o.step(1, 1.0)
        assert o.list_covers_cutoff()
    assert o.stats()["rebuilds"] >= 4


def test_step_equals_manual_velocity_verlet():
    """one oracle step against the three textbook lines written out with numpy and oracle forces."""
    w = workloads.config(0, scale=5)
    o, o2 = Oracle(w), Oracle(w)
    f0 = o2.compute_forces()[0]
    m = 63.546 * workloads.AMU_TO_EV_FS2_PER_A2
    vh = w.velocities + 0.5 * 1.0 / m * f0
    x1 = w.positions - w.box * np.floor(w.positions / w.box) + 1.0 * vh
    o2.set_positions(x1)
    f1 = o2.compute_forces()[0]
    o.step(1, 1.0)
    d = o.positions() - x1
    d -= np.round(d / w.box) * w.box
    assert np.abs(d).max() < 1e-13 and np.abs(o.velocities() - (vh + 0.5 / m * f1)).max() < 1e-15


# ---------------------------------------------------------------- errors and edge cases
def test_error_codes():
    w = workloads.config(0, scale=2)                                   # L = 7.23 < 2 r_l
    with pytest.raises(OracleError) as ei:
        Oracle(w)
    assert ei.value.code == -2
    w = workloads.config(0, scale=3)                                   # L = 10.8: brute force ok, 27-cell stencil not
    o = Oracle(w)
    o.build_neighbors(brute_force=True)
    with pytest.raises(OracleError) as ei:
        o.build_neighbors(brute_force=False)
    assert ei.value.code == -2
    w = workloads.config(0, scale=5)
    with pytest.raises(OracleError) as ei:
        Oracle(w, max_neighbors=20).build_neighbors()
    assert ei.value.code == -3
    w.positions[1] = w.positions[0]
    with pytest.raises(OracleError) as ei:
        Oracle(w).compute_forces()
    assert ei.value.code == -4
    with pytest.raises(OracleError):
        Oracle(w, types=np.full(w.n_atoms, 3, np.int32))


def test_isolated_atom_and_empty_neighbourhood():
    o = big_box_cluster([[0, 0, 0], [8.0, 0, 0]])                      # farther apart than r_l
    f, e, vir = o.compute_forces()
    assert np.all(f == 0) and np.all(e == 0) and np.all(vir == 0)
    assert np.all(o.neighbors()[0] == 0)


# ---------------------------------------------------------------- binary alloys (PAPER.md:78 rho^(ab), V^(ab))
def _alloy_energy_numpy(pos, types, tb, cutoff, pair_cutoff=None, pair_taper_on=None, nt=2):
    """eq.(1) with type-pair parameters written out in numpy (direct double loop, float64); index [ti*nt + tj]."""
    ron0 = tb["taper_on"]
    etot, n = 0.0, len(pos)
    for i in range(n):
        rho = pair = 0.0
        for j in range(n):
            if i == j:
                continue
            r = float(np.sqrt(((pos[i] - pos[j]) ** 2).sum()))
            k = types[i] * nt + types[j]
            rc = cutoff if pair_cutoff is None else pair_cutoff[k]
            ron = ron0 if pair_taper_on is None else pair_taper_on[k]
            if r >= rc:
                continue
            t = min(max((r - ron) / (rc - ron), 0.0), 1.0)
            s = 1.0 - t ** 3 * (10.0 - 15.0 * t + 6.0 * t * t)
            x = r / tb["r0"][k] - 1.0
            rho += tb["xi"][k] ** 2 * np.exp(-2.0 * tb["q"][k] * x) * s
            pair += 2.0 * tb["A"][k] * np.exp(-tb["p"][k] * x) * s
        etot += -np.sqrt(rho) + 0.5 * pair
    return etot


def test_alloy_energy_and_forces_against_numpy_definition():
    """type-pair indexing of every parameter: energy from the definition, forces from its central differences."""
    w = workloads.alloy(workloads.config(0, scale=5), 11)
    rng = np.random.default_rng(3)
    idx = rng.choice(w.n_atoms, 24, replace=False)
    pos = w.positions[idx] * 0.55 + 20.0                # a dense random cluster in a big box, both types present
    types = w.types[idx]
    assert 4 < types.sum() < 20
    kw = dict(pot_kind=0, mass=w.mass, tbsma=w.tbsma, box=np.full(3, 60.0), cutoff=4.9, skin=0.3,
              velocities=np.zeros((24, 3)), types=types, n_boxes=1)
    f, e, _ = Oracle(positions=pos, **kw).compute_forces()
    eref = _alloy_energy_numpy(pos, types, w.tbsma, 4.9)
    assert abs(e.sum() - eref) < 1e-12 * abs(eref)
    h = 1e-4
    for a, c in ((0, 0), (5, 1), (17, 2)):
        def E(dh):
            p2 = pos.copy(); p2[a, c] += dh
            return _alloy_energy_numpy(p2, types, w.tbsma, 4.9)
        fd = -((8 * (E(h) - E(-h)) - (E(2 * h) - E(-2 * h))) / (12 * h))
        assert abs(fd - f[a, c]) < 2e-8 * max(1.0, abs(f[a, c]))


@pytest.mark.parametrize("cfg", ["0", "1"])
def test_alloy_reduces_to_one_species_and_label_swap(cfg):
    base = workloads.config(cfg, scale=5 if cfg == "0" else 7)
    w = workloads.alloy(base, 5)
    # (a) identical parameter sets for every pair == the one-species system, whatever the labels
    same = workloads.Workload(**{**w.__dict__})
    if cfg == "0":
        same.tbsma = {k: (np.repeat(base.tbsma[k], 4) if k != "taper_on" else base.tbsma[k]) for k in base.tbsma}
    else:
        t = base.tables
        same.tables = {**t, **{k: np.tile(t[k], 4) for k in ("f_val", "f_der", "phi_val", "phi_der")},
                       **{k: np.tile(t[k], 2) for k in ("F_val", "F_der")}}
    f1, e1, v1 = Oracle(same).compute_forces()
    f0, e0, v0 = Oracle(base).compute_forces()
    assert np.array_equal(f1, f0) and np.array_equal(e1, e0)
    # (b) swapping the labels 0 <-> 1 together with the parameter blocks changes nothing
    sw = workloads.Workload(**{**w.__dict__})
    sw.types = (1 - w.types).astype(np.int32)
    sw.mass = w.mass[::-1].copy()
    if cfg == "0":
        sw.tbsma = {k: (w.tbsma[k][[3, 2, 1, 0]] if k != "taper_on" else w.tbsma[k]) for k in w.tbsma}
    else:
        t, nr, nrho = w.tables, w.tables["nr"], w.tables["nrho"]
        blk = lambda a, n, order: np.concatenate([a[i * n:(i + 1) * n] for i in order])
        sw.tables = {**t, **{k: blk(t[k], nr, [3, 2, 1, 0]) for k in ("f_val", "f_der", "phi_val", "phi_der")},
                     **{k: blk(t[k], nrho, [1, 0]) for k in ("F_val", "F_der")}}
    fa, ea, va = Oracle(w).compute_forces()
    fb, eb, vb = Oracle(sw).compute_forces()
    assert np.array_equal(fa, fb) and np.array_equal(ea, eb)
    assert not np.allclose(fa, f0, atol=1e-3)            # and the alloy is not the one-species system
    # (c) alloy forces sum to zero and the run conserves momentum with two masses
    assert np.abs(fa.sum(0)).max() < 1e-11
    o = Oracle(w)
    p0 = (o.velocities() * w.mass[w.types][:, None]).sum(0)
    o.step(20, w.dt)
    p1 = (o.velocities() * w.mass[w.types][:, None]).sum(0)
    assert np.abs(p1 - p0).max() < 1e-12 * np.abs(o.velocities() * w.mass[w.types][:, None]).sum()


# ---------------------------------------------------------------- electron-bath thermostat, eq.(4)
KB = 8.617333262e-5
AMU = 103.642696526805


def _free_atoms(speeds, masses=(63.546, 107.8682)):
    """atoms further apart than the cut-off (no forces), two species, prescribed speeds along random directions"""
    n = len(speeds)
    rng = np.random.default_rng(8)
    grid = np.array([[i, j, k] for i in range(3) for j in range(3) for k in range(3)], float)[:n] * 13.0 + 3.0
    u = rng.standard_normal((n, 3)); u /= np.linalg.norm(u, axis=1)[:, None]
    types = (np.arange(n) % 2).astype(np.int32)
    tb = workloads.alloy(workloads.config(0, scale=5), 1).tbsma
    return dict(pot_kind=0, mass=np.array(masses), tbsma=tb, box=np.full(3, 39.0), positions=grid, cutoff=4.9, skin=0.3,
                velocities=u * np.asarray(speeds)[:, None], types=types, n_boxes=1), types


def test_thermostat_free_atoms_closed_form():
    """no forces: |v|^2(t) = c2 + (|v0|^2 - c2) exp(-2t/tau), c2 = 3 k_B T_e/m, direction unchanged; first order in dt"""
    Te, tau, T = 450.0, 80.0, 120.0
    speeds = np.array([0.001, 0.004, 0.008, 0.002, 0.012, 0.0005, 0.006, 0.003])
    kw, types = _free_atoms(speeds)
    m = np.array(kw["mass"])[types] * AMU
    c2 = 3 * KB * Te / m
    exact = np.sqrt(c2 + (speeds ** 2 - c2) * np.exp(-2 * T / tau))
    err = []
    for dt in (0.5, 0.25):
        o = Oracle(**kw)
        o.set_thermostat(Te, tau)
        o.step(int(round(T / dt)), dt)
        v = o.velocities()
        s = np.linalg.norm(v, axis=1)
        assert np.abs(np.cross(v / s[:, None], kw["velocities"] / speeds[:, None])).max() < 1e-12     # same direction
        err.append(np.abs(s - exact).max())
        assert err[-1] < 2e-2 * exact.max() * dt
    assert 1.7 < err[0] / err[1] < 2.3
    # atoms hotter than the bath slow down, colder ones speed up
    assert np.all((s < speeds) == (speeds ** 2 > c2))


def test_thermostat_off_limits_and_crystal_temperature():
    w = workloads.config(0, scale=5)
    a, b, c = Oracle(w), Oracle(w), Oracle(w)
    b.set_thermostat(300.0, 1e30)                       # infinitely slow exchange == no thermostat
    c.set_thermostat(300.0, 0.0)                        # tau <= 0: off
    for o in (a, b, c):
        o.step(30, 1.0)
    assert np.abs(a.positions() - b.positions()).max() < 1e-13 and np.array_equal(a.positions(), c.positions())
    # a 300 K crystal coupled to a 900 K bath heats up towards it (equipartition halves the initial kinetic T first)
    o = Oracle(w)
    o.set_thermostat(900.0, 40.0)
    o.step(600, 1.0)
    temps = []
    for _ in range(10):
        o.step(20, 1.0)
        temps.append(2 * o.energies()[1].sum() / (3 * w.n_atoms * KB))
    assert 750.0 < np.mean(temps) < 1050.0
    # an atom at rest feels no damping (no division by zero)
    kw, _ = _free_atoms(np.array([0.0, 0.002]))
    o = Oracle(**kw); o.set_thermostat(300.0, 50.0); o.step(5, 1.0)
    assert np.all(o.velocities()[0] == 0.0) and np.all(np.isfinite(o.velocities()))


# ---------------------------------------------------------------- Berendsen barostat, eq.(5)-(6)
def test_pressure_closed_forms(pins):
    """eq.(6): the virial part on a perfect lattice (= -dE/dV from the lattice-sum pin) and the ideal-gas part"""
    w = perfect_cu(6)
    o = Oracle(w, velocities=np.zeros_like(w.velocities))
    a = 3.615
    assert abs(o.pressure() - 4 * pins["cu49.W"] / (3 * a ** 3)) < 1e-15          # N W_i / (3 V), 4 atoms per a^3
    assert abs(o.pressure() * 160.21766208 - 0.66154) < 1e-4                        # GPa, SURVEY.md section 8(c)
    kw, types = _free_atoms(np.array([0.003, 0.004, 0.002, 0.005]))
    m = np.array(kw["mass"])[types] * AMU
    ek = 0.5 * (m * np.array([0.003, 0.004, 0.002, 0.005]) ** 2).sum()
    assert abs(Oracle(**kw).pressure() - (2.0 / 3.0) * ek / 39.0 ** 3) < 1e-20      # no forces: P V = N k_B T = 2/3 E_kin


def test_barostat_one_step_formula_and_relaxation_to_the_pinned_lattice_constant(pins):
    w = perfect_cu(6)
    v0 = np.zeros_like(w.velocities)
    # one step, atoms at rest on the perfect lattice: mu = cbrt(1 - dt/tau (P0 - P)) exactly, box and coordinates scaled
    o = Oracle(w, velocities=v0)
    P, P0, tau, dt = o.pressure(), -0.002, 5.0, 1.0
    o.set_barostat(P0, tau)
    x0 = o.positions()
    o.step(1, dt)
    mu = np.cbrt(1.0 - dt / tau * (P0 - P))
    assert mu > 1.0                                                                # P > P0: the box grows
    assert np.abs(o.box() / w.box - mu).max() < 1e-15 and np.abs(o.positions() - mu * x0).max() < 1e-12
    # P0 = 0: the box relaxes to the minimum of the closed-form E(a): the pinned equilibrium lattice constant
    o = Oracle(w, velocities=v0)
    o.set_barostat(0.0, 1.75)                                                       # dt/tau ~ 0.5/B, B ~ 0.87 eV/A^3
    o.step(80, 1.0)
    assert abs(o.box()[0] / 6 - pins["cu49.a_eq"]) < 1e-9
    assert abs(o.pressure()) < 1e-12 and np.abs(o.compute_forces()[0]).max() < 1e-10
    assert abs(o.energies()[0].sum() / w.n_atoms - pins["cu49.E_eq"]) < 1e-12
    # off by default / tau <= 0; refuses batched boxes
    a, b = Oracle(workloads.config(0)), Oracle(workloads.config(0))
    b.set_barostat(0.0, 0.0)
    a.step(10, 1.0); b.step(10, 1.0)
    assert np.array_equal(a.positions(), b.positions()) and np.array_equal(b.box(), workloads.config(0).box)
    with pytest.raises(OracleError):
        Oracle(workloads.config(2, scale=2)).set_barostat(0.0, 5.0)
    # a read-only query between steps does not change the trajectory (reading B1: the next first half-kick keeps the
    # forces of the unscaled coordinates whether or not energies / pressure / forces were asked for in between)
    a, b = Oracle(workloads.config(0)), Oracle(workloads.config(0))
    for o in (a, b):
        o.set_barostat(0.0, 20.0)
    for _ in range(6):
        a.step(5, 1.0); b.step(5, 1.0)
        fq = b.compute_forces()[0]; b.energies(); b.pressure(); fq2 = b.compute_forces()[0]
        assert np.array_equal(fq, fq2)
    assert np.array_equal(a.positions(), b.positions()) and np.array_equal(a.velocities(), b.velocities())
    assert np.abs(fq - Oracle(workloads.config(0), positions=b.positions(), box=b.box()).compute_forces()[0]).max() < 1e-12
    # thermal run under pressure control keeps the list valid (x_ref is not scaled: the rebuild rule sees the scaling)
    o = Oracle(workloads.config(0))
    o.set_barostat(0.0, 20.0)
    for _ in range(8):
        o.step(10, 1.0)
        assert o.list_covers_cutoff()


def test_pair_cutoffs_against_numpy_definition_and_defaults():
    """the paper's RCUT(ity,jty): per-pair cut-offs and switches"""
    w = workloads.alloy(workloads.config(0, scale=5), 11, pair_cutoffs=True)
    rng = np.random.default_rng(3)
    idx = rng.choice(w.n_atoms, 24, replace=False)
    pos = w.positions[idx] * 0.6 + 20.0
    types = w.types[idx]
    kw = dict(pot_kind=0, mass=w.mass, tbsma=w.tbsma, box=np.full(3, 60.0), cutoff=4.9, skin=0.3, velocities=np.zeros((24, 3)),
              types=types, n_boxes=1)
    f, e, _ = Oracle(positions=pos, pair_cutoff=w.pair_cutoff, pair_taper_on=w.pair_taper_on, **kw).compute_forces()
    eref = _alloy_energy_numpy(pos, types, w.tbsma, 4.9, w.pair_cutoff, w.pair_taper_on)
    assert abs(e.sum() - eref) < 1e-12 * abs(eref)
    e_glob = Oracle(positions=pos, **kw).compute_forces()[1].sum()
    assert abs(e_glob - eref) > 1e-6                       # the pair cut-offs do change the energy of this cluster
    h = 1e-4
    for a, c in ((1, 0), (9, 2)):
        def E(dh):
            p2 = pos.copy(); p2[a, c] += dh
            return _alloy_energy_numpy(p2, types, w.tbsma, 4.9, w.pair_cutoff, w.pair_taper_on)
        fd = -((8 * (E(h) - E(-h)) - (E(2 * h) - E(-2 * h))) / (12 * h))
        assert abs(fd - f[a, c]) < 2e-8 * max(1.0, abs(f[a, c]))
    # pair cut-offs equal to the global ones == no pair cut-offs, bit for bit; tables: strict per-pair cut
    for cfg, sc in (("0", 5), ("1", 7)):
        w0 = workloads.alloy(workloads.config(cfg, scale=sc), 5)
        same = Oracle(w0, pair_cutoff=np.full(4, w0.cutoff), pair_taper_on=None if cfg == "1" else np.full(4, w0.tbsma["taper_on"]))
        assert np.array_equal(same.compute_forces()[0], Oracle(w0).compute_forces()[0])
    wt = workloads.alloy(workloads.config(1, scale=7), 5, pair_cutoffs=True)
    ft = Oracle(wt).compute_forces()[0]
    assert np.abs(ft.sum(0)).max() < 1e-11 and not np.allclose(ft, Oracle(workloads.alloy(workloads.config(1, scale=7), 5)).compute_forces()[0])
    with pytest.raises(OracleError):                       # larger than the list cut-off, or asymmetric
        Oracle(w0, pair_cutoff=np.full(4, 1.01 * w0.cutoff))
    with pytest.raises(OracleError):
        Oracle(w0, pair_cutoff=np.array([5.0, 4.8, 4.9, 5.0]))


# ---------------------------------------------------------------- three and four species (MD_MAX_TYPES = 4)
@pytest.mark.parametrize("nt", [3, 4])
def test_multi_species_energy_and_forces_against_numpy_definition(nt):
    """[ti*nt + tj] indexing with nt > 2 (a 2-type test cannot tell ti*nt+tj from ti*2+tj or from tj*nt+ti on a
    symmetric table): energy from the definition, forces from its central differences, per-pair cut-offs included."""
    w = workloads.alloy(workloads.config(0, scale=5), 11, n_types=nt, pair_cutoffs=True)
    rng = np.random.default_rng(3)
    idx = rng.choice(w.n_atoms, 28, replace=False)
    pos = w.positions[idx] * 0.57 + 20.0
    types = w.types[idx]
    assert len(np.unique(types)) == nt
    kw = dict(pot_kind=0, mass=w.mass, tbsma=w.tbsma, box=np.full(3, 60.0), cutoff=4.9, skin=0.3, velocities=np.zeros((28, 3)),
              types=types, n_boxes=1, pair_cutoff=w.pair_cutoff, pair_taper_on=w.pair_taper_on)
    f, e, _ = Oracle(positions=pos, **kw).compute_forces()
    eref = _alloy_energy_numpy(pos, types, w.tbsma, 4.9, w.pair_cutoff, w.pair_taper_on, nt=nt)
    assert abs(e.sum() - eref) < 1e-12 * abs(eref)
    h = 1e-4
    for a, c in ((0, 0), (7, 1), (19, 2), (27, 0)):
        def E(dh):
            p2 = pos.copy(); p2[a, c] += dh
            return _alloy_energy_numpy(p2, types, w.tbsma, 4.9, w.pair_cutoff, w.pair_taper_on, nt=nt)
        fd = -((8 * (E(h) - E(-h)) - (E(2 * h) - E(-2 * h))) / (12 * h))
        assert abs(fd - f[a, c]) < 2e-8 * max(1.0, abs(f[a, c]))


@pytest.mark.parametrize("cfg,nt", [("0", 3), ("1", 3), ("0", 4), ("1", 4)])
def test_multi_species_label_permutation(cfg, nt):
    """re-labelling the species cyclically (t -> t+1 mod nt) together with every parameter block / table / mass / pair
    cut-off changes nothing, bit for bit: catches a transposed or mis-strided type-pair index in any array."""
    w = workloads.alloy(workloads.config(cfg, scale=5 if cfg == "0" else 7), 5, n_types=nt, pair_cutoffs=True)
    new_of_old = (np.arange(nt) + 1) % nt
    old_of_new = np.argsort(new_of_old)
    pair_src = [old_of_new[s] * nt + old_of_new[t] for s in range(nt) for t in range(nt)]      # new block (s,t) <- old block
    sw = workloads.Workload(**{**w.__dict__})
    sw.types = new_of_old[w.types].astype(np.int32)
    sw.mass = w.mass[old_of_new].copy()
    sw.pair_cutoff = w.pair_cutoff[pair_src].copy()
    if cfg == "0":
        sw.tbsma = {k: (w.tbsma[k][pair_src].copy() if k != "taper_on" else w.tbsma[k]) for k in w.tbsma}
        sw.pair_taper_on = w.pair_taper_on[pair_src].copy()
    else:
        t, nr, nrho = w.tables, w.tables["nr"], w.tables["nrho"]
        blk = lambda a, n, order: np.concatenate([a[i * n:(i + 1) * n] for i in order])
        sw.tables = {**t, **{k: blk(t[k], nr, pair_src) for k in ("f_val", "f_der", "phi_val", "phi_der")},
                     **{k: blk(t[k], nrho, old_of_new) for k in ("F_val", "F_der")}}
    fa, ea, va = Oracle(w).compute_forces()
    fb, eb, vb = Oracle(sw).compute_forces()
    assert np.array_equal(fa, fb) and np.array_equal(ea, eb) and np.array_equal(va, vb)
    one = workloads.config(cfg, scale=5 if cfg == "0" else 7)
    assert not np.allclose(fa, Oracle(one).compute_forces()[0], atol=1e-3)
    assert np.abs(fa.sum(0)).max() < 1e-11
    oa, ob = Oracle(w), Oracle(sw)
    oa.step(15, w.dt); ob.step(15, w.dt)
    assert np.array_equal(oa.positions(), ob.positions())                      # masses follow the labels too


# ---------------------------------------------------------------- F(rho) above the last table node (reading A8)
def test_embedding_linear_continuation_above_rho_max(pins):
    """rho >= rho_max: F = F(rho_max) + F'(rho_max)(rho - rho_max), F' = F'(rho_max).  Fe-form EAM tabulated only up to
    rho_max = 8 while the perfect bcc lattice has rho = 10.76: closed form from tests/golden/make_lattice_pins.py."""
    w = workloads.bcc_eam(6, 2.855, 2.4725, 5.0, "Fe", sigma=0.0, temperature=0.0, rho_max=8.0)
    o = Oracle(w)
    f, e, vir = o.compute_forces()
    rho, fp = o.densities()
    assert np.abs(rho - pins["fe.rho"]).max() < 1e-11 and rho.min() > 8.0
    assert np.abs(e - pins["fe_rhomax8.E"]).max() < 1e-11
    assert np.abs(fp - pins["fe_rhomax8.Fp"]).max() < 1e-15
    assert abs(vir[0, :3].sum() / w.n_atoms - pins["fe_rhomax8.W"]) < 2e-8
    assert np.abs(f).max() < 1e-12
    # the two branches join continuously and forces stay the gradient of the energy across the junction: a jittered
    # crystal whose densities straddle rho_max
    wj = workloads.bcc_eam(6, 2.855, 2.4725, 5.0, "Fe", sigma=0.05, temperature=0.0, rho_max=10.76, seed=77)
    oj = Oracle(wj)
    fj, ej, _ = oj.compute_forces()
    rj = oj.densities()[0]
    assert (rj > 10.76).sum() > 20 and (rj < 10.76).sum() > 20
    h = 1e-4
    for a, c in ((3, 0), (100, 1), (211, 2)):
        def E(dh):
            p2 = wj.positions.copy(); p2[a, c] += dh
            return Oracle(wj, positions=p2).compute_forces()[1].sum()
        fd = -((8 * (E(h) - E(-h)) - (E(2 * h) - E(-2 * h))) / (12 * h))
        assert abs(fd - fj[a, c]) < 5e-8 * max(1.0, abs(fj[a, c]))


# ---------------------------------------------------------------- the oracle under the sanitizers
def test_oracle_under_address_and_undefined_sanitizers(tmp_path):
    """eam_oracle.c compiled with -fsanitize=address,undefined and driven from a small C main over both potential
    kinds, batched boxes, rebuilds and the getters: no heap error, no undefined behaviour."""
    import os
    import subprocess
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    exe = str(tmp_path / "oracle_asan")
    cmd = ["gcc", "-O1", "-g", "-std=c11", "-ffp-contract=off", "-fopenmp", "-fsanitize=address,undefined",
           "-fno-sanitize-recover=undefined", "-I", os.path.join(root, "oracle"), os.path.join(root, "tests", "oracle_asan_main.c"),
           os.path.join(root, "oracle", "eam_oracle.c"), "-lm", "-o", exe]
    subprocess.run(cmd, check=True)
    env = {**os.environ, "ASAN_OPTIONS": "detect_leaks=1:abort_on_error=0", "OMP_NUM_THREADS": "2"}
    r = subprocess.run([exe], capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode == 0, r.stdout[-2000:] + r.stderr[-4000:]
    assert "runtime error" not in r.stderr and "AddressSanitizer" not in r.stderr and "LeakSanitizer" not in r.stderr
    assert "asan-main ok" in r.stdout


# --------------------------------------------------------------------------------------
# Gear predictor-corrector (reading G1)
# --------------------------------------------------------------------------------------
def _smooth_cluster():
    """Four Cu atoms 2.4-2.9 A apart in the 21.7 A box of config 0: every pair stays inside the taper onset (4.4 A), so
    the potential is analytic along the trajectory and an integrator shows its formal order."""
    w = workloads.config(0)
    x = np.array([[5, 5, 5], [7.5, 5.1, 5.0], [6.2, 7.2, 5.1], [6.3, 5.8, 7.1]], dtype=np.float64)
    v = np.array([[0.01, 0, 0.005], [-0.01, 0.004, 0], [0, -0.006, 0.003], [0.0, 0.002, -0.008]])
    return w, dict(positions=x, velocities=v, types=np.zeros(4, np.int32))


def _run(w, kw, kind, dt, t_end):
    o = Oracle(w, **kw)
    o.set_integrator(kind)
    o.step(int(round(t_end / dt)), dt)
    return o


def test_gear_order_of_accuracy_and_agreement_with_velocity_verlet():
    """The five-value Gear scheme with coefficients (19/120, 3/4, 1, 1/2, 1/12) converges with the fifth power of dt on
    a smooth potential (halving dt divides the error by ~32); a wrong coefficient (19/90 for 19/120, a wrong Pascal
    entry of the predictor) or a start-up with zero higher derivatives leaves second to fourth order (ratio 4 ... 20).
    Both integrators converge to the same trajectory."""
    w, kw = _smooth_cluster()
    T = 32.0
    ref = _run(w, kw, 1, 1.0 / 32, T).positions()
    err = [np.abs(_run(w, kw, 1, dt, T).positions() - ref).max() for dt in (2.0, 1.0, 0.5)]
    assert err[0] < 5e-6 and 26.0 < err[0] / err[1] < 40.0 and 26.0 < err[1] / err[2] < 40.0
    vv = [np.abs(_run(w, kw, 0, dt, T).positions() - ref).max() for dt in (1.0, 0.5)]
    assert 3.5 < vv[0] / vv[1] < 4.5                                   # velocity-Verlet: second order, same limit
    assert np.abs(_run(w, kw, 0, 1.0 / 64, T).positions() - ref).max() < 2e-8


def test_gear_free_flight_momentum_and_energy():
    w, kw = _smooth_cluster()
    # atoms out of each other's reach: straight lines
    far = dict(kw, positions=np.array([[1, 1, 1], [11, 1.5, 2], [2, 12, 3], [12, 11, 13]], dtype=np.float64))
    o = _run(w, far, 1, 1.0, 40.0)
    assert np.abs(o.positions() - (far["positions"] + 40.0 * far["velocities"])).max() < 1e-12
    assert np.abs(o.velocities() - far["velocities"]).max() < 1e-15
    # crystal at 300 K: total momentum constant, energy conserved far better than by velocity-Verlet at the same dt,
    # rebuilds as often as velocity-Verlet (the skin/2 rule acts on the predicted positions)
    w0 = workloads.config(0)
    m = w0.mass[0]
    res = {}
    for kind in (0, 1):
        o = Oracle(w0)
        o.set_integrator(kind)
        e0 = sum(e.sum() for e in o.energies())
        p0 = m * o.velocities().sum(axis=0)
        o.step(100, 1.0)
        res[kind] = abs(sum(e.sum() for e in o.energies()) - e0) / w0.n_atoms
        assert np.abs(m * o.velocities().sum(axis=0) - p0).max() < 1e-10
        assert o.stats()["rebuilds"] >= 4 and o.list_covers_cutoff()
    assert res[1] < 1e-7 and res[1] < 0.05 * res[0]
    # one step is not the same as velocity-Verlet's (the corrector also moves the positions)
    a, b = Oracle(w0), Oracle(w0)
    b.set_integrator(1)
    a.step(1, 1.0); b.step(1, 1.0)
    d = np.abs(a.positions() - b.positions()).max()
    assert 1e-9 < d < 1e-4


def test_gear_refuses_thermostat_and_barostat():
    w0 = workloads.config(0)
    o = Oracle(w0)
    o.set_integrator(1)
    with pytest.raises(OracleError):
        o.set_thermostat(300.0, 100.0)
    with pytest.raises(OracleError):
        o.set_barostat(0.0, 1e4)
    o.set_integrator(0)
    o.set_thermostat(300.0, 100.0)
    with pytest.raises(OracleError):
        o.set_integrator(1)
