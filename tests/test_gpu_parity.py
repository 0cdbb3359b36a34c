"""Parity of the CUDA path (through the C ABI) with the CPU oracle, element by element, on the same seeded
inputs.  Tolerances are BASELINE.json's north_star: neighbour pair sets bit-exact; |dF| <= 1e-9 eV/A per
component; total energy relative error <= 1e-12; positions after 100 steps within 1e-8 A."""
import numpy as np
import pytest

import workloads

pytestmark = pytest.mark.gpu

F_TOL, E_REL, X_TOL = 1e-9, 1e-12, 1e-8


@pytest.fixture(scope="module")
def md():
    import torch
    assert torch.cuda.is_available(), "these tests need the B200"
    import paper_1212_6332_b200 as m
    m.lib()
    return m


def oracle_of(w, **kw):
    from oracle import Oracle
    return Oracle(w, **kw)


CASES = {
    "cfg0": lambda: workloads.config(0),                                   # 864 Cu, 4^3 cells, 7 tiles of 128 + ragged tail
    "cfg0_perm": lambda: workloads.permuted(workloads.config(0), 99)[0],   # caller order != any lattice order
    "cfg1_small": lambda: workloads.config(1, scale=10),                   # 2000 Fe, tables, 5^3 cells
    "cfg2_small": lambda: workloads.config(2, scale=7),                    # 7 boxes x 500: 3^3 cells each, images everywhere
    "cfg3a_small": lambda: workloads.config("3a", scale=12),               # 6912 Cu
    "cfg3b_small": lambda: workloads.config("3b", scale=12),               # 6.5 A cut-off, ~134 list entries
    "cfg4_small": lambda: workloads.config(4, scale=12),                   # W tables + PKA
    "noncubic": lambda: _noncubic(),
    # binary alloys: every type-pair parameter set / table differs, two masses
    "alloy_tbsma": lambda: workloads.alloy(workloads.config("3a", scale=10), 21),           # 4000 atoms
    "alloy_tbsma_boxes": lambda: workloads.alloy(workloads.config(2, scale=5), 22, 0.3),    # 5 boxes x 500, 30 % type 1
    "alloy_tables": lambda: workloads.alloy(workloads.config(1, scale=10), 23),             # 2000 atoms, 4 pair tables
    # per-pair cut-offs, the paper's RCUT(ity,jty): r_c, 0.93 r_c, 0.97 r_c
    "alloy_tbsma_rcut": lambda: workloads.alloy(workloads.config("3a", scale=10), 24, pair_cutoffs=True),
    "alloy_tables_rcut": lambda: workloads.alloy(workloads.config(1, scale=10), 25, pair_cutoffs=True),
    # three and four species (MD_MAX_TYPES = 4): every one of the n(n+1)/2 parameter sets / tables / cut-offs differs
    "alloy3_tbsma_rcut": lambda: workloads.alloy(workloads.config("3a", scale=10), 26, n_types=3, pair_cutoffs=True),
    "alloy4_tbsma": lambda: workloads.alloy(workloads.config("3a", scale=10), 27, n_types=4),
    "alloy4_tbsma_boxes_rcut": lambda: workloads.alloy(workloads.config(2, scale=5), 28, n_types=4, pair_cutoffs=True),
    "alloy3_tables": lambda: workloads.alloy(workloads.config(1, scale=10), 29, n_types=3),
    "alloy4_tables_rcut": lambda: workloads.alloy(workloads.config(1, scale=10), 30, n_types=4, pair_cutoffs=True),
    # prefactors that cannot be folded into the exponent (xi = 0 for one pair / for all: the kernels' FOLD = false variants)
    "tbsma_xi0_cross": lambda: _xi0(workloads.alloy(workloads.config("3a", scale=10), 31), cross_only=True),
    "born_mayer": lambda: _xi0(workloads.config("3a", scale=10), cross_only=False),
    "born_mayer_boxes": lambda: _xi0(workloads.config(2, scale=6), cross_only=False),
    # F(rho) above the last node of its table (reading A8): every atom / about half of the atoms on the linear continuation
    "cfg1_rhomax8": lambda: workloads.bcc_eam(10, 2.855, 2.4725, 5.0, "Fe", seed=41, rho_max=8.0),
    "cfg1_rhomax_mid": lambda: workloads.bcc_eam(10, 2.855, 2.4725, 5.0, "Fe", seed=42, rho_max=10.76),
}
NEW_VARIANT_CASES = ["alloy3_tbsma_rcut", "alloy4_tbsma", "alloy4_tbsma_boxes_rcut", "alloy3_tables", "alloy4_tables_rcut",
                     "tbsma_xi0_cross", "born_mayer", "born_mayer_boxes", "cfg1_rhomax8", "cfg1_rhomax_mid"]


def _xi0(w, cross_only):
    """xi = 0: no many-body term for that pair (all pairs: a Born-Mayer pair potential, PAPER.md:75 with F = 0)."""
    w.tbsma = {k: (np.array(v, dtype=np.float64, copy=True) if k != "taper_on" else v) for k, v in w.tbsma.items()}
    if cross_only:
        w.tbsma["xi"][[1, 2]] = 0.0
    else:
        w.tbsma["xi"][:] = 0.0
    w.name += "_xi0"
    return w


def _noncubic():
    w = workloads.config(0, scale=5)
    s = np.array([1.0, 1.13, 1.31])
    w.box = w.box * s
    w.positions = w.positions * s + np.array([40.0, -33.0, 1000.0])        # far outside the box: the build wraps
    return w


@pytest.mark.parametrize("case", list(CASES))
def test_neighbor_pair_sets_bit_exact(md, case):
    w = CASES[case]()
    o = oracle_of(w)
    o.build_neighbors()
    oc, ol = o.neighbors(stride=192)
    g = md.MDSystem(w)
    g.build_neighbors()
    gc, gl = g.neighbors(stride=192)
    assert np.array_equal(gc, oc)
    assert np.array_equal(gl, ol)
    st = g.stats()
    assert st["max_neighbors"] == oc.max() and st["error_flags"] == 0 and st["rebuilds"] == 1
    # device-pointer outputs give the same thing
    dc, dl = g.neighbors(stride=192, device_out=True)
    assert np.array_equal(dc.cpu().numpy(), oc) and np.array_equal(dl.cpu().numpy(), ol)
    # wrapped positions agree bit for bit with the oracle's wrap
    assert np.array_equal(g.positions(), o.positions())


@pytest.mark.parametrize("case", list(CASES))
def test_density_force_energy_virial(md, case):
    w = CASES[case]()
    o = oracle_of(w)
    of, oe, ow = o.compute_forces()
    orho, ofp = o.densities()
    g = md.MDSystem(w)
    gf, ge, gw = g.compute_forces()
    grho, gfp = g.densities()
    assert np.abs(grho - orho).max() <= 1e-12 * np.abs(orho).max()
    assert np.abs(gfp - ofp).max() <= 1e-12 * np.abs(ofp).max()
    assert np.abs(gf - of).max() <= F_TOL
    assert np.abs(ge - oe).max() <= 1e-12 * np.abs(oe).max()
    if case.startswith("cfg1_rhomax"):                       # the case does reach the continuation branch
        rmax = w.tables["drho"] * (w.tables["nrho"] - 1)
        assert (orho >= rmax).sum() > 100 and ((orho < rmax).sum() > 100 or case == "cfg1_rhomax8")
    oep, oek = o.energies()
    gep, gek = g.energies()
    assert np.abs(gep - oep).max() <= E_REL * np.abs(oep).max()
    assert np.abs(gek - oek).max() <= E_REL * max(np.abs(oek).max(), 1e-300)
    assert np.abs(gw - ow).max() <= 1e-11 * np.abs(ow).max()
    # device outputs
    df, de, dw = g.compute_forces(device_out=True)
    assert np.array_equal(df.cpu().numpy(), gf) and np.array_equal(de.cpu().numpy(), ge) and np.array_equal(dw.cpu().numpy(), gw)


@pytest.mark.parametrize("case,nsteps", [("cfg0", 100), ("cfg0_perm", 100), ("cfg1_small", 100), ("cfg2_small", 100),
                                         ("cfg3b_small", 40), ("cfg4_small", 100), ("alloy_tbsma", 100),
                                         ("alloy_tbsma_boxes", 60), ("alloy_tables", 100), ("alloy_tbsma_rcut", 100),
                                         ("alloy_tables_rcut", 100)] + [(c, 60) for c in NEW_VARIANT_CASES])
def test_trajectory(md, case, nsteps):
    w = CASES[case]()
    o = oracle_of(w)
    g = md.MDSystem(w)
    e0 = sum(x.sum() for x in g.energies())
    o.step(nsteps, w.dt)
    g.step(nsteps, w.dt)
    ox, gx = o.positions(), g.positions()
    d = gx - ox
    d -= np.round(d / w.box) * w.box            # the two sides may have wrapped at different steps
    assert np.abs(d).max() <= X_TOL
    assert np.abs(g.velocities() - o.velocities()).max() <= 1e-9
    so, sg = o.stats(), g.stats()
    assert sg["steps"] == nsteps and sg["error_flags"] == 0
    assert abs(sg["rebuilds"] - so["rebuilds"]) <= 1
    oep, oek = o.energies()
    gep, gek = g.energies()
    assert abs((gep.sum() + gek.sum()) - (oep.sum() + oek.sum())) <= 1e-10 * abs(oep.sum())
    if case.startswith("cfg0"):
        assert abs(gep.sum() + gek.sum() - e0) / w.n_atoms < 5e-6          # NVE on the device too
    # the list the device holds now is the oracle's list for the device's current positions
    g.build_neighbors()
    o2 = oracle_of(w, positions=g.positions())
    o2.build_neighbors()
    assert np.array_equal(g.neighbors(192)[1], o2.neighbors(192)[1])


def test_step_with_observables_matches_plain_step(md):
    w = CASES["cfg0"]()
    a, b = md.MDSystem(w), md.MDSystem(w)
    b.set_option(md.MD_OPT_STEP_OBSERVABLES, 1)
    a.step(25, 1.0)
    b.step(25, 1.0)
    # same arithmetic up to the contraction choices the compiler makes in the two kernel variants
    assert np.abs(a.positions() - b.positions()).max() < 1e-11 and np.abs(a.velocities() - b.velocities()).max() < 1e-12


@pytest.mark.parametrize("variant", [1, 2, 3, 4])
@pytest.mark.parametrize("case", ["cfg0_perm", "cfg1_small", "cfg2_small", "cfg3b_small", "cfg4_small", "alloy_tbsma",
                                  "alloy_tables", "alloy_tbsma_rcut", "alloy_tables_rcut"] + NEW_VARIANT_CASES)
def test_both_pass_variants(md, case, variant):
    """One thread per atom (what large systems run), 8 / 32 lanes per atom (small systems) and 4 lanes per atom (long
    rows), forced on the same input."""
    w = CASES[case]()
    o = oracle_of(w)
    of, oe, ow = o.compute_forces()
    orho, ofp = o.densities()
    g = md.MDSystem(w)
    g.set_option(md.MD_OPT_FORCE_VARIANT, variant)
    gf, ge, gw = g.compute_forces()
    grho, gfp = g.densities()
    assert np.abs(grho - orho).max() <= 1e-12 * np.abs(orho).max()
    assert np.abs(gfp - ofp).max() <= 1e-12 * np.abs(ofp).max()
    assert np.abs(gf - of).max() <= F_TOL
    assert np.abs(ge - oe).max() <= 1e-12 * np.abs(oe).max()
    assert np.abs(gw - ow).max() <= 1e-11 * np.abs(ow).max()
    o.step(30, w.dt)
    g.step(30, w.dt)
    d = g.positions() - o.positions()
    d -= np.round(d / w.box) * w.box
    assert np.abs(d).max() <= X_TOL and g.stats()["error_flags"] == 0


@pytest.mark.parametrize("case", ["cfg0", "cfg2_small", "cfg4_small"])
def test_graph_step_equals_plain_launches(md, case):
    """md_step as a CUDA graph with the rebuild in a conditional node runs the same kernels as the plain launches."""
    w = CASES[case]()
    a, b = md.MDSystem(w), md.MDSystem(w)
    b.set_option(md.MD_OPT_GRAPH, 0)
    for n in (1, 7, 40):
        a.step(n, w.dt)
        b.step(n, w.dt)
    assert np.array_equal(a.positions(), b.positions()) and np.array_equal(a.velocities(), b.velocities())
    sa, sb = a.stats(), b.stats()
    assert sa["rebuilds"] == sb["rebuilds"] and sa["rebuilds"] >= 2 and sa["error_flags"] == 0
    if w.n_atoms > 4096:                                           # per-step IF nodes: the chain is launched only when a rebuild is due
        assert sa["kernel_launches"] < sb["kernel_launches"]       # (loop graphs of small systems also count the passes that return at once)
    assert sa["graph_active"] == 1 and sb["graph_active"] == 0
    # a different dt re-builds the graph
    a.step(5, 0.5 * w.dt)
    b.step(5, 0.5 * w.dt)
    assert np.array_equal(a.positions(), b.positions())


@pytest.mark.parametrize("half", [1, 2, 3])
@pytest.mark.parametrize("case", ["cfg0_perm", "cfg1_small", "cfg2_small", "cfg3a_small", "cfg3b_small", "cfg4_small", "noncubic",
                                  "alloy_tbsma_boxes", "alloy_tables_rcut", "alloy4_tbsma_boxes_rcut", "alloy3_tables", "born_mayer",
                                  "tbsma_xi0_cross", "cfg1_rhomax_mid"])
def test_half_list_passes(md, case, half):
    """Row f2, Newton's third law: every undirected pair evaluated once, by the atom that owns it; the
    partner's share arrives by 64-bit integer reductions.  Density pass (1), force pass (2) or both (3) against the
    full-list oracle, same tolerances; bit-identical from run to run; the list itself is unchanged as a set."""
    w = CASES[case]()
    o = oracle_of(w)
    of, oe, ow = o.compute_forces()
    orho, ofp = o.densities()

    def run():
        g = md.MDSystem(w)
        g.set_option(md.MD_OPT_FORCE_VARIANT, 1)            # half passes need one thread per atom
        g.set_option(md.MD_OPT_HALF_LIST, half)
        gf, ge, gw = g.compute_forces()
        grho, gfp = g.densities()
        g.step(30, w.dt)
        return g, gf, ge, gw, grho, gfp, g.positions(), g.velocities()

    g, gf, ge, gw, grho, gfp, gx, gv = run()
    assert np.abs(grho - orho).max() <= 1e-12 * np.abs(orho).max()
    assert np.abs(gfp - ofp).max() <= 1e-12 * np.abs(ofp).max()
    assert np.abs(gf - of).max() <= F_TOL
    assert np.abs(ge - oe).max() <= 1e-12 * np.abs(oe).max()
    assert np.abs(gw - ow).max() <= 1e-11 * np.abs(ow).max()
    o.step(30, w.dt)
    d = gx - o.positions()
    d -= np.round(d / w.box) * w.box
    assert np.abs(d).max() <= X_TOL and g.stats()["error_flags"] == 0
    g.build_neighbors()
    o2 = oracle_of(w, positions=g.positions())
    o2.build_neighbors()
    assert np.array_equal(g.neighbors(192)[1], o2.neighbors(192)[1])
    _, gf2, ge2, gw2, _, _, gx2, gv2 = run()
    assert np.array_equal(gf, gf2) and np.array_equal(ge, ge2) and np.array_equal(gw, gw2)
    assert np.array_equal(gx, gx2) and np.array_equal(gv, gv2)
    # switching the option off again gives back the full-list passes
    g.set_option(md.MD_OPT_HALF_LIST, 0)
    gf3 = g.compute_forces()[0]
    assert np.abs(gf3 - oracle_of(w, positions=g.positions()).compute_forces()[0]).max() <= F_TOL


@pytest.mark.parametrize("zfine", [1, 2, 4])
@pytest.mark.parametrize("case", ["cfg0_perm", "cfg2_small", "cfg3b_small", "cfg4_small", "noncubic", "alloy_tbsma_boxes"])
def test_cell_grids(md, case, zfine, monkeypatch):
    """The list build with cubic cells and with cells 2 or 4 times thinner in z and a z window per column (the default
    depends on the box size): the same pair sets, forces and trajectory."""
    monkeypatch.setenv("MD_CELL_ZFINE", str(zfine))
    w = CASES[case]()
    o = oracle_of(w)
    g = md.MDSystem(w)
    g.build_neighbors()
    o.build_neighbors()
    assert np.array_equal(g.neighbors(192)[1], o.neighbors(192)[1])
    gf, ge, gw = g.compute_forces()
    of, oe, ow = o.compute_forces()
    assert np.abs(gf - of).max() <= F_TOL and np.abs(ge - oe).max() <= 1e-12 * np.abs(oe).max()
    g.step(40, w.dt)
    o.step(40, w.dt)
    d = g.positions() - o.positions()
    d -= np.round(d / w.box) * w.box
    assert np.abs(d).max() <= X_TOL and g.stats()["error_flags"] == 0 and g.stats()["rebuilds"] >= 2
    g.build_neighbors()
    o2 = oracle_of(w, positions=g.positions())
    o2.build_neighbors()
    assert np.array_equal(g.neighbors(192)[1], o2.neighbors(192)[1])


@pytest.mark.parametrize("case", ["cfg0", "cfg2_small", "cfg4_small", "alloy_tables_rcut"])
@pytest.mark.parametrize("graph", [1, 0])
def test_chained_steps_equal_single_steps(md, case, graph):
    """md_step(n) chains the steps (the force pass of a step performs the next step's first half-kick, drift and
    displacement check; several steps per CUDA graph); n calls of md_step(1) do not.  Same bits either way."""
    w = CASES[case]()
    a, b = md.MDSystem(w), md.MDSystem(w)
    for s in (a, b):
        s.set_option(md.MD_OPT_GRAPH, graph)
    a.step(43, w.dt)                                  # 5 graphs of 8 steps + one of 3
    for _ in range(43):
        b.step(1, w.dt)
    assert np.array_equal(a.positions(), b.positions()) and np.array_equal(a.velocities(), b.velocities())
    sa, sb = a.stats(), b.stats()
    assert sa["rebuilds"] == sb["rebuilds"] and sa["rebuilds"] >= 2 and sa["error_flags"] == 0
    assert sa["graph_active"] == graph and sa["kernel_launches"] > 0
    if not graph:                                     # (loop graphs of small systems also count the passes that return at once)
        assert sa["kernel_launches"] < sb["kernel_launches"]
    fa, fb = a.compute_forces()[0], b.compute_forces()[0]
    assert np.array_equal(fa, fb)


@pytest.mark.parametrize("case,variant", [("cfg0", 0), ("alloy_tbsma", 1), ("alloy_tables", 2), ("cfg2_small", 0)])
def test_thermostat_trajectory(md, case, variant):
    """eq.(4) electron-bath thermostat (row f1): same half-kicks as the oracle, through the graph and the plain path."""
    w = CASES[case]()
    o = oracle_of(w)
    g = md.MDSystem(w)
    g.set_option(md.MD_OPT_FORCE_VARIANT, variant)
    g.step(10, w.dt)                                   # first without: setting the thermostat must re-build the step graph
    o.step(10, w.dt)
    for x in (o, g):
        x.set_thermostat(900.0, 60.0)
    o.step(90, w.dt)
    g.step(90, w.dt)
    d = g.positions() - o.positions()
    d -= np.round(d / w.box) * w.box
    assert np.abs(d).max() <= X_TOL
    assert np.abs(g.velocities() - o.velocities()).max() <= 1e-9
    ek_o, ek_g = o.energies()[1].sum(), g.energies()[1].sum()
    assert abs(ek_g - ek_o) <= 1e-10 * ek_o
    # the bath is hotter than the crystal: it has heated up, and switching the thermostat off restores plain NVE steps
    w0 = CASES[case]()
    ref = oracle_of(w0); ref.step(100, w.dt)
    assert ek_o > 1.05 * ref.energies()[1].sum()
    for x in (o, g):
        x.set_thermostat(0.0, 0.0)
    o.step(10, w.dt); g.step(10, w.dt)
    d = g.positions() - o.positions()
    d -= np.round(d / w.box) * w.box
    assert np.abs(d).max() <= X_TOL and g.stats()["error_flags"] == 0
    with pytest.raises(md.MDError):
        g.set_thermostat(-1.0, 10.0)


@pytest.mark.parametrize("case,graph", [("cfg0", 1), ("cfg3a_small", 1), ("alloy_tables", 0), ("noncubic", 1)])
def test_barostat_trajectory(md, case, graph):
    """eq.(5)-(6) Berendsen barostat (row f1): box, coordinates and pressure follow the oracle's, step by step."""
    w = CASES[case]()
    if case == "noncubic":
        w.positions = w.positions - np.array([40.0, -33.0, 1000.0])      # scaling acts on the coordinates as given
    o = oracle_of(w)
    g = md.MDSystem(w)
    g.set_option(md.MD_OPT_GRAPH, graph)
    assert abs(g.pressure() - o.pressure()) <= 1e-12 * abs(o.pressure())
    P0 = 0.0 if w.pot_kind == 0 else o.pressure()        # the synthetic Fe-form EAM sits at -33 GPa: hold it there
    for x in (o, g):
        x.set_barostat(P0, 15.0)
        x.set_thermostat(500.0, 100.0)
    for n in (1, 59):
        o.step(n, w.dt)
        g.step(n, w.dt)
    assert np.abs(g.box() / o.box() - 1.0).max() <= 1e-13
    assert np.abs(g.box() / w.box - 1.0).max() > 1e-5     # the box did move
    d = g.positions() - o.positions()
    d -= np.round(d / o.box()) * o.box()
    assert np.abs(d).max() <= X_TOL
    assert abs(g.pressure() - o.pressure()) <= 1e-10 * max(abs(o.pressure()), 1e-3)
    gep, gek = g.energies()
    oep, oek = o.energies()
    assert abs(gep.sum() - oep.sum()) <= 1e-11 * abs(oep.sum()) and abs(gek.sum() - oek.sum()) <= 1e-10 * oek.sum()
    assert g.stats()["error_flags"] == 0
    # the list the device holds is the oracle's list for the device's positions and box
    g.build_neighbors()
    w2 = CASES[case]()
    w2.box = g.box()
    o2 = oracle_of(w2, positions=g.positions())
    o2.build_neighbors()
    assert np.array_equal(g.neighbors(192)[1], o2.neighbors(192)[1])


@pytest.mark.parametrize("graph", [0, 1])
def test_barostat_queries_do_not_change_the_trajectory(md, graph):
    """reading B1: after a scaled step the next first half-kick keeps the forces of the unscaled coordinates; asking for
    forces / energies / pressure in between re-evaluates them at the scaled coordinates without touching that."""
    w = CASES["cfg0"]()
    a, b, o = md.MDSystem(w), md.MDSystem(w), oracle_of(w)
    for x in (a, b, o):
        x.set_barostat(0.0, 20.0)
    a.set_option(md.MD_OPT_GRAPH, graph); b.set_option(md.MD_OPT_GRAPH, graph)
    for _ in range(6):
        a.step(5, 1.0); b.step(5, 1.0); o.step(5, 1.0)
        fq = b.compute_forces()[0]; b.energies(); b.pressure()
        assert np.array_equal(fq, b.compute_forces(device_out=True)[0].cpu().numpy())
        assert np.abs(fq - o.compute_forces()[0]).max() <= F_TOL
    assert np.array_equal(a.positions(), b.positions()) and np.array_equal(a.velocities(), b.velocities())
    d = b.positions() - o.positions()
    d -= np.round(d / o.box()) * o.box()
    assert np.abs(d).max() <= X_TOL and b.stats()["graph_active"] == graph and b.stats()["graph_error"] == 0


def test_barostat_relaxes_perfect_lattice_to_closed_form_and_guards(md):
    """P0 = 0 on a perfect Cu lattice at rest: the box converges to the minimum of the closed-form E(a)
    (tests/golden/lattice_pins.txt cu49.a_eq, mpmath), on the device as in the oracle."""
    pins = dict(l.split(" = ") for l in open(__import__("os").path.join(__import__("os").path.dirname(__file__), "golden", "lattice_pins.txt"))
                if " = " in l)
    w = workloads.cu_fcc(6, sigma=0.0, temperature=0.0)
    w.velocities = np.zeros_like(w.velocities)
    g = md.MDSystem(w)
    g.set_barostat(0.0, 1.75)
    g.step(80, 1.0)
    assert abs(g.box()[0] / 6 - float(pins["cu49.a_eq"])) < 1e-9 and abs(g.pressure()) < 1e-11
    assert abs(g.energies()[0].sum() / w.n_atoms - float(pins["cu49.E_eq"])) < 1e-12
    # a huge external pressure shrinks the cells below cutoff + skin: sticky flag, MD_EBOX
    g = md.MDSystem(workloads.config(0))
    g.set_barostat(5.0, 20.0)
    with pytest.raises(md.MDError) as ei:
        g.step(40, 1.0)
        g.stats(); g.positions()
    assert ei.value.code == md.MD_EBOX
    with pytest.raises(md.MDError):
        md.MDSystem(workloads.config(2, scale=2)).set_barostat(0.0, 5.0)


def test_two_systems_interleaved_and_profile_toggle(md):
    """every system owns its step graph and conditional handle; MD_OPT_PROFILE switches to plain launches and back"""
    w1, w2 = CASES["cfg0"](), CASES["cfg3a_small"]()
    a, b, ra, rb = md.MDSystem(w1), md.MDSystem(w2), md.MDSystem(w1), md.MDSystem(w2)
    for n in (3, 17, 30):
        a.step(n, 1.0)
        b.step(n, 1.0)
    ra.step(50, 1.0)
    rb.step(50, 1.0)
    assert np.array_equal(a.positions(), ra.positions()) and np.array_equal(b.positions(), rb.positions())
    a.set_option(md.MD_OPT_PROFILE, 1)
    a.step(5, 1.0)
    pr = a.profile()
    assert pr["force"][0] == 1 and pr["force_chained"][0] == 4      # one graph-sized group of 5 steps: 4 chained passes + the last
    a.set_option(md.MD_OPT_PROFILE, 0)
    a.step(5, 1.0)
    ra.step(10, 1.0)
    assert np.array_equal(a.positions(), ra.positions()) and a.stats()["error_flags"] == 0


@pytest.mark.parametrize("case", ["cfg0_perm", "cfg2_small", "cfg4_small", "alloy_tbsma_rcut"])
def test_garbage_in_the_workspace_is_never_read(md, case, monkeypatch):
    """the caller's allocation arrives uninitialised: pre-fill it with 0xAB (a list entry of that pattern would index far
    outside every array) and require the same results as the oracle"""
    monkeypatch.setenv("MD_POISON_WORKSPACE", "1")
    w = CASES[case]()
    o, g = oracle_of(w), md.MDSystem(w)
    gf, ge, gw = g.compute_forces()
    of, oe, ow = o.compute_forces()
    assert np.abs(gf - of).max() <= F_TOL and np.abs(ge - oe).max() <= 1e-12 * np.abs(oe).max()
    o.step(40, w.dt)
    g.step(40, w.dt)
    d = g.positions() - o.positions()
    d -= np.round(d / w.box) * w.box
    assert np.abs(d).max() <= X_TOL and g.stats()["error_flags"] == 0
    assert np.array_equal(g.neighbors(192)[1][:, :4] >= -1, np.ones((w.n_atoms, 4), bool))


def test_run_to_run_determinism(md):
    w = CASES["cfg2_small"]()
    res = []
    for _ in range(2):
        g = md.MDSystem(w)
        g.step(30, 1.0)
        res.append((g.positions(), g.compute_forces()[0], g.energies()[0]))
    assert np.array_equal(res[0][0], res[1][0]) and np.array_equal(res[0][1], res[1][1]) and np.array_equal(res[0][2], res[1][2])


def test_set_get_roundtrip_and_device_inputs(md):
    import torch
    w = CASES["cfg0_perm"]()
    g = md.MDSystem(w)
    assert np.array_equal(g.velocities(), w.velocities)
    g.build_neighbors()
    x = g.positions()
    v2 = np.random.default_rng(0).standard_normal(x.shape) * 0.01
    g.set_velocities(torch.from_numpy(v2).cuda())
    assert np.array_equal(g.velocities(), v2)
    f0 = g.compute_forces()[0]
    g.set_positions(x + 0.01)                    # rigid shift below skin/2: list kept, forces unchanged
    f1 = g.compute_forces()[0]
    assert g.stats()["rebuilds"] == 1 and np.abs(f1 - f0).max() < 1e-10
    g.set_positions(torch.from_numpy(x + w.box * np.array([1.0, -2.0, 3.0])).cuda())   # other periodic image
    assert np.abs(g.compute_forces()[0] - f0).max() < 1e-10 and g.stats()["rebuilds"] == 1
    g.set_positions(x + np.array([0.2, 0.0, 0.0]))   # beyond skin/2: must rebuild
    f2 = g.compute_forces()[0]
    assert g.stats()["rebuilds"] == 2 and np.abs(f2 - f0).max() < 1e-10
    # a system created from device tensors equals one created from host arrays
    gd = md.MDSystem(w, positions=torch.from_numpy(w.positions).cuda(), velocities=torch.from_numpy(w.velocities).cuda(),
                     types=torch.from_numpy(w.types).cuda())
    assert np.array_equal(gd.compute_forces()[0], md.MDSystem(w).compute_forces()[0])


def test_set_get_state(md):
    """md_set_state / md_get_state: one call for positions and velocities; an echoed state keeps the forces (no second
    evaluation, bit-identical trajectory); changed coordinates invalidate them."""
    w = CASES["cfg3a_small"]()
    a, b = md.MDSystem(w), md.MDSystem(w)
    a.step(30, w.dt)
    for it in range(30):
        x, v = b.get_state()
        assert np.array_equal(x, b.positions()) and np.array_equal(v, b.velocities())
        l0 = b.stats()["kernel_launches"]
        b.set_state(x, v)
        b.step(1, w.dt)
        if it:      # (the first step of a new system evaluates its initial forces)
            assert b.stats()["kernel_launches"] - l0 <= 6 + 10     # set, drift, density, force (+ a rebuild): no extra force evaluation
    assert np.array_equal(a.positions(), b.positions()) and np.array_equal(a.velocities(), b.velocities())
    # velocities only
    x, v = b.get_state()
    b.set_state(None, 0.5 * v)
    assert np.array_equal(b.velocities(), 0.5 * v) and np.array_equal(b.positions(), x)
    # changed positions: the next call evaluates the forces for them (against the oracle)
    x2 = x + 0.01 * np.sin(np.arange(x.size).reshape(x.shape))
    b.set_state(x2, v)
    o = oracle_of(w, positions=x2, velocities=v)
    assert np.abs(b.compute_forces()[0] - o.compute_forces()[0]).max() <= F_TOL
    # device tensors
    xt, vt = b.get_state(device_out=True)
    b.set_state(xt, vt)
    assert np.array_equal(xt.cpu().numpy(), b.positions())


@pytest.mark.parametrize("case", ["cfg3a_small", "cfg4_small", "alloy_tbsma_boxes", "cfg0"])
def test_step_get_state_equals_step_then_get_state(md, case, monkeypatch):
    """md_step_get_state(n, dt, x, v): the download of the positions runs beside the two passes of the last step; the state it
    returns and the trajectory it leaves are those of md_step(n) + md_get_state, bit for bit (pinned and pageable host
    buffers, across rebuilds, echoed back through md_set_state as bench.py's end-to-end leg does; device buffers, the
    predictor-corrector integrator and a barostat take the plain path)."""
    import torch
    monkeypatch.setenv("MD_FORK_MIN_ATOMS", "0")                              # these systems are below the size from which the call forks
    w = CASES[case]()
    a, b = md.MDSystem(w), md.MDSystem(w)
    n = w.n_atoms
    px, pv = torch.empty((n, 3), dtype=torch.float64).pin_memory().numpy(), torch.empty((n, 3), dtype=torch.float64).pin_memory().numpy()
    rebuilds = 0
    for it, k in enumerate([1, 1, 5, 1, 9, 1, 1, 16, 1, 3]):
        a.step(k, w.dt)
        xa, va = a.get_state()
        if it % 3 == 2:
            xb, vb = b.step_get_state(k, w.dt)                            # pageable numpy buffers
        else:
            xb, vb = b.step_get_state(k, w.dt, out=(px, pv))               # pinned
        assert np.array_equal(xa, xb) and np.array_equal(va, vb)
        if it % 2:
            b.set_state(xb, vb)                                            # echo: the forces stay valid
        rebuilds = b.stats()["rebuilds"]
    assert rebuilds >= 2 and a.stats()["rebuilds"] == rebuilds and b.stats()["error_flags"] == 0
    assert np.array_equal(a.positions(), b.positions()) and np.array_equal(a.velocities(), b.velocities())
    assert np.array_equal(a.compute_forces()[0], b.compute_forces()[0])
    # positions only / velocities only / device tensors
    a.step(2, w.dt)
    xb, _ = b.step_get_state(2, w.dt, out=(px, None))
    assert np.array_equal(a.positions(), xb)
    a.step(1, w.dt)
    _, vb = b.step_get_state(1, w.dt, out=(None, pv))
    assert np.array_equal(a.velocities(), vb)
    a.step(2, w.dt)
    xt, vt = b.step_get_state(2, w.dt, device_out=True)
    assert np.array_equal(a.positions(), xt.cpu().numpy()) and np.array_equal(a.velocities(), vt.cpu().numpy())
    with pytest.raises(md.MDError):
        b.step_get_state(0, w.dt)
    # the predictor-corrector integrator: plain path, same answers as step + get_state
    c, d = md.MDSystem(w), md.MDSystem(w)
    c.set_integrator(md.MD_INT_GEAR5); d.set_integrator(md.MD_INT_GEAR5)
    c.step(3, w.dt)
    xd, vd = d.step_get_state(3, w.dt, out=(px, pv))
    assert np.array_equal(c.positions(), xd) and np.array_equal(c.velocities(), vd)


@pytest.mark.parametrize("case,nsteps", [("cfg0", 100), ("cfg0_perm", 60), ("cfg1_small", 60), ("cfg2_small", 60), ("cfg3b_small", 40),
                                         ("cfg4_small", 60), ("alloy_tbsma_boxes", 60), ("alloy4_tables_rcut", 60)])
def test_gear_predictor_corrector_trajectory(md, case, nsteps):
    """Row f4, the paper's predictor-corrector integration as the five-value Gear scheme: the
    same start-up, predictor, skin/2 rule on the predicted positions, and corrector as the oracle."""
    w = CASES[case]()
    o = oracle_of(w)
    g = md.MDSystem(w)
    o.set_integrator(1)
    g.set_integrator(md.MD_INT_GEAR5)
    e0 = sum(x.sum() for x in g.energies())
    for n in (1, nsteps - 1):                       # (two calls: the derivative arrays carry over)
        o.step(n, w.dt)
        g.step(n, w.dt)
    d = g.positions() - o.positions()
    d -= np.round(d / w.box) * w.box
    assert np.abs(d).max() <= X_TOL
    assert np.abs(g.velocities() - o.velocities()).max() <= 1e-9
    so, sg = o.stats(), g.stats()
    assert sg["steps"] == nsteps and sg["error_flags"] == 0 and sg["graph_active"] == 0
    assert abs(sg["rebuilds"] - so["rebuilds"]) <= 1 and sg["rebuilds"] >= 2
    oep, oek = o.energies()
    gep, gek = g.energies()
    assert abs((gep.sum() + gek.sum()) - (oep.sum() + oek.sum())) <= 1e-10 * abs(oep.sum())
    if case == "cfg0":
        assert abs(gep.sum() + gek.sum() - e0) / w.n_atoms < 1e-7          # two orders better than velocity-Verlet at this dt
    # new velocities restart the scheme (a, j, s are rebuilt from the new state), on both sides alike
    v = 0.9 * g.velocities()
    g.set_velocities(v)
    o.set_velocities(v)
    g.step(10, w.dt)
    o.step(10, w.dt)
    d = g.positions() - o.positions()
    d -= np.round(d / w.box) * w.box
    assert np.abs(d).max() <= X_TOL
    # back to velocity-Verlet
    g.set_integrator(md.MD_INT_VERLET)
    o.set_integrator(0)
    g.step(10, w.dt)
    o.step(10, w.dt)
    d = g.positions() - o.positions()
    d -= np.round(d / w.box) * w.box
    assert np.abs(d).max() <= X_TOL and g.stats()["error_flags"] == 0


def test_gear_refusals_and_determinism(md):
    w = CASES["cfg3a_small"]()
    g = md.MDSystem(w)
    g.set_integrator(md.MD_INT_GEAR5)
    with pytest.raises(md.MDError):
        g.set_thermostat(300.0, 100.0)
    with pytest.raises(md.MDError):
        g.set_barostat(0.0, 1e4)
    with pytest.raises(md.MDError):
        g.set_integrator(7)
    g.step(30, 1.0)
    h = md.MDSystem(w)
    h.set_integrator(md.MD_INT_GEAR5)
    h.step(30, 1.0)
    assert np.array_equal(g.positions(), h.positions()) and np.array_equal(g.velocities(), h.velocities())
    t = md.MDSystem(w)
    t.set_thermostat(300.0, 100.0)
    with pytest.raises(md.MDError):
        t.set_integrator(md.MD_INT_GEAR5)


def test_prepare_step_is_only_setup(md):
    """md_prepare_step builds the graphs md_step will replay: no step is taken and the trajectory is the same bits."""
    w = CASES["cfg3a_small"]()
    a, b = md.MDSystem(w), md.MDSystem(w)
    x0 = a.positions()
    a.prepare_step(37, w.dt)
    assert np.array_equal(a.positions(), x0) and a.stats()["steps"] == 0
    a.step(37, w.dt)
    b.step(37, w.dt)
    assert np.array_equal(a.positions(), b.positions()) and np.array_equal(a.velocities(), b.velocities())
    assert a.stats()["graph_active"] == 1 and a.stats()["rebuilds"] == b.stats()["rebuilds"]
    a.set_option(md.MD_OPT_GRAPH, 0)
    a.prepare_step(5, w.dt)                              # nothing to prepare: still fine
    a.step(5, w.dt)
    b.step(5, w.dt)
    assert np.array_equal(a.positions(), b.positions())


def test_diagnostics_run(md):
    rate, mhz = md.fp64_dfma_rate()
    assert rate > 1e12 and mhz > 500
    g = md.probe_table_gather()
    assert len(g) == 4 and all(0.5 < v < 1e4 for v in g)


def test_error_codes(md):
    w = workloads.config(0, scale=4)             # L = 14.46 < 3 * 5.2
    with pytest.raises(md.MDError) as ei:
        md.MDSystem(w)
    assert ei.value.code == md.MD_EBOX
    w = workloads.config(0, scale=5)
    g = md.MDSystem(w, max_neighbors=20)
    g.build_neighbors()
    with pytest.raises(md.MDError) as ei:
        g.neighbors()
    assert ei.value.code == md.MD_EOVERFLOW and g.stats()["error_flags"] & md.MD_FLAG_OVERFLOW
    w.positions[1] = w.positions[0]
    g = md.MDSystem(w)
    with pytest.raises(md.MDError) as ei:
        g.compute_forces()
    assert ei.value.code == md.MD_ENONFINITE
    w = workloads.config(0, scale=5)
    w.positions[7, 1] = np.nan
    g = md.MDSystem(w)
    with pytest.raises(md.MDError) as ei:
        g.compute_forces()
    assert ei.value.code == md.MD_ENONFINITE
    w = workloads.config(0, scale=5)
    with pytest.raises(md.MDError) as ei:
        md.MDSystem(w, types=np.full(w.n_atoms, 2, np.int32))
    assert ei.value.code == md.MD_EINVAL
    g = md.MDSystem(w)
    with pytest.raises(md.MDError) as ei:
        g.neighbors()
    assert ei.value.code == md.MD_ESTATE


def test_list_build_at_the_edge_of_the_list_cutoff(md):
    """Pairs whose separation straddles r_l = r_c + skin by relative amounts from 1e-16 to 1e-5, at coordinates up to 590 A
    (where a float coordinate is rounded by up to 3e-5 A) and across the periodic boundary.  In boxes of this size the list
    build classifies the candidates on float copies of the coordinates and takes the canonical double-precision test
    (reading A3) inside the rounding band only (md_neighbor.cu): the pair sets must still be the
    oracle's, which takes every decision in double precision (brute force over all pairs here)."""
    rng = np.random.default_rng(12126332 + 77)
    L, rc, skin, K = 590.0, 4.9, 0.3, 3000
    rl = rc + skin
    a = rng.uniform(0.0, L, (K, 3))
    face = rng.integers(0, 3, K // 4)                                         # a quarter of the pairs at a face of the box
    a[np.arange(K // 4), face] = np.where(rng.random(K // 4) < 0.5, rng.uniform(0.0, 2.0, K // 4), rng.uniform(L - 2.0, L, K // 4))
    u = rng.normal(size=(K, 3))
    u /= np.linalg.norm(u, axis=1)[:, None]
    delta = 10.0 ** rng.uniform(-16.0, -5.0, K) * rng.choice([-1.0, 1.0], K)
    delta[:50] = 0.0                                                          # as close to r_l as the rounding of b allows
    b = a + (rl * (1.0 + delta))[:, None] * u                                 # some b lie outside [0, L): the build wraps them
    pos = np.concatenate([a, b])
    kw = dict(box=np.full(3, L), cutoff=rc, skin=skin, n_boxes=1, pot_kind=0, mass=np.array([63.546]), tbsma=workloads.cu_tbsma_params(rc),
              positions=pos, types=np.zeros(2 * K, np.int32))
    o = oracle_of(None, velocities=np.zeros_like(pos), **kw)
    o.build_neighbors(brute_force=True)
    oc, ol = o.neighbors(stride=16)
    g = md.MDSystem(velocities=None, **kw)
    g.build_neighbors()
    gc, gl = g.neighbors(stride=16)
    assert np.array_equal(gc, oc) and np.array_equal(gl, ol)
    assert 0.3 * K < oc[:K].sum() < 0.7 * K and g.stats()["error_flags"] == 0   # about half of the pairs are listed: the edge is straddled


def test_sparse_and_tiny_systems(md):
    """degenerate inputs: atoms with no neighbour at all, a box holding two atoms, a one-atom box batch."""
    base = dict(box=np.full(3, 40.0), velocities=None, cutoff=4.9, skin=0.3, n_boxes=1, pot_kind=0,
                mass=np.array([63.546]), tbsma=workloads.cu_tbsma_params(4.9))
    pos = np.array([[1.0, 1.0, 1.0], [20.0, 20.0, 20.0]])
    g = md.MDSystem(positions=pos, types=np.zeros(2, np.int32), **base)
    f, e, wv = g.compute_forces()
    assert np.all(f == 0) and np.all(e == 0) and np.all(wv == 0) and np.all(g.neighbors()[0] == 0)
    pos = np.array([[39.5, 0.2, 20.0], [1.5, 39.9, 20.0]])                # neighbours only through the periodic images
    g = md.MDSystem(positions=pos, types=np.zeros(2, np.int32), **base)
    o = oracle_of(None, positions=pos, types=np.zeros(2, np.int32), velocities=np.zeros((2, 3)), **{k: v for k, v in base.items() if k != "velocities"})
    assert np.abs(g.compute_forces()[0] - o.compute_forces()[0]).max() < 1e-12 and np.abs(g.compute_forces()[0]).max() > 0.1
    pos = np.tile(np.array([[3.0, 4.0, 5.0]]), (6, 1))                     # 6 boxes x 1 atom: never a neighbour
    g = md.MDSystem(positions=pos, types=np.zeros(6, np.int32), **{**base, "n_boxes": 6})
    assert np.all(g.compute_forces()[0] == 0) and g.energies()[0].shape == (6,)
