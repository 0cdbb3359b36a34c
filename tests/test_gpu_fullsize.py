"""Parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (md_step through the C ABI,
default options): the CUDA path against the CPU oracle on the same seeded inputs, every atom compared.

The oracle (OpenMP over atoms) needs about 0.25 s per step per million atoms, so the step counts are bounded;
tolerances are north_star's: pair sets bit-exact, |dF| <= 1e-9 eV/A, total energy 1e-12 relative, positions 1e-8 A.
"""
import numpy as np
import pytest

import workloads

pytestmark = pytest.mark.gpu

F_TOL, E_REL, X_TOL = 1e-9, 1e-12, 1e-8

#        config  steps  list stride
FULL = [("1", 100, 96),       # 65,536 Fe, tables
        ("2", 40, 96),        # 2048 boxes x 500 Cu, every pair of a box crosses the 3x3x3 stencil
        ("3a", 100, 96),      # 1,048,576 Cu, r_c 4.9: the bench workload
        ("3b", 20, 192),      # r_c 6.5, ~134 list entries
        ("4", 20, 96)]        # 4,194,304 W, tables, 2 keV PKA: a rebuild every other step


@pytest.fixture(scope="module")
def md():
    import torch
    assert torch.cuda.is_available(), "these tests need the B200"
    import paper_1212_6332_b200 as m
    m.lib()
    return m


@pytest.mark.parametrize("cfg,nsteps,stride", FULL)
def test_full_size(md, cfg, nsteps, stride):
    from oracle import Oracle
    w = workloads.config(cfg)
    o, g = Oracle(w), md.MDSystem(w)

    # neighbour pair sets, every atom, bit-exact
    o.build_neighbors()
    g.build_neighbors()
    oc, ol = o.neighbors(stride=stride)
    gc, gl = g.neighbors(stride=stride)
    assert np.array_equal(gc, oc)
    assert np.array_equal(gl, ol)
    del ol, gl

    # densities, forces, per-atom energies, virial
    of, oe, ow = o.compute_forces()
    gf, ge, gw = g.compute_forces()
    orho, ofp = o.densities()
    grho, gfp = g.densities()
    assert np.abs(grho - orho).max() <= 1e-12 * np.abs(orho).max()
    assert np.abs(gfp - ofp).max() <= 1e-12 * np.abs(ofp).max()
    assert np.abs(gf - of).max() <= F_TOL
    assert np.abs(ge - oe).max() <= 1e-12 * np.abs(oe).max()
    oep, oek = o.energies()
    gep, gek = g.energies()
    assert np.abs(gep - oep).max() <= E_REL * np.abs(oep).max()
    assert abs(gep.sum() - oep.sum()) <= E_REL * abs(oep.sum())
    assert np.abs(gw - ow).max() <= 1e-11 * np.abs(ow).max()
    del of, gf, oe, ge

    # the trajectory, as bench.py runs it
    o.step(nsteps, w.dt)
    g.step(nsteps, w.dt)
    d = g.positions() - o.positions()
    d -= np.round(d / w.box) * w.box            # the two sides may have wrapped at different steps
    assert np.abs(d).max() <= X_TOL
    assert np.abs(g.velocities() - o.velocities()).max() <= 1e-9
    so, sg = o.stats(), g.stats()
    assert sg["steps"] == nsteps and sg["error_flags"] == 0
    assert abs(sg["rebuilds"] - so["rebuilds"]) <= 1
    if cfg == "4":
        assert sg["rebuilds"] >= nsteps // 3     # the cascade does stress the rebuild rate


def test_sixteen_million_atoms(md):
    """north_star: one B200's memory holds multi-million-atom systems directly.  Cu fcc 160^3 = 16,384,000 atoms
    (workspace ~10 GB): every force component and the per-atom energies against the oracle, then a few steps."""
    from oracle import Oracle
    w = workloads.config("3a", scale=160)
    assert w.n_atoms == 16_384_000
    o, g = Oracle(w), md.MDSystem(w)
    of, oe, ow = o.compute_forces()
    gf, ge, gw = g.compute_forces()
    assert np.abs(gf - of).max() <= F_TOL
    assert np.abs(ge - oe).max() <= 1e-12 * np.abs(oe).max()
    assert abs(ge.sum() - oe.sum()) <= E_REL * abs(oe.sum())
    assert np.abs(gw - ow).max() <= 1e-11 * np.abs(ow).max()
    st = g.stats()
    assert st["error_flags"] == 0 and st["max_neighbors"] == o.stats()["max_neighbors"]
    assert st["list_entries"] == int(o.neighbors(stride=96)[0].sum())          # same number of listed pairs
    del of, gf, oe, ge
    o.step(3, w.dt)
    g.step(3, w.dt)
    d = g.positions() - o.positions()
    d -= np.round(d / w.box) * w.box
    assert np.abs(d).max() <= X_TOL and g.stats()["error_flags"] == 0


def test_thermostat_and_barostat_at_full_size(md):
    """rows f1a/f1b on the bench workload: 1,048,576 Cu atoms, eq.(4) bath at 600 K and eq.(5) pressure control at P0 = 0."""
    from oracle import Oracle
    w = workloads.config("3a")
    o, g = Oracle(w), md.MDSystem(w)
    for x in (o, g):
        x.set_thermostat(600.0, 80.0)
        x.set_barostat(0.0, 20.0)
    o.step(30, w.dt)
    g.step(30, w.dt)
    assert np.abs(g.box() / o.box() - 1.0).max() <= 1e-13 and np.abs(g.box() / w.box - 1.0).max() > 1e-6
    d = g.positions() - o.positions()
    d -= np.round(d / o.box()) * o.box()
    assert np.abs(d).max() <= X_TOL
    assert np.abs(g.velocities() - o.velocities()).max() <= 1e-9
    assert abs(g.pressure() - o.pressure()) <= 1e-10 * max(abs(o.pressure()), 1e-3)
    assert g.stats()["error_flags"] == 0
