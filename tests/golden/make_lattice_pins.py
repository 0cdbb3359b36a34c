"""Closed-form pins for the oracle, independent of oracle/ and of the CUDA path.

For a PERFECT crystal every atom is equivalent, so eq.(1) of the paper
collapses to a sum over neighbour shells:

    E_i = F( sum_s n_s f(r_s) ) + 1/2 sum_s n_s V(r_s),      r_s = a sqrt(m_s) / 2,

with n_s the number of lattice vectors of squared length m_s (a/2)^2 (enumerated exactly in
integers).  The virial trace per atom follows from homogeneous strain, W_i = -a dE_i/da
(eq.(6): pressure from sum f.r).  Everything is evaluated with mpmath at
40 significant digits, so the numbers written to lattice_pins.txt are exact to double
precision.  The dimer lines are eq.(1) for two atoms.  This script is the only writer of
tests/golden/lattice_pins.txt:

    python tests/golden/make_lattice_pins.py
"""
import itertools
import os
from collections import Counter

from mpmath import diff, exp, findroot, mp, mpf, sqrt

mp.dps = 40


def shells(kind, a, rmax):
    """[(m, count)] with r = a sqrt(m)/2 < rmax; integer enumeration in half-lattice units."""
    c = Counter()
    n = int(rmax / a) + 2
    basis = [(0, 0, 0), (0, 1, 1), (1, 0, 1), (1, 1, 0)] if kind == "fcc" else [(0, 0, 0), (1, 1, 1)]
    for i, j, k in itertools.product(range(-n, n + 1), repeat=3):
        for b in basis:
            x, y, z = 2 * i + b[0], 2 * j + b[1], 2 * k + b[2]
            m = x * x + y * y + z * z
            if m and mpf(m) / 4 * a * a < rmax * rmax:
                c[m] += 1
    return sorted(c.items())


def switch(r, ron, rc):
    if r <= ron:
        return mpf(1)
    if r >= rc:
        return mpf(0)
    t = (r - ron) / (rc - ron)
    return 1 - t ** 3 * (10 - 15 * t + 6 * t * t)


CU = dict(A=mpf("0.0855"), xi=mpf("1.224"), p=mpf("10.96"), q=mpf("2.278"), r0=mpf("2.5562"))


def tbsma(a, rc, ron, aref):
    rep = rho = mpf(0)
    for m, cnt in shells("fcc", aref, rc + mpf("0.5")):
        r = a * sqrt(mpf(m)) / 2
        if r >= rc:
            continue
        s = switch(r, ron, rc)
        rep += cnt * CU["A"] * exp(-CU["p"] * (r / CU["r0"] - 1)) * s
        rho += cnt * CU["xi"] ** 2 * exp(-2 * CU["q"] * (r / CU["r0"] - 1)) * s
    return rep - sqrt(rho), rep, rho


def eam(a, rc, re, aref):
    rho = pair = mpf(0)
    for m, cnt in shells("bcc", aref, rc + mpf("0.5")):
        r = a * sqrt(mpf(m)) / 2
        if r >= rc:
            continue
        x = r / re - 1
        rho += cnt * exp(-6 * x)
        pair += cnt * (mpf("0.4") * exp(-8 * x) - mpf("0.6") * exp(-4 * x))
    return -mpf("2.5") * sqrt(rho / 20) + pair / 2, pair / 2, rho


def main():
    out = ["# closed-form lattice sums, mpmath 40 digits; written by tests/golden/make_lattice_pins.py",
           "# eq.(1) PAPER.md:75 on a perfect crystal; virial = -a dE/da (eq.(6) PAPER.md:105-111)"]

    def put(k, v):
        out.append(f"{k} = {mp.nstr(v, 20)}")

    a = mpf("3.615")
    for tag, rc, ron in (("cu49", mpf("4.9"), mpf("4.4")), ("cu65", mpf("6.5"), mpf("6.0"))):
        E, rep, rho = tbsma(a, rc, ron, a)
        put(f"{tag}.E", E); put(f"{tag}.rep", rep); put(f"{tag}.rho", rho); put(f"{tag}.Fp", -1 / (2 * sqrt(rho)))
        put(f"{tag}.W", -a * diff(lambda x: tbsma(x, rc, ron, a)[0], a))
        aeq = findroot(lambda x: diff(lambda y: tbsma(y, rc, ron, a)[0], x), a)
        put(f"{tag}.a_eq", aeq); put(f"{tag}.E_eq", tbsma(aeq, rc, ron, a)[0])
        put(f"{tag}.n_in_cutoff", sum(c for m, c in shells("fcc", a, rc)))
        put(f"{tag}.n_in_list", sum(c for m, c in shells("fcc", a, rc + mpf("0.3"))))
    for tag, a, rc, re in (("fe", mpf("2.855"), mpf("5.0"), mpf("2.4725")), ("w", mpf("3.165"), mpf("5.5"), mpf("2.741"))):
        E, pair, rho = eam(a, rc, re, a)
        put(f"{tag}.E", E); put(f"{tag}.pair", pair); put(f"{tag}.rho", rho)
        put(f"{tag}.Fp", -mpf("2.5") / (2 * sqrt(20 * rho)))
        put(f"{tag}.W", -a * diff(lambda x: eam(x, rc, re, a)[0], a))
        put(f"{tag}.n_in_cutoff", sum(c for m, c in shells("bcc", a, rc)))
        put(f"{tag}.n_in_list", sum(c for m, c in shells("bcc", a, rc + mpf("0.3"))))

    # F(rho) above the last node of its table (reading A8: linear continuation F(rho_max) + F'(rho_max)(rho - rho_max)):
    # the Fe-form EAM with rho_max = 8 < rho_lattice = 10.76, so every atom of the perfect crystal sits on the continuation
    a, rc, re, rmax = mpf("2.855"), mpf("5.0"), mpf("2.4725"), mpf(8)
    _, pair, rho = eam(a, rc, re, a)
    Fmax, Fpmax = -mpf("2.5") * sqrt(rmax / 20), -mpf("2.5") / (2 * sqrt(20 * rmax))
    put("fe_rhomax8.E", Fmax + Fpmax * (rho - rmax) + pair); put("fe_rhomax8.Fp", Fpmax)

    def e_cont(x):
        _, pr, rh = eam(x, rc, re, a)
        return Fmax + Fpmax * (rh - rmax) + pr
    put("fe_rhomax8.W", -a * diff(e_cont, a))

    # Cu dimer, eq.(1) for two atoms: E = 2 [ F(f(r)) + V(r)/2 ], force on atom 1 along (r1-r2)/r is -dE/dr
    def dimer(r, ron=mpf("4.4"), rc=mpf("4.9")):
        s, x = switch(r, ron, rc), r / CU["r0"] - 1
        return 2 * CU["A"] * exp(-CU["p"] * x) * s - 2 * sqrt(CU["xi"] ** 2 * exp(-2 * CU["q"] * x) * s)
    for tag, r in (("dimer25", mpf("2.5")), ("dimer46", mpf("4.6"))):
        put(f"{tag}.E", dimer(r)); put(f"{tag}.F", -diff(dimer, r))
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "lattice_pins.txt")
    with open(path, "w") as fh:
        fh.write("\n".join(out) + "\n")
    print("\n".join(out))


if __name__ == "__main__":
    main()
