"""Pins for f2 (Eq. 16-18): the oracle's finite-T Thomas-Fermi average atom, the
norm-conserving pseudo-density, the Eq. 18 inversion, the radial transform, the table interpolation, and the tabulated
pseudopotential inside the 3D SCF.  No GPU.  P:NNN = PAPER.md line."""
import os

import mpmath as mp
import numpy as np
import pytest

import arche_inputs as ai

PI = np.pi
HA = 27.211386245988
GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _const(name):
    for line in open(os.path.join(GOLD, "constants.txt")):
        if line.startswith(name + " "):
            return float(line.split()[1])
    raise KeyError(name)


def _al():
    rho = 2.7 / (26.98 * 1.66053906660e-24) * (0.529177210903e-8) ** 3      # ions per bohr^3 at 2.7 g/cc
    return 13.0, (3.0 / (4.0 * PI * rho)) ** (1.0 / 3.0), 100.0 / HA


@pytest.fixture(scope="module")
def al_atom(orc):
    Z, rws, kT = _al()
    r, n, mu, it = orc.aa_solve(Z, rws, kT, 0, 601)
    return dict(Z=Z, rws=rws, kT=kT, r=r, n=n, mu=mu, it=it, n0=(2 * Z) ** 1.5 / (3 * PI ** 2))


def test_fd_wide_range(orc):
    """oracle_fd_wide: closed forms outside the quadrature's range against the polylogarithm, and continuity where it
    hands over to oracle_fd (eta = -40 and 500)"""
    mp.mp.dps = 40
    for tj in (-1, 1, 3):
        j = mp.mpf(tj) / 2
        for eta in (-300.0, -41.0, 501.0, 2.0e3, 1.0e5):
            if eta > 0:    # Li_s(-e^eta) directly is unstable for huge eta: use the reflection-free Sommerfeld series in mp
                ref = mp.quad(lambda t: t ** j / (mp.exp(t - eta) + 1), [0, eta - 60, eta, eta + 60, eta + 200])
            else:
                ref = -mp.gamma(j + 1) * mp.polylog(j + 1, -mp.exp(eta))
            assert abs(orc.fd_wide(tj, eta) / float(mp.re(ref)) - 1) < 2e-13, (tj, eta)
        for eta in (-40.0, 500.0):
            assert abs(orc.fd_wide(tj, eta - 1e-9) / orc.fd_wide(tj, eta + 1e-9) - 1) < 1e-8
            assert abs(orc.fd_wide(tj, np.nextafter(eta, 1e9)) / orc.fd(tj, eta)[0] - 1) < 5e-13


def test_average_atom_solves_eq9_in_the_sphere(orc, al_atom):
    """neutrality, the Thomas-Fermi relation with a potential rebuilt here by numpy quadrature, zero electrostatic
    potential at r_ws (neutral sphere), and the nuclear limit r^(3/2) n -> (2Z)^(3/2)/(3 pi^2)"""
    a = al_atom; r, n, Z, kT = a["r"], a["n"], a["Z"], a["kT"]
    x = np.sqrt(r)
    g1 = 8 * PI * x ** 5 * n
    Q = np.concatenate([[0.0], np.cumsum(0.5 * (g1[1:] + g1[:-1]) * np.diff(x))])
    assert abs(Q[-1] / Z - 1) < 2e-5                                   # trapezoid here; the oracle's Simpson is exact to 1e-13
    g2 = 8 * PI * x ** 3 * n; g2[0] = 8 * PI * a["n0"]
    I2 = np.concatenate([[0.0], np.cumsum(0.5 * (g2[1:] + g2[:-1]) * np.diff(x))])
    V = -Z / r[1:] + Q[1:] / r[1:] + (I2[-1] - I2[1:])
    assert abs(V[-1]) < 1e-4                                           # neutral sphere: potential vanishes at r_ws
    cTF = np.sqrt(2.0) / PI ** 2 * kT ** 1.5
    for i in (5, 60, 200, 450, 599):
        assert abs(cTF * orc.fd_wide(1, (a["mu"] - V[i - 1]) / kT) / n[i] - 1) < 2e-4, i
    assert abs(n[1] * r[1] ** 1.5 / a["n0"] - 1) < 1e-3
    assert a["it"] < 60                                                # More's mixing converges the atom quickly


def test_average_atom_energy_against_the_papers_number(orc, al_atom):
    """P:215 prints -6550 eV for Al at rho_0, 100 eV with the Coulomb potential.  K_e + E_en + E_H of the oracle's TF
    atom (no XC) is -6649.2 eV, grid-converged to 1e-6: within 2% of the paper's value (its model [21] is only cited)."""
    a = al_atom
    E = orc.aa_energy(a["kT"], 0, a["r"], a["n"], a["n0"], None, a["Z"])
    assert abs(E.sum() * HA / _const("paper_aa_energy_al_coulomb_eV") - 1) < 0.02
    r2, n2, mu2, _ = orc.aa_solve(a["Z"], a["rws"], a["kT"], 0, 301)
    E2 = orc.aa_energy(a["kT"], 0, r2, n2, a["n0"], None, a["Z"])
    assert abs(E2.sum() / E.sum() - 1) < 1e-6 and abs(mu2 / a["mu"] - 1) < 1e-6
    # virial-like sanity of the parts: kinetic > 0, electron-nucleus < 0 and dominant, Hartree > 0
    assert E[0] > 0 and E[2] > 0 and E[1] < -(E[0] + E[2])


def test_eq18_inverts_the_average_atom_back_to_the_coulomb_potential(orc, al_atom):
    """Eq. 18 applied to the average-atom density itself must return the potential it was solved in, -Z/r, at every
    radius: pins the inverse Fermi-Dirac function, both Hartree integrals and the sign of every term of Eq. 18"""
    a = al_atom
    V = orc.aa_invert(a["kT"], 0, a["r"], a["n"], a["n0"], a["mu"])
    assert np.abs(V[2:] * a["r"][2:] / a["Z"] + 1).max() < 1e-9


# ---------------------------------------------------------------- Eq. 16-17: pseudo-density; Eq. 18: pseudopotential
@pytest.mark.parametrize("frac", [0.17, 0.5])
def test_norm_conserving_pseudo_density_and_potential(orc, al_atom, frac):
    a = al_atom; r, n = a["r"], a["n"]
    N = len(r); x = np.sqrt(r); h = x[1]
    ic = int(round((N - 1) * np.sqrt(frac)))
    ps, (ca, cb, cc) = orc.aa_pseudize(r, n, ic)
    assert np.array_equal(ps[ic + 1:], n[ic + 1:])                           # Eq. 16, r >= r_cut
    f = lambda rr: np.exp(ca + cb * rr ** 2 + cc * rr ** 4)
    assert abs(f(r[ic]) / n[ic] - 1) < 1e-12                                 # Eq. 17, value
    # slope: analytic derivative of the exponential form against a one-sided difference of n OUTSIDE r_cut
    dps = (2 * cb * r[ic] + 4 * cc * r[ic] ** 3) * f(r[ic])
    dn_out = (-3 * n[ic] + 4 * n[ic + 1] - n[ic + 2]) / (2 * h) / (2 * x[ic])   # dn/dr = (dn/dx)/(2x)
    assert abs(dps / dn_out - 1) < 5e-4
    # norm conservation: charge inside r_cut (Simpson by hand on an even number of panels)
    m = ic if ic % 2 == 0 else ic - 1
    w = np.ones(m + 1); w[1:-1:2] = 4; w[2:-1:2] = 2
    q = lambda d: (w * 8 * PI * x[:m + 1] ** 5 * d[:m + 1]).sum() * h / 3
    if m == ic:
        assert abs(q(ps) / q(n) - 1) < 1e-9
    assert ps[1] < n[1] and np.all(ps > 0)                                   # "less polarized in the vicinity of the nucleus"
    # Eq. 18: Coulomb beyond r_cut, finite and smooth at the nucleus
    V = orc.aa_invert(a["kT"], 0, r, ps, 0.0, a["mu"])
    assert np.abs(V[ic:] * r[ic:] / a["Z"] + 1).max() < 1e-6
    assert np.isfinite(V[1]) and abs(V[1] - V[2]) < 1e-3 * abs(V[1]) and V[1] > -a["Z"] / r[3]


def test_pseudo_atom_energy_fixes_the_cutoff_fraction(orc, al_atom):
    """The paper does not give r_cut/r_ws but prints the pseudo-atom energy of Al at rho_0, 100 eV: -2971 eV
    (P:215).  The energy of the pseudo-atom rises monotonically with r_cut; it equals the paper's value at
    r_cut = 0.17 r_ws (reading A22), within the 2% by which the Coulomb-atom energies differ."""
    a = al_atom; r, n = a["r"], a["n"]; N = len(r)
    E = []
    for frac in (0.12, 0.17, 0.25):
        ic = int(round((N - 1) * np.sqrt(frac)))
        ps, _ = orc.aa_pseudize(r, n, ic)
        V = orc.aa_invert(a["kT"], 0, r, ps, 0.0, a["mu"])
        E.append(orc.aa_energy(a["kT"], 0, r, ps, 0.0, V, a["Z"]).sum() * HA)
    assert E[0] < E[1] < E[2]
    assert abs(E[1] / _const("paper_aa_energy_al_pseudo_eV") - 1) < 0.03, E


def test_radial_transform_of_a_gaussian(orc):
    """f(r) = exp(-r^2/(2 s^2)):  int f 4 pi r^2 sinc(2 pi k r) dr = (2 pi s^2)^(3/2) exp(-2 pi^2 s^2 k^2) (P:146 convention)"""
    N = 801; R = 9.0; s = 0.7
    x = np.linspace(0, np.sqrt(R), N); r = x * x
    k = np.array([0.0, 0.05, 0.3, 0.9])
    got = orc.radial_ft(r, np.exp(-r * r / (2 * s * s)), N - 1, k)
    ref = (2 * PI * s * s) ** 1.5 * np.exp(-2 * PI ** 2 * s * s * k * k)
    assert np.abs(got - ref).max() < 1e-9 * ref[0]


def test_table_interpolation_rule(orc):
    """cubic Lagrange through four nodes: exact for cubics (value and derivative), including the clamped end intervals"""
    dk = 0.05; k = dk * np.arange(12)
    p = lambda q: 0.3 - 1.1 * q + 2.0 * q * q - 0.7 * q ** 3
    dp = lambda q: -1.1 + 4.0 * q - 2.1 * q * q
    tab = np.ascontiguousarray(p(k))
    import ctypes as C
    for q in (0.0, 0.012, 0.05, 0.261, 0.5, 0.549):
        d = C.c_double()
        v = orc.lib().oracle_table_interp(len(tab), dk, tab.ctypes.data_as(C.POINTER(C.c_double)), q, C.byref(d))
        assert abs(v - p(q)) < 1e-14 and abs(d.value - dp(q)) < 1e-12, q


# ---------------------------------------------------------------- the table inside the 3D SCF
def _ashcroft_table(rc, dk, nk):
    """non-Coulomb part of the Ashcroft form factor per unit charge: -cos(2 pi k rc)/(pi k^2) = -1/(pi k^2) + Du(k)"""
    k = dk * np.arange(nk)
    du = np.empty(nk)
    du[1:] = (1.0 - np.cos(2 * PI * k[1:] * rc)) / (PI * k[1:] ** 2)
    du[0] = 2 * PI * rc * rc                                           # limit k -> 0 = alpha_s/Z of Eq. 55
    return du


def test_ashcroft_recovered_from_a_synthetic_table(orc):
    """psp = 1 fed the Ashcroft form factor as a table must reproduce psp = 0: potential, energies (incl. the k = 0
    constant E_ie0 from Du(0)), density, forces and the stress table, to the interpolation error of the cubic"""
    cfg = ai.make_small(n_ions=3, cell=[7.0, 7.6, 8.3], grid=(12, 12, 12), T_eV=10.0, seed=5, dmin=2.5)
    kw = dict(init_mode=0, scf_tol_F=1e-12, scf_tol_dn=1e-11, scf_max_iter=400)
    dk = 0.002; nk = int(1.6 / dk) + 4
    oa = orc.Oracle(cfg, **kw); ra = oa.scf_solve(cfg["pos"])
    ot = orc.Oracle(cfg, psp_table=_ashcroft_table(1.12, dk, nk), psp_dk=dk, **kw); rt = ot.scf_solve(cfg["pos"])
    assert ra["converged"] and rt["converged"] and ra["scf_iters"] == rt["scf_iters"]
    assert np.abs(ot.get_complex("Vhat_ie") - oa.get_complex("Vhat_ie")).max() < 1e-8 * np.abs(oa.get_complex("Vhat_ie")).max()
    for key in ("F_total", "E_ie", "E_ie0", "E_H", "mu"):
        assert abs(rt[key] - ra[key]) < 1e-8 * max(1.0, abs(ra[key])), key
    assert abs(rt["E_ie0"] / ra["E_ie0"] - 1) < 1e-14
    assert np.abs(ot.get_real("n_a") - oa.get_real("n_a")).max() < 1e-8 * oa.get_real("n_a").max()
    assert np.abs(ot.forces() - oa.forces()).max() < 1e-7 * np.abs(oa.forces()).max()
    sa, st = oa.stress(), ot.stress()
    assert np.abs(st["ie"] - sa["ie"]).max() < 1e-6 * np.abs(sa["ie"]).max() and abs(st["P"] / sa["P"] - 1) < 1e-6
    # a table that does not reach the largest |k| of the grid is refused
    with pytest.raises(ValueError):
        orc.Oracle(cfg, psp_table=_ashcroft_table(1.12, dk, 100), psp_dk=dk, **kw)


@pytest.fixture(scope="module")
def hydrogen(orc):
    """dense hydrogen: 4 protons, r_ws = 1.5 bohr, kT = 2 Ha, 16^3 grid; average-atom pseudopotential with
    r_cut = 0.5 r_ws from the oracle's own generator"""
    Z, rws, kT, n = 1.0, 1.5, 2.0, 401
    r, dens, mu, _ = orc.aa_solve(Z, rws, kT, 0, n)
    ic = int(round((n - 1) * np.sqrt(0.5)))
    ps, abc = orc.aa_pseudize(r, dens, ic)
    V = orc.aa_invert(kT, 0, r, ps, 0.0, mu)
    dV = np.zeros(n); dV[1:] = V[1:] + Z / r[1:]
    dk = 0.02; k = dk * np.arange(int(4.0 / dk) + 3)
    table = orc.radial_ft(r, dV, ic, k) / Z
    L = (4 * 4.0 / 3.0 * PI * rws ** 3) ** (1.0 / 3.0)
    cfg = ai.make_small(n_ions=4, cell=[L, L, L], grid=(16, 16, 16), seed=17, dmin=1.2)
    cfg["Z"] = np.full(4, Z); cfg["kT"] = kT; cfg["xc"] = 0
    return dict(cfg=cfg, table=table, dk=dk, Z=Z, rws=rws, kT=kT, n=n, ic=ic, mu=mu, abc=abc)


def test_average_atom_pseudopotential_in_the_scf_forces_and_stress(orc, hydrogen):
    """the paper's pseudopotential path end to end: SCF with the tabulated form factor; the forces are minus the
    gradient of the re-converged free energy and the diagonal stress its strain derivative (pins the table lookup in
    V_ie, the force sum, E_ie0 = (N_e/|Omega|) sum_j Z_j Du(0) and the derivative of the interpolant in sigma^ie)"""
    h_ = hydrogen; cfg = h_["cfg"]
    alpha = orc.ewald_alpha(cfg["cell"], cfg["grid"])
    kw = dict(psp_table=h_["table"], psp_dk=h_["dk"], ewald_alpha=alpha, init_mode=0, scf_tol_F=1e-12, scf_tol_dn=1e-12,
              scf_max_iter=400)
    o = orc.Oracle(cfg, **kw)
    pos = cfg["pos"]
    r = o.scf_solve(pos); assert r["converged"] == 1
    F = o.forces()
    dV = float(np.prod(cfg["cell"])) / 16 ** 3
    assert abs(o.get_real("n_a").sum() * dV - 4.0) < 1e-12
    def fd(j, c, h):
        p = pos.copy(); p[j, c] += h; fp = o.scf_solve(p)["F_total"]
        p[j, c] -= 2 * h; fm = o.scf_solve(p)["F_total"]
        return -(fp - fm) / (2 * h)
    for j, c in ((0, 0), (3, 2)):
        rich = (4 * fd(j, c, 1e-3) - fd(j, c, 2e-3)) / 3
        assert abs(rich - F[j, c]) < 2e-7 * np.abs(F).max(), (j, c, rich, F[j, c])
    o.scf_solve(pos); s = o.stress()
    vol = float(np.prod(cfg["cell"])); e = 2e-4
    def strained(mu_, eps):
        c2 = dict(cfg); cell = np.array(cfg["cell"], float); p2 = pos.copy()
        cell[mu_] *= 1 + eps; p2[:, mu_] *= 1 + eps
        c2["cell"] = cell
        return orc.Oracle(c2, **kw).scf_solve(p2)["F_total"]
    dF = (strained(1, e) - strained(1, -e)) / (2 * e * vol)
    assert abs(dF - s["total"][1]) < 2e-6 * abs(s["total"][1]), (dF, s["total"][1])


def test_product_generator_agrees_with_the_oracle(orc, hydrogen):
    """paper_2606_13283_b200/aa_pseudopotential.py (numpy pre-processing shipped with the product) and the oracle's C
    generator are independent codes: same chemical potential, same a, b, c, same table"""
    from paper_2606_13283_b200 import aa_pseudopotential as aa
    h_ = hydrogen
    rho = 3.0 / (4.0 * PI * h_["rws"] ** 3)
    tab = aa.make_table(h_["Z"], rho, h_["kT"], k_max=4.0, dk=h_["dk"], xc=0, rcut_frac=0.5, n=h_["n"])
    assert abs(tab["mu"] / h_["mu"] - 1) < 1e-9
    assert np.abs(np.array(tab["abc"]) / h_["abc"] - 1).max() < 1e-7
    m = min(len(tab["table"]), len(h_["table"]))
    assert np.abs(tab["table"][:m] - h_["table"][:m]).max() < 1e-9 * np.abs(h_["table"]).max()
    # its Fermi-Dirac evaluation against the oracle's quadrature
    for tj in (-1, 1, 3):
        eta = np.array([-35.0, -29.0, -3.0, 0.0, 4.0, 31.0, 59.0, 61.0, 400.0])
        assert np.abs(aa.fermi_dirac(tj, eta) / np.array([orc.fd_wide(tj, e) for e in eta]) - 1).max() < 1e-11
