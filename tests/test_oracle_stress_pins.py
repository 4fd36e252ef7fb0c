"""Pins for the oracle's stress tensor and pressure (no GPU).  P:NNN = PAPER.md line.

The stress formulas are pinned against what they must equal:
strain derivatives of the energies.  Nothing below evaluates a stress formula; every expected value is a finite
difference of an energy (the oracle's own converged F for the diagonal, definitions of the individual energy terms
under a general, sheared cell for all six components) or a textbook identity (ideal Fermi gas, P = -dF/dV).
"""
import math

import numpy as np
import pytest

import arche_inputs as ai

PI = np.pi
VOIGT = [(0, 0), (1, 1), (2, 2), (1, 2), (0, 2), (0, 1)]


def _solve(orc, cfg, pos, **kw):
    o = orc.Oracle(cfg, **kw)
    r = o.scf_solve(pos)
    assert r["rc"] == 0 and r["converged"], r
    return o, r


# ---------------------------------------------------------------- uniform gas (Eq. 39, Eq. 34)
@pytest.mark.parametrize("xc", [0, 1])
def test_uniform_gas_pressure_is_minus_dF_dV(orc, xc):
    """No ions, N_e electrons on a neutralising background: the density is uniform, F = F_0 + E_xc, and
    P = -dF/dV at fixed N_e, T.  With xc = 0 this is the ideal Fermi gas, P = 2 K_e/(3|Omega|)."""
    kT = 10.0 / ai.HARTREE_EV
    Ne, L, h = 6.0, 7.0, 1e-4

    def run(scale):
        cfg = dict(cell=[L * scale, L, L], grid=[6, 6, 6], Z=np.zeros(0), mass=np.zeros(0), kT=kT, xc=xc)
        o = orc.Oracle(cfg, n_electrons=Ne, init_mode=0)
        r = o.scf_solve(np.zeros((0, 3)))
        assert r["converged"]
        return o, r

    o, r = run(1.0)
    s = o.stress()
    vol = L ** 3
    dFdV = (run(1 + h)[1]["F_total"] - run(1 - h)[1]["F_total"]) / (2 * h * vol)
    assert abs(s["P"] + dFdV) < 2e-7 * abs(s["P"])
    assert np.allclose(s["total"][:3], -s["P"], rtol=0, atol=1e-14) and np.abs(s["total"][3:]).max() < 1e-20
    if xc == 0:
        assert abs(s["P"] - 2 * r["K_e"] / (3 * vol)) < 1e-14
        assert np.all(s["xc"] == 0)
    for row in ("i", "pp", "pm", "je", "ie"):
        assert np.all(s[row] == 0), row
    assert np.abs(s["ee"]).max() < 1e-20


# ---------------------------------------------------------------- full SCF: diagonal = dF/d(eps_mm)/|Omega|
def _strained(cfg, mu, e):
    c = dict(cfg)
    cell = np.array(cfg["cell"], dtype=float).copy(); pos = cfg["pos"].copy()
    cell[mu] *= 1 + e; pos[:, mu] *= 1 + e
    c["cell"] = cell; c["pos"] = pos
    return c


@pytest.mark.parametrize("xc", [0, 1])
def test_diagonal_stress_is_strain_derivative_of_converged_free_energy(orc, xc):
    """F is stationary in n at the fixed point, so dF/d(eps) at fixed scaled ion coordinates is the explicit
    derivative the stress formulas state (sigma^e + sigma^xc + sigma^ii + sigma^ee + sigma^ie, sigma^i = 0)."""
    cfg = ai.make_small(n_ions=3, cell=[7.0, 7.6, 8.3], grid=(12, 12, 12), T_eV=10.0, seed=5, dmin=2.5)
    cfg["xc"] = xc
    alpha = orc.ewald_alpha(cfg["cell"], cfg["grid"])
    kw = dict(ewald_alpha=alpha, init_mode=0, scf_tol_F=1e-12, scf_tol_dn=1e-11, scf_max_iter=400)
    o, r = _solve(orc, cfg, cfg["pos"], **kw)
    assert o.get_real("n_a").max() < 0.2      # below n* = 3/(4 pi): no PZ81 branch flip under the strain
    s = o.stress()
    vol = float(np.prod(cfg["cell"]))
    h = 2e-4
    for mu in (range(3) if xc == 1 else (1,)):     # the xc = 0 run repeats one axis only (CPU time)
        cp, cm = _strained(cfg, mu, h), _strained(cfg, mu, -h)
        Fp = _solve(orc, cp, cp["pos"], **kw)[1]["F_total"]
        Fm = _solve(orc, cm, cm["pos"], **kw)[1]["F_total"]
        fd = (Fp - Fm) / (2 * h * vol)
        assert abs(fd - s["total"][mu]) < 2e-6 * abs(s["total"][mu]) + 1e-9, (mu, fd, s["total"][mu])
    assert abs(s["P"] + s["total"][:3].sum() / 3) < 1e-16
    assert np.allclose(s["total"], sum(s[k] for k in ("i", "e", "xc", "pp", "pm", "je", "ee", "ie")), rtol=0, atol=1e-15)
    if xc == 0:
        assert np.all(s["xc"] == 0)


# ---------------------------------------------------------------- every term, all six components
def _term_energies(eps, cfg, alpha, rc, S, nh, kidx, dij, zz):
    """U_pp, U_pm (without the constant self term), U_je, E_H, E_ie (+ its k = 0 term) of P:377-405, P:453-456,
    P:465-469 for the cell strained by the 3x3 matrix eps (any entries, shear included) at fixed scaled ion
    coordinates and fixed nhat(k), S_Z(k): r -> (1 + eps) r, k -> (1 + eps)^-T k, |Omega| -> |Omega| det(1 + eps)."""
    A = np.eye(3) + eps
    vol = float(np.prod(cfg["cell"])) * np.linalg.det(A)
    k = (kidx / np.asarray(cfg["cell"], dtype=float)) @ np.linalg.inv(A)
    k2 = (k * k).sum(-1)
    nz = k2 > 0
    k2s = np.where(nz, k2, 1.0)
    r = np.linalg.norm(dij @ A.T, axis=-1)
    Q = cfg["Z"].sum()
    erfc = np.vectorize(math.erfc)
    va = np.exp(-PI * PI * k2s / alpha ** 2) / (PI * k2s)
    vps = -np.cos(2 * PI * np.sqrt(k2s) * rc) / (PI * k2s)
    return {
        "pp": float((zz * erfc(alpha * r) / r).sum()),
        "pm": float((va * np.abs(S) ** 2)[nz].sum() / (2 * vol)),
        "je": -PI * Q * Q / (2 * alpha ** 2 * vol),
        "ee": float((np.abs(nh) ** 2 / (PI * k2s))[nz].sum() / (2 * vol)),
        "ie": float((np.conj(nh) * S * vps).real[nz].sum() / vol + Q / vol * (2 * PI * cfg["Z"] * rc * rc).sum()),
    }


def test_every_stress_term_is_the_strain_derivative_of_its_energy(orc):
    """sigma^X_mn = (1/|Omega|) dE_X/d(eps_mn) for X in pp, pm, je, ee, ie and all six (m, n), off-diagonal ones
    through a sheared cell, on a converged density of an anisotropic cell with even and odd-factor grid sizes."""
    cfg = ai.make_small(n_ions=3, cell=[7.0, 7.6, 8.3], grid=(12, 8, 9), T_eV=10.0, seed=5, dmin=2.5)
    alpha = 1.3 * orc.ewald_alpha(cfg["cell"], cfg["grid"])
    o, r = _solve(orc, cfg, cfg["pos"], ewald_alpha=alpha, init_mode=0, scf_max_iter=400, scf_tol_dn=1e-9)
    s = o.stress()
    S, nh = o.get_complex("S_Z"), o.get_complex("nhat_a")
    nx, ny, nz = (int(v) for v in cfg["grid"])
    m = lambda N: np.where(np.arange(N) <= N // 2, np.arange(N), np.arange(N) - N)
    kidx = np.stack(np.meshgrid(m(nz), m(ny), m(nx), indexing="ij")[::-1], axis=-1).astype(float)   # [z][y][x][xyz]
    cell = np.asarray(cfg["cell"], dtype=float)
    iu = np.triu_indices(len(cfg["Z"]), 1)
    d = cfg["pos"][iu[0]] - cfg["pos"][iu[1]]
    d -= cell * np.rint(d / cell)                                                       # minimum image
    zz = cfg["Z"][iu[0]] * cfg["Z"][iu[1]]
    vol = float(np.prod(cell))
    h = 1e-5
    for q, (mu, nu) in enumerate(VOIGT):
        e = np.zeros((3, 3)); e[mu, nu] = h
        Ep = _term_energies(e, cfg, alpha, cfg["psp_rc"], S, nh, kidx, d, zz)
        Em = _term_energies(-e, cfg, alpha, cfg["psp_rc"], S, nh, kidx, d, zz)
        for X in ("pp", "pm", "je", "ee", "ie"):
            fd = (Ep[X] - Em[X]) / (2 * h * vol)
            scale = np.abs(s[X]).max()
            assert abs(fd - s[X][q]) < 1e-8 * scale + 1e-12, (X, mu, nu, fd, s[X][q])
    assert np.abs(s["pm"][3:]).max() > 1e-6 and np.abs(s["ie"][3:]).max() > 1e-6    # the shear components are exercised
    # the unstrained energies are the ones the solve reported
    E0 = _term_energies(np.zeros((3, 3)), cfg, alpha, cfg["psp_rc"], S, nh, kidx, d, zz)
    assert abs(E0["ee"] - r["E_H"]) < 1e-12 and abs(E0["ie"] - r["E_ie"] - r["E_ie0"]) < 1e-12
    assert abs(E0["pp"] + E0["pm"] - alpha / math.sqrt(PI) * (cfg["Z"] ** 2).sum() + E0["je"] - r["U_ii"]) < 1e-12


def test_ion_kinetic_stress_trace_is_twice_the_kinetic_energy(orc):
    """P:353-357 (Eq. 36-37): -|Omega| tr(sigma^i) = 2 K^i, with K^i as the MD step reports it; off-diagonal
    components change sign with one velocity component."""
    cfg = ai.make_small(n_ions=3, L=7.0, grid=(8, 8, 8), T_eV=10.0, seed=3, dmin=2.5)
    o = orc.Oracle(cfg, init_mode=0, scf_tol_dn=1e-8)
    pos, vel = cfg["pos"].copy(), cfg["vel"].copy()
    r = o.md_step(cfg["dt"], pos, vel)
    s = o.stress(vel)
    vol = float(np.prod(cfg["cell"]))
    assert abs(-vol * s["i"][:3].sum() - 2 * r["K_i"]) < 1e-14 * r["K_i"]
    v2 = vel.copy(); v2[:, 0] *= -1
    s2 = o.stress(v2)
    assert np.allclose(s2["i"], s["i"] * np.array([1, 1, 1, 1, -1, -1]), rtol=1e-15, atol=0)
    assert np.allclose(s["total"] - s["i"], o.stress()["total"], rtol=0, atol=1e-15)
    with pytest.raises(RuntimeError):
        orc.Oracle(cfg).stress()
