"""Pins for the oracle's forces and MD step (no GPU).  P:NNN = PAPER.md line."""
import numpy as np

import arche_inputs as ai

PI = np.pi


def _mk(orc, cfg, **kw):
    kw.setdefault("scf_tol_dn", 1e-12); kw.setdefault("scf_tol_F", 1e-9); kw.setdefault("scf_max_iter", 400)
    return orc.Oracle(cfg, **kw)


def test_force_ie_fixed_density_is_minus_gradient(orc):
    # E_ie(R) = (1/|O|) Re sum_k conj(nhat) v(k) S_Z(k;R) at fixed density; F^ie (Eq. 56, reading A17)
    cfg = ai.make_small(n_ions=3, L=7.0, grid=(10, 12, 8), seed=1)
    cell, grid, pos, Z, rc = cfg["cell"], cfg["grid"], cfg["pos"], np.array([3.0, 1.0, 2.0]), 1.12
    rng = np.random.default_rng(11)
    n = 0.03 + 0.01 * rng.random((8, 12, 10))
    nh = orc.fft3d(n, -1) * cell.prod() / n.size
    def m(N):
        i = np.arange(N); return np.where(i <= N // 2, i, i - N)
    kz, ky, kx = np.meshgrid(m(8) / cell[2], m(12) / cell[1], m(10) / cell[0], indexing="ij")
    kk = np.sqrt(kx ** 2 + ky ** 2 + kz ** 2)
    v = np.vectorize(lambda k: orc.vps_unit(k, rc))(kk)
    def E(p):
        return (np.conj(nh) * v * orc.structure_factor(cell, grid, p, Z)).real.sum() / cell.prod()
    F = orc.force_ie(cell, grid, pos, Z, rc, nh)
    h = 1e-4
    for j in range(3):
        for c in range(3):
            p = pos.copy(); p[j, c] += h; ep = E(p); p[j, c] -= 2 * h; em = E(p)
            assert abs(-(ep - em) / (2 * h) - F[j, c]) < 1e-7 * abs(F).max()


def test_total_force_is_minus_gradient_of_converged_free_energy(orc):
    # Hellmann-Feynman on the grid: F_j = -dF/dR_j with re-converged SCF (pin P7). This ties together the
    # coefficients of F0, E_xc, E_H, E_ie, U_ii and the SCF equations (a wrong factor in any breaks it).
    cfg = ai.make_small(n_ions=3, L=7.5, grid=(12, 12, 12), T_eV=8.0, seed=2)
    o = _mk(orc, cfg, init_mode=0)
    pos = cfg["pos"]
    r = o.scf_solve(pos); assert r["converged"] == 1
    F = o.forces()
    def fd(j, c, h):
        p = pos.copy(); p[j, c] += h; fp = o.scf_solve(p)["F_total"]
        p[j, c] -= 2 * h; fm = o.scf_solve(p)["F_total"]
        return -(fp - fm) / (2 * h)
    for j, c in ((0, 0), (2, 1)):
        rich = (4 * fd(j, c, 1e-3) - fd(j, c, 2e-3)) / 3       # Richardson: the FD error is O(h^2)
        assert abs(rich - F[j, c]) < 2e-7 * abs(F).max(), (j, c)


def test_translation_permutation_and_lattice_symmetry(orc):
    cfg = ai.make_small(n_ions=3, L=7.5, grid=(12, 12, 12), T_eV=8.0, seed=4)
    o = _mk(orc, cfg, init_mode=0)
    pos = cfg["pos"]
    r0 = o.scf_solve(pos); F0 = o.forces(); n0 = o.get_real("n_a")
    # shift by a grid vector: density rolls, energies and forces unchanged (pin P8)
    d = cfg["cell"] / cfg["grid"] * np.array([2, -3, 5])
    r1 = o.scf_solve(pos + d); F1 = o.forces(); n1 = o.get_real("n_a")
    assert abs(r1["F_total"] - r0["F_total"]) < 1e-10 * abs(r0["F_total"])
    assert abs(F1 - F0).max() < 1e-9 * abs(F0).max()
    assert abs(np.roll(n0, (5, -3, 2), axis=(0, 1, 2)) - n1).max() < 1e-10 * n0.max()
    # permutation of (identical) ions
    perm = [2, 0, 1]
    r2 = o.scf_solve(pos[perm]); F2 = o.forces()
    assert abs(r2["F_total"] - r0["F_total"]) < 1e-11 * abs(r0["F_total"])
    assert abs(F2 - F0[perm]).max() < 1e-9 * abs(F0).max()
    # one ion sitting on a grid point: inversion symmetry about it -> zero force (a lattice with pairs at exactly
    # L/2 would not do: the minimum-image convention of P:385 keeps only one of the two equidistant images)
    cfg2 = dict(cfg); cfg2["Z"] = np.full(1, 3.0); cfg2["mass"] = np.full(1, 1e4)
    o2 = _mk(orc, cfg2, init_mode=0)
    o2.scf_solve(cfg["cell"] / cfg["grid"] * np.array([[3.0, 7.0, 10.0]]))
    assert abs(o2.forces()).max() < 1e-11


def test_md_energy_conservation_and_reversibility(orc):
    cfg = ai.make_small(n_ions=3, L=7.5, grid=(12, 12, 12), T_eV=8.0, seed=5)
    cfg["mass"] = np.full(3, 2000.0)          # light ions so that a few steps move them visibly
    drift = []
    for dt in (8.0, 4.0):
        o = _mk(orc, cfg, init_mode=1, scf_tol_dn=1e-10)
        pos = cfg["pos"].copy(); vel = cfg["vel"].copy() * 3.0
        r = o.scf_solve(pos); o.forces()
        E0 = r["F_total"] + 0.5 * (cfg["mass"][:, None] * vel ** 2).sum()
        nst = int(16 / dt)
        for _ in range(nst):
            r = o.md_step(dt, pos, vel)
        drift.append(abs(r["F_total"] + r["K_i"] - E0))
        if dt == 4.0:                          # time reversal
            vel *= -1
            for _ in range(nst):
                o.md_step(dt, pos, vel)
            assert abs(pos - cfg["pos"]).max() < 1e-7
    assert drift[1] < 0.4 * drift[0]                          # O(dt^2) integrator


def test_one_center_init_reduces_iterations(orc):
    # soft target from P:315-321 (Fig. 3): profile initialisation needs fewer iterations than uniform start
    cfg = ai.make_small(n_ions=4, L=8.0, grid=(12, 12, 12), T_eV=10.0, seed=6)
    its = {}
    for mode in (0, 1):
        o = _mk(orc, cfg, init_mode=mode, scf_tol_dn=1e-9)
        pos = cfg["pos"].copy()
        o.scf_solve(pos)
        pos[:, 0] += 0.05
        its[mode] = o.scf_solve(pos)["scf_iters"]
    assert its[1] < its[0]


def test_structure_factor_and_ionic_potential_do_not_depend_on_the_grid(orc):
    """S_Z(k) = sum_j Z_j exp(-2 pi i k.R_j) and Vhat_ie(k) = v(k) S_Z(k) are functions of the
    integer wave vector m (k = m/L) and the ions only: the same cell on an 8^3 and a 12 x 10 x 14 grid must give the
    same values at every |m_i| <= 3 (off both grids' Nyquist planes).  This is what the sampled full-size GPU test of
    the c5 sweep relies on."""
    cfg = ai.make_config("c1")
    a = dict(cfg); a["grid"] = np.array([8, 8, 8])
    b = dict(cfg); b["grid"] = np.array([12, 10, 14])
    oa = orc.Oracle(a); ob = orc.Oracle(b)
    oa.scf_begin(cfg["pos"]); ob.scf_begin(cfg["pos"])
    m = np.arange(-3, 4)
    for name in ("S_Z", "Vhat_ie"):
        fa = oa.get_complex(name)[np.ix_(m % 8, m % 8, m % 8)]          # [iz][iy][ix]
        fb = ob.get_complex(name)[np.ix_(m % 14, m % 10, m % 12)]
        assert np.abs(fa - fb).max() <= 1e-13 * np.abs(fb).max(), name
    # and the definition itself at one wave vector, written out
    mz, my, mx = 2, -1, 3
    k = np.array([mx, my, mz]) / np.asarray(cfg["cell"])
    direct = np.sum(cfg["Z"] * np.exp(-2j * np.pi * (cfg["pos"] @ k)))
    assert abs(oa.get_complex("S_Z")[mz % 8, my % 8, mx % 8] - direct) < 1e-12 * abs(cfg["Z"].sum())
