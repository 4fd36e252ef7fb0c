"""Pins for the oracle's Ewald sum, SCF fixed point, forces and MD (no GPU).  P:NNN = PAPER.md line."""
import os

import numpy as np
import pytest

import arche_inputs as ai

GOLD = os.path.join(os.path.dirname(__file__), "golden")
PI = np.pi


def _const(name):
    for line in open(os.path.join(GOLD, "constants.txt")):
        if line.startswith(name + " "):
            return float(line.split()[1])
    raise KeyError(name)


# ---------------------------------------------------------------- Ewald
def test_ewald_madelung_single_charge(orc):
    L = 5.0; cell = [L, L, L]; grid = np.array([24, 24, 24])
    U, F = orc.ewald(cell, grid, np.array([[1.3, 2.2, 0.4]]), np.array([2.0]))
    assert abs(U.sum() * L / 4.0 - _const("madelung_sc_jellium")) < 1e-9
    assert abs(F).max() < 1e-10


def test_ewald_nacl_and_cscl(orc):
    a = 6.0; cell = [a, a, a]; grid = np.array([24, 24, 24])
    fcc = np.array([[0, 0, 0], [.5, .5, 0], [.5, 0, .5], [0, .5, .5]])
    pos = np.vstack([fcc, fcc + [.5, 0, 0]]) * a
    Z = np.array([1.0] * 4 + [-1.0] * 4)
    U, F = orc.ewald(cell, grid, pos, Z)
    assert abs(U.sum() / 4 * (a / 2) + _const("madelung_nacl")) < 1e-8   # 4 ion pairs per cell
    assert abs(F).max() < 1e-8      # truncation (asymmetric Nyquist set of P:142), not round-off
    pos = np.array([[0, 0, 0], [.5, .5, .5]]) * a
    U, F = orc.ewald(cell, grid, pos, np.array([1.0, -1.0]))
    assert abs(U.sum() * (a * np.sqrt(3) / 2) + _const("madelung_cscl")) < 1e-8


def test_ewald_alpha_independence_forces_fd(orc):
    cfg = ai.make_small(n_ions=5, L=7.0, grid=(20, 20, 20), seed=3)
    cell, grid, pos, Z = cfg["cell"], cfg["grid"], cfg["pos"], np.array([3.0, 1.0, 2.0, 3.0, 1.5])
    a0 = orc.ewald_alpha(cell, grid)
    U0, F0 = orc.ewald(cell, grid, pos, Z, a0)
    U1, F1 = orc.ewald(cell, grid, pos, Z, 0.9 * a0)
    assert abs(U0.sum() - U1.sum()) < 1e-8 * abs(U0.sum())
    assert abs(F0 - F1).max() < 1e-8
    assert abs(F0.sum(0)).max() < 1e-11                     # Newton's third law
    h = 1e-4
    for j, c in ((0, 0), (2, 1), (4, 2)):
        p = pos.copy(); p[j, c] += h; Up = orc.ewald(cell, grid, p, Z, a0)[0].sum()
        p[j, c] -= 2 * h; Um = orc.ewald(cell, grid, p, Z, a0)[0].sum()
        assert abs(-(Up - Um) / (2 * h) - F0[j, c]) < 2e-7 * abs(F0).max()


def test_gaussian_hartree_equals_ewald_reciprocal(orc):
    # rho = sum_j Z_j periodic Gaussians of width sigma: (1/2|O|) sum_k |rho_hat|^2/(pi k^2) equals the Ewald
    # reciprocal sum with alpha = 1/(2 sigma) (+ self term): pins FFT normalisation, Poisson kernel, Eq. 42-43.
    L = 6.0; N = 24; sigma = 0.55; cell = np.array([L, L, L]); grid = np.array([N, N, N], dtype=np.int32)
    pos = np.array([[1.0, 2.0, 3.0], [4.2, 0.7, 2.1], [2.9, 5.1, 5.0]]); Z = np.array([1.0, 2.0, 0.5])
    x = np.arange(N) * L / N
    zz, yy, xx = np.meshgrid(x, x, x, indexing="ij")
    rho = np.zeros((N, N, N))
    for Zj, p in zip(Z, pos):
        g = 1.0
        for coord, pc in ((xx, p[0]), (yy, p[1]), (zz, p[2])):
            g1 = sum(np.exp(-((coord - pc + s * L) ** 2) / (2 * sigma ** 2)) for s in range(-3, 4))
            g = g * g1 / np.sqrt(2 * PI * sigma ** 2)
        rho += Zj * g
    dV = L ** 3 / N ** 3
    rh = orc.fft3d(rho, -1) * dV
    i = np.arange(N); m = np.where(i <= N // 2, i, i - N) / L
    kz, ky, kx = np.meshgrid(m, m, m, indexing="ij")
    k2 = kx ** 2 + ky ** 2 + kz ** 2; k2[0, 0, 0] = 1.0
    w = 1.0 / (PI * k2); w[0, 0, 0] = 0.0
    EH = 0.5 / L ** 3 * (abs(rh) ** 2 * w).sum()
    alpha = 1.0 / (2 * sigma)
    U, _ = orc.ewald(cell, grid, pos, Z, alpha)
    assert abs(EH - (U[1] + alpha / np.sqrt(PI) * (Z ** 2).sum())) < 1e-9 * EH


# ---------------------------------------------------------------- uniform gas (pin P2)
@pytest.mark.parametrize("xc", [0, 1])
def test_uniform_gas_closed_form(orc, xc):
    cfg = dict(cell=[5.0, 6.0, 7.0], grid=[6, 8, 10], Z=np.zeros(0), mass=np.zeros(0), kT=0.4)
    Ne = 9.0
    o = orc.Oracle(cfg, n_electrons=Ne, xc=xc)
    o.scf_begin(np.zeros((0, 3)))
    r1 = o.scf_iter(); r2 = o.scf_iter()
    vol = 210.0; n0 = Ne / vol; kT = 0.4
    cTF = np.sqrt(2) / PI ** 2 * kT ** 1.5
    eta0 = orc.fd_half_inverse(n0 / cTF)
    exc, vxc = orc.xc(n0, xc)
    assert abs(o.get_real("n_a") - n0).max() < 1e-14
    assert r2["dn_l2"] < 1e-14 and r2["converged"] == 1
    assert abs(r2["mu"] - (kT * eta0 + vxc)) < 1e-12
    f0 = kT * cTF * (eta0 * orc.fd(1, eta0)[0] - 2 / 3 * orc.fd(3, eta0)[0])
    assert abs(r2["F_total"] - vol * (f0 + n0 * exc)) < 1e-11
    assert abs(r2["E_H"]) < 1e-20 and r2["U_ii"] == 0.0
    assert abs(r2["K_e"] - vol * kT * cTF * orc.fd(3, eta0)[0]) < 1e-11


def test_uniform_gas_limits(orc):
    # degenerate: K_e/V -> (3/10)(3 pi^2)^{2/3} n^{5/3}; classical: K_e/V -> (3/2) n kT  (Eq. 38)
    for kT, n0, ref, tol in ((1e-3, 0.03, 0.3 * (3 * PI ** 2) ** (2 / 3) * 0.03 ** (5 / 3), 2e-3),
                             (50.0, 0.03, 1.5 * 0.03 * 50.0, 2e-3)):
        cfg = dict(cell=[4.0, 4.0, 4.0], grid=[4, 4, 4], Z=np.zeros(0), mass=np.zeros(0), kT=kT)
        o = orc.Oracle(cfg, n_electrons=n0 * 64.0, xc=0)
        o.scf_begin(np.zeros((0, 3)))
        r = o.scf_iter()
        assert abs(r["K_e"] / 64.0 / ref - 1) < tol


# ---------------------------------------------------------------- linear response (pin P5) and mixing (P9)
def test_linear_response_and_neutrality(orc):
    kT = 0.5; cell = np.array([6.0, 7.0, 5.0]); grid = np.array([10, 12, 8], dtype=np.int32)
    Ne = 6.0; eps = 1e-6
    cfg = dict(cell=cell, grid=grid, Z=np.array([eps]), mass=np.array([1.0]), kT=kT)
    o = orc.Oracle(cfg, n_electrons=Ne, xc=0, scf_tol_dn=1e-13, scf_tol_F=1e-9, scf_max_iter=300)
    r = o.scf_solve(np.array([[1.1, 2.3, 0.9]]))
    assert r["converged"] == 1
    na = o.get_real("n_a"); dV = cell.prod() / grid.prod()
    assert abs(na.sum() * dV - Ne) < 1e-12 * Ne and na.min() > 0
    n0 = Ne / cell.prod(); cTF = np.sqrt(2) / PI ** 2 * kT ** 1.5
    eta0 = orc.fd_half_inverse(n0 / cTF)
    chi = cTF * orc.fd(-1, eta0)[0] / (2 * kT)
    nh = o.get_complex("nhat_a"); vie = o.get_complex("Vhat_ie")
    def m(N):
        i = np.arange(N); return np.where(i <= N // 2, i, i - N)
    kz, ky, kx = np.meshgrid(m(8) / cell[2], m(12) / cell[1], m(10) / cell[0], indexing="ij")
    k2 = kx ** 2 + ky ** 2 + kz ** 2
    # exclude k=0 and the Nyquist planes (real-part rule, reading A6, symmetrises those)
    mask = (k2 > 0) & (np.abs(kx) < 5 / cell[0]) & (np.abs(ky) < 6 / cell[1]) & (np.abs(kz) < 4 / cell[2])
    pred = -chi * vie[mask] / (1 + chi / (PI * k2[mask]))
    assert abs(nh[mask] - pred).max() < 2e-5 * abs(pred).max()


def test_more_mixing_single_mode_closed_form(orc):
    # n_i = n0 + a cos(2 pi k.r), no ions, no xc: w = lambda/(1+lambda), lambda = chi/(pi k^2), and the mode is
    # annihilated to O(a^2) (Eq. 30-31)
    kT = 0.3; cell = np.array([8.0, 8.0, 8.0]); N = 8
    cfg = dict(cell=cell, grid=[N, N, N], Z=np.zeros(0), mass=np.zeros(0), kT=kT)
    Ne = 10.0; n0 = Ne / 512.0
    o = orc.Oracle(cfg, n_electrons=Ne, xc=0, mix_warmup=0)
    o.scf_begin(np.zeros((0, 3)))
    x = np.arange(N) * 1.0
    zz, yy, xx = np.meshgrid(x, x, x, indexing="ij")
    a = 1e-6 * n0
    o.set_input_density(n0 + a * np.cos(2 * PI * (2 * xx - yy) / 8.0))
    r = o.scf_iter()
    cTF = np.sqrt(2) / PI ** 2 * kT ** 1.5
    chi = cTF * orc.fd(-1, orc.fd_half_inverse(n0 / cTF))[0] / (2 * kT)
    lam = chi / (PI * (4 + 1) / 64.0)
    assert abs(r["w_last"] - lam / (1 + lam)) < 1e-5
    assert 0 <= r["w_last"] < 1
    assert abs(o.get_real("n_i") - n0).max() < 1e-4 * a
