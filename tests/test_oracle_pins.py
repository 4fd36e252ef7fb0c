"""Pins for the CPU oracle (no GPU): every oracle function is checked against something other than
itself -- library evaluations (mpmath polylog, numpy.fft), closed forms, textbook constants,
invariants and finite differences.  Citations: P:NNN = PAPER.md line NNN.
"""
import os

import mpmath as mp
import numpy as np
import pytest

import arche_inputs as ai

GOLD = os.path.join(os.path.dirname(__file__), "golden")
PI = np.pi


def _gold_constants():
    d = {}
    for line in open(os.path.join(GOLD, "constants.txt")):
        if line.strip() and not line.startswith("#"):
            k, v = line.split()
            d[k] = float(v)
    return d


# ---------------------------------------------------------------- Fermi-Dirac integrals
def test_fd_golden_values(orc):
    for line in open(os.path.join(GOLD, "fermi_dirac_values.txt")):
        if not line.strip() or line.startswith("#"):
            continue
        tj, eta, val = line.split()
        got = orc.fd(int(tj), float(eta))[0]
        assert abs(got / float(val) - 1) < 2e-14, (tj, eta, got)


def test_fd_vs_polylog(orc):
    mp.mp.dps = 30
    for tj in (-1, 1, 3):
        j = mp.mpf(tj) / 2
        for eta in (-40.0, -12.5, -3.0, -0.7, 0.0, 0.9, 2.5, 7.0, 15.0, 33.0, 80.0, 250.0):
            ref = -mp.gamma(j + 1) * mp.polylog(j + 1, -mp.exp(eta))
            got = orc.fd(tj, eta)[0]
            assert abs(got / float(mp.re(ref)) - 1) < 5e-14, (tj, eta)


def test_fd_limits_and_derivative(orc):
    from math import gamma
    for tj in (-1, 1, 3):
        j = tj / 2
        # classical limit Gamma(j+1) e^eta; degenerate (Sommerfeld) limit
        assert abs(orc.fd(tj, -35.0)[0] / (gamma(j + 1) * np.exp(-35.0)) - 1) < 1e-13
        eta = 400.0
        somm = eta ** (j + 1) / (j + 1) * (1 + PI ** 2 * j * (j + 1) / (6 * eta ** 2))
        assert abs(orc.fd(tj, eta)[0] / somm - 1) < 1e-8
    # I_j' = j I_{j-1}: central differences of I_{1/2} and I_{3/2}
    for eta in (-4.0, 0.3, 6.0, 40.0):
        h = 1e-4
        d12 = (orc.fd(1, eta + h)[0] - orc.fd(1, eta - h)[0]) / (2 * h)
        d32 = (orc.fd(3, eta + h)[0] - orc.fd(3, eta - h)[0]) / (2 * h)
        assert abs(d12 / (0.5 * orc.fd(-1, eta)[0]) - 1) < 1e-7
        assert abs(d32 / (1.5 * orc.fd(1, eta)[0]) - 1) < 1e-7


def test_fd_inverse(orc):
    for eta in (-8.0, -0.5, 0.27601, 3.0, 25.0, 120.0):
        y = orc.fd(1, eta)[0]
        assert abs(orc.fd_half_inverse(y) - eta) < 1e-11 * max(1.0, abs(eta))


# ---------------------------------------------------------------- FFT
@pytest.mark.parametrize("shape", [(4, 6, 8), (9, 5, 12), (16, 12, 18)])
def test_fft_vs_numpy_and_definition(orc, shape):
    rng = np.random.default_rng(3)
    a = rng.standard_normal(shape) + 1j * rng.standard_normal(shape)
    ref = np.fft.fftn(a)
    assert abs(orc.fft3d(a, -1) - ref).max() < 1e-12 * abs(ref).max()
    assert abs(orc.fft3d(a, -1, naive=True) - ref).max() < 1e-12 * abs(ref).max()
    assert abs(orc.fft3d(a, +1) - np.fft.ifftn(a) * a.size).max() < 1e-12 * abs(ref).max()
    assert abs(orc.fft3d(orc.fft3d(a, -1), +1) / a.size - a).max() < 1e-13


def test_fft_single_mode(orc):
    # f(r) = cos(2 pi k.r) with k = (2/Lx, -1/Ly, 3/Lz): only +-k are non-zero, each N_g/2
    nz, ny, nx = 8, 6, 10
    z, y, x = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    f = np.cos(2 * PI * (2 * x / nx - 1 * y / ny + 3 * z / nz))
    F = orc.fft3d(f, -1)
    ng = f.size
    assert abs(F[3, ny - 1, 2] - ng / 2) < 1e-10 and abs(F[nz - 3, 1, nx - 2] - ng / 2) < 1e-10
    F[3, ny - 1, 2] = 0; F[nz - 3, 1, nx - 2] = 0
    assert abs(F).max() < 1e-10


# ---------------------------------------------------------------- XC (reading D5)
def test_xc_potential_is_derivative_of_energy(orc):
    for n in (1e-4, 3e-3, 0.05, 0.2, 0.3, 1.7, 40.0):
        h = 1e-5 * n
        ep, _ = orc.xc(n + h); em, _ = orc.xc(n - h)
        dfdn = ((n + h) * ep - (n - h) * em) / (2 * h)
        assert abs(dfdn / orc.xc(n)[1] - 1) < 1e-8, n


def test_xc_reference_points(orc):
    # exchange-only part: Dirac exchange eps_x = -(3/4)(3 n/pi)^{1/3}; correlation: Ceperley-Alder
    # unpolarised energies (Ry -> Ha) that PZ81 fits: rs=2: -0.0902 Ry, rs=5: -0.0563 Ry, rs=10: -0.0372 Ry
    for rs, ec_ry in ((2.0, -0.0902), (5.0, -0.0563), (10.0, -0.0372)):
        n = 3 / (4 * PI * rs ** 3)
        ex = -0.75 * (3 * n / PI) ** (1 / 3)
        assert abs((orc.xc(n)[0] - ex) - ec_ry / 2) < 4e-4
    # high-density (Gell-Mann--Brueckner) leading term (1-ln2)/pi^2 ln rs
    n1 = 3 / (4 * PI * 0.01 ** 3); n2 = 3 / (4 * PI * 0.001 ** 3)
    ec1 = orc.xc(n1)[0] + 0.75 * (3 * n1 / PI) ** (1 / 3)
    ec2 = orc.xc(n2)[0] + 0.75 * (3 * n2 / PI) ** (1 / 3)
    assert abs((ec1 - ec2) / np.log(10.0) - (1 - np.log(2)) / PI ** 2) < 2e-4
    # the two PZ81 branches meet at rs=1 up to the known small jump (~3e-5 Ha)
    ns = 3 / (4 * PI)
    assert abs(orc.xc(ns * (1 + 1e-9))[0] - orc.xc(ns * (1 - 1e-9))[0]) < 5e-5
    assert orc.xc(0.1, 0) == (0.0, 0.0)


# ---------------------------------------------------------------- structure factor
def test_structure_factor_properties(orc):
    cell = np.array([7.0, 9.0, 5.0]); grid = np.array([6, 8, 4], dtype=np.int32)
    rng = np.random.default_rng(5)
    pos = rng.random((5, 3)) * cell; Z = np.array([1.0, 2.0, 3.0, 1.5, 0.5])
    S = orc.structure_factor(cell, grid, pos, Z)
    assert abs(S[0, 0, 0] - Z.sum()) < 1e-13
    # independent evaluation with numpy broadcasting over the literal index set of P:142
    def m(N):
        i = np.arange(N); return np.where(i <= N // 2, i, i - N)
    kz, ky, kx = np.meshgrid(m(4) / cell[2], m(8) / cell[1], m(6) / cell[0], indexing="ij")
    ref = sum(Zj * np.exp(-2j * PI * (kx * p[0] + ky * p[1] + kz * p[2])) for Zj, p in zip(Z, pos))
    assert abs(S - ref).max() < 1e-12
    # one ion at the origin: S = Z everywhere; a rigid shift multiplies by a phase
    S1 = orc.structure_factor(cell, grid, np.zeros((1, 3)), np.array([2.0]))
    assert abs(S1 - 2.0).max() < 1e-14
    d = np.array([0.3, -1.1, 0.7])
    S2 = orc.structure_factor(cell, grid, pos + d, Z)
    assert abs(S2 - S * np.exp(-2j * PI * (kx * d[0] + ky * d[1] + kz * d[2]))).max() < 1e-12
    # a lattice translation leaves S unchanged
    assert abs(orc.structure_factor(cell, grid, pos + cell * np.array([1, -2, 3]), Z) - S).max() < 1e-11


def test_ashcroft_form_factor_is_transform_of_empty_core(orc):
    # V(r) = -1/r (r > rc), 0 inside: radial transform 4 pi int r^2 V(r) sin(2 pi k r)/(2 pi k r) dr with
    # a convergence factor exp(-eps r) -> -cos(2 pi k rc)/(pi k^2)
    mp.mp.dps = 30
    rc = 1.12
    for k in (0.05, 0.3, 1.1):
        eps = mp.mpf("1e-9")
        # closed form of int_rc^inf exp(-eps r) sin(q r) dr
        q = 2 * mp.pi * k
        integral = mp.e ** (-eps * rc) * (eps * mp.sin(q * rc) + q * mp.cos(q * rc)) / (eps ** 2 + q ** 2)
        ref = -4 * mp.pi / q * integral
        assert abs(orc.vps_unit(k, rc) / float(ref) - 1) < 1e-7
    assert orc.vps_unit(0.0, rc) == 0.0
