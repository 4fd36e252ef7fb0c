"""Pre-processing for SURVEY.md 8(f2): the norm-conserving local pseudopotential of PAPER.md:179-215 from a
finite-temperature Thomas-Fermi average atom, as the form-factor TABLE the C ABI takes (arche_params.psp = 1).

    tab = make_table(Z, rho_ion, kT, k_max, dk)          # dict: dk, table (Du(k_m) per unit charge), r_cut, mu, ...
    Arche(cfg, psp_table=tab["table"], psp_dk=tab["dk"])

This is host-side pre-processing (the paper's own pre-processing is Python); nothing here runs per MD step.
Plain numpy; it shares no code with oracle/ (tests compare the two tables).  Steps, in the paper's order:
  1. average-atom density n(r) of one nucleus Z in a neutral sphere r_ws (4/3 pi rho r_ws^3 = 1): Eq. 9 with
     V = -Z/r + V_H[n] + V_xc(n), mu from neutrality, SCF with the mixing of More et al.;
  2. pseudo-density exp(a + b r^2 + c r^4) inside r_cut (Eq. 16) with value, slope and charge matched (Eq. 17);
  3. pseudopotential by inverting Eq. 9 for the pseudo-density (Eq. 18); it is -Z/r beyond r_cut;
  4. Du(k) = (1/Z) int_0^r_cut (V_s(r) + Z/r) 4 pi r^2 sin(2 pi k r)/(2 pi k r) dr on the uniform grid k_m = m dk.
Radial grid uniform in x = sqrt(r); Simpson's rule in x.  r_cut/r_ws defaults to 0.17, the value at which the
pseudo-atom energy of Al at 2.7 g/cc, 100 eV equals the paper's -2971 eV (reading A22).
"""
from __future__ import annotations

import numpy as np

_GLX, _GLW = np.polynomial.legendre.leggauss(48)


def fermi_dirac(twice_j: int, eta) -> np.ndarray:
    """I_j(eta) = int_0^inf t^j/(exp(t-eta)+1) dt, j = twice_j/2, vectorised: two-term series below -30, Sommerfeld
    expansion above 60, composite Gauss-Legendre in s = sqrt(t) in between (panels refined around the Fermi edge)."""
    eta = np.atleast_1d(np.asarray(eta, dtype=np.float64))
    j = 0.5 * twice_j
    out = np.empty_like(eta)
    from math import gamma, pi
    lo = eta < -30.0
    x = np.exp(eta[lo])
    out[lo] = gamma(j + 1) * x * (1.0 - x / 2.0 ** (j + 1) + x * x / 3.0 ** (j + 1))
    hi = eta > 60.0
    e2 = 1.0 / eta[hi] ** 2
    p1 = (j + 1) * j; p2 = p1 * (j - 1) * (j - 2); p3 = p2 * (j - 3) * (j - 4); p4 = p3 * (j - 5) * (j - 6)
    c1 = pi ** 2 / 6; c2 = 7 * pi ** 4 / 360; c3 = 31 * pi ** 6 / 15120; c4 = 127 * pi ** 8 / 604800
    out[hi] = eta[hi] ** (j + 1) / (j + 1) * (1 + e2 * (c1 * p1 + e2 * (c2 * p2 + e2 * (c3 * p3 + e2 * c4 * p4))))
    mid = ~(lo | hi)
    if mid.any():
        e = eta[mid]
        s0 = np.sqrt(np.maximum(e, 0.0))
        # panels in s: [0, s0 - d], [s0 - d, s0], [s0, s0 + d], ..., tail to sqrt(max(eta,0) + 70); d ~ edge width 2/s0
        edges = [np.zeros_like(e)]
        d = np.minimum(s0, 4.0 / np.maximum(s0, 1.0))
        for f in (-1.0, -0.5, 0.0):
            edges.append(np.maximum(s0 + f * d, 0.0))
        top = np.sqrt(np.maximum(e, 0.0) + 70.0)
        for f in (0.25, 0.5, 0.75, 1.0):
            edges.append(s0 + f * (top - s0))
        acc = np.zeros_like(e)
        for a, b in zip(edges[:-1], edges[1:]):
            h = 0.5 * (b - a)[:, None]
            s = 0.5 * (a + b)[:, None] + h * _GLX[None, :]
            arg = np.minimum(s * s - e[:, None], 700.0)
            f = 2.0 * s ** (twice_j + 1) / (np.exp(arg) + 1.0)
            acc += (h * f * _GLW[None, :]).sum(1)
        out[mid] = acc
    return out


def fermi_dirac_half_inverse(y) -> np.ndarray:
    """eta with I_{1/2}(eta) = y: Newton on log y (I_{1/2}' = I_{-1/2}/2), started from the two limits"""
    y = np.atleast_1d(np.asarray(y, dtype=np.float64))
    eta = np.where(y < 1.0, np.log(y / 0.8862269254527580), (1.5 * y) ** (2.0 / 3.0))
    for _ in range(60):
        f = fermi_dirac(1, eta)
        step = (np.log(f) - np.log(y)) * f / (0.5 * fermi_dirac(-1, eta))
        eta = eta - step
        if np.all(np.abs(step) <= 1e-13 * np.maximum(1.0, np.abs(eta))):
            break
    return eta


def _pz81(n, xc):
    """V_xc and eps_xc of Perdew-Zunger 1981 (xc = 1 as printed, 2 with C, D from its continuity conditions); 0: none"""
    n = np.asarray(n, dtype=np.float64)
    if xc == 0:
        return np.zeros_like(n), np.zeros_like(n)
    pos = n > 0
    ns = np.where(pos, n, 1.0)
    rs = (3.0 / (4.0 * np.pi * ns)) ** (1.0 / 3.0)
    ex = -0.75 * (3.0 * ns / np.pi) ** (1.0 / 3.0)
    g, b1, b2, A, B = -0.1423, 1.0529, 0.3334, 0.0311, -0.048
    C, D = 0.0020, -0.0116
    if xc == 2:
        den1 = 1 + b1 + b2
        D = g / den1 - B
        C = -g * (0.5 * b1 + b2) / den1 ** 2 - A - D
    sq = np.sqrt(rs); den = 1 + b1 * sq + b2 * rs
    ec_hi = g / den; vc_hi = ec_hi * (1 + 7.0 / 6.0 * b1 * sq + 4.0 / 3.0 * b2 * rs) / den
    l = np.log(rs)
    ec_lo = A * l + B + C * rs * l + D * rs
    vc_lo = A * l + (B - A / 3) + 2.0 / 3.0 * C * rs * l + (2 * D - C) / 3 * rs
    ec = np.where(rs >= 1, ec_hi, ec_lo); vc = np.where(rs >= 1, vc_hi, vc_lo)
    return np.where(pos, 4.0 / 3.0 * ex + vc, 0.0), np.where(pos, ex + ec, 0.0)


def _simpson_cum(g, h):
    """cumulative integral on a uniform grid: Simpson on even nodes, chained from a three-point start on odd nodes"""
    F = np.zeros_like(g)
    F[1] = h * (5 * g[0] + 8 * g[1] - g[2]) / 12
    for i in range(2, len(g)):
        F[i] = F[i - 2] + h * (g[i - 2] + 4 * g[i - 1] + g[i]) / 3
    return F


def _hartree(x, dens, n0lim):
    h = x[1]; r = x * x
    g1 = 8 * np.pi * x ** 5 * dens
    g2 = 8 * np.pi * x ** 3 * dens; g2[0] = 8 * np.pi * n0lim
    Q = _simpson_cum(g1, h); I2 = _simpson_cum(g2, h)
    VH = I2[-1] - I2
    VH[1:] += Q[1:] / r[1:]
    return VH, Q


def average_atom(Z, r_ws, kT, xc=0, n=801, tol=1e-11, max_iter=500):
    """finite-T Thomas-Fermi average atom: returns x (= sqrt r) grid, density (entry 0 stands for the r^(-3/2) singularity),
    mu, iterations"""
    assert n % 2 == 1
    x = np.linspace(0.0, np.sqrt(r_ws), n); h = x[1]; r = x * x
    cTF = np.sqrt(2.0) / np.pi ** 2 * kT ** 1.5
    w5 = 8 * np.pi * x ** 5
    dens = np.full(n, 3 * Z / (4 * np.pi * r_ws ** 3)); dens[0] = 0.0
    n0lim_true = (2 * Z) ** 1.5 / (3 * np.pi ** 2); n0lim = 0.0
    mu = 0.0
    for it in range(1, max_iter + 1):
        VH, _ = _hartree(x, dens, n0lim)
        vxc, _ = _pz81(dens, xc)
        V = np.empty(n); V[1:] = -Z / r[1:] + VH[1:] + vxc[1:]; V[0] = V[1]

        def count(m):
            f = w5 * cTF * fermi_dirac(1, (m - V) / kT); f[0] = 0.0
            return _simpson_cum(f, h)[-1] - Z
        if it == 1:
            lo, hi = V[-1] - 60 * kT - 10 - 10 * Z * Z, V[-1] + 60 * kT + 10 * Z
        else:
            lo, hi = mu - 5 * kT - 1, mu + 5 * kT + 1
        flo, fhi = count(lo), count(hi)
        while flo > 0: lo -= 10 * kT + 10; flo = count(lo)
        while fhi < 0: hi += 10 * kT + 10; fhi = count(hi)
        for _ in range(200):                     # Illinois
            m = (lo * fhi - hi * flo) / (fhi - flo)
            fm = count(m)
            if abs(fm) <= 1e-13 * Z or hi - lo <= 4e-16 * max(abs(lo), abs(hi)):
                break
            if fm > 0: hi, fhi, flo = m, fm, flo * 0.5
            else: lo, flo, fhi = m, fm, fhi * 0.5
        mu = m
        eta = (mu - V) / kT
        na = cTF * fermi_dirac(1, eta); na[0] = 0.0
        chi = cTF * 0.5 * fermi_dirac(-1, eta) / kT
        dn = dens - na
        dVH, _ = _hartree(x, dn, 0.0)
        U = _simpson_cum(w5 * dn * dVH, h)[-1]
        kk = np.where(chi > 0, dn * dn / np.where(chi > 0, chi, 1.0), 0.0); kk[0] = 0.0
        K = _simpson_cum(w5 * kk, h)[-1]
        w = 0.5 if it <= 3 else (U / (K + U) if K + U > 0 else 0.0)      # Eq. 30-31, radial form
        res = np.sqrt((x[1:] ** 5 * dn[1:] ** 2).sum() / (x[1:] ** 5 * na[1:] ** 2).sum())
        dens = na + w * dn
        n0lim = n0lim_true
        if res < tol:
            break
    return x, na, mu, it


def pseudize(x, dens, ic):
    """Eq. 16-17 with r_cut = x[ic]^2"""
    from scipy.optimize import brentq
    h = x[1]; r = x * x; rc = r[ic]
    dndx = (dens[ic - 2] - 8 * dens[ic - 1] + 8 * dens[ic + 1] - dens[ic + 2]) / (12 * h)
    L = np.log(dens[ic]); s = dndx / (2 * x[ic]) / dens[ic]
    w5 = 8 * np.pi * x[:ic + 1] ** 5
    g = w5 * dens[:ic + 1]; g[0] = 0.0
    Q = _simpson_cum(g, h)[-1]

    def coeff(c):
        b = (s - 4 * c * rc ** 3) / (2 * rc)
        return L - b * rc ** 2 - c * rc ** 4, b

    def f(c):
        a, b = coeff(c)
        rr = r[:ic + 1]
        return _simpson_cum(w5 * np.exp(a + b * rr ** 2 + c * rr ** 4), h)[-1] - Q
    c = brentq(f, -50 / rc ** 4, 50 / rc ** 4, xtol=1e-15 / rc ** 4, rtol=1e-15)
    a, b = coeff(c)
    ps = dens.copy(); ps[:ic + 1] = np.exp(a + b * r[:ic + 1] ** 2 + c * r[:ic + 1] ** 4)
    return ps, (a, b, c)


def invert(x, dens, n0lim, mu, kT, xc=0):
    """Eq. 18: V_ext with which `dens` solves Eq. 9 in the sphere"""
    cTF = np.sqrt(2.0) / np.pi ** 2 * kT ** 1.5
    VH, _ = _hartree(x, dens, n0lim)
    vxc, _ = _pz81(dens, xc)
    V = np.empty_like(x)
    V[1:] = mu - kT * fermi_dirac_half_inverse(dens[1:] / cTF) - VH[1:] - vxc[1:]
    V[0] = V[1]
    return V


def make_table(Z, rho_ion, kT, k_max, dk=0.01, xc=0, rcut_frac=0.17, n=801):
    """Du(k_m), m = 0..ceil(k_max/dk)+2, for arche_params.h_psp_table (per unit charge).  rho_ion in ions/bohr^3."""
    r_ws = (3.0 / (4.0 * np.pi * rho_ion)) ** (1.0 / 3.0)
    x, dens, mu, it = average_atom(Z, r_ws, kT, xc, n)
    ic = int(round((n - 1) * np.sqrt(rcut_frac)))
    ps, abc = pseudize(x, dens, ic)
    V = invert(x, ps, 0.0, mu, kT, xc)
    r = x * x; h = x[1]
    dV = np.zeros(ic + 1); dV[1:] = V[1:ic + 1] + Z / r[1:ic + 1]          # non-Coulomb part inside r_cut
    nk = int(np.ceil(k_max / dk)) + 3
    k = dk * np.arange(nk)
    q = 2 * np.pi * k[:, None] * r[None, :ic + 1]
    sinc = np.where(q > 1e-6, np.sin(q) / np.where(q > 1e-6, q, 1.0), 1.0 - q * q / 6.0)
    g = 8 * np.pi * x[None, :ic + 1] ** 5 * dV[None, :] * sinc
    table = np.array([_simpson_cum(row, h)[-1] for row in g]) / Z
    return dict(dk=dk, table=table, r_ws=r_ws, r_cut=r[ic], mu=mu, abc=abc, iters=it, x=x, n_aa=dens, n_ps=ps, V_ps=V)
