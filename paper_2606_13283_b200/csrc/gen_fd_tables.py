#!/usr/bin/env python3
"""Generate fd_tables.h: piecewise polynomial fits of the Fermi-Dirac integrals
I_j(eta) = int_0^inf t^j/(exp(t-eta)+1) dt, j = -1/2, 1/2, 3/2 (Eq. 9), for the CUDA path.

Run by hand (needs mpmath; a few minutes on 8 cores):  python paper_2606_13283_b200/csrc/gen_fd_tables.py
The generated header is committed, so building the library needs no mpmath.

Method (own fits; no published coefficient table is used; nothing here is shared with oracle/):
  reference values: I_j(eta) = -Gamma(j+1) Li_{j+1}(-e^eta) with mpmath at 40 digits;
  segment 0          (eta <= ETA_A):        I_j = x * P(t), x = e^eta on [0, e^ETA_A]   (P absorbs Gamma(j+1));
  segments 1..NB+1   (ETA_A < eta < ETA_C): I_j = P(t), segments of width W CENTRED on eta_k = ETA_A + k W, k = 0..NB
                     (k = rint((eta - ETA_A)/W): the device gets k and t = (eta - eta_k)/W from one magic-number
                     addition, no float<->int conversion; the first and last segment are used on one half only);
  segment NB+2       (eta >= ETA_C):        I_j = eta^(j+1) * P(t), t from u = 1/eta^2 on [0, 1/ETA_C^2].
Every P is a polynomial in t on [-1/2, 1/2] (t = (x - centre)/width).
The poles of the Fermi function sit at eta +- i pi, so a Chebyshev interpolant on a segment of half-width h
converges like rho^-n with rho = pi/h + sqrt((pi/h)^2 + 1): W = 0.25 gives rho = 50 and degree 9 reaches 1e-16.
Region B reaches down to eta = -24 so that hot, dilute plasmas (eta << 0) never pay for an exp() per grid point.
Each P is the Chebyshev interpolant of degree FD_NC-1 converted to monomials in t.

Mixed precision (the table reads, not the FMAs, bound the device kernels: 64 bytes per function and point instead of
96): the monomial coefficients fall like rho^-k, so the tail c_6..c_9 (relative weight <= 50^-6 = 6e-11) is stored
and summed in fp32 -- B(t) = c6 + t (c7 + t (c8 + t c9)), four floats -- and the head c_0..c_5 in fp64, the Horner
recurrence simply continuing from (double)B(t): six DFMAs per function.  The fp32 rounding of the tail (1e-7 of
6e-11) is far below one fp64 ulp of the result.  The header stores the tail already rounded to fp32.  The script
checks every segment in simulated device arithmetic (fp32 tail, fp64 head) against mpmath and fails if the
relative error exceeds 1e-15.
"""
import os
import sys
from multiprocessing import Pool

import mpmath as mp
import numpy as np

mp.mp.dps = 40
NC = 10
NC_LO = 6      # c_0..c_5 in fp64; c_6..c_9 in fp32
ETA_A = -24.0
ETA_C = 40.0
W = 0.25
NB = int(round((ETA_C - ETA_A) / W))
TJ = (-1, 1, 3)


def I(tj, eta):
    j = mp.mpf(tj) / 2
    return mp.re(-mp.gamma(j + 1) * mp.polylog(j + 1, -mp.exp(eta)))


def cheb_to_mono(f, n):
    """monomial coefficients (in t on [-1,1]) of the degree n-1 Chebyshev interpolant of f"""
    nodes = [mp.cos(mp.pi * (i + mp.mpf(1) / 2) / n) for i in range(n)]
    fv = [f(x) for x in nodes]
    c = []
    for m in range(n):
        s = sum(fv[i] * mp.cos(mp.pi * m * (i + mp.mpf(1) / 2) / n) for i in range(n))
        c.append(2 * s / n)
    c[0] /= 2
    T = [[mp.mpf(1)], [mp.mpf(0), mp.mpf(1)]]
    for k in range(2, n):
        a = [mp.mpf(0)] + [2 * x for x in T[k - 1]]
        b = T[k - 2] + [mp.mpf(0)] * (len(a) - len(T[k - 2]))
        T.append([x - y for x, y in zip(a, b)])
    mono = [mp.mpf(0)] * n
    for k in range(n):
        for p, x in enumerate(T[k]):
            mono[p] += c[k] * x
    return mono


def horner_f64(co, t):
    """the device evaluation: fp32 Horner of the tail in float(t), then the fp64 Horner of the head continues from it"""
    tf = np.float32(t)
    b = np.float32(co[-1])
    for c in co[-2:NC_LO - 1:-1]:
        b = np.float32(b * tf + np.float32(c))
    acc = np.float64(b)
    for c in co[NC_LO - 1::-1]:
        acc = acc * np.float64(t) + np.float64(c)
    return acc


def seg_geometry(s):
    """(kind, centre, 1/width) of segment s in its own variable; t = (x - centre)/width in [-1/2, 1/2]"""
    if s == 0:
        xa = float(mp.exp(ETA_A))
        return "A", xa / 2, 1 / xa
    if s == NB + 2:
        um = 1.0 / ETA_C ** 2
        return "C", um / 2, 1 / um
    return "B", ETA_A + W * (s - 1), 1 / W


def fit_segment(s):
    mp.mp.dps = 40
    kind, c, ih = seg_geometry(s)
    co = {}
    for tj in TJ:
        j = mp.mpf(tj) / 2
        if kind == "A":
            def f(t):
                x = mp.mpf(c) + t / mp.mpf(ih)
                return I(tj, mp.log(x)) / x if x > 0 else mp.gamma(j + 1)
        elif kind == "B":
            def f(t):
                return I(tj, mp.mpf(c) + t / mp.mpf(ih))
        else:
            def f(t):
                u = mp.mpf(c) + t / mp.mpf(ih)
                if u <= 0:
                    return 1 / (j + 1)
                eta = 1 / mp.sqrt(u)
                return I(tj, eta) / eta ** (j + 1)
        mono = cheb_to_mono(lambda x: f(x / 2), NC)          # interpolant in x = 2t on [-1, 1]
        co[tj] = [m * mp.mpf(2) ** k for k, m in enumerate(mono)]   # -> monomials in t
    # verification in simulated double precision
    rng = np.random.default_rng(1000 + s)
    worst = 0.0
    for tj in TJ:
        cf = [float(x) for x in co[tj][:NC_LO]] + [float(np.float32(float(x))) for x in co[tj][NC_LO:]]
        for t in np.concatenate([rng.uniform(-0.5, 0.5, 24), [-0.5, 0.5, 0.0]]):
            v = np.float64(c) + np.float64(t) / np.float64(ih)
            tt = (v - np.float64(c)) * np.float64(ih)
            if kind == "A":
                if v <= 0:
                    continue
                eta = mp.log(mp.mpf(float(v))); val = v * horner_f64(cf, tt)
            elif kind == "B":
                eta = mp.mpf(float(v)); val = horner_f64(cf, tt)
            else:
                if v <= 1e-9:
                    continue
                eta = 1 / mp.sqrt(mp.mpf(float(v)))
                val = horner_f64(cf, tt) * float(eta ** (mp.mpf(tj) / 2 + 1))
            worst = max(worst, float(abs(mp.mpf(float(val)) / I(tj, eta) - 1)))
    out = {tj: [mp.nstr(x, 19, min_fixed=0, max_fixed=0) for x in co[tj][:NC_LO]] +
                [repr(float(np.float32(float(x)))) for x in co[tj][NC_LO:]] for tj in TJ}
    return s, out, worst


def main():
    with Pool(os.cpu_count()) as pool:
        res = pool.map(fit_segment, range(NB + 3), chunksize=1)
    res.sort()
    worst = max(r[2] for r in res)
    print("max rel err %.2e" % worst, file=sys.stderr)
    assert worst < 1e-15, worst
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "fd_tables.h")
    with open(out, "w") as fh:
        fh.write("// GENERATED by gen_fd_tables.py -- do not edit.  Piecewise fits of I_{-1/2}, I_{1/2}, I_{3/2}\n")
        fh.write("// (PAPER.md:124).  Max relative error of the device evaluation (fp32 tail, fp64 head) vs mpmath: %.2e\n" % worst)
        fh.write("#pragma once\n#define FD_NC %d\n#define FD_NC_LO %d\n#define FD_NB %d\n#define FD_NSEG %d\n" % (NC, NC_LO, NB, NB + 3))
        fh.write("#define FD_ETA_A %r\n#define FD_ETA_C %r\n#define FD_INV_W %r\n" % (ETA_A, ETA_C, 1.0 / W))
        ka, ca, iha = seg_geometry(0)
        kc, cc, ihc = seg_geometry(NB + 2)
        fh.write("#define FD_A_CENTER %r\n#define FD_A_INVW %r\n#define FD_C_CENTER %r\n#define FD_C_INVW %r\n"
                 % (ca, iha, cc, ihc))
        fh.write("// [function: -1/2, 1/2, 3/2][segment][monomial power of t in [-1/2,1/2]]; segment 0 = region A,\n")
        fh.write("// 1 + k (k = 0..FD_NB) = region B centred on FD_ETA_A + k/FD_INV_W, FD_NB+2 = region C.\n")
        fh.write("// Powers >= FD_NC_LO are exactly representable in fp32 (the device keeps them as floats).\n")
        fh.write("static const double FD_COEF[3][FD_NSEG][FD_NC] = {\n")
        for tj in TJ:
            fh.write("  { // I_{%d/2}\n" % tj)
            for s, co, _ in res:
                fh.write("    {%s},\n" % ", ".join(co[tj]))
            fh.write("  },\n")
        fh.write("};\n")
    print("wrote", out, "max rel err %.2e" % worst)


if __name__ == "__main__":
    main()
