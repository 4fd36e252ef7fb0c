"""Constructs an SCF problem whose converged density puts ONE grid point on the PZ81 branch point n* = 3/(4 pi)
(r_s = 1), where the published parametrisation is discontinuous (reading A13): a tiny cell with one ion
and N_e electrons on a uniform background; N_e is tuned by regula falsi / bisection on n(g0; N_e) - n* using oracle
solves only.  Shared by the oracle pin (tests/test_oracle_scf_pins.py) and the GPU parity test."""
import numpy as np

NSTAR = 3.0 / (4.0 * np.pi)
KW = dict(scf_tol_F=1e-12, scf_tol_dn=1e-11, scf_max_iter=300, init_mode=0)


def base_cfg():
    return dict(cell=np.array([3.0, 3.2, 3.4]), grid=np.array([4, 4, 4], dtype=np.int32), Z=np.array([1.0]),
                mass=np.array([1.0e4]), kT=10.0 / 27.211386245988, pos=np.array([[0.4, 1.1, 2.0]]))


def find_flip_case(orc):
    """returns (cfg, Ne_flip, Ne_below, Ne_above, g0): a solve at Ne_flip shows the branch flip at flat index g0; the
    solves at Ne_below / Ne_above converge smoothly with n(g0) on either side of n*"""
    cfg = base_cfg()
    vol = float(np.prod(cfg["cell"]))

    def solve(Ne):
        o = orc.Oracle(cfg, n_electrons=Ne, **KW)
        r = o.scf_solve(cfg["pos"])
        return r, o.get_real("n_a").ravel()

    Ne0 = NSTAR * vol
    _, n = solve(Ne0)
    g0 = int(np.argmin(np.abs(n - NSTAR)))
    a, b = 0.97 * Ne0, 1.03 * Ne0
    (ra, na), (rb, nb) = solve(a), solve(b)
    fa, fb = na[g0] - NSTAR, nb[g0] - NSTAR
    assert fa < 0 < fb and ra["flip_seen"] == 0 and rb["flip_seen"] == 0 and ra["converged"] and rb["converged"]
    below, above = a, b
    for it in range(60):
        x = (a * fb - b * fa) / (fb - fa) if it % 2 == 0 else 0.5 * (a + b)
        r, n = solve(x)
        if r["flip_seen"] or not r["converged"]:
            return cfg, x, below, above, g0
        fx = n[g0] - NSTAR
        if fx < 0:
            a, fa = x, fx
        else:
            b, fb = x, fx
    raise AssertionError("no branch flip found")
