"""CPU ORACLE -- TEST INFRASTRUCTURE ONLY.

ctypes wrapper around oracle/arche_oracle.c (plain fp64 C written from PAPER.md).  Only tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline / `--impl reference` legs may import this.
It shares no code with paper_2606_13283_b200/.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "liboracle.so")
_SRC = os.path.join(_HERE, "arche_oracle.c")
_SRC_AA = os.path.join(_HERE, "aa_pseudopotential.c")


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2 -fopenmp). Building the checker is not using it."""
    hdr = os.path.join(_HERE, "arche_oracle.h")
    stale = (not os.path.exists(_SO)) or any(
        os.path.getmtime(f) > os.path.getmtime(_SO) for f in (_SRC, _SRC_AA, hdr))
    if force or stale:
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=gnu11",
                               "-o", _SO, _SRC, _SRC_AA, "-lm"])
    return _SO


class Params(C.Structure):
    _fields_ = [("cell", C.c_double * 3), ("grid", C.c_int * 3), ("n_ions", C.c_int),
                ("Z", C.POINTER(C.c_double)), ("mass", C.POINTER(C.c_double)), ("kT", C.c_double),
                ("xc", C.c_int), ("psp_rc", C.c_double), ("init_mode", C.c_int),
                ("mix_mode", C.c_int), ("mix_w_fixed", C.c_double), ("mix_warmup", C.c_int),
                ("scf_tol_F", C.c_double), ("scf_tol_dn", C.c_double), ("scf_max_iter", C.c_int),
                ("scf_fixed_iter", C.c_int), ("ewald_alpha", C.c_double),
                ("n_electrons", C.c_double), ("mix_mu_tol", C.c_double), ("psp", C.c_int), ("psp_nk", C.c_int),
                ("psp_dk", C.c_double), ("mix_chi_floor", C.c_double), ("psp_table", C.POINTER(C.c_double)),
                ("ensemble", C.c_int)]


class Result(C.Structure):
    _fields_ = [(k, C.c_double) for k in ("mu", "F_total", "F0", "E_H", "E_xc", "E_ie", "E_ie0",
                                          "U_ii", "K_e", "K_i", "dn_l2", "w_last", "U_mix",
                                          "K_mix", "tol_F_eff", "tol_dn_eff")] + \
               [(k, C.c_int) for k in ("scf_iters", "mu_evals", "converged", "flip_seen")]

    def asdict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        dp = C.POINTER(C.c_double)
        ip = C.POINTER(C.c_int)
        L.oracle_fd.restype = C.c_double
        L.oracle_fd.argtypes = [C.c_int, C.c_double]
        L.oracle_fd_half_inverse.restype = C.c_double
        L.oracle_fd_half_inverse.argtypes = [C.c_double]
        L.oracle_fft3d.argtypes = [C.c_int, C.c_int, C.c_int, dp, C.c_int]
        L.oracle_dft3d_naive.argtypes = [C.c_int, C.c_int, C.c_int, dp, C.c_int]
        L.oracle_xc.argtypes = [C.c_int, C.c_double, dp, dp]
        L.oracle_structure_factor.argtypes = [dp, ip, C.c_int, dp, dp, dp]
        L.oracle_table_interp.restype = C.c_double
        L.oracle_table_interp.argtypes = [C.c_int, C.c_double, dp, C.c_double, dp]
        L.oracle_vps_unit.restype = C.c_double
        L.oracle_vps_unit.argtypes = [C.c_double, C.c_double]
        L.oracle_ewald_alpha.restype = C.c_double
        L.oracle_ewald_alpha.argtypes = [dp, ip]
        L.oracle_ewald.argtypes = [dp, ip, C.c_int, dp, dp, C.c_double, dp, dp]
        L.oracle_force_ie.argtypes = [dp, ip, C.c_int, dp, dp, C.c_double, dp, dp]
        L.oracle_init.argtypes = [C.POINTER(Params), C.POINTER(C.c_void_p)]
        L.oracle_destroy.argtypes = [C.c_void_p]
        L.oracle_scf_begin.argtypes = [C.c_void_p, dp]
        L.oracle_set_input_density.argtypes = [C.c_void_p, dp]
        L.oracle_set_profile.argtypes = [C.c_void_p, dp]
        L.oracle_scf_iter.argtypes = [C.c_void_p, C.POINTER(Result)]
        L.oracle_scf_solve.argtypes = [C.c_void_p, dp, C.POINTER(Result)]
        L.oracle_forces.argtypes = [C.c_void_p, dp]
        L.oracle_md_step.argtypes = [C.c_void_p, C.c_double, dp, dp, C.POINTER(Result)]
        L.oracle_stress.argtypes = [C.c_void_p, dp, dp]
        L.oracle_isokinetic_kick.argtypes = [C.c_int, dp, dp, C.c_double, dp]
        L.oracle_get_real.argtypes = [C.c_void_p, C.c_int, dp]
        L.oracle_get_complex.argtypes = [C.c_void_p, C.c_int, dp]
        L.oracle_num_threads.restype = C.c_int
        L.oracle_fd_wide.restype = C.c_double
        L.oracle_fd_wide.argtypes = [C.c_int, C.c_double]
        L.oracle_fd_half_inverse_wide.restype = C.c_double
        L.oracle_fd_half_inverse_wide.argtypes = [C.c_double]
        L.oracle_aa_solve.argtypes = [C.c_double, C.c_double, C.c_double, C.c_int, C.c_int, dp, dp, dp, ip]
        L.oracle_aa_pseudize.argtypes = [C.c_int, dp, dp, C.c_int, dp, dp]
        L.oracle_aa_invert.argtypes = [C.c_double, C.c_int, C.c_int, dp, dp, C.c_double, C.c_double, dp]
        L.oracle_radial_ft.argtypes = [C.c_int, dp, dp, C.c_int, C.c_int, dp, dp]
        L.oracle_aa_energy.argtypes = [C.c_double, C.c_int, C.c_int, dp, dp, C.c_double, dp, C.c_double, dp]
        _lib = L
    return _lib


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _ip(a):
    return a.ctypes.data_as(C.POINTER(C.c_int))


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def fd(twice_j: int, eta) -> np.ndarray:
    """I_{twice_j/2}(eta) by adaptive quadrature."""
    e = np.atleast_1d(np.asarray(eta, dtype=np.float64))
    return np.array([lib().oracle_fd(int(twice_j), float(x)) for x in e.ravel()]).reshape(e.shape)


def fd_half_inverse(y: float) -> float:
    return lib().oracle_fd_half_inverse(float(y))


def fft3d(a: np.ndarray, sign: int, naive: bool = False) -> np.ndarray:
    """Unnormalised 3D DFT of a[z,y,x] (complex128); sign=-1 forward."""
    b = np.ascontiguousarray(a, dtype=np.complex128).copy()
    nz, ny, nx = b.shape
    f = lib().oracle_dft3d_naive if naive else lib().oracle_fft3d
    f(nx, ny, nz, _dp(b.view(np.float64)), int(sign))
    return b


def xc(n: float, kind: int = 1):
    e, v = C.c_double(), C.c_double()
    lib().oracle_xc(kind, float(n), C.byref(e), C.byref(v))
    return e.value, v.value


def structure_factor(cell, grid, pos, Z) -> np.ndarray:
    cell = _f64(cell); grid = np.ascontiguousarray(grid, dtype=np.int32)
    pos = _f64(pos); Z = _f64(Z)
    S = np.empty((grid[2], grid[1], grid[0]), dtype=np.complex128)
    lib().oracle_structure_factor(_dp(cell), _ip(grid), len(Z), _dp(pos), _dp(Z), _dp(S.view(np.float64)))
    return S


def vps_unit(k: float, rc: float) -> float:
    return lib().oracle_vps_unit(float(k), float(rc))


def ewald_alpha(cell, grid) -> float:
    cell = _f64(cell); grid = np.ascontiguousarray(grid, dtype=np.int32)
    return lib().oracle_ewald_alpha(_dp(cell), _ip(grid))


def ewald(cell, grid, pos, Z, alpha=None):
    """Returns (U_pp, U_pm, U_je), F[n,3]."""
    cell = _f64(cell); grid = np.ascontiguousarray(grid, dtype=np.int32)
    pos = _f64(pos); Z = _f64(Z)
    if alpha is None:
        alpha = ewald_alpha(cell, grid)
    U = np.zeros(3); F = np.zeros((len(Z), 3))
    lib().oracle_ewald(_dp(cell), _ip(grid), len(Z), _dp(pos), _dp(Z), float(alpha), _dp(U), _dp(F))
    return U, F


def force_ie(cell, grid, pos, Z, rc, nhat) -> np.ndarray:
    cell = _f64(cell); grid = np.ascontiguousarray(grid, dtype=np.int32)
    pos = _f64(pos); Z = _f64(Z)
    nh = np.ascontiguousarray(nhat, dtype=np.complex128)
    F = np.zeros((len(Z), 3))
    lib().oracle_force_ie(_dp(cell), _ip(grid), len(Z), _dp(pos), _dp(Z), float(rc),
                          _dp(nh.view(np.float64)), _dp(F))
    return F


# ---- f2: average-atom pseudopotential (aa_pseudopotential.c)
def isokinetic_kick(mass, F, t, vel) -> np.ndarray:
    """Exact constant-force flow of the Gaussian isokinetic equations over a time t (reading A23); returns the new velocities."""
    m = _f64(mass); f = _f64(F); v = _f64(vel).copy()
    lib().oracle_isokinetic_kick(len(m), _dp(m), _dp(f), float(t), _dp(v))
    return v


def fd_wide(twice_j, eta):
    return lib().oracle_fd_wide(int(twice_j), float(eta))


def aa_solve(Z, r_ws, kT, xc=0, n=1201):
    r = np.zeros(n); dens = np.zeros(n); mu = C.c_double(); it = C.c_int()
    rc = lib().oracle_aa_solve(float(Z), float(r_ws), float(kT), int(xc), n, _dp(r), _dp(dens), C.byref(mu), C.byref(it))
    if rc != 0:
        raise RuntimeError(f"oracle_aa_solve: {rc} after {it.value} iterations")
    return r, dens, mu.value, it.value


def aa_pseudize(r, n_aa, ic):
    n_ps = np.zeros_like(r); abc = np.zeros(3)
    rc = lib().oracle_aa_pseudize(len(r), _dp(_f64(r)), _dp(_f64(n_aa)), int(ic), _dp(n_ps), _dp(abc))
    if rc != 0:
        raise RuntimeError(f"oracle_aa_pseudize: {rc}")
    return n_ps, abc


def aa_invert(kT, xc, r, dens, n0lim, mu):
    V = np.zeros_like(r)
    lib().oracle_aa_invert(float(kT), int(xc), len(r), _dp(_f64(r)), _dp(_f64(dens)), float(n0lim), float(mu), _dp(V))
    return V


def radial_ft(r, f, ic, k):
    k = _f64(np.atleast_1d(k)); out = np.zeros_like(k)
    lib().oracle_radial_ft(len(r), _dp(_f64(r)), _dp(_f64(f)), int(ic), len(k), _dp(k), _dp(out))
    return out


def aa_energy(kT, xc, r, dens, n0lim, V_ext, Z):
    out = np.zeros(4)
    v = None if V_ext is None else _dp(_f64(V_ext))
    lib().oracle_aa_energy(float(kT), int(xc), len(r), _dp(_f64(r)), _dp(_f64(dens)), float(n0lim), v, float(Z), _dp(out))
    return out


STRESS_ROWS = ("i", "e", "xc", "pp", "pm", "je", "ee", "ie", "total")


class Oracle:
    """SCF/MD context (mirrors the C-ABI of the product, with host arrays)."""

    def __init__(self, cfg: dict, **over):
        p = dict(xc=1, psp_rc=1.12, init_mode=1, mix_mode=1, mix_w_fixed=0.95, mix_warmup=3,
                 scf_tol_F=1e-10, scf_tol_dn=1e-12, scf_max_iter=500, scf_fixed_iter=0,
                 ewald_alpha=0.0, n_electrons=0.0, mix_mu_tol=0.0, mix_chi_floor=0.0, ensemble=0)
        for k in p:
            if k in cfg:
                p[k] = cfg[k]
        p.update(over)
        table = p.pop("psp_table", cfg.get("psp_table")); dk = p.pop("psp_dk", cfg.get("psp_dk", 0.0))
        self.cell = _f64(cfg["cell"]); self.grid = np.ascontiguousarray(cfg["grid"], dtype=np.int32)
        self._Z = _f64(cfg["Z"]); self._m = _f64(cfg["mass"])
        self.n_ions = len(self._Z)
        P = Params()
        P.cell[:] = list(self.cell); P.grid[:] = [int(g) for g in self.grid]
        P.n_ions = self.n_ions; P.Z = _dp(self._Z); P.mass = _dp(self._m); P.kT = float(cfg["kT"])
        for k, v in p.items():
            setattr(P, k, v)
        if table is not None:                     # f2: tabulated form factor (non-Coulomb part per unit charge)
            self._tab = _f64(table)
            P.psp = 1; P.psp_nk = len(self._tab); P.psp_dk = float(dk); P.psp_table = _dp(self._tab)
        self.params = P
        self._h = C.c_void_p()
        rc = lib().oracle_init(C.byref(P), C.byref(self._h))
        if rc != 0:
            raise ValueError(f"oracle_init failed: {rc}")
        self.shape = (int(self.grid[2]), int(self.grid[1]), int(self.grid[0]))

    def close(self):
        if self._h:
            lib().oracle_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def scf_begin(self, pos):
        lib().oracle_scf_begin(self._h, _dp(_f64(pos)))

    def set_input_density(self, n_i):
        lib().oracle_set_input_density(self._h, _dp(_f64(n_i)))

    def set_profile(self, ghat):
        g = np.ascontiguousarray(ghat, dtype=np.complex128)
        assert g.shape == self.shape
        lib().oracle_set_profile(self._h, _dp(g.view(np.float64)))

    def scf_iter(self) -> dict:
        r = Result()
        lib().oracle_scf_iter(self._h, C.byref(r))
        return r.asdict()

    def scf_solve(self, pos) -> dict:
        r = Result()
        rc = lib().oracle_scf_solve(self._h, _dp(_f64(pos)), C.byref(r))
        d = r.asdict(); d["rc"] = rc
        return d

    def forces(self) -> np.ndarray:
        F = np.zeros((self.n_ions, 3))
        rc = lib().oracle_forces(self._h, _dp(F))
        if rc != 0:
            raise RuntimeError("oracle_forces before a solve")
        return F

    def stress(self, vel=None) -> dict:
        """Stress tensor of the last solve: {'i','e','xc','pp','pm','je','ee','ie','total'} ->
        [xx, yy, zz, yz, xz, xy], and 'P' = -tr(total)/3."""
        out = np.zeros(55)
        v = None if vel is None else _dp(_f64(vel))
        rc = lib().oracle_stress(self._h, v, _dp(out))
        if rc != 0:
            raise RuntimeError("oracle_stress before a solve")
        d = {k: out[6 * r:6 * r + 6].copy() for r, k in enumerate(STRESS_ROWS)}
        d["P"] = float(out[54])
        return d

    def md_step(self, dt, pos, vel) -> dict:
        """pos, vel: float64 C-contiguous arrays, updated in place."""
        assert pos.flags.c_contiguous and vel.flags.c_contiguous and pos.dtype == np.float64
        r = Result()
        rc = lib().oracle_md_step(self._h, float(dt), _dp(pos), _dp(vel), C.byref(r))
        d = r.asdict(); d["rc"] = rc
        return d

    def get_real(self, which: str) -> np.ndarray:
        idx = {"n_a": 0, "n_i": 1, "V_i": 2}[which]
        a = np.empty(self.shape)
        lib().oracle_get_real(self._h, idx, _dp(a))
        return a

    def get_complex(self, which: str) -> np.ndarray:
        idx = {"nhat_a": 0, "Vhat_ie": 1, "S_Z": 2, "ghat": 3, "nhat_i": 4}[which]
        a = np.empty(self.shape, dtype=np.complex128)
        lib().oracle_get_complex(self._h, idx, _dp(a.view(np.float64)))
        return a
