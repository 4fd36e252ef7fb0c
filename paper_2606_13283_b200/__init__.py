"""paper_2606_13283_b200 -- B200-native (sm_100a, fp64 CUDA) hot path of Arche's orbital-free MD:
finite-temperature Thomas-Fermi SCF on a periodic grid + per-MD-step ion-grid work (arXiv 2606.13283).

This package is a thin ctypes binding over the C ABI in include/arche.h: it marshals arguments and lets
PyTorch own device memory and streams.  Every step of the path runs in the CUDA kernels of csrc/.
There is no CPU fallback: if the library is missing or no CUDA device is present the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from .build import LIB, build

__all__ = ["Arche", "ArcheError", "load", "SYMBOLS", "Params", "Result"]

SYMBOLS = ["arche_workspace_bytes", "arche_scf_init", "arche_destroy", "arche_last_error", "arche_scf_solve",
           "arche_scf_begin", "arche_scf_iter", "arche_set_input_density", "arche_forces", "arche_stress", "arche_md_step",
           "arche_md_step_host", "arche_get_real", "arche_get_complex", "arche_get_density", "arche_fft3d",
           "arche_rfft3d_forward", "arche_rfft3d_inverse",
           "arche_fermi_dirac", "arche_launch_count", "arche_profile_enable", "arche_profile_get", "arche_is_fused", "arche_is_persistent",
           "arche_peak_fp64", "arche_peak_l2", "arche_set_scf_iterations", "arche_fft3d_static",
           "arche_fft3d_slab_scatter", "arche_fft3d_slab_finish", "arche_slab_alloc", "arche_slab_free",
           "arche_ipc_export", "arche_ipc_open", "arche_ipc_close"]

ERRORS = {-1: "ARCHE_EINVAL", -2: "ARCHE_ENOMEM", -3: "ARCHE_ENOCONV", -4: "ARCHE_ENAN", -5: "ARCHE_ECUDA"}


class ArcheError(RuntimeError):
    pass


class Params(C.Structure):
    _fields_ = [("cell", C.c_double * 3), ("grid", C.c_int * 3), ("n_ions", C.c_int),
                ("h_Z", C.c_void_p), ("h_mass", C.c_void_p), ("kT", C.c_double), ("xc", C.c_int),
                ("psp_rc", C.c_double), ("init_mode", C.c_int), ("mix_mode", C.c_int),
                ("mix_w_fixed", C.c_double), ("mix_warmup", C.c_int), ("scf_tol_F", C.c_double),
                ("scf_tol_dn", C.c_double), ("scf_max_iter", C.c_int), ("scf_fixed_iter", C.c_int),
                ("ewald_alpha", C.c_double), ("n_electrons", C.c_double), ("psp", C.c_int), ("psp_nk", C.c_int),
                ("psp_dk", C.c_double), ("h_psp_table", C.c_void_p), ("mix_mu_tol", C.c_double), ("mix_chi_floor", C.c_double),
                ("ensemble", C.c_int), ("d_workspace", C.c_void_p),
                ("workspace_bytes", C.c_size_t), ("stream", C.c_void_p)]


class Result(C.Structure):
    _fields_ = [(k, C.c_double) for k in ("mu", "F_total", "F0", "E_H", "E_xc", "E_ie", "E_ie0", "U_ii", "K_e",
                                          "K_i", "dn_l2", "w_last", "U_mix", "K_mix", "tol_F_eff", "tol_dn_eff")] + \
               [(k, C.c_int) for k in ("scf_iters", "mu_evals", "converged", "flip_seen", "F_evals")]

    def asdict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


_lib = None


def load(rebuild_if_stale: bool = True):
    """dlopen the C-ABI library (building it in-tree first if the sources are newer). Fails loudly."""
    global _lib
    if _lib is not None:
        return _lib
    path = build() if rebuild_if_stale else LIB
    if not os.path.exists(path):
        raise ArcheError(f"CUDA library missing: {path} (run python -m paper_2606_13283_b200.build)")
    L = C.CDLL(path)
    vp, dp = C.c_void_p, C.c_void_p
    L.arche_workspace_bytes.restype = C.c_size_t
    L.arche_workspace_bytes.argtypes = [C.POINTER(Params)]
    L.arche_scf_init.argtypes = [C.POINTER(Params), C.POINTER(vp)]
    L.arche_destroy.argtypes = [vp]; L.arche_destroy.restype = None
    L.arche_last_error.argtypes = [vp]; L.arche_last_error.restype = C.c_char_p
    L.arche_scf_solve.argtypes = [vp, dp, C.POINTER(Result)]
    L.arche_scf_begin.argtypes = [vp, dp]
    L.arche_scf_iter.argtypes = [vp, C.POINTER(Result)]
    L.arche_set_input_density.argtypes = [vp, dp]
    L.arche_forces.argtypes = [vp, dp]
    L.arche_stress.argtypes = [vp, dp, C.POINTER(C.c_double)]
    L.arche_md_step.argtypes = [vp, C.c_double, dp, dp, C.POINTER(Result)]
    L.arche_md_step_host.argtypes = [vp, C.c_double, dp, dp, dp, C.POINTER(Result)]
    L.arche_get_real.argtypes = [vp, C.c_int, dp]
    L.arche_get_complex.argtypes = [vp, C.c_int, dp]
    L.arche_get_density.argtypes = [vp, dp]
    L.arche_fft3d.argtypes = [vp, dp, dp, dp, C.c_int]
    L.arche_fft3d_static.argtypes = [vp, dp, dp, C.c_int]
    L.arche_rfft3d_forward.argtypes = [vp, dp, dp]
    L.arche_rfft3d_inverse.argtypes = [vp, dp, dp]
    L.arche_fermi_dirac.argtypes = [vp, C.c_int, dp, dp, C.c_size_t]
    L.arche_launch_count.argtypes = [vp]; L.arche_launch_count.restype = C.c_longlong
    L.arche_profile_enable.argtypes = [vp, C.c_int]
    L.arche_is_fused.argtypes = [vp]
    L.arche_is_persistent.argtypes = [vp]
    L.arche_profile_get.argtypes = [vp, C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_longlong)]
    L.arche_peak_fp64.argtypes = [vp, C.c_double, C.POINTER(C.c_double), C.POINTER(C.c_double)]
    L.arche_peak_l2.argtypes = [vp, C.POINTER(C.c_double)]
    L.arche_set_scf_iterations.argtypes = [vp, C.c_int, C.c_int]
    L.arche_fft3d_slab_scatter.argtypes = [vp, vp, vp, C.POINTER(vp), C.c_int, C.c_int, C.c_int]
    L.arche_fft3d_slab_finish.argtypes = [vp, vp, C.c_int, C.c_int]
    L.arche_slab_alloc.argtypes = [C.c_size_t, C.POINTER(vp)]
    L.arche_slab_free.argtypes = [vp]
    L.arche_ipc_export.argtypes = [vp, C.c_char_p]
    L.arche_ipc_open.argtypes = [C.c_char_p, C.POINTER(vp)]
    L.arche_ipc_close.argtypes = [vp]
    _lib = L
    return L


_DEFAULTS = dict(xc=1, psp_rc=1.12, init_mode=1, mix_mode=1, mix_w_fixed=0.95, mix_warmup=3, scf_tol_F=1e-10,
                 scf_tol_dn=1e-12, scf_max_iter=500, scf_fixed_iter=0, ewald_alpha=0.0, n_electrons=0.0, mix_mu_tol=0.0, mix_chi_floor=0.0,
                 ensemble=0)


class Arche:
    """One SCF/MD context on the current CUDA device; torch owns the workspace and the stream."""

    def __init__(self, cfg: dict, device="cuda:0", stream=None, **over):
        import torch
        if not torch.cuda.is_available():
            raise ArcheError("no CUDA device: the Arche hot path has no CPU fallback")
        self.torch = torch
        self.lib = load()
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        p = dict(_DEFAULTS)
        for k in p:
            if k in cfg:
                p[k] = cfg[k]
        p.update(over)
        table = p.pop("psp_table", cfg.get("psp_table")); dk = p.pop("psp_dk", cfg.get("psp_dk", 0.0))
        self._Z = np.ascontiguousarray(cfg["Z"], dtype=np.float64)
        self._m = np.ascontiguousarray(cfg["mass"], dtype=np.float64)
        self.n_ions = len(self._Z)
        self.grid = [int(g) for g in cfg["grid"]]
        self.shape = (self.grid[2], self.grid[1], self.grid[0])
        self.ng = self.grid[0] * self.grid[1] * self.grid[2]
        P = Params()
        P.cell[:] = [float(x) for x in cfg["cell"]]
        P.grid[:] = self.grid
        P.n_ions = self.n_ions
        P.h_Z = self._Z.ctypes.data if self.n_ions else None
        P.h_mass = self._m.ctypes.data if self.n_ions else None
        P.kT = float(cfg["kT"])
        for k, v in p.items():
            setattr(P, k, v)
        if table is not None:                     # f2: tabulated form factor (non-Coulomb part per unit charge)
            self._tab = np.ascontiguousarray(table, dtype=np.float64)
            P.psp = 1; P.psp_nk = len(self._tab); P.psp_dk = float(dk); P.h_psp_table = self._tab.ctypes.data
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        P.stream = self.stream.cuda_stream
        nbytes = self.lib.arche_workspace_bytes(C.byref(P))
        if nbytes == 0:
            raise ArcheError("arche_workspace_bytes: invalid parameters")
        self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        ptr = (self.workspace.data_ptr() + 255) & ~255
        P.d_workspace = ptr
        P.workspace_bytes = nbytes
        self.params = P
        self._h = C.c_void_p()
        rc = self.lib.arche_scf_init(C.byref(P), C.byref(self._h))
        if rc != 0:
            raise ArcheError(f"arche_scf_init failed: {ERRORS.get(rc, rc)}")

    # -- helpers
    def _check(self, rc, allow_noconv=True):
        if rc == 0 or (allow_noconv and rc == -3):
            return rc
        msg = self.lib.arche_last_error(self._h)
        raise ArcheError(f"{ERRORS.get(rc, rc)}: {msg.decode() if msg else ''}")

    def _dev(self, a):
        t = self.torch
        if isinstance(a, t.Tensor):
            assert a.is_cuda and a.dtype in (t.float64, t.complex128) and a.is_contiguous()
            return a
        return t.as_tensor(np.ascontiguousarray(a, dtype=np.float64), device=self.device)

    def close(self):
        if getattr(self, "_h", None):
            self.lib.arche_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- the C-ABI calls
    def scf_solve(self, pos) -> dict:
        d = self._dev(pos); r = Result()
        with self.torch.cuda.stream(self.stream):
            rc = self._check(self.lib.arche_scf_solve(self._h, d.data_ptr(), C.byref(r)))
        out = r.asdict(); out["rc"] = rc
        return out

    def scf_begin(self, pos):
        d = self._dev(pos)
        self._check(self.lib.arche_scf_begin(self._h, d.data_ptr() if self.n_ions else None))

    def scf_iter(self) -> dict:
        r = Result()
        self._check(self.lib.arche_scf_iter(self._h, C.byref(r)))
        return r.asdict()

    def set_scf_iterations(self, max_iter: int = 0, fixed_iter: int = 0):
        self._check(self.lib.arche_set_scf_iterations(self._h, int(max_iter), int(fixed_iter)))

    def set_input_density(self, n):
        d = self._dev(n)
        self._check(self.lib.arche_set_input_density(self._h, d.data_ptr()))

    def forces(self, out=None):
        t = self.torch
        F = out if out is not None else t.empty((self.n_ions, 3), dtype=t.float64, device=self.device)
        self._check(self.lib.arche_forces(self._h, F.data_ptr()))
        return F

    STRESS_ROWS = ("i", "e", "xc", "pp", "pm", "je", "ee", "ie", "total")

    def stress(self, vel=None) -> dict:
        """Stress tensor of the last solve (include/arche.h: arche_stress): row name -> [xx, yy, zz, yz, xz, xy]
        (numpy), and 'P' = -tr(total)/3.  vel: CUDA float64 tensor [n_ions,3] or None."""
        import numpy as np
        out = (C.c_double * 55)()
        self._check(self.lib.arche_stress(self._h, None if vel is None else vel.data_ptr(), out))
        a = np.array(out[:])
        d = {k: a[6 * r:6 * r + 6].copy() for r, k in enumerate(self.STRESS_ROWS)}
        d["P"] = float(a[54])
        return d

    def md_step(self, dt, pos, vel) -> dict:
        """pos, vel: CUDA float64 tensors [n_ions,3], updated in place."""
        r = Result()
        rc = self._check(self.lib.arche_md_step(self._h, float(dt), pos.data_ptr(), vel.data_ptr(), C.byref(r)))
        out = r.asdict(); out["rc"] = rc
        return out

    def md_step_host(self, dt, pos, vel, F=None) -> dict:
        """pos, vel (and F): host float64 arrays (numpy or pinned torch CPU tensors), updated in place."""
        r = Result()
        ptr = lambda a: a.ctypes.data if isinstance(a, np.ndarray) else a.data_ptr()
        rc = self._check(self.lib.arche_md_step_host(self._h, float(dt), ptr(pos), ptr(vel),
                                                     ptr(F) if F is not None else None, C.byref(r)))
        out = r.asdict(); out["rc"] = rc
        return out

    def get_real(self, which: str):
        t = self.torch
        a = t.empty(self.shape, dtype=t.float64, device=self.device)
        self._check(self.lib.arche_get_real(self._h, {"n_a": 0, "n_i": 1, "V_i": 2}[which], a.data_ptr()))
        return a

    def get_complex(self, which: str):
        t = self.torch
        a = t.empty(self.shape, dtype=t.complex128, device=self.device)
        idx = {"nhat_a": 0, "Vhat_ie": 1, "S_Z": 2, "ghat": 3, "nhat_i": 4}[which]
        self._check(self.lib.arche_get_complex(self._h, idx, a.data_ptr()))
        return a

    def fft3d(self, a, sign: int):
        t = self.torch
        a = a.to(device=self.device, dtype=t.complex128).contiguous()
        out = t.empty_like(a); scratch = t.empty_like(a)
        self._check(self.lib.arche_fft3d(self._h, a.data_ptr(), out.data_ptr(), scratch.data_ptr(), int(sign)))
        return out

    def fft3d_static(self, a, sign: int, out=None):
        """arche_fft3d_static: no scratch argument, nothing allocated inside the call (grids up to 64^3 points)"""
        t = self.torch
        a = a.to(device=self.device, dtype=t.complex128).contiguous()
        if out is None:
            out = t.empty_like(a)
        self._check(self.lib.arche_fft3d_static(self._h, a.data_ptr(), out.data_ptr(), int(sign)))
        return out

    def fft3d_slab_scatter(self, d_in, d_scratch, peers, rank: int, sign: int):
        """arche_fft3d_slab_scatter: d_in / d_scratch / peers[q] are device addresses (int); see include/arche.h"""
        arr = (C.c_void_p * len(peers))(*[int(p) for p in peers])
        self._check(self.lib.arche_fft3d_slab_scatter(self._h, int(d_in), int(d_scratch) if d_scratch else None, arr,
                                                      len(peers), int(rank), int(sign)))

    def fft3d_slab_finish(self, d_slab, n_ranks: int, sign: int):
        self._check(self.lib.arche_fft3d_slab_finish(self._h, int(d_slab), int(n_ranks), int(sign)))

    def rfft3d_forward(self, a):
        """real [nz,ny,nx] -> full unnormalised complex spectrum, through the SCF's own r2c passes"""
        t = self.torch
        a = a.to(device=self.device, dtype=t.float64).contiguous()
        out = t.empty(self.shape, dtype=t.complex128, device=self.device)
        self._check(self.lib.arche_rfft3d_forward(self._h, a.data_ptr(), out.data_ptr()))
        return out

    def rfft3d_inverse(self, ahat):
        """Hermitian complex spectrum [nz,ny,nx] -> real unnormalised inverse transform (c2r passes)"""
        t = self.torch
        ahat = ahat.to(device=self.device, dtype=t.complex128).contiguous()
        out = t.empty(self.shape, dtype=t.float64, device=self.device)
        self._check(self.lib.arche_rfft3d_inverse(self._h, ahat.data_ptr(), out.data_ptr()))
        return out

    def fermi_dirac(self, twice_j: int, eta):
        t = self.torch
        e = self._dev(eta); out = t.empty_like(e)
        self._check(self.lib.arche_fermi_dirac(self._h, int(twice_j), e.data_ptr(), out.data_ptr(), e.numel()))
        return out

    PROFILE_CLASSES = ("fft_inv_z_potential", "fft_y", "fft_inv_x_vi", "mu_pass", "density", "fft_fwd_x_real",
                       "fft_fwd_z_reduce", "mix", "structure_factor", "force", "ewald_pp", "other",
                       "potential_g", "vi_r", "density_r", "reduce_g", "stress_fields")

    def is_fused(self) -> bool:
        return bool(self.lib.arche_is_fused(self._h))

    def is_persistent(self) -> bool:
        return bool(self.lib.arche_is_persistent(self._h))

    def profile_enable(self, on: bool = True):
        self._check(self.lib.arche_profile_enable(self._h, int(on)))

    def profile_get(self) -> dict:
        out = {}
        for i, name in enumerate(self.PROFILE_CLASSES):
            ms, n = C.c_double(), C.c_longlong()
            self._check(self.lib.arche_profile_get(self._h, i, C.byref(ms), C.byref(n)))
            out[name] = (ms.value, n.value)
        return out

    def peak_fp64(self, seconds: float = 1.0) -> dict:
        """measured fp64 FMA rate of the vector pipe (TFLOP/s): sustained over `seconds`, and the best single launch"""
        out = (C.c_double * 2)(); ms = C.c_double()
        self._check(self.lib.arche_peak_fp64(self._h, float(seconds), out, C.byref(ms)))
        return {"sustained_tflops": out[0], "burst_tflops": out[1], "ran_ms": ms.value}

    def peak_l2(self) -> float:
        """measured L2 read bandwidth (GB/s)"""
        v = C.c_double()
        self._check(self.lib.arche_peak_l2(self._h, C.byref(v)))
        return v.value

    def launch_count(self) -> int:
        return int(self.lib.arche_launch_count(self._h))

    def sync(self):
        self.stream.synchronize()
