"""Seeded synthetic workload generator shared by the oracle tests, the GPU tests and bench.py.

This module holds *data recipes only* (cells, positions, velocities, masses): none of the
method's arithmetic lives here, so both the CPU oracle (`oracle/`) and the CUDA path
(`paper_2606_13283_b200/`) may consume its arrays without sharing code.

The recipes are the five configurations of BASELINE.json (aluminium-like plasmas; they stand in
for the paper's own Al/H/O production runs, which are not public data).
DESIGN.md section "Input recipe" restates them.
"""
from __future__ import annotations

import numpy as np

# CODATA-2018 unit conversions (units only, no physics of the method).
HARTREE_EV = 27.211386245988
AMU_ME = 1822.888486209          # electron masses per atomic mass unit
FS_AU = 41.341373335             # atomic time units per femtosecond
BOHR_ANG = 0.529177210903
AMU_G = 1.66053906660e-24
SEED_BASE = 1328300

AL_MASS_U = 26.98
AL_Z = 3.0
ASHCROFT_RC = 1.12

_FCC_BASIS = np.array([[0.0, 0.0, 0.0], [0.5, 0.5, 0.0], [0.5, 0.0, 0.5], [0.0, 0.5, 0.5]])


def _cubic_L(n_ions: int, rho_gcc: float) -> float:
    vol_cm3 = n_ions * AL_MASS_U * AMU_G / rho_gcc
    return (vol_cm3 * 1e24) ** (1.0 / 3.0) / BOHR_ANG


def _fcc_sites(reps, a):
    sites = []
    for ix in range(reps[0]):
        for iy in range(reps[1]):
            for iz in range(reps[2]):
                for b in _FCC_BASIS:
                    sites.append(((ix + b[0]) * a, (iy + b[1]) * a, (iz + b[2]) * a, ix, iy, iz))
    return np.array(sites)


def _maxwell(rng, n, kT, mass):
    v = rng.standard_normal((n, 3)) * np.sqrt(kT / mass)[:, None]
    v -= (mass[:, None] * v).sum(0) / mass.sum()          # remove centre-of-mass drift once
    return v


def _random_positions(rng, n, L, dmin):
    pos = np.empty((n, 3))
    k = 0
    while k < n:
        p = rng.random(3) * L
        if dmin > 0.0 and k > 0:
            d = pos[:k] - p
            d -= L * np.rint(d / L)
            if (np.einsum("ij,ij->i", d, d) < dmin * dmin).any():
                continue
        pos[k] = p
        k += 1
    return pos


def make_config(name: str, grid: int | None = None) -> dict:
    """Return the workload `name` in {"c1","c2","c3","c4","c5"} as plain numpy arrays.

    Keys: cell[3] (bohr), grid[3], pos[n,3] (bohr), vel[n,3] (a.u.), Z[n], mass[n] (m_e),
    kT (Ha), dt (a.u.), n_steps, init_mode, and the common functional choices.
    """
    name = name.lower()
    num = int(name[1])
    rng = np.random.Generator(np.random.PCG64(SEED_BASE + num))
    a_fcc = (4 * AL_MASS_U * AMU_G / 2.7 * 1e24) ** (1.0 / 3.0) / BOHR_ANG   # 7.65117 bohr
    if num == 1:
        # 16 ions in the cubic 2.7 g/cc cell: the fcc sites of the four "even" (ix+iy+iz even)
        # conventional cells of a 2x2x2 replication with a = L/2 (reading R-C1).
        L = _cubic_L(16, 2.7)
        s = _fcc_sites((2, 2, 2), L / 2)
        keep = ((s[:, 3] + s[:, 4] + s[:, 5]) % 2) == 0
        pos = s[keep, :3] + rng.standard_normal((16, 3)) * 0.2
        cell = [L, L, L]; g = 32; T = 10.0; dt_fs = 0.5; steps = 5
    elif num == 2:
        pos = _fcc_sites((4, 4, 2), a_fcc)[:, :3]
        pos = pos + rng.standard_normal(pos.shape) * 0.3
        cell = [4 * a_fcc, 4 * a_fcc, 2 * a_fcc]; g = 64; T = 10.0; dt_fs = 0.5; steps = 100
    elif num == 3:
        L = _cubic_L(256, 10.0)
        pos = _random_positions(rng, 256, L, 1.0)
        cell = [L, L, L]; g = 128; T = 100.0; dt_fs = 0.1; steps = 200
    elif num == 4:
        pos = _fcc_sites((8, 8, 4), a_fcc)[:, :3]
        pos = pos + rng.standard_normal(pos.shape) * 0.3
        cell = [8 * a_fcc, 8 * a_fcc, 4 * a_fcc]; g = 192; T = 1.0; dt_fs = 1.0; steps = 50
    elif num == 5:
        L = _cubic_L(2000, 2.7)
        pos = _random_positions(rng, 2000, L, 0.0)
        cell = [L, L, L]; g = 384 if grid is None else grid; T = 50.0; dt_fs = 0.5; steps = 1
    else:
        raise ValueError(name)
    if grid is not None:
        g = grid
    n = pos.shape[0]
    cell = np.array(cell, dtype=np.float64)
    pos = np.mod(pos, cell)
    mass = np.full(n, AL_MASS_U * AMU_ME)
    kT = T / HARTREE_EV
    vel = _maxwell(rng, n, kT, mass)
    return dict(name=name, cell=cell, grid=np.array([g, g, g], dtype=np.int32),
                pos=np.ascontiguousarray(pos), vel=np.ascontiguousarray(vel),
                Z=np.full(n, AL_Z), mass=mass, kT=kT, T_eV=T, dt=dt_fs * FS_AU, n_steps=steps,
                xc=1, psp_rc=ASHCROFT_RC, init_mode=1, mix_mode=1)


def make_small(n_ions=4, L=8.0, grid=(12, 12, 12), T_eV=10.0, seed=7, cell=None, dmin=1.5) -> dict:
    """Small random test cell (used by pins and parity tests); grid sizes may be any 2^a 3^b."""
    rng = np.random.Generator(np.random.PCG64(SEED_BASE + 100 + seed))
    cell = np.array([L, L, L] if cell is None else cell, dtype=np.float64)
    pos = np.empty((n_ions, 3))
    k = 0
    while k < n_ions:
        p = rng.random(3) * cell
        d = pos[:k] - p
        d -= cell * np.rint(d / cell)
        if k and (np.einsum("ij,ij->i", d, d) < dmin * dmin).any():
            continue
        pos[k] = p; k += 1
    mass = np.full(n_ions, AL_MASS_U * AMU_ME)
    kT = T_eV / HARTREE_EV
    return dict(name=f"small{seed}", cell=cell, grid=np.array(grid, dtype=np.int32), pos=pos,
                vel=_maxwell(rng, n_ions, kT, mass), Z=np.full(n_ions, AL_Z), mass=mass, kT=kT,
                T_eV=T_eV, dt=0.5 * FS_AU, n_steps=3, xc=1, psp_rc=ASHCROFT_RC, init_mode=1,
                mix_mode=1)
