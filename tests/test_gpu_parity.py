"""GPU-vs-oracle parity through the C ABI (run on the B200 box: pytest -m gpu).

Tolerances (BASELINE.json north_star): relative 1e-10 on density and free energy, 1e-8 on forces.
Index/flag quantities (iteration counts under scf_fixed_iter) must be equal.
"""
import numpy as np
import pytest

import arche_inputs as ai

pytestmark = pytest.mark.gpu

TOL_N = 1e-10
TOL_F = 1e-10
TOL_FORCE = 1e-8


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU test run without a CUDA device")
    return torch


def _gpu(cfg, **kw):
    from paper_2606_13283_b200 import Arche
    return Arche(cfg, **kw)


def _rel(a, b):
    return float(np.abs(a - b).max() / np.abs(b).max())


TOL_STRESS = 1e-10


def _check_stress(sg, so):
    """every row of the 9 x 6 table and P, relative 1e-10 of the largest term entering (the total and the
    off-diagonal components are sums with cancellation)"""
    big = max(np.abs(so[k]).max() for k in so if k != "P")
    for k in so:
        if k == "P":
            assert abs(sg[k] - so[k]) < TOL_STRESS * big, (k, sg[k], so[k])
            continue
        scale = big if k == "total" else max(np.abs(so[k]).max(), 1e-300)
        assert np.abs(sg[k] - so[k]).max() <= TOL_STRESS * scale + 1e-16 * big, (k, sg[k], so[k])   # + round-off of rows that vanish


def test_fermi_dirac_parity(orc, torch_cuda):
    cfg = ai.make_small()
    g = _gpu(cfg)
    eta = np.concatenate([np.linspace(-60, 0, 301), np.linspace(0, 20, 801), np.linspace(20, 400, 401),
                          [-0.0, 1e-300, 19.999999999, 20.0, 20.000000001, 2.0, 4.0, 7.0, 10.0, 14.0]])
    for tj in (-1, 1, 3):
        got = g.fermi_dirac(tj, eta).cpu().numpy()
        ref = orc.fd(tj, eta)
        assert np.abs(got / ref - 1).max() < 2e-14, tj


@pytest.mark.parametrize("shape", [(4, 4, 4), (8, 12, 16), (24, 16, 36), (32, 32, 32), (48, 64, 96), (16, 18, 128)])
def test_fft3d_parity(orc, torch_cuda, shape):
    torch = torch_cuda
    nz, ny, nx = shape
    cfg = ai.make_small(grid=(nx, ny, nz))
    g = _gpu(cfg)
    rng = np.random.default_rng(nx + 7 * ny + 13 * nz)
    a = rng.standard_normal(shape) + 1j * rng.standard_normal(shape)
    for sign in (-1, +1):
        got = g.fft3d(torch.as_tensor(a), sign).cpu().numpy()
        ref = orc.fft3d(a, sign)
        assert np.abs(got - ref).max() < 1e-13 * np.abs(ref).max() * np.log2(a.size)


@pytest.mark.parametrize("shape", [(8, 12, 16), (9, 12, 18), (32, 64, 128), (64, 128, 32), (128, 32, 64), (32, 192, 256),
                                   (256, 32, 192), (16, 384, 32), (384, 16, 64), (32, 32, 384), (18, 64, 48), (9, 9, 16), (27, 9, 12)])
def test_real_fft_pair_parity(orc, torch_cuda, shape):
    """the r2c / c2r transform pair the SCF uses (register two-stage kernels on 32..384, generic radix kernels and
    mixed dispatch otherwise), against the oracle's full complex transform of the same real field"""
    torch = torch_cuda
    nz, ny, nx = shape
    cfg = ai.make_small(grid=(nx, ny, nz))
    g = _gpu(cfg)
    rng = np.random.default_rng(3 * nx + 7 * ny + 13 * nz)
    a = rng.standard_normal(shape)
    ref = orc.fft3d(a.astype(np.complex128), -1)
    got = g.rfft3d_forward(torch.as_tensor(a)).cpu().numpy()
    tol = 1e-13 * np.abs(ref).max() * np.log2(a.size)
    assert np.abs(got - ref).max() < tol
    back = g.rfft3d_inverse(torch.as_tensor(ref)).cpu().numpy()
    assert np.abs(back - a * a.size).max() < 1e-13 * a.size * np.abs(a).max() * np.log2(a.size)


def test_structure_factor_and_ionic_potential(orc, torch_cuda):
    cfg = ai.make_small(n_ions=7, L=9.0, grid=(24, 16, 12), cell=[9.0, 7.0, 6.0], seed=3)
    cfg["Z"] = np.array([3.0, 1.0, 2.0, 3.0, 1.5, 3.0, 0.5])
    g = _gpu(cfg); o = orc.Oracle(cfg)
    pos = cfg["pos"] + cfg["cell"] * np.array([2, -1, 0])          # unwrapped positions are legal
    g.scf_begin(pos); o.scf_begin(pos)
    for name in ("S_Z", "Vhat_ie"):
        assert _rel(g.get_complex(name).cpu().numpy(), o.get_complex(name)) < 1e-12


@pytest.mark.parametrize("feed", ["copy-engine", "global-loads"])
@pytest.mark.parametrize("grid,n_ions", [((128, 16, 8), 256), ((192, 8, 8), 256), ((256, 8, 12), 256), ((384, 12, 8), 256),
                                         ((384, 9, 6), 261)])
def test_structure_factor_register_tiled(orc, torch_cuda, monkeypatch, grid, n_ions, feed):
    """the register-tiled structure-factor kernels (2, 3 or 4 kx columns x 8 rows per thread, column kx = nx/2 left to
    the Nyquist-plane kernel) on long-x cells with 256 ions: S_Z, V_ie and the Ewald energy against the oracle.
    "copy-engine": structure_factor_tma_kernel (a_j rows by cp.async.bulk, every (columns, row groups) instantiation; the
    last case has an ion count that is no multiple of the stage and a row count that is no multiple of the block's rows);
    "global-loads": structure_factor_tiled_kernel (ARCHE_SF_TMA=0)."""
    if feed == "global-loads":
        monkeypatch.setenv("ARCHE_SF_TMA", "0")
    cfg = ai.make_small(n_ions=n_ions, grid=grid, cell=[40.0, 8.0, 8.0], seed=31, dmin=0.8)
    cfg["Z"] = np.full(n_ions, 0.25)                   # weak ions: a dense cell the oracle's quadrature handles quickly
    g = _gpu(cfg); o = orc.Oracle(cfg)
    g.scf_begin(cfg["pos"]); o.scf_begin(cfg["pos"])
    for name in ("S_Z", "Vhat_ie"):
        assert _rel(g.get_complex(name).cpu().numpy(), o.get_complex(name)) < 1e-11
    rg = g.scf_iter(); ro = o.scf_iter()
    assert abs(rg["U_ii"] - ro["U_ii"]) < 1e-10 * abs(ro["U_ii"])
    assert abs(rg["E_ie"] - ro["E_ie"]) < 1e-10 * abs(ro["E_ie"])


@pytest.fixture(params=["fused", "streamed"])
def pointwise_mode(request, monkeypatch):
    """both forms of the pointwise work: fused into the FFT passes (default on L2-resident grids) and streaming
    kernels around plain passes (default on large grids); ARCHE_FUSE is read by arche_scf_init"""
    monkeypatch.setenv("ARCHE_FUSE", "1" if request.param == "fused" else "0")
    return request.param


@pytest.mark.parametrize("xc", [0, 1, 2])
def test_single_scf_iteration(orc, torch_cuda, xc, pointwise_mode):
    cfg = ai.make_small(n_ions=4, L=8.0, grid=(16, 12, 24), T_eV=10.0, seed=8)
    g = _gpu(cfg, xc=xc); o = orc.Oracle(cfg, xc=xc)
    assert g.is_fused() == (pointwise_mode == "fused")
    g.scf_begin(cfg["pos"]); o.scf_begin(cfg["pos"])
    for it in range(3):
        rg = g.scf_iter(); ro = o.scf_iter()
        assert _rel(g.get_real("V_i").cpu().numpy(), o.get_real("V_i")) < 1e-11
        assert _rel(g.get_real("n_a").cpu().numpy(), o.get_real("n_a")) < TOL_N
        assert _rel(g.get_real("n_i").cpu().numpy(), o.get_real("n_i")) < TOL_N
        assert _rel(g.get_complex("nhat_a").cpu().numpy(), o.get_complex("nhat_a")) < TOL_N
        for k in ("mu", "F_total", "F0", "E_H", "E_xc", "E_ie", "E_ie0", "U_ii", "K_e", "w_last"):
            assert abs(rg[k] - ro[k]) <= TOL_F * max(1.0, abs(ro[k])), (it, k, rg[k], ro[k])
        assert abs(rg["U_mix"] / ro["U_mix"] - 1) < 1e-9 and abs(rg["K_mix"] / ro["K_mix"] - 1) < 1e-9
        assert rg["scf_iters"] == ro["scf_iters"] == it + 1
    dV = float(np.prod(cfg["cell"]) / np.prod(cfg["grid"]))
    assert abs(g.get_real("n_a").sum().item() * dV - cfg["Z"].sum()) < 1e-12 * cfg["Z"].sum()   # neutrality


@pytest.mark.parametrize("T_eV", [1.0, 100.0])
def test_temperature_extremes(orc, torch_cuda, T_eV):
    """degenerate (T = 1 eV: eta up to several hundred, asymptotic Fermi-Dirac region, vanishing density in the
    classically forbidden cores) and hot dilute (T = 100 eV: eta << 0) plasmas, three iterations field by field"""
    cfg = ai.make_small(n_ions=4, L=8.0, grid=(16, 16, 16), T_eV=T_eV, seed=21)
    g = _gpu(cfg); o = orc.Oracle(cfg)
    g.scf_begin(cfg["pos"]); o.scf_begin(cfg["pos"])
    for it in range(3):
        rg = g.scf_iter(); ro = o.scf_iter()
        assert _rel(g.get_real("V_i").cpu().numpy(), o.get_real("V_i")) < 1e-11
        assert _rel(g.get_real("n_a").cpu().numpy(), o.get_real("n_a")) < TOL_N
        for k in ("mu", "F_total", "F0", "E_H", "E_xc", "E_ie", "K_e", "w_last"):
            assert abs(rg[k] - ro[k]) <= TOL_F * max(1.0, abs(ro[k])), (T_eV, it, k, rg[k], ro[k])


def _solve_pair(orc, cfg, **kw):
    o = orc.Oracle(cfg, **kw)
    ro = o.scf_solve(cfg["pos"])
    assert ro["converged"] == 1
    g = _gpu(cfg, scf_fixed_iter=ro["scf_iters"], **kw)      # replay the same number of iterations (reading D4)
    rg = g.scf_solve(cfg["pos"])
    return g, o, rg, ro


@pytest.mark.parametrize("name,iters", [("c2", 3), ("c3", 2)])
def test_full_size_configs_iterations_and_forces(orc, torch_cuda, name, iters):
    """BASELINE.json configs[1] (128 ions, 64^3: fused passes, register FFT kernels) and configs[2] (256 ions, 128^3:
    streamed pointwise kernels) at their full sizes and in the launch configuration bench.py times: a few SCF
    iterations from the uniform start, every field and scalar against the oracle, then the forces on that density."""
    cfg = ai.make_config(name)
    kw = dict(mix_warmup=3, mix_w_fixed=0.95)
    g = _gpu(cfg, **kw); o = orc.Oracle(cfg, **kw)
    assert g.is_fused() == (name == "c2")
    g.scf_begin(cfg["pos"]); o.scf_begin(cfg["pos"])
    for name_c in ("S_Z", "Vhat_ie"):
        assert _rel(g.get_complex(name_c).cpu().numpy(), o.get_complex(name_c)) < 1e-11
    for it in range(iters):
        rg = g.scf_iter(); ro = o.scf_iter()
        for k in ("mu", "F_total", "F0", "E_H", "E_xc", "E_ie", "U_ii", "K_e", "w_last"):
            assert abs(rg[k] - ro[k]) <= TOL_F * max(1.0, abs(ro[k])), (it, k, rg[k], ro[k])
    assert _rel(g.get_real("n_a").cpu().numpy(), o.get_real("n_a")) < TOL_N
    assert _rel(g.get_real("n_i").cpu().numpy(), o.get_real("n_i")) < TOL_N
    assert _rel(g.get_complex("nhat_a").cpu().numpy(), o.get_complex("nhat_a")) < TOL_N
    Fg = g.forces().cpu().numpy(); Fo = o.forces()
    assert np.abs(Fg - Fo).max() < TOL_FORCE * np.abs(Fo).max()
    import torch
    _check_stress(g.stress(torch.as_tensor(cfg["vel"], device="cuda")), o.stress(cfg["vel"]))
    dV = float(np.prod(cfg["cell"]) / np.prod(cfg["grid"]))
    assert abs(g.get_real("n_a").sum().item() * dV - cfg["Z"].sum()) < 1e-12 * cfg["Z"].sum()


def test_c2_solve_in_one_cooperative_launch(orc, torch_cuda, monkeypatch):
    """configs[1] through arche_scf_solve: on 32^3 / 64^3 grids the whole solve runs in one persistent cooperative
    kernel (scf_persistent.cuh).  Ten iterations replayed against the oracle, and against the per-pass form."""
    cfg = ai.make_config("c2")
    kw = dict(mix_warmup=3, mix_w_fixed=0.95, scf_fixed_iter=10)
    o = orc.Oracle(cfg, **kw); ro = o.scf_solve(cfg["pos"])
    g = _gpu(cfg, **kw)
    l0 = g.launch_count(); rg = g.scf_solve(cfg["pos"]); launches = g.launch_count() - l0
    assert launches < 20, launches                       # per-MD-step kernels + ONE launch for the ten iterations
    assert rg["scf_iters"] == ro["scf_iters"] == 10
    na = g.get_real("n_a").cpu().numpy()
    assert _rel(na, o.get_real("n_a")) < TOL_N
    assert _rel(g.get_real("n_i").cpu().numpy(), o.get_real("n_i")) < TOL_N
    for k in ("mu", "F_total", "F0", "E_H", "E_xc", "E_ie", "K_e", "w_last"):
        assert abs(rg[k] - ro[k]) <= TOL_F * max(1.0, abs(ro[k])), (k, rg[k], ro[k])
    Fg = g.forces().cpu().numpy(); Fo = o.forces()
    assert np.abs(Fg - Fo).max() < TOL_FORCE * np.abs(Fo).max()
    monkeypatch.setenv("ARCHE_PERSIST", "0")
    g2 = _gpu(cfg, **kw)
    l0 = g2.launch_count(); r2 = g2.scf_solve(cfg["pos"])
    assert g2.launch_count() - l0 > 70                   # 7 launches per iteration
    assert _rel(g2.get_real("n_a").cpu().numpy(), na) < 1e-13 and abs(r2["F_total"] - rg["F_total"]) < 1e-12 * abs(rg["F_total"])


def test_converged_solve_and_forces(orc, torch_cuda, pointwise_mode):
    cfg = ai.make_small(n_ions=5, L=9.0, grid=(24, 16, 18), cell=[9.0, 7.5, 8.0], T_eV=10.0, seed=9)
    g, o, rg, ro = _solve_pair(orc, cfg, scf_tol_dn=1e-11, init_mode=0)
    assert rg["scf_iters"] == ro["scf_iters"]
    assert _rel(g.get_real("n_a").cpu().numpy(), o.get_real("n_a")) < TOL_N
    assert abs(rg["F_total"] - ro["F_total"]) < TOL_F * abs(ro["F_total"])
    Fg = g.forces().cpu().numpy(); Fo = o.forces()
    assert np.abs(Fg - Fo).max() < TOL_FORCE * np.abs(Fo).max()
    # the GPU's own stop rule ends at the same iteration
    g2 = _gpu(cfg, scf_tol_dn=1e-11, init_mode=0)
    r2 = g2.scf_solve(cfg["pos"])
    assert r2["converged"] == 1 and abs(r2["scf_iters"] - ro["scf_iters"]) <= 1
    assert _rel(g.get_complex("ghat").cpu().numpy(), o.get_complex("ghat")) < 1e-8


@pytest.mark.parametrize("grid,cell,xc", [((24, 16, 18), [9.0, 7.5, 8.0], 1), ((12, 8, 9), [7.0, 7.6, 8.3], 1),
                                          ((9, 27, 16), [6.5, 9.0, 8.0], 0), ((32, 32, 32), [9.0, 9.5, 10.0], 1)])
def test_stress_tensor_and_pressure(orc, torch_cuda, grid, cell, xc):
    """f1: all nine rows x six components + P against the oracle on a converged density; anisotropic
    cells so that every off-diagonal component is non-zero; even sizes (Nyquist planes on every axis, where the half
    spectrum needs S2 and the sign flips), odd sizes, mixed; with and without velocities."""
    torch = torch_cuda
    cfg = ai.make_small(n_ions=5, grid=grid, cell=cell, T_eV=10.0, seed=11, dmin=2.0)
    cfg["xc"] = xc
    g, o, rg, ro = _solve_pair(orc, cfg, scf_tol_dn=1e-10, init_mode=0)
    so = o.stress(cfg["vel"])
    sg = g.stress(torch.as_tensor(cfg["vel"], device="cuda"))
    _check_stress(sg, so)
    for row in ("pp", "pm", "ee", "ie", "i"):
        assert np.abs(so[row][3:]).min() > 0          # the shear components are exercised
    _check_stress(g.stress(), o.stress())
    assert abs(sg["P"] + sg["total"][:3].sum() / 3) < 1e-15


def test_stress_edge_cases(orc, torch_cuda):
    from paper_2606_13283_b200 import ArcheError
    cfg = dict(cell=[5.0, 6.0, 7.0], grid=[8, 12, 16], Z=np.zeros(0), mass=np.zeros(0), kT=0.4)
    g = _gpu(cfg, n_electrons=9.0); o = orc.Oracle(cfg, n_electrons=9.0)
    with pytest.raises(ArcheError):
        g.stress()                                                  # before any solve
    rg = g.scf_solve(np.zeros((0, 3))); ro = o.scf_solve(np.zeros((0, 3)))
    sg, so = g.stress(), o.stress()                                 # uniform gas: only sigma^e and sigma^xc
    _check_stress(sg, so)
    assert abs(sg["P"] - (2 * rg["K_e"] / (3 * 210.0) - sg["xc"][0])) < 1e-15
    for row in ("i", "pp", "pm", "je", "ie"):
        assert np.all(sg[row] == 0), row


def test_c1_md_trajectory(orc, torch_cuda):
    """BASELINE.json config 1: 16 Al ions, 32^3, T = 10 eV, 5 velocity-Verlet steps of 0.5 fs."""
    torch = torch_cuda
    cfg = ai.make_config("c1")
    kw = dict(scf_tol_F=1e-10, scf_tol_dn=1e-9, scf_max_iter=300)
    o = orc.Oracle(cfg, **kw)
    g = _gpu(cfg, **kw)
    po = cfg["pos"].copy(); vo = cfg["vel"].copy()
    pg = torch.as_tensor(cfg["pos"].copy(), device="cuda"); vg = torch.as_tensor(cfg["vel"].copy(), device="cuda")
    for step in range(cfg["n_steps"]):
        ro = o.md_step(cfg["dt"], po, vo)
        rg = g.md_step(cfg["dt"], pg, vg)
        assert abs(rg["scf_iters"] - ro["scf_iters"]) <= 1, step
        assert abs(rg["F_total"] - ro["F_total"]) < 1e-9 * abs(ro["F_total"])
        assert abs(rg["K_i"] - ro["K_i"]) < 1e-9 * abs(ro["K_i"])
        assert np.abs(pg.cpu().numpy() - po).max() < 1e-9
        Fo = o.forces(); Fg = g.forces().cpu().numpy()
        assert np.abs(Fg - Fo).max() < 1e-6 * np.abs(Fo).max()    # free stop rule: residual-limited, not round-off
    # host-buffer variant gives the same step as the device-pointer one
    g2 = _gpu(cfg, **kw)
    ph = cfg["pos"].copy(); vh = cfg["vel"].copy(); Fh = np.zeros_like(ph)
    g3 = _gpu(cfg, **kw)
    pd = torch.as_tensor(cfg["pos"].copy(), device="cuda"); vd = torch.as_tensor(cfg["vel"].copy(), device="cuda")
    g2.md_step_host(cfg["dt"], ph, vh, Fh); g3.md_step(cfg["dt"], pd, vd)
    assert np.array_equal(ph, pd.cpu().numpy()) and np.array_equal(Fh, g3.forces().cpu().numpy())


def test_uniform_gas_and_edge_cases(orc, torch_cuda):
    from paper_2606_13283_b200 import ArcheError
    cfg = dict(cell=[5.0, 6.0, 7.0], grid=[8, 12, 16], Z=np.zeros(0), mass=np.zeros(0), kT=0.4)
    g = _gpu(cfg, n_electrons=9.0); o = orc.Oracle(cfg, n_electrons=9.0)
    g.scf_begin(np.zeros((0, 3))); o.scf_begin(np.zeros((0, 3)))
    rg = g.scf_iter(); ro = o.scf_iter()
    assert abs(rg["mu"] - ro["mu"]) < 1e-12 and abs(rg["F_total"] - ro["F_total"]) < 1e-11
    assert np.abs(g.get_real("n_a").cpu().numpy() - 9.0 / 210.0).max() < 1e-15
    with pytest.raises(ArcheError):
        _gpu(dict(cfg, grid=[7, 12, 16]), n_electrons=9.0)        # 7 is not 2^a 3^b
    c2 = ai.make_small()
    g2 = _gpu(c2)
    with pytest.raises(ArcheError):
        g2.forces()                                                 # before any solve


def test_c5_large_grid_streamed_form_properties_and_sampled_oracle(orc, torch_cuda):
    """BASELINE.json configs[4] (2000 ions, T = 50 eV) at 192^3: fields beyond the L2, streamed pointwise kernels, the
    register-tiled structure-factor kernel -- the launch configuration bench.py --workload c5 times.  The oracle cannot
    do this size in seconds, so: (a) S_Z(k) and Vhat_ie(k) depend on the integer wave vector m and the ions only, not
    on the grid, hence the oracle on an 8^3 grid of the same cell gives their values at all |m_i| <= 3 (343 sampled
    outputs, away from any Nyquist plane); (b) properties that hold at any size after two SCF iterations: charge
    neutrality, nhat_a(0) = N_e, Parseval between n_a and nhat_a, n_a > 0."""
    torch = torch_cuda
    cfg = ai.make_config("c5", grid=192)
    g = _gpu(cfg)
    assert not g.is_fused()
    g.scf_begin(cfg["pos"])
    small = dict(cfg); small["grid"] = np.array([8, 8, 8])
    o = orc.Oracle(small)
    o.scf_begin(cfg["pos"])
    m = np.arange(-3, 4)
    for name in ("S_Z", "Vhat_ie"):
        big = g.get_complex(name).cpu().numpy(); ref = o.get_complex(name)
        sub_g = big[np.ix_(m % 192, m % 192, m % 192)]; sub_o = ref[np.ix_(m % 8, m % 8, m % 8)]
        assert _rel(sub_g, sub_o) < 1e-11, name
        del big
    Ne = float(cfg["Z"].sum()); vol = float(np.prod(cfg["cell"])); dV = vol / 192 ** 3
    for _ in range(2):
        r = g.scf_iter()
    n_a = g.get_real("n_a")
    assert float(n_a.min()) > 0.0
    assert abs(float(n_a.sum()) * dV - Ne) < 1e-12 * Ne
    nh = g.get_complex("nhat_a")
    assert abs(complex(nh[0, 0, 0]) - Ne) < 1e-12 * Ne
    lhs = float((n_a * n_a).sum()) * dV; rhs = float((nh.real ** 2 + nh.imag ** 2).sum()) / vol
    assert abs(lhs - rhs) < 1e-12 * lhs
    assert np.isfinite(r["mu"]) and np.isfinite(r["F_total"])


def test_determinism(orc, torch_cuda):
    cfg = ai.make_small(n_ions=4, L=8.0, grid=(16, 16, 16), seed=12)
    r = []
    for _ in range(2):
        g = _gpu(cfg, scf_fixed_iter=6)
        res = g.scf_solve(cfg["pos"])
        r.append((res["F_total"], res["mu"], g.get_real("n_a").cpu().numpy(), g.forces().cpu().numpy()))
    assert r[0][0] == r[1][0] and r[0][1] == r[1][1]
    assert np.array_equal(r[0][2], r[1][2]) and np.array_equal(r[0][3], r[1][3])


def test_tabulated_pseudopotential(orc, torch_cuda):
    """f2: the average-atom norm-conserving pseudopotential as a form-factor table (arche_params.psp = 1).
    Dense hydrogen (4 protons, r_ws = 1.5 bohr, kT = 2 Ha, 16^3), table from the oracle-side generator (test data, like
    the positions): V_ie, three iterations field by field, forces, the stress table; and the Ashcroft potential fed as
    a table must reproduce psp = 0 on the device as well."""
    torch = torch_cuda
    Z, rws, kT, n = 1.0, 1.5, 2.0, 401
    r, dens, mu, _ = orc.aa_solve(Z, rws, kT, 0, n)
    ic = int(round((n - 1) * np.sqrt(0.5)))
    ps, _ = orc.aa_pseudize(r, dens, ic)
    V = orc.aa_invert(kT, 0, r, ps, 0.0, mu)
    dVr = np.zeros(n); dVr[1:] = V[1:] + Z / r[1:]
    dk = 0.02
    table = orc.radial_ft(r, dVr, ic, dk * np.arange(int(4.0 / dk) + 3)) / Z
    L = (4 * 4.0 / 3.0 * np.pi * rws ** 3) ** (1.0 / 3.0)
    cfg = ai.make_small(n_ions=4, cell=[L, L * 1.1, L / 1.1], grid=(16, 12, 18), seed=17, dmin=1.2)
    cfg["Z"] = np.full(4, Z); cfg["kT"] = kT; cfg["xc"] = 0
    kw = dict(psp_table=table, psp_dk=dk)
    g = _gpu(cfg, **kw); o = orc.Oracle(cfg, **kw)
    g.scf_begin(cfg["pos"]); o.scf_begin(cfg["pos"])
    assert _rel(g.get_complex("Vhat_ie").cpu().numpy(), o.get_complex("Vhat_ie")) < 1e-12
    for it in range(3):
        rg = g.scf_iter(); ro = o.scf_iter()
        assert _rel(g.get_real("n_a").cpu().numpy(), o.get_real("n_a")) < TOL_N
        for k in ("mu", "F_total", "E_ie", "E_ie0", "E_H", "U_ii", "w_last"):
            assert abs(rg[k] - ro[k]) <= TOL_F * max(1.0, abs(ro[k])), (it, k, rg[k], ro[k])
    Fg = g.forces().cpu().numpy(); Fo = o.forces()
    assert np.abs(Fg - Fo).max() < TOL_FORCE * np.abs(Fo).max()
    _check_stress(g.stress(torch.as_tensor(cfg["vel"], device="cuda")), o.stress(cfg["vel"]))
    # Ashcroft as a table against the built-in Ashcroft path, both on the device
    c2 = ai.make_small(n_ions=3, cell=[7.0, 7.6, 8.3], grid=(12, 12, 12), T_eV=10.0, seed=5, dmin=2.5)
    kk = 0.002 * np.arange(int(1.6 / 0.002) + 4)
    du = np.empty_like(kk); du[1:] = (1 - np.cos(2 * np.pi * kk[1:] * 1.12)) / (np.pi * kk[1:] ** 2); du[0] = 2 * np.pi * 1.12 ** 2
    ga = _gpu(c2, scf_fixed_iter=12); gt = _gpu(c2, scf_fixed_iter=12, psp_table=du, psp_dk=0.002)
    ra = ga.scf_solve(c2["pos"]); rt = gt.scf_solve(c2["pos"])
    assert abs(rt["F_total"] - ra["F_total"]) < 1e-8 * abs(ra["F_total"]) and abs(rt["E_ie0"] / ra["E_ie0"] - 1) < 1e-14
    assert np.abs((gt.forces() - ga.forces()).cpu().numpy()).max() < 1e-7 * float(ga.forces().abs().max())
    from paper_2606_13283_b200 import ArcheError
    with pytest.raises(ArcheError):
        _gpu(c2, psp_table=du[:100], psp_dk=0.002)                  # the table does not cover the grid's largest |k|
