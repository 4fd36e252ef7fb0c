"""Pins of the oracle's isokinetic integrator (ref. [48]; reading A23).

The oracle's closed-form constant-force flow is checked against what the Gaussian isokinetic equations of motion
m dv/dt = F - alpha m v, alpha = sum F.v / sum m v^2 fix by themselves: conservation of K, the group property of an
exact flow, a numerical integration of the ODE written out here, and the textbook one-particle solution."""
import numpy as np
import pytest

import arche_inputs as ai
import oracle


def _case(n, seed):
    rng = np.random.default_rng(seed)
    m = rng.uniform(1.0e3, 5.0e4, n)
    v = rng.normal(0, 1e-3, (n, 3))
    F = rng.normal(0, 2e-2, (n, 3))
    return m, v, F


def _K(m, v):
    return 0.5 * float(np.sum(m[:, None] * v * v))


@pytest.mark.parametrize("n,t", [(1, 40.0), (2, 7.5), (7, 20.0), (64, 300.0)])
def test_kinetic_energy_is_conserved(n, t):
    m, v, F = _case(n, 11 + n)
    v1 = oracle.isokinetic_kick(m, F, t, v)
    assert abs(_K(m, v1) - _K(m, v)) < 1e-14 * _K(m, v)
    assert np.abs(v1 - v).max() > 1e-3 * np.abs(v).max()          # the map is not the identity


def test_flow_has_the_group_property():
    m, v, F = _case(9, 3)
    t1, t2 = 13.0, 29.0
    a = oracle.isokinetic_kick(m, F, t1 + t2, v)
    b = oracle.isokinetic_kick(m, F, t2, oracle.isokinetic_kick(m, F, t1, v))
    assert np.abs(a - b).max() < 1e-13 * np.abs(a).max()
    back = oracle.isokinetic_kick(m, F, -(t1 + t2), a)              # and the inverse element
    assert np.abs(back - v).max() < 1e-13 * np.abs(v).max()


def test_against_runge_kutta_of_the_equations_of_motion():
    m, v0, F = _case(5, 21)
    t = 50.0

    def rhs(v):
        alpha = np.sum(F * v) / np.sum(m[:, None] * v * v)
        return F / m[:, None] - alpha * v

    nstep = 4000
    h = t / nstep
    v = v0.copy()
    for _ in range(nstep):
        k1 = rhs(v); k2 = rhs(v + 0.5 * h * k1); k3 = rhs(v + 0.5 * h * k2); k4 = rhs(v + h * k3)
        v = v + (h / 6.0) * (k1 + 2 * k2 + 2 * k3 + k4)
    v1 = oracle.isokinetic_kick(m, F, t, v0)
    assert np.abs(v1 - v).max() < 1e-10 * np.abs(v).max()


def test_one_particle_turns_towards_the_force():
    # one particle, speed u, constant force f at angle theta to v: tan(theta(t)/2) = tan(theta_0/2) exp(-f t/(m u))
    m = np.array([2.0e4]); u = 2.0e-3; f = 0.05
    for th0 in (0.5 * np.pi, 2.0, 0.3):
        v0 = np.array([[u * np.cos(th0), u * np.sin(th0), 0.0]])
        F = np.array([[f, 0.0, 0.0]])
        for t in (100.0, 1000.0, 4000.0):
            v1 = oracle.isokinetic_kick(m, F, t, v0)[0]
            th = np.arctan2(v1[1], v1[0])
            assert abs(np.tan(th / 2) - np.tan(th0 / 2) * np.exp(-f * t / (m[0] * u))) < 1e-12
            assert abs(np.hypot(v1[0], v1[1]) - u) < 1e-15 and v1[2] == 0.0


def test_first_order_in_t_is_the_constrained_acceleration():
    m, v, F = _case(6, 5)
    alpha = np.sum(F * v) / np.sum(m[:, None] * v * v)
    acc = F / m[:, None] - alpha * v
    errs = []
    for t in (1.0, 0.5, 0.25):
        errs.append(np.abs(oracle.isokinetic_kick(m, F, t, v) - (v + t * acc)).max())
    assert errs[0] / errs[1] == pytest.approx(4.0, rel=0.05) and errs[1] / errs[2] == pytest.approx(4.0, rel=0.05)


def test_md_step_conserves_K_and_is_time_reversible():
    cfg = ai.make_small(n_ions=4, L=8.0, grid=(12, 12, 12), T_eV=10.0, seed=31)
    kw = dict(scf_tol_dn=1e-11, scf_max_iter=400, ensemble=1)
    o = oracle.Oracle(cfg, **kw)
    pos = cfg["pos"].copy(); vel = cfg["vel"].copy()
    K0 = _K(cfg["mass"], vel)
    for _ in range(3):
        r = o.md_step(cfg["dt"], pos, vel)
        assert abs(r["K_i"] - K0) < 1e-13 * K0
    assert np.abs(pos - cfg["pos"]).max() > 1e-3
    o2 = oracle.Oracle(cfg, **kw)                                   # fresh context: forces at the turning point
    vel *= -1.0
    for _ in range(3):
        o2.md_step(cfg["dt"], pos, vel)
    assert np.abs(pos - cfg["pos"]).max() < 1e-7                    # limited by the SCF tolerance of the forces
    assert np.abs(vel + cfg["vel"]).max() < 1e-7 * np.abs(cfg["vel"]).max() + 1e-11


def test_reduces_to_velocity_verlet_to_second_order():
    cfg = ai.make_small(n_ions=3, L=7.0, grid=(12, 12, 12), T_eV=10.0, seed=32)
    d = []
    for dt in (cfg["dt"], 0.5 * cfg["dt"]):
        out = []
        for ens in (0, 1):
            o = oracle.Oracle(cfg, scf_tol_dn=1e-11, scf_max_iter=400, ensemble=ens)
            pos = cfg["pos"].copy(); vel = cfg["vel"].copy()
            o.md_step(dt, pos, vel)
            out.append(pos)
        d.append(np.abs(out[0] - out[1]).max())
    # positions after one step differ by the constraint term alpha v dt^2/2
    assert d[0] > 0 and d[0] / d[1] == pytest.approx(4.0, rel=0.1)
