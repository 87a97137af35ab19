"""Pins for oracle O7 (Shu-Osher SSP-RK3; north_star 'Runge-Kutta stage update')."""
import numpy as np

from paper_1804_09101_b200 import configs, inputs


def gauge_wave_state(oracle, sd, t):
    xyz = oracle.coords(sd)
    psi, Pi, Phi, *_ = inputs.gauge_wave(xyz, t)
    return inputs.pack_fields(psi, Pi, Phi)


def test_third_order_on_gauge_wave(oracle):
    """Harmonic gauge wave (O(1) time dependence, H_a = 0) on a 12^3 block to T = 0.02 with dt = T/n,
    n = 1,2,4,8.  The spatial truncation error (~1.6e-5 at N=12) is common to all runs, so the order of
    the time integrator is read from successive differences: |u_n - u_2n| falls ~8x per halving
    (order 3); against the ANALYTIC solution every run is within the spatial error."""
    sd = configs.block(12, (-1.0, -1.0, -1.0), (1.0, 1.0, 1.0), gamma=(1.0, -1.0, 1.0))
    P = oracle.num_points(sd)
    H = np.zeros((4, P))
    dH = np.zeros((12, P))
    T = 0.02
    u0 = gauge_wave_state(oracle, sd, 0.0)
    exact = gauge_wave_state(oracle, sd, T)
    us = [oracle.rk3(sd, u0, H, T / n, n, dH=dH) for n in (1, 2, 4, 8)]
    d = [np.abs(us[i] - us[i + 1]).max() for i in range(3)]
    assert d[0] > 1e-7
    assert 6.0 < d[0] / d[1] < 9.5 and 6.0 < d[1] / d[2] < 9.5
    assert all(np.abs(u - exact).max() < 5e-5 for u in us)
    assert np.abs(u0 - exact).max() > 1e-3           # the solution really moved


def test_one_step_equals_three_rhs_calls(oracle):
    """The step is exactly the Shu-Osher combination of three O5 evaluations (composition pin)."""
    cfg = configs.c1()
    sd = cfg["descs"][0]
    xyz = oracle.coords(sd)
    (u0,), (H,) = inputs.initial_data([sd], [xyz], cfg["spin"], cfg["amplitude"], cfg["id"])
    dt = 0.01
    u1 = u0 + dt * oracle.rhs(sd, u0, H)
    u2 = 0.75 * u0 + 0.25 * (u1 + dt * oracle.rhs(sd, u1, H))
    u3 = u0 / 3 + (2.0 / 3.0) * (u2 + dt * oracle.rhs(sd, u2, H))
    un = oracle.rk3(sd, u0, H, dt, 1)
    assert np.abs(un - u3).max() < 1e-15
    # FROZEN outer face: those points never move
    P = xyz.shape[1]
    outer = np.arange(P).reshape(8, -1)[-1]
    assert np.array_equal(un[:, outer], u0[:, outer])


def test_stationary_ks_stays_put(oracle):
    """Stationary Kerr-Schild on the C1 shell: 20 steps move the state by no more than dt*steps*|RHS| ~ truncation."""
    sd = configs.shell(12, 6, 1.8, 5.0, face=(0, 1))
    xyz = oracle.coords(sd)
    u0 = inputs.pack_fields(*inputs.kerr_schild(xyz, 1.0, 0.0))
    H = inputs.kerr_schild_gauge_source(xyz, 1.0, 0.0)
    k0 = np.abs(oracle.rhs(sd, u0, H)).max()
    dt = 0.25 * configs.min_spacing([sd])
    u = oracle.rk3(sd, u0, H, dt, 20)
    assert np.abs(u - u0).max() < 3 * 20 * dt * k0


def test_dH_null_uses_spectral_gradient(oracle):
    sd = configs.block(8, (3.0, -1.0, -1.0), (5.0, 1.0, 1.0))
    xyz = oracle.coords(sd)
    u = inputs.pack_fields(*inputs.kerr_schild(xyz, 1.0, 0.4))
    H = inputs.kerr_schild_gauge_source(xyz, 1.0, 0.4)
    g = oracle.gradient(sd, H)                       # [3,4,P] -> dH[i*4+a]
    a = oracle.rhs(sd, u, H)
    b = oracle.rhs(sd, u, H, dH=g.reshape(12, -1))
    assert np.abs(a - b).max() < 1e-15
