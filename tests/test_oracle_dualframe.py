"""Pins for oracle O14, the dual-frame right-hand side (NEXT-4): fields at fixed GRID points, equations in inertial
coordinates:  d_t u|_xbar = F[u, Jm dbar u] + v^i (Jm dbar u)_i  with Jm_i^k = d xbar^k / d x^i and v the grid velocity."""
import numpy as np
import pytest

from paper_1804_09101_b200 import configs, inputs
from test_oracle_rhs import GAMMAS, cstep, random_point


def test_identity_map_is_the_single_frame_rhs(oracle):
    psi, Pi, Phi, dpsi, dPi, dPhi, H, dH = random_point(3)
    a = oracle.rhs_point(psi, Pi, Phi, dpsi, dPi, dPhi, H, dH, (1.0, -1.0, 1.0))
    b = oracle.rhs_point_map(psi, Pi, Phi, dpsi, dPi, dPhi, H, dH, (1.0, -1.0, 1.0), np.eye(3), np.zeros(3))
    for x, y in zip(a, b):
        assert np.array_equal(x, y)


def test_gauge_wave_is_stationary_in_the_comoving_grid(oracle):
    """The harmonic gauge wave H(x - t) moves along +x at speed 1.  On a grid that moves with it (x = xbar + t: Jm = 1, v = (1,0,0))
    every field is constant at the grid points: the dual-frame RHS vanishes although the single-frame one is O(1)."""
    pts = np.array([[0.13, -0.4, 0.2], [-0.77, 0.1, 0.9], [0.5, 0.5, -0.5]]).T
    t = 0.3
    psi, Pi, Phi, dtpsi, dtPi, dtPhi = inputs.gauge_wave(pts, t)
    dPi = cstep(lambda z: inputs.gauge_wave(z, t)[1], pts)
    dPhi = cstep(lambda z: inputs.gauge_wave(z, t)[2], pts)
    assert np.abs(dtPi).max() > 0.05
    for gam in GAMMAS:
        for p in range(pts.shape[1]):
            o = oracle.rhs_point_map(psi[..., p], Pi[..., p], Phi[..., p], Phi[..., p], dPi[..., p], dPhi[..., p], np.zeros(4), np.zeros((3, 4)),
                                     gam, np.eye(3), np.array([1.0, 0.0, 0.0]))
            for x in o:
                assert np.abs(x).max() < 1e-14
            # moving the other way doubles the time derivative instead: the sign of the advection term is pinned
            o = oracle.rhs_point_map(psi[..., p], Pi[..., p], Phi[..., p], Phi[..., p], dPi[..., p], dPhi[..., p], np.zeros(4), np.zeros((3, 4)),
                                     gam, np.eye(3), np.array([-1.0, 0.0, 0.0]))
            assert np.abs(o[1] - 2 * dtPi[..., p]).max() < 1e-14


def test_stretched_grid_recovers_the_inertial_derivative(oracle):
    """x = a xbar (a static stretch): grid-frame derivatives are a times the inertial ones, Jm = 1/a undoes it (a and 1/a swapped fails):
    the gauge wave's analytic time derivatives come back."""
    pts = np.array([[0.2, 0.1, -0.3], [-0.6, 0.4, 0.7]]).T
    t, a = 0.1, 1.7
    psi, Pi, Phi, dtpsi, dtPi, dtPhi = inputs.gauge_wave(pts, t)
    dPi = cstep(lambda z: inputs.gauge_wave(z, t)[1], pts)
    dPhi = cstep(lambda z: inputs.gauge_wave(z, t)[2], pts)
    for p in range(pts.shape[1]):
        o = oracle.rhs_point_map(psi[..., p], Pi[..., p], Phi[..., p], a * Phi[..., p], a * dPi[..., p], a * dPhi[..., p], np.zeros(4),
                                 np.zeros((3, 4)), (1.0, -1.0, 1.0), np.eye(3) / a, np.zeros(3))
        assert np.abs(o[1] - dtPi[..., p]).max() < 1e-14 and np.abs(o[2] - dtPhi[..., p]).max() < 1e-14
        bad = oracle.rhs_point_map(psi[..., p], Pi[..., p], Phi[..., p], a * Phi[..., p], a * dPi[..., p], a * dPhi[..., p], np.zeros(4),
                                   np.zeros((3, 4)), (1.0, -1.0, 1.0), np.eye(3) * a, np.zeros(3))
        assert np.abs(bad[1] - dtPi[..., p]).max() > 1e-2


def test_kerr_schild_in_a_rotating_grid(oracle):
    """Stationary Kerr-Schild data (spin along z) seen from a grid rotating rigidly about z: the inertial-frame RHS vanishes, so the
    time derivative at a grid point is the field sampled along its circle, d/dt u(R_z(Omega t) xbar) = Omega d/dalpha u(R_z(alpha) x)
    at alpha = 0 (complex step in alpha) - with v = Omega z^ x x and analytic derivatives, to rounding."""
    a, Om = 0.6, 0.37
    pts = np.array([[2.0, 0.3, -1.1], [-3.0, 2.5, 0.7], [0.4, -2.2, 2.9]]).T
    psi, Pi, Phi = inputs.kerr_schild(pts, 1.0, a)
    dPi = cstep(lambda z: inputs.kerr_schild(z, 1.0, a)[1], pts)
    dPhi = cstep(lambda z: inputs.kerr_schild(z, 1.0, a)[2], pts)
    H = inputs.kerr_schild_gauge_source(pts, 1.0, a)
    dH = cstep(lambda z: inputs.kerr_schild_gauge_source(z, 1.0, a), pts)

    def along_circle(k):       # d/dalpha of field k at alpha = 0, complex step
        h = 1e-30
        al = 1j * h
        R = np.array([[np.cos(al), -np.sin(al), 0], [np.sin(al), np.cos(al), 0], [0, 0, 1]])
        return np.imag(inputs.kerr_schild(R @ pts.astype(complex), 1.0, a)[k]) / h

    ref = [Om * along_circle(k) for k in range(3)]
    for p in range(pts.shape[1]):
        v = Om * np.array([-pts[1, p], pts[0, p], 0.0])
        o = oracle.rhs_point_map(psi[..., p], Pi[..., p], Phi[..., p], Phi[..., p], dPi[..., p], dPhi[..., p], H[:, p], dH[..., p],
                                 (1.0, -1.0, 1.0), np.eye(3), v)
        for k in range(3):
            assert np.abs(o[k] - ref[k][..., p]).max() < 1e-12
        assert np.abs(ref[1][..., p]).max() > 1e-3


def test_structure_and_subdomain_level(oracle):
    """General Jm, v: the result is F[Jm d] + v.(Jm d) composed here from the single-frame oracle call; the subdomain-level routine is
    the point-level one on the oracle's own spectral gradient, zero on FROZEN faces; the RK3 variant is three such evaluations."""
    rng = np.random.default_rng(8)
    psi, Pi, Phi, dpsi, dPi, dPhi, H, dH = random_point(5)
    J, v = np.eye(3) + 0.2 * rng.standard_normal((3, 3)), rng.standard_normal(3)
    o = oracle.rhs_point_map(psi, Pi, Phi, dpsi, dPi, dPhi, H, dH, (1.0, -0.5, 2.0), J, v)
    td = lambda d: np.einsum("ik,k...->i...", J, d)
    f = oracle.rhs_point(psi, Pi, Phi, td(dpsi), td(dPi), td(dPhi), H, dH, (1.0, -0.5, 2.0))
    adv = [np.einsum("i,i...->...", v, td(dpsi)), np.einsum("i,i...->...", v, td(dPi)), np.einsum("i,ij...->j...", v, td(dPhi))]
    for x, y, z in zip(o, f, adv):
        assert np.abs(x - (y + z)).max() < 1e-13
    sd = configs.block([6, 5, 7], (3.0, -1.0, -1.0), (5.0, 1.0, 1.0), face=(1, 0, 0, 0, 0, 0))
    xyz = oracle.coords(sd)
    P = xyz.shape[1]
    us, Hs = inputs.initial_data([sd], [xyz], 0.3, 1e-3, 41)
    dHs = cstep(lambda z: inputs.kerr_schild_gauge_source(z, 1.0, 0.3), xyz).reshape(12, P)
    Jm = np.repeat(J.reshape(9, 1), P, axis=1) * (1 + 0.05 * np.sin(xyz[0]))
    vv = np.stack([0.3 * xyz[1], -0.2 * xyz[0], 0.1 + 0 * xyz[2]])
    k = oracle.rhs_map(sd, us[0], Hs[0], dHs, Jm, vv)
    g = oracle.gradient(sd, us[0])
    psi_, Pi_, Phi_ = inputs.unpack_fields(us[0])
    gp = [inputs.unpack_fields(g[i]) for i in range(3)]
    for p in (50, 101, P - 1):
        dps = np.stack([gp[i][0][..., p] for i in range(3)]); dPi_p = np.stack([gp[i][1][..., p] for i in range(3)])
        dPh = np.stack([gp[i][2][..., p] for i in range(3)])
        o = oracle.rhs_point_map(psi_[..., p], Pi_[..., p], Phi_[..., p], dps, dPi_p, dPh, Hs[0][:, p], dHs[:, p].reshape(3, 4), sd["gamma"],
                                 Jm[:, p].reshape(3, 3), vv[:, p])
        ref = inputs.pack_fields(o[0][..., None], o[1][..., None], o[2][..., None])[:, 0]
        assert np.abs(k[:, p] - ref).max() < 1e-13
    assert np.all(k[:, :35] == 0.0)              # the FROZEN -x face (i0 = 0: the first 5 * 7 points) holds the grid-frame value
    dt = 1e-3
    u1 = oracle.rhs_map(sd, us[0], Hs[0], dHs, Jm, vv, dt=dt, nsteps=1)
    f = lambda u: oracle.rhs_map(sd, u, Hs[0], dHs, Jm, vv)
    a1 = us[0] + dt * f(us[0]); a2 = 0.75 * us[0] + 0.25 * (a1 + dt * f(a1)); a3 = us[0] / 3 + (2.0 / 3.0) * (a2 + dt * f(a2))
    assert np.abs(u1 - a3).max() < 1e-14
