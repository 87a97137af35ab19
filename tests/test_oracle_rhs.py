"""Pins for oracle O5 (GH right-hand side), O8 (constraints) — SURVEY.md §8(c) pin table.

The paper does not print the evolved equations, so these pins are what fix them:
(i) exact Kerr-Schild data is stationary (the paper's own test problem), with
derivatives supplied analytically (complex step) so no truncation error hides a wrong term;
(iii) the harmonic gauge wave has O(1) analytic time derivatives and pins every sign stationarity
cannot; the damping terms vanish in both and get dedicated homogeneous-data cases.
"""
import numpy as np
import pytest

from paper_1804_09101_b200 import configs, inputs

PTS = np.array([[2.0, 0.3, -1.1], [-3.0, 2.5, 0.7], [0.4, -2.2, 2.9], [5.0, 5.0, 5.0], [1.5, 1.0, 0.2]]).T
GAMMAS = [(0.0, 0.0, 0.0), (1.0, -1.0, 1.0), (3.0, -1.0, 2.0), (0.7, 0.4, -1.3)]


def cstep(fun, xyz, h=1e-30):
    out = []
    for i in range(3):
        z = xyz.astype(complex)
        z[i] += 1j * h
        out.append(np.imag(fun(z)) / h)
    return np.stack(out)


def ks_point_data(a, M=1.0, pts=PTS):
    psi, Pi, Phi = inputs.kerr_schild(pts, M, a)
    dPi = cstep(lambda z: inputs.kerr_schild(z, M, a)[1], pts)          # [k,a,b,P]
    dPhi = cstep(lambda z: inputs.kerr_schild(z, M, a)[2], pts)         # [k,i,a,b,P]
    H = inputs.kerr_schild_gauge_source(pts, M, a)
    dH = cstep(lambda z: inputs.kerr_schild_gauge_source(z, M, a), pts)  # [i,b,P]
    return psi, Pi, Phi, dPi, dPhi, H, dH


@pytest.mark.parametrize("a", [0.0, 0.5, 0.7, 0.9])
def test_kerr_schild_stationary_with_analytic_derivatives(oracle, a):
    psi, Pi, Phi, dPi, dPhi, H, dH = ks_point_data(a)
    for gam in GAMMAS:
        for p in range(PTS.shape[1]):
            o = oracle.rhs_point(psi[..., p], Pi[..., p], Phi[..., p], Phi[..., p], dPi[..., p], dPhi[..., p], H[:, p], dH[..., p], gam)
            for name, v in zip(("dtpsi", "dtPi", "dtPhi"), o):
                assert np.abs(v).max() < 1e-12, (a, gam, p, name, np.abs(v).max())


@pytest.mark.parametrize("a", [0.0, 0.6])
def test_gamma_a_matches_analytic_gauge_source(oracle, a):
    """Gamma_a from O5's Christoffel trace equals -H_a from the closed form Gamma^a = 2 d_j (H l^a l^j):
    so C_a = H_a + Gamma_a vanishes; also C_iab = 0 and C_ijab = 0 with analytic derivatives."""
    psi, Pi, Phi, dPi, dPhi, H, dH = ks_point_data(a)
    for p in range(PTS.shape[1]):
        Ca, Ciab, Cijab = oracle.constraints_point(psi[..., p], Pi[..., p], Phi[..., p], Phi[..., p], dPhi[..., p], H[:, p])
        assert np.abs(Ca).max() < 1e-14 and np.abs(Ciab).max() == 0 and np.abs(Cijab).max() < 1e-14
    if a == 0.0:  # Schwarzschild: Gamma^0 = -2M/r^2, Gamma^i = 2 M x^i / r^3  (SURVEY pin)
        r = np.sqrt((PTS**2).sum(0))
        Gup = np.stack([-2 / r**2, *(2 * PTS / r**3)])
        Glow = np.einsum("abp,bp->ap", psi, Gup)
        assert np.abs(H + Glow).max() < 1e-14


def test_gauge_wave(oracle):
    """RHS == analytic d_t(psi,Pi,Phi) for the harmonic gauge wave, H_a = 0, any gamma (constraints vanish)."""
    pts = np.array([[0.13, -0.4, 0.2], [-0.77, 0.1, 0.9], [0.5, 0.5, -0.5]]).T
    t = 0.3
    psi, Pi, Phi, dtpsi, dtPi, dtPhi = inputs.gauge_wave(pts, t)
    dPi = cstep(lambda z: inputs.gauge_wave(z, t)[1], pts)
    dPhi = cstep(lambda z: inputs.gauge_wave(z, t)[2], pts)
    assert np.abs(dtPi).max() > 0.05
    for gam in GAMMAS:
        for p in range(pts.shape[1]):
            o = oracle.rhs_point(psi[..., p], Pi[..., p], Phi[..., p], Phi[..., p], dPi[..., p], dPhi[..., p], np.zeros(4), np.zeros((3, 4)), gam)
            assert np.abs(o[0] - dtpsi[..., p]).max() < 1e-14
            assert np.abs(o[1] - dtPi[..., p]).max() < 1e-14
            assert np.abs(o[2] - dtPhi[..., p]).max() < 1e-14
            Ca, _, _ = oracle.constraints_point(psi[..., p], Pi[..., p], Phi[..., p], Phi[..., p], dPhi[..., p], np.zeros(4))
            assert np.abs(Ca).max() < 1e-15   # harmonic: Gamma_a = 0


def minkowski():
    psi = np.diag([-1.0, 1.0, 1.0, 1.0])
    return psi, np.zeros((4, 4)), np.zeros((3, 4, 4)), np.zeros((3, 4, 4)), np.zeros((3, 4, 4)), np.zeros((3, 3, 4, 4))


def test_damping_terms_homogeneous(oracle):
    """Minkowski, spatially homogeneous data, H_a = 0 (SURVEY pin): only Pi_00 = p gives
    dt Pi_00 = -gamma0 p/2 + p^2 and dt psi_00 = -p; only Phi_y23 = q gives dt Phi_y23 = -gamma2 q."""
    g0, g1, g2 = 3.0, -1.0, 2.0
    p = 0.37
    psi, Pi, Phi, dpsi, dPi, dPhi = minkowski()
    Pi[0, 0] = p
    o = oracle.rhs_point(psi, Pi, Phi, dpsi, dPi, dPhi, np.zeros(4), np.zeros((3, 4)), (g0, g1, g2))
    assert abs(o[1][0, 0] - (-g0 * p / 2 + p * p)) < 1e-15 and abs(o[0][0, 0] + p) < 1e-15
    q = -0.21
    psi, Pi, Phi, dpsi, dPi, dPhi = minkowski()
    Phi[1, 2, 3] = Phi[1, 3, 2] = q
    o = oracle.rhs_point(psi, Pi, Phi, dpsi, dPi, dPhi, np.zeros(4), np.zeros((3, 4)), (g0, g1, g2))
    assert abs(o[2][1, 2, 3] + g2 * q) < 1e-15


def random_point(seed):
    rng = np.random.default_rng(seed)
    sym = lambda m: 0.5 * (m + np.swapaxes(m, -1, -2))
    psi = np.diag([-1.0, 1.0, 1.0, 1.0]) + 0.2 * sym(rng.standard_normal((4, 4)))
    Pi = sym(rng.standard_normal((4, 4)))
    Phi = sym(rng.standard_normal((3, 4, 4)))
    dpsi = sym(rng.standard_normal((3, 4, 4)))
    dPi = sym(rng.standard_normal((3, 4, 4)))
    dPhi = sym(rng.standard_normal((3, 3, 4, 4)))
    return psi, Pi, Phi, dpsi, dPi, dPhi, rng.standard_normal(4), rng.standard_normal((3, 4))


def test_gamma_structure(oracle):
    """With gamma1 = -1, dt psi does not see the spectral d_k psi at all; the RHS is affine in gamma0, gamma2
    and in gamma1*gamma2 (SURVEY pin); outputs are symmetric in (a,b) for symmetric inputs."""
    psi, Pi, Phi, dpsi, dPi, dPhi, H, dH = random_point(11)
    a = oracle.rhs_point(psi, Pi, Phi, dpsi, dPi, dPhi, H, dH, (1.0, -1.0, 1.0))
    b = oracle.rhs_point(psi, Pi, Phi, 100 * dpsi + 7, dPi, dPhi, H, dH, (1.0, -1.0, 1.0))
    assert np.abs(a[0] - b[0]).max() < 1e-15
    for o in a:
        assert np.abs(o - np.swapaxes(o, -1, -2)).max() < 1e-14
    f = lambda g: np.concatenate([x.ravel() for x in oracle.rhs_point(psi, Pi, Phi, dpsi, dPi, dPhi, H, dH, g)])
    base = f((0.0, 0.0, 0.0))
    assert np.abs(f((2.0, 0.0, 0.0)) - base - 2 * (f((1.0, 0.0, 0.0)) - base)).max() < 1e-13   # affine in gamma0
    assert np.abs(f((0.0, 0.0, 2.0)) - base - 2 * (f((0.0, 0.0, 1.0)) - base)).max() < 1e-13   # affine in gamma2 (g1=0)
    # g1 enters dt Pi only through g1*g2: (g1,g2) = (2,3) and (3,2) give the same dt Pi
    p1 = oracle.rhs_point(psi, Pi, Phi, dpsi, dPi, dPhi, H, dH, (0.5, 2.0, 3.0))[1]
    p2 = oracle.rhs_point(psi, Pi, Phi, dpsi, dPi, dPhi, H, dH, (0.5, 3.0, 2.0))[1]
    q0 = oracle.rhs_point(psi, Pi, Phi, dpsi, dPi, dPhi, H, dH, (0.5, 0.0, 3.0))[1]
    q2 = oracle.rhs_point(psi, Pi, Phi, dpsi, dPi, dPhi, H, dH, (0.5, 0.0, 2.0))[1]
    assert np.abs((p1 - q0) - (p2 - q2)).max() < 1e-13


def test_linearised_principal_part(oracle):
    """Around Minkowski with Pi = Phi = 0 the RHS is linear in the derivative inputs with the textbook
    principal part: dt Pi = -delta^{ki} d_k Phi_iab + g1 g2 * 0,  dt Phi_i = -d_i Pi + g2 d_i psi,  dt psi = 0 (shift = 0)."""
    psi, Pi, Phi, dpsi, dPi, dPhi = minkowski()
    rng = np.random.default_rng(5)
    sym = lambda m: 0.5 * (m + np.swapaxes(m, -1, -2))
    dpsi, dPi, dPhi = sym(rng.standard_normal((3, 4, 4))), sym(rng.standard_normal((3, 4, 4))), sym(rng.standard_normal((3, 3, 4, 4)))
    g = (0.0, 0.3, 1.7)
    o = oracle.rhs_point(psi, Pi, Phi, dpsi, dPi, dPhi, np.zeros(4), np.zeros((3, 4)), g)
    assert np.abs(o[0]).max() < 1e-15
    assert np.abs(o[1] + np.einsum("kkab->ab", dPhi)).max() < 1e-14
    assert np.abs(o[2] - (-dPi + g[2] * dpsi)).max() < 1e-14


def test_stationary_ks_spectral_convergence_shell(oracle):
    """(ii) with spectral derivatives on the C1 geometry, a = 0: residual decays ~x100 per Delta N_r = 4 and
    does not depend on L for L >= 4 (fields band-limited to l <= 3); dt psi == 0 with gamma1 = -1.
    Survey's measured values: N_r=8: max|dtPi| 1.6e-3, |dtPhi| 1.9e-3, |C_iab| 6.3e-4;
    N_r=12: 1.7e-5 / 2.0e-5 / 3.9e-6."""
    res = {}
    for nr, L in [(8, 4), (8, 8), (12, 4)]:
        sd = configs.shell(nr, L, 1.8, 5.0)
        xyz = oracle.coords(sd)
        u = inputs.pack_fields(*inputs.kerr_schild(xyz, 1.0, 0.0))
        H = inputs.kerr_schild_gauge_source(xyz, 1.0, 0.0)
        k = oracle.rhs(sd, u, H)
        _, maxs, _ = oracle.constraints(sd, u, H)
        res[(nr, L)] = (np.abs(k[:10]).max(), np.abs(k[10:20]).max(), np.abs(k[20:]).max(), maxs)
    assert res[(8, 4)][0] < 1e-15 and res[(12, 4)][0] < 1e-15
    assert abs(res[(8, 4)][1] / res[(8, 8)][1] - 1) < 1e-2 and abs(res[(8, 4)][2] / res[(8, 8)][2] - 1) < 1e-2
    assert 1.2e-3 < res[(8, 8)][1] < 2.0e-3 and 1.5e-3 < res[(8, 8)][2] < 2.4e-3     # 1.6e-3 / 1.9e-3
    assert 1.3e-5 < res[(12, 4)][1] < 2.1e-5 and 1.6e-5 < res[(12, 4)][2] < 2.4e-5   # 1.7e-5 / 2.0e-5
    assert 5e-4 < res[(8, 8)][3][1] < 8e-4 and 3e-6 < res[(12, 4)][3][1] < 5e-6      # C_iab 6.3e-4 / 3.9e-6
    assert res[(8, 8)][3][0] < 1e-14                                                # C_a == 0


def test_stationary_ks_spectral_convergence_block(oracle):
    """C2 geometry (block [3,11]x[-4,4]^2, a = 0.5): survey's values max|dtPi| N=8: 2.7e-2, 12: 6.6e-3, 16: 1.1e-3."""
    vals = []
    for n in (8, 12, 16):
        sd = configs.block(n, (3.0, -4.0, -4.0), (11.0, 4.0, 4.0))
        xyz = oracle.coords(sd)
        u = inputs.pack_fields(*inputs.kerr_schild(xyz, 1.0, 0.5))
        H = inputs.kerr_schild_gauge_source(xyz, 1.0, 0.5)
        vals.append(np.abs(oracle.rhs(sd, u, H)[10:20]).max())
    assert 2.0e-2 < vals[0] < 3.4e-2 and 5.0e-3 < vals[1] < 8.2e-3 and 0.8e-3 < vals[2] < 1.4e-3


def test_symmetry_preserved_full_arrays(oracle):
    """The 16-component oracle keeps dt psi_ab and dt Pi_ab symmetric to rounding on perturbed data."""
    cfg = configs.c1()
    sd = cfg["descs"][0]
    xyz = oracle.coords(sd)
    us, Hs = inputs.initial_data([sd], [xyz], cfg["spin"], cfg["amplitude"], cfg["id"])
    out = oracle.rhs_full(sd, us[0], Hs[0])
    P = xyz.shape[1]
    dpsi, dPi, dPhi = out[:16].reshape(4, 4, P), out[16:32].reshape(4, 4, P), out[32:].reshape(3, 4, 4, P)
    assert np.abs(dpsi - dpsi.swapaxes(0, 1)).max() < 1e-15
    assert np.abs(dPi - dPi.swapaxes(0, 1)).max() < 1e-14
    assert np.abs(dPhi - dPhi.swapaxes(1, 2)).max() < 1e-14
    # packed output == upper triangle of the full one, with FREE faces
    sd_free = dict(sd, face=[0] * 6)
    k = oracle.rhs(sd_free, us[0], Hs[0])
    assert np.array_equal(k[:10], np.stack([dpsi[a, b] for a, b in inputs.SYM_PAIRS]))


def test_constraint_linearity_and_frozen_faces(oracle):
    """O8: on perturbed data C_iab = (spectral d_i of delta psi) - delta Phi_i + C_iab(unperturbed), by linearity;
    O6: FROZEN faces zero all 50 RHS components exactly there and nowhere else."""
    sd = configs.block([6, 5, 7], (3.0, -1.0, -1.0), (5.0, 1.0, 1.0), face=(1, 0, 0, 1, 0, 0))
    xyz = oracle.coords(sd)
    u0 = inputs.pack_fields(*inputs.kerr_schild(xyz, 1.0, 0.3))
    H = inputs.kerr_schild_gauge_source(xyz, 1.0, 0.3)
    du = inputs.block_perturbation(sd["lo"], sd["hi"], xyz, 1e-3, 99, deg=3)
    _, _, C0 = oracle.constraints(sd, u0, H, fields=True)
    _, _, C1 = oracle.constraints(sd, u0 + du, H, fields=True)
    g = oracle.gradient(sd, du[:10])
    for i in range(3):
        assert np.abs((C1 - C0)[4 + 10 * i : 14 + 10 * i] - (g[i] - du[20 + 10 * i : 30 + 10 * i])).max() < 1e-14
    k = oracle.rhs(sd, u0 + du, H)
    idx = np.arange(xyz.shape[1]).reshape(6, 5, 7)
    on = np.zeros((6, 5, 7), bool)
    on[0, :, :] = True
    on[:, -1, :] = True
    assert np.all(k[:, on.ravel()] == 0.0)
    assert np.all(np.abs(k[10:20, ~on.ravel()]).max(axis=0) > 0)
    sums, maxs, _ = oracle.constraints(sd, u0 + du, H)
    norms = oracle.constraint_norms([sd], [u0 + du], [H])
    assert np.allclose(norms[:, 0], np.sqrt(sums / (xyz.shape[1] * np.array([4, 30, 30]))))
    assert np.allclose(norms[1], [np.sqrt((C1[4:34] ** 2).mean()), np.abs(C1[4:34]).max()])


def _poly_phi(sd, xyz, seed, deg=3):
    """Seeded polynomial dPhi_iab (degree <= deg per axis in the block's reference coordinates) and its ANALYTIC Cartesian
    gradient, both from the monomial coefficients in numpy (nothing of the oracle): -> Phi[30, P], grad[3, 30, P]."""
    rng = np.random.default_rng(seed)
    lo, hi = np.array(sd["lo"]), np.array(sd["hi"])
    X = (2 * xyz - (lo + hi)[:, None]) / (hi - lo)[:, None]          # reference cube coordinates
    c = rng.uniform(-1, 1, (30, deg + 1, deg + 1, deg + 1))
    pw = [np.stack([X[a] ** p for p in range(deg + 1)]) for a in range(3)]                                   # X^p
    dpw = [np.stack([p * X[a] ** max(p - 1, 0) for p in range(deg + 1)]) * (2 / (hi[a] - lo[a])) for a in range(3)]  # d/dx_a X^p
    Phi = np.einsum("cpqr,pn,qn,rn->cn", c, pw[0], pw[1], pw[2])
    grad = np.stack([np.einsum("cpqr,pn,qn,rn->cn", c, *(dpw[b] if b == a else pw[b] for b in range(3))) for a in range(3)])
    return Phi, grad


def test_c_ijab_on_non_vanishing_data(oracle):
    """O8, the C_ijab part: C_ijab = d_i Phi_jab - d_j Phi_iab must equal the ANALYTIC curl
    of a seeded polynomial Phi on a block, component by component for the pairs (x,y), (x,z), (y,z) in that order; a wrong
    pair table, a dropped pair or a repeated index fails (the three curls differ).  Both as absolute values (Minkowski psi,
    Phi = polynomial) and by linearity on top of exact Kerr-Schild data; sums[2] / maxs[2] against their numpy restatement."""
    sd = configs.block([6, 5, 7], (3.0, -1.0, -1.5), (5.0, 1.0, 1.0))
    xyz = oracle.coords(sd)
    P = xyz.shape[1]
    dPhi, g = _poly_phi(sd, xyz, 314)
    # analytic curl rows in the oracle's documented order: 34 + 10 q + s, q = 0, 1, 2 for (i,j) = (0,1), (0,2), (1,2)
    curl = np.concatenate([g[i][10 * j:10 * j + 10] - g[j][10 * i:10 * i + 10] for i, j in ((0, 1), (0, 2), (1, 2))])
    assert min(np.abs(curl[10 * q:10 * q + 10] - curl[10 * r:10 * r + 10]).max() for q, r in ((0, 1), (0, 2), (1, 2))) > 0.1
    # (a) Minkowski metric, Pi = 0, Phi = the polynomial, H = 0
    psi = np.broadcast_to(np.diag([-1.0, 1.0, 1.0, 1.0])[..., None], (4, 4, P))
    u = inputs.pack_fields(psi, np.zeros((4, 4, P)), np.zeros((3, 4, 4, P)))
    u[20:50] = dPhi
    sums, maxs, C = oracle.constraints(sd, u, np.zeros((4, P)), fields=True)
    scale = np.abs(curl).max()
    assert np.abs(C[34:64] - curl).max() < 1e-13 * scale
    assert np.abs(C[4:34] + dPhi).max() < 1e-15            # C_iab = d_i psi - Phi_i with constant psi
    assert abs(sums[2] - (C[34:64] ** 2).sum()) <= 1e-14 * sums[2] and maxs[2] == np.abs(C[34:64]).max()
    assert abs(sums[1] - (C[4:34] ** 2).sum()) <= 1e-14 * sums[1] and maxs[1] == np.abs(C[4:34]).max()
    # (b) on top of exact Kerr-Schild data, by linearity (the unperturbed C_ijab is the truncation error of d_i Phi_j)
    u0 = inputs.pack_fields(*inputs.kerr_schild(xyz, 1.0, 0.4))
    H = inputs.kerr_schild_gauge_source(xyz, 1.0, 0.4)
    u1 = u0.copy()
    u1[20:50] += 1e-2 * dPhi
    _, _, C0 = oracle.constraints(sd, u0, H, fields=True)
    s1, m1, C1 = oracle.constraints(sd, u1, H, fields=True)
    assert np.abs((C1 - C0)[34:64] - 1e-2 * curl).max() < 1e-13 * 1e-2 * scale
    assert abs(s1[2] - (C1[34:64] ** 2).sum()) <= 1e-14 * s1[2] and m1[2] == np.abs(C1[34:64]).max()
    # the point-level function: antisymmetric in (i,j), zero diagonal, upper pairs = the analytic curl at a point
    p = 17
    full = lambda a: np.array([[a[inputs.SYM_PAIRS.index((min(x, y), max(x, y)))] for y in range(4)] for x in range(4)])
    dPhi_p = np.array([[full(g[k][10 * i:10 * i + 10, p]) for i in range(3)] for k in range(3)])      # [k][i][a][b] = d_k Phi_iab
    _, _, Cij = oracle.constraints_point(np.diag([-1.0, 1.0, 1.0, 1.0]), np.zeros((4, 4)), np.zeros((3, 4, 4)), np.zeros((3, 4, 4)),
                                         dPhi_p, np.zeros(4))
    assert np.abs(Cij + Cij.swapaxes(0, 1)).max() == 0 and np.abs(Cij[[0, 1, 2], [0, 1, 2]]).max() == 0
    for q, (i, j) in enumerate(((0, 1), (0, 2), (1, 2))):
        assert np.abs(Cij[i, j] - full(curl[10 * q:10 * q + 10, p])).max() < 1e-15 * scale


def test_stated_conventions(oracle):
    """The three conventions DESIGN.md fixes and calls 'parity unpinned' (S16 unweighted RMS normalisation, S2 default gamma's,
    S22 the VALUE of the interface penalty): no mathematics decides them, so these asserts only keep the oracle, the configs and
    the documents saying the same thing."""
    assert configs.GAMMA_DEFAULT == [1.0, -1.0, 1.0]                                                   # S2
    sd = configs.block([4, 3, 5], (3.0, -1.0, -1.0), (5.0, 1.0, 1.0))
    xyz = oracle.coords(sd)
    P = xyz.shape[1]
    u = inputs.pack_fields(np.broadcast_to(np.diag([-1.0, 1.0, 1.0, 1.0])[..., None], (4, 4, P)), np.zeros((4, 4, P)), np.zeros((3, 4, 4, P)))
    u[20:50] = 0.5                                                                                    # C_iab = -0.5 everywhere
    norms = oracle.constraint_norms([sd, sd], [u, u], [np.zeros((4, P))] * 2)
    assert abs(norms[1, 0] - 0.5) < 1e-15 and norms[1, 1] == 0.5                                       # S16: unweighted RMS over points x 30
    # S22: p = (N_r - 1)^2 / (r_out - r_in): a unit jump in psi_tt across an outer interface face of flat space with shift
    # pointing inwards (v0 = -(1+g1) n.N < 0 only if n.N > 0: use gamma1 = 0 and an outward shift) changes d_t psi_tt by p v0
    sh = configs.shell(5, 2, 2.0, 4.0, face=(0, 3), gamma=[0.0, 0.0, 0.0])
    xs = oracle.coords(sh)
    Ps = xs.shape[1]
    psi = np.broadcast_to(np.diag([-1.0, 1.0, 1.0, 1.0])[..., None], (4, 4, Ps)).copy()
    r = np.sqrt((xs ** 2).sum(0))
    beta = 0.3
    for i in range(3):
        psi[0, i + 1] = psi[i + 1, 0] = beta * xs[i] / r                                               # N^i = beta r^: n.N = beta > 0
    psi[0, 0] = -1.0 + beta ** 2
    us = inputs.pack_fields(psi, np.zeros((4, 4, Ps)), np.zeros((3, 4, 4, Ps)))
    pl = 3 * 6
    nbr = us[:, :pl].copy()
    nbr[:] = us[:, -pl:]
    k0 = oracle.rhs_ifc(sh, us, np.zeros((4, Ps)), nbr_out=nbr)
    nbr[0] -= 1.0                                                                                     # own - neighbour = +1 in psi_tt
    k1 = oracle.rhs_ifc(sh, us, np.zeros((4, Ps)), nbr_out=nbr)
    pen = (5 - 1) ** 2 / (4.0 - 2.0)
    assert np.abs((k1 - k0)[0, -pl:] - pen * (-(1 + 0.0) * beta)).max() < 1e-13
    assert np.abs((k1 - k0)[:, :-pl]).max() == 0
