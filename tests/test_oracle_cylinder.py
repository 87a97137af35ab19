"""Pins for oracle O15: the cylindrical-shell topology (PAPER.md:79, 564 name it for binary runs and give no formulas; DESIGN.md
reading S25: I1(rho) x I1(z) x S1(phi), axis along z, Chebyshev-Gauss-Lobatto in rho and z, uniform Fourier in phi).  What fixes
it without another implementation: the textbook Fourier differentiation matrix, exactness on single modes and on Cartesian
polynomials, the grid's closed form, stationarity of exact Kerr-Schild data, and the face treatment re-derived from the point
functions (O10) with the face normals written out here."""
import numpy as np
import pytest

from paper_1804_09101_b200 import configs, inputs
from domain_util import build_case


# ---- Fourier line ------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("N", [4, 7, 12, 17])
def test_fourier_derivative_matches_textbook_matrix(oracle, N):
    """delta inputs trace the matrix: D_jk = (1/2)(-1)^(j-k) cot((j-k) pi/N) for even N,
    (1/2)(-1)^(j-k) / sin((j-k) pi/N) for odd N, zero diagonal (the periodic cardinal-function derivative)."""
    D = np.stack([oracle.fourier_derivative_line(e) for e in np.eye(N)], axis=1)
    j, k = np.meshgrid(np.arange(N), np.arange(N), indexing="ij")
    d = (j - k).astype(float)
    with np.errstate(divide="ignore", invalid="ignore"):
        ref = 0.5 * (-1.0) ** (j - k) * (1.0 / np.tan(d * np.pi / N) if N % 2 == 0 else 1.0 / np.sin(d * np.pi / N))
    ref[j == k] = 0.0
    assert np.abs(D - ref).max() < 1e-13
    assert np.abs(D + D.T).max() < 1e-13            # antisymmetric
    assert np.abs(D.sum(1)).max() < 1e-13           # constants are annihilated


@pytest.mark.parametrize("N", [8, 9])
def test_fourier_derivative_single_modes(oracle, N):
    phi = 2 * np.pi * np.arange(N) / N
    for m in range(0, (N + 1) // 2):              # every mode below Nyquist, with a phase
        u = np.cos(m * phi + 0.3)
        assert np.abs(oracle.fourier_derivative_line(u) + m * np.sin(m * phi + 0.3)).max() < 1e-13, m
    if N % 2 == 0:                                  # the Nyquist mode of an even N: its derivative vanishes at the nodes
        assert np.abs(oracle.fourier_derivative_line(np.cos(N // 2 * phi))).max() < 1e-13
    # an unresolved mode aliases (m = N - 1 looks like m = -1): the result is the derivative of the alias, not of the input
    u = np.sin((N - 1) * phi)
    assert np.abs(oracle.fourier_derivative_line(u) - (-np.cos(phi))).max() < 1e-13


# ---- grid ----------------------------------------------------------------------------------------------------------------
def test_cylinder_coords(oracle):
    sd = configs.cylinder((5, 4, 6), 2.0, 6.0, -1.0, 3.0, center=(1.0, 2.0, 3.0))
    xyz = oracle.coords(sd) - np.array(sd["center"])[:, None]
    rho = np.hypot(xyz[0], xyz[1]).reshape(5, 4, 6)
    assert np.allclose(rho[:, 0, 0], 2.0 + 4.0 * (oracle.cheb_nodes(5) + 1) / 2, atol=1e-14)      # rho slowest
    assert np.abs(rho - rho[:, :1, :1]).max() < 1e-14
    z = xyz[2].reshape(5, 4, 6)
    assert np.allclose(z[0, :, 0], -1.0 + 4.0 * (oracle.cheb_nodes(4) + 1) / 2, atol=1e-14)
    assert np.abs(z - z[:1, :, :1]).max() < 1e-14
    ph = np.arctan2(xyz[1], xyz[0]).reshape(5, 4, 6) % (2 * np.pi)
    assert np.allclose(ph[2, 1], 2 * np.pi * np.arange(6) / 6, atol=1e-13)                          # phi fastest
    assert configs.num_points(sd) == 120


# ---- gradient --------------------------------------------------------------------------------------------------------------
CYL_POLYS = [  # (f, df/dx, df/dy, df/dz): x^a y^b z^c with a + b <= 3 (needs N_rho >= 4, N_phi >= 7), c <= 3 (N_z >= 4)
    (lambda x, y, z: x, lambda x, y, z: 1 + 0 * x, lambda x, y, z: 0 * x, lambda x, y, z: 0 * x),
    (lambda x, y, z: y, lambda x, y, z: 0 * x, lambda x, y, z: 1 + 0 * x, lambda x, y, z: 0 * x),
    (lambda x, y, z: z, lambda x, y, z: 0 * x, lambda x, y, z: 0 * x, lambda x, y, z: 1 + 0 * x),
    (lambda x, y, z: x * y, lambda x, y, z: y, lambda x, y, z: x, lambda x, y, z: 0 * x),
    (lambda x, y, z: x * x - y * y, lambda x, y, z: 2 * x, lambda x, y, z: -2 * y, lambda x, y, z: 0 * x),
    (lambda x, y, z: x * x * y + z, lambda x, y, z: 2 * x * y, lambda x, y, z: x * x, lambda x, y, z: 1 + 0 * x),
    (lambda x, y, z: z**3 - 2 * x * y * z, lambda x, y, z: -2 * y * z, lambda x, y, z: -2 * x * z, lambda x, y, z: 3 * z * z - 2 * x * y),
    (lambda x, y, z: y**3 * z * z, lambda x, y, z: 0 * x, lambda x, y, z: 3 * y * y * z * z, lambda x, y, z: 2 * y**3 * z),
]


@pytest.mark.parametrize("n", [(4, 4, 7), (6, 5, 8), (5, 7, 12)])
def test_cylinder_cartesian_polynomials(oracle, n):
    """x^a y^b z^c = rho^(a+b) cos^a sin^b z^c: a polynomial of degree a+b in rho, c in z and a trigonometric polynomial of
    degree a+b in phi - all resolved, so the Cartesian gradient is exact.  (Each monomial fails under a different mistake:
    x, y under a wrong sign or a cos/sin swap in the Jacobian, z under an exchange of the z and phi slots, x y and x^2 - y^2
    under a missing 1/rho, the cubic ones under a wrong map factor.)"""
    sd = configs.cylinder(n, 1.5, 4.0, -2.0, 1.0, center=(0.3, -0.2, 0.1))
    xyz = oracle.coords(sd)
    x, y, z = xyz - np.array(sd["center"])[:, None]
    u = np.stack([f(x, y, z) for f, *_ in CYL_POLYS])
    g = oracle.gradient(sd, u)
    for c, (_, fx, fy, fz) in enumerate(CYL_POLYS):
        for d, fd in enumerate((fx, fy, fz)):
            assert np.abs(g[d, c] - fd(x, y, z)).max() < 2e-12, (c, d)


def test_cylinder_gradient_converges_on_smooth_data(oracle):
    errs = []
    for n in (6, 10, 14):
        sd = configs.cylinder((n, n, 2 * n), 2.0, 4.0, -1.0, 1.0)
        x, y, z = oracle.coords(sd)
        u = np.exp(0.3 * x - 0.2 * y + 0.25 * z)[None]
        g = oracle.gradient(sd, u)
        errs.append(max(np.abs(g[0, 0] - 0.3 * u[0]).max(), np.abs(g[1, 0] + 0.2 * u[0]).max(), np.abs(g[2, 0] - 0.25 * u[0]).max()))
    assert errs[1] < 1e-3 * errs[0] and errs[2] < 1e-11


# ---- spectral filter ---------------------------------------------------------------------------------------------------------
def _cheb_T(k, x):
    return np.cos(k * np.arccos(np.clip(x, -1, 1)))


def test_cylinder_filter_single_modes(oracle):
    """T_a(rho~) T_b(z~) cos(m phi + d) is an eigenfunction: it comes back scaled by sigma_rho[a] sigma_z[b] sigma_phi[m]
    (the Nyquist mode of an even N_phi included); sigma = 1 is the identity."""
    n = (6, 5, 8)
    sd = configs.cylinder(n, 2.0, 5.0, -1.0, 2.0)
    xyz = oracle.coords(sd)
    rho, z, ph = np.hypot(xyz[0], xyz[1]), xyz[2], np.arctan2(xyz[1], xyz[0])
    xr, xz = (rho - 2.0) / 3.0 * 2 - 1, (z + 1.0) / 3.0 * 2 - 1
    rng = np.random.default_rng(7)
    sig = [rng.uniform(0.2, 1.0, n[0]), rng.uniform(0.2, 1.0, n[1]), rng.uniform(0.2, 1.0, n[2] // 2 + 1)]
    cases = [(0, 0, 0), (3, 0, 0), (0, 4, 0), (0, 0, 3), (5, 2, 1), (2, 3, 4)]
    u = np.stack([_cheb_T(a, xr) * _cheb_T(b, xz) * (np.cos(m * ph + 0.4) if m < 4 else np.cos(m * ph)) for a, b, m in cases])
    out = oracle.spectral_filter(sd, u, sig)
    for c, (a, b, m) in enumerate(cases):
        assert np.abs(out[c] - sig[0][a] * sig[1][b] * sig[2][m] * u[c]).max() < 1e-13, (a, b, m)
    ones = [np.ones(n[0]), np.ones(n[1]), np.ones(n[2] // 2 + 1)]
    v = rng.standard_normal((2, u.shape[1]))
    assert np.abs(oracle.spectral_filter(sd, v, ones) - v).max() < 1e-13
    # odd N_phi: no Nyquist mode, the top mode (N-1)/2 is an ordinary one
    sd7 = configs.cylinder((4, 4, 7), 2.0, 5.0, -1.0, 2.0)
    x7 = oracle.coords(sd7)
    p7 = np.arctan2(x7[1], x7[0])
    s7 = [np.ones(4), np.ones(4), np.array([1.0, 0.9, 0.5, 0.25])]
    assert np.abs(oracle.spectral_filter(sd7, np.sin(3 * p7)[None], s7) - 0.25 * np.sin(3 * p7)).max() < 1e-13


# ---- RHS on the new topology -----------------------------------------------------------------------------------------------
def test_stationary_ks_converges_on_a_cylinder(oracle):
    """Exact Kerr-Schild data (a = 0.5, the hole on the axis inside the hollow) is stationary: the RHS with spectral derivatives
    decays exponentially with the resolution; dt psi == 0 to rounding with gamma1 = -1."""
    vals = []
    for n in (8, 12, 16):
        sd = configs.cylinder((n, n, 2 * n), 3.0, 7.0, -2.0, 2.0)
        xyz = oracle.coords(sd)
        u = inputs.pack_fields(*inputs.kerr_schild(xyz, 1.0, 0.5))
        H = inputs.kerr_schild_gauge_source(xyz, 1.0, 0.5)
        k = oracle.rhs(sd, u, H)
        vals.append((np.abs(k[:10]).max(), np.abs(k[10:]).max()))
    assert all(v[0] < 1e-14 for v in vals)
    assert vals[1][1] < 0.05 * vals[0][1] and vals[2][1] < 0.05 * vals[1][1] and vals[2][1] < 1e-5, vals


def test_cylinder_rhs_equals_point_function_on_its_gradient(oracle):
    """Interior points: the subdomain RHS is the point function O5 applied to the state and the subdomain's own gradient
    (nothing topology-specific hides in between)."""
    cfg = {"id": 41, "spin": 0.4, "amplitude": 1e-3, "descs": [configs.cylinder((5, 4, 8), 3.0, 6.0, -1.0, 1.5, gamma=[0.7, 0.4, -1.3])]}
    descs, coords, us, Hs = build_case(cfg, oracle)
    sd, u, H = descs[0], us[0], Hs[0]
    k = oracle.rhs(sd, u, H)
    g = oracle.gradient(sd, u)
    gH = oracle.gradient(sd, H)
    for p in (0, 37, 101, 159):
        full = lambda t10: np.array([[t10[inputs.SYM_PAIRS.index((min(a, b), max(a, b)))] for b in range(4)] for a in range(4)])
        psi, Pi = full(u[:10, p]), full(u[10:20, p])
        Phi = np.stack([full(u[20 + 10 * i:30 + 10 * i, p]) for i in range(3)])
        dpsi = np.stack([full(g[kk, :10, p]) for kk in range(3)])
        dPi = np.stack([full(g[kk, 10:20, p]) for kk in range(3)])
        dPhi = np.stack([[full(g[kk, 20 + 10 * i:30 + 10 * i, p]) for i in range(3)] for kk in range(3)])
        a, b, c = oracle.rhs_point(psi, Pi, Phi, dpsi, dPi, dPhi, H[:, p], gH[:, :, p], sd["gamma"])
        ref = np.concatenate([[a[x, y] for x, y in inputs.SYM_PAIRS], [b[x, y] for x, y in inputs.SYM_PAIRS]] +
                             [[c[i, x, y] for x, y in inputs.SYM_PAIRS] for i in range(3)])
        assert np.abs(k[:, p] - ref).max() < 1e-14, p


def test_cylinder_faces(oracle):
    """O6 / O10 on the four faces (phi is periodic: no face there).  FROZEN zeroes exactly the face points; CHARACTERISTIC equals
    the point function O10 applied to the unflagged RHS with the outward normals written out here: -+ (cos phi, sin phi, 0) on
    the rho faces, -+ z^ on the z faces, applied in face order at edges."""
    n = (5, 4, 6)
    cfg = {"id": 42, "spin": 0.3, "amplitude": 1e-3, "descs": [configs.cylinder(n, 3.0, 6.0, -1.0, 1.5, center=(0.2, -0.1, 0.3))]}
    descs, coords, us, Hs = build_case(cfg, oracle)
    sd, u, H, xyz = descs[0], us[0], Hs[0], coords[0]
    free = oracle.rhs(sd, u, H)
    k = oracle.rhs(dict(sd, face=[1, 0, 0, 1, 0, 0]), u, H)
    on = np.zeros(n, bool)
    on[0, :, :] = True
    on[:, -1, :] = True
    assert np.all(k[:, on.ravel()] == 0.0) and np.array_equal(k[:, ~on.ravel()], free[:, ~on.ravel()])
    assert np.all(np.abs(free[10:20]).max(axis=0) > 0)          # ... so the k = 0 and k = N_phi - 1 columns are not "faces"
    kc = oracle.rhs(dict(sd, face=[2, 2, 2, 2, 0, 0]), u, H)
    rel = xyz - np.array(sd["center"])[:, None]
    full = lambda t10: np.array([[t10[inputs.SYM_PAIRS.index((min(a, b), max(a, b)))] for b in range(4)] for a in range(4)])
    pack = lambda t: np.array([t[x, y] for x, y in inputs.SYM_PAIRS])
    idx = np.arange(np.prod(n)).reshape(n)
    checked = 0
    for i in range(n[0]):
        for j in range(n[1]):
            for kk in (0, 1, 4):
                p = idx[i, j, kk]
                rho = np.hypot(rel[0, p], rel[1, p])
                dirs = []
                if i == 0: dirs.append([-rel[0, p] / rho, -rel[1, p] / rho, 0.0])
                if i == n[0] - 1: dirs.append([rel[0, p] / rho, rel[1, p] / rho, 0.0])
                if j == 0: dirs.append([0.0, 0.0, -1.0])
                if j == n[1] - 1: dirs.append([0.0, 0.0, 1.0])
                a, b = full(free[:10, p]), full(free[10:20, p])
                c = np.stack([full(free[20 + 10 * q:30 + 10 * q, p]) for q in range(3)])
                for s in dirs:
                    a, b, c, _ = oracle.char_bc_point(full(u[:10, p]), sd["gamma"], s, a, b, c)
                ref = np.concatenate([pack(a), pack(b)] + [pack(c[q]) for q in range(3)])
                assert np.abs(kc[:, p] - ref).max() < 1e-14, (i, j, kk)
                checked += len(dirs)
    assert checked > 50 and np.abs(kc - free).max() > 1e-6      # the condition did act
