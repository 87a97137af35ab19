"""Pins of the oracle's characteristic boundary condition (O10, NEXT-2 (i); the paper's ApplyBCs).
The paper prints no formulas, so the characteristic fields and speeds are pinned against the oracle's own, independently
pinned right-hand side: feeding it derivatives d_k u = n_k w isolates the principal part -A^n w, and every characteristic
eigenvector must come back multiplied by minus its speed."""
import numpy as np
import pytest

from paper_1804_09101_b200 import inputs


def _full(v10):
    m = np.zeros((4, 4))
    for s, (a, b) in enumerate(inputs.SYM_PAIRS):
        m[a, b] = m[b, a] = v10[s]
    return m


def _point(xyz, spin):
    psi, Pi, Phi = inputs.kerr_schild(np.array(xyz, dtype=float).reshape(3, 1), 1.0, spin)
    return psi[:, :, 0], Pi[:, :, 0], Phi[:, :, :, 0]


def _normal(oracle, psi, s):
    ginv, lapse, shift, _ = oracle.geometry_point(psi)
    ginv = np.asarray(ginv).reshape(3, 3)
    nd = np.asarray(s) / np.sqrt(np.asarray(s) @ ginv @ np.asarray(s))
    return nd, ginv @ nd, float(lapse), np.asarray(shift)


@pytest.mark.parametrize("gamma", [(1.0, -1.0, 1.0), (3.0, -0.4, 2.0), (0.0, 0.0, 0.0)])
def test_characteristic_fields_are_eigenvectors_of_the_principal_part(oracle, gamma):
    rng = np.random.default_rng(3)
    psi, Pi, Phi = _point([2.3, -1.1, 0.7], 0.6)
    H, dH = rng.standard_normal(4), rng.standard_normal((3, 4))
    s = rng.standard_normal(3)
    nd, nu, N, shift = _normal(oracle, psi, s)
    nN = float(nd @ shift)
    speeds = {"0": -(1 + gamma[1]) * nN, "1p": -nN + N, "1m": -nN - N, "2": -nN}

    def principal(wpsi, wPi, wPhi):
        d = lambda w: np.stack([nd[k] * w for k in range(3)])                       # d_k u = n_k w
        a1 = oracle.rhs_point(psi, Pi, Phi, d(wpsi), d(wPi), np.stack([nd[k] * wPhi for k in range(3)]), H, dH, gamma)
        z = np.zeros((3, 4, 4))
        a0 = oracle.rhs_point(psi, Pi, Phi, z, z, np.zeros((3, 3, 4, 4)), H, dH, gamma)
        return [x - y for x, y in zip(a1, a0)]

    X = _full(rng.standard_normal(10))
    Y = np.stack([_full(rng.standard_normal(10)) for _ in range(3)])
    Y = Y - nd[:, None, None] * np.einsum("k,kab->ab", nu, Y)[None]                   # n^i Y_i = 0
    cases = {"1p": (0 * X, 0.5 * X, 0.5 * nd[:, None, None] * X), "1m": (0 * X, 0.5 * X, -0.5 * nd[:, None, None] * X),
             "2": (0 * X, 0 * X, Y), "0": (X, gamma[2] * X, 0 * Y)}
    for name, w in cases.items():
        got = principal(*w)
        for g, e in zip(got, w):
            assert np.max(np.abs(g + speeds[name] * e)) < 2e-13, name
    # and the oracle reports exactly these speeds
    _, _, _, sp = oracle.char_bc_point(psi, gamma, s, X, X, Y)
    assert np.allclose(sp, [speeds["0"], speeds["1p"], speeds["1m"], speeds["2"]], rtol=1e-14, atol=1e-15)


def test_freezing_acts_only_on_incoming_fields(oracle):
    rng = np.random.default_rng(9)
    gamma = (1.0, -0.3, 2.0)
    psi, _, _ = _point([2.6, 0.4, -0.9], 0.5)                # outside the horizon: u1- comes in through an outward normal
    s = np.array([2.6, 0.4, -0.9])
    nd, nu, N, shift = _normal(oracle, psi, s)
    a, b, c = _full(rng.standard_normal(10)), _full(rng.standard_normal(10)), np.stack([_full(rng.standard_normal(10)) for _ in range(3)])
    a2, b2, c2, sp = oracle.char_bc_point(psi, gamma, s, a, b, c)
    assert sp[1] > 0 and sp[2] < 0                              # v1+ out, v1- in

    def fields(dpsi, dPi, dPhi):
        nPhi = np.einsum("i,iab->ab", nu, dPhi)
        return dpsi, dPi + nPhi - gamma[2] * dpsi, dPi - nPhi - gamma[2] * dpsi, dPhi - nd[:, None, None] * nPhi[None]

    before, after = fields(a, b, c), fields(a2, b2, c2)
    for k, v in enumerate(sp):
        if v < 0:
            assert np.max(np.abs(after[k])) < 1e-14            # frozen
        else:
            assert np.max(np.abs(after[k] - before[k])) < 1e-14  # untouched
    # projecting twice changes nothing more
    a3, b3, c3, _ = oracle.char_bc_point(psi, gamma, s, a2, b2, c2)
    assert max(np.max(np.abs(a3 - a2)), np.max(np.abs(b3 - b2)), np.max(np.abs(c3 - c2))) < 1e-14


def test_excision_face_inside_the_horizon_needs_no_condition(oracle):
    """Schwarzschild in Kerr-Schild coordinates, r = 1.8 < 2M, outward normal of the inner face = -r^: every speed is >= 0, so the
    condition is the identity ('excision: nothing')."""
    rng = np.random.default_rng(1)
    x = np.array([1.8, 0.0, 0.0])
    psi, _, _ = _point(x, 0.0)
    a, b, c = _full(rng.standard_normal(10)), _full(rng.standard_normal(10)), np.stack([_full(rng.standard_normal(10)) for _ in range(3)])
    a2, b2, c2, sp = oracle.char_bc_point(psi, (1.0, -1.0, 1.0), -x, a, b, c)
    assert np.all(sp >= 0)
    assert max(np.max(np.abs(a2 - a)), np.max(np.abs(b2 - b)), np.max(np.abs(c2 - c))) < 1e-14
    # closed form there: n_k N^k = -sqrt(2M/r) / ... : v1- = sqrt(g^rr)(2M/r) ... - N;  check against N and N^r of the golden file
    N, Nr = (1 + 2 / 1.8) ** -0.5, (2 / 1.8) / (1 + 2 / 1.8)
    assert sp[2] == pytest.approx(Nr / np.sqrt(1 / (1 + 2 / 1.8)) - N, rel=1e-13)


def test_minkowski_speeds(oracle):
    eta = np.diag([-1.0, 1.0, 1.0, 1.0])
    z = np.zeros((4, 4))
    _, _, _, sp = oracle.char_bc_point(eta, (1.0, -1.0, 1.0), [1.0, 0.0, 0.0], z, z, np.zeros((3, 4, 4)))
    assert np.array_equal(sp, [0.0, 1.0, -1.0, 0.0]) or np.allclose(sp, [0.0, 1.0, -1.0, 0.0], atol=0)
