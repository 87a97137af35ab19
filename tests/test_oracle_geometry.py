"""Pins for oracle O4 (3+1 geometry from psi_ab) and for the analytic input generator itself."""
import numpy as np

from paper_1804_09101_b200 import inputs

PTS = np.array([[2.0, 0.3, -1.1], [-3.0, 2.5, 0.7], [0.4, -2.2, 2.9], [5.0, 5.0, 5.0]]).T  # [3,P]


def cstep(fun, xyz, h=1e-30):
    """exact first derivatives by the complex step: d_i f = Im f(x + i h e_i)/h"""
    out = []
    for i in range(3):
        z = xyz.astype(complex)
        z[i] += 1j * h
        out.append(np.imag(fun(z)) / h)
    return np.stack(out)


def test_schwarzschild_closed_forms(oracle):
    M = 1.3
    psi, Pi, Phi = inputs.kerr_schild(PTS, M, 0.0)
    r = np.sqrt((PTS**2).sum(0))
    for p in range(PTS.shape[1]):
        ginv, lapse, shift, psiinv = oracle.geometry_point(psi[:, :, p])
        assert abs(lapse - (1 + 2 * M / r[p]) ** -0.5) < 1e-15
        assert np.abs(shift - 2 * M * PTS[:, p] / (r[p] ** 2 * (1 + 2 * M / r[p]))).max() < 1e-15
        assert np.abs(psiinv @ psi[:, :, p] - np.eye(4)).max() < 1e-14
        assert np.abs(ginv @ psi[1:, 1:, p] - np.eye(3)).max() < 1e-14


def test_kerr_lapse_shift_and_inverse(oracle):
    for a in (0.5, 0.9):
        psi, Pi, Phi = inputs.kerr_schild(PTS, 1.0, a)
        N, Ni = inputs.kerr_schild_lapse_shift(PTS, 1.0, a)
        for p in range(PTS.shape[1]):
            ginv, lapse, shift, psiinv = oracle.geometry_point(psi[:, :, p])
            assert abs(lapse - N[p]) < 1e-15 and np.abs(shift - Ni[:, p]).max() < 1e-15
            assert np.abs(psiinv - np.linalg.inv(psi[:, :, p])).max() < 1e-13   # library inverse
            assert abs(np.linalg.det(psi[:, :, p]) + 1.0) < 1e-13              # Kerr-Schild: sqrt(-g) = 1


def test_input_generator_gradients_by_complex_step():
    """The analytic Phi_iab = d_i psi_ab coded in inputs.kerr_schild equals the complex-step derivative."""
    for a in (0.0, 0.5, 0.9):
        psi, Pi, Phi = inputs.kerr_schild(PTS, 1.0, a)
        d = cstep(lambda z: inputs.kerr_schild(z, 1.0, a)[0], PTS)
        assert np.abs(d - Phi).max() < 1e-14
        assert np.abs(psi - np.swapaxes(psi, 0, 1)).max() < 1e-15


def test_kerr_solves_defining_relations():
    """r solves the Kerr-Schild quartic, l is null w.r.t. eta, H is harmonic off the ring (Laplace H = 0)."""
    a = 0.7
    H, l, dH, dl = inputs._ks_scalars(PTS, 1.0, a)
    x, y, z = PTS
    r = z / l[3]
    assert np.abs((x * x + y * y) / (r * r + a * a) + z * z / (r * r) - 1).max() < 1e-14
    assert np.abs(l[1] ** 2 + l[2] ** 2 + l[3] ** 2 - 1).max() < 1e-14
    lap = sum(cstep(lambda zz, i=i: inputs._ks_scalars(zz, 1.0, a)[2][i], PTS)[i] for i in range(3))
    assert np.abs(lap).max() < 1e-13


def test_lapse_shift_gradient_identities(oracle):
    """SURVEY O4 pin: d_i N = -1/2 N t^c t^d Phi_icd and d_i N^k = N g^{jk} t^c Phi_ijc hold on spinning
    Kerr-Schild data (they are identities of the 3+1 split given Phi = d psi)."""
    a = 0.6
    psi, Pi, Phi = inputs.kerr_schild(PTS, 1.0, a)
    dN = cstep(lambda z: inputs.kerr_schild_lapse_shift(z, 1.0, a)[0], PTS)        # [i,P]
    dNk = cstep(lambda z: inputs.kerr_schild_lapse_shift(z, 1.0, a)[1], PTS)       # [i,k,P]
    for p in range(PTS.shape[1]):
        ginv, N, shift, psiinv = oracle.geometry_point(psi[:, :, p])
        t = np.array([1 / N, *(-shift / N)])
        for i in range(3):
            assert abs(dN[i, p] + 0.5 * N * t @ Phi[i, :, :, p] @ t) < 1e-14
            for k in range(3):
                rhs = N * sum(ginv[j, k] * (t @ Phi[i, j + 1, :, p]) for j in range(3))
                assert abs(dNk[i, k, p] - rhs) < 1e-14
