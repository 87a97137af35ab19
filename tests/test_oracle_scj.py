"""Pins for oracle O13, SpatialCoordJac (NEXT-4; §3.3, Eqs. 9-11): the coordinate change of a tensor's
spatial indices only.  With Lambda = diag(1, J) the result is the tensor law T' = Lambda x ... x Lambda T, restated here with
numpy einsum on FULL arrays; the oracle itself follows the paper's order (purely spatial part first, then one index
timelike, ...) with successive single-index contractions."""
import os

import numpy as np
import pytest

from paper_1804_09101_b200 import inputs

RANK = {"a": 1, "aa": 2, "ab": 2, "abb": 3}
SYM = inputs.SYM_PAIRS            # the packed order 00,01,02,03,11,...


def _golden():
    out = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "opcount_spatialcoordjac.txt")) as f:
        for ln in f:
            if ln.strip() and not ln.startswith("#"):
                k, v = ln.split()
                out[k] = float(v)
    return out


def _rand_tensor(structure, rng):
    r = RANK[structure]
    T = rng.standard_normal((4,) * r)
    if structure == "aa":
        T = 0.5 * (T + T.T)
    if structure == "abb":
        T = 0.5 * (T + T.swapaxes(1, 2))
    return T


def _law(structure, J, T):
    Lam = np.eye(4)
    Lam[1:, 1:] = J
    r = RANK[structure]
    if r == 1:
        return np.einsum("ak,k->a", Lam, T)
    if r == 2:
        return np.einsum("ak,bl,kl->ab", Lam, Lam, T)
    return np.einsum("ak,bl,cm,klm->abc", Lam, Lam, Lam, T)


def _rot(axis, ang):
    c, s = np.cos(ang), np.sin(ang)
    i, j = [(1, 2), (2, 0), (0, 1)][axis]
    R = np.eye(3)
    R[i, i], R[i, j], R[j, i], R[j, j] = c, -s, s, c
    return R


@pytest.mark.parametrize("structure", ["a", "aa", "ab", "abb"])
def test_identity_rotation_general_and_composition(oracle, structure):
    rng = np.random.default_rng(42)
    T = _rand_tensor(structure, rng)
    out, _ = oracle.scj_point(structure, np.eye(3), T)
    assert np.array_equal(out, T)                                   # J = 1 is the identity
    R = _rot(2, 0.7) @ _rot(0, -1.1) @ _rot(1, 0.3)
    for J in (R, rng.standard_normal((3, 3))):                      # a rotation and a general (non-orthogonal, non-symmetric) J
        out, _ = oracle.scj_point(structure, J, T)
        ref = _law(structure, J, T)
        assert np.abs(out - ref).max() < 1e-14 * max(1.0, np.abs(ref).max())
        # a transposed Jacobian is a different result: the pin sees the index order of J_i^k
        assert np.abs(oracle.scj_point(structure, J.T, T)[0] - ref).max() > 1e-3
    J1, J2 = rng.standard_normal((3, 3)), rng.standard_normal((3, 3))
    two = oracle.scj_point(structure, J1, oracle.scj_point(structure, J2, T)[0])[0]
    one = oracle.scj_point(structure, J1 @ J2, T)[0]
    assert np.abs(two - one).max() < 1e-13 * np.abs(one).max()      # composition J1 o J2
    back = oracle.scj_point(structure, np.linalg.inv(J1), oracle.scj_point(structure, J1, T)[0])[0]
    assert np.abs(back - T).max() < 1e-12 * np.abs(T).max()


def test_time_components(oracle):
    """Eqs. 10-11 and the null-op: the purely timelike component is untouched; T'_0j sees only T_0l, T'_i0 only T_k0."""
    rng = np.random.default_rng(7)
    J = rng.standard_normal((3, 3))
    T = rng.standard_normal((4, 4))
    out, _ = oracle.scj_point("ab", J, T)
    assert out[0, 0] == T[0, 0]
    assert np.abs(out[0, 1:] - J @ T[0, 1:]).max() < 1e-15 and np.abs(out[1:, 0] - J @ T[1:, 0]).max() < 1e-15
    assert np.abs(out[1:, 1:] - J @ T[1:, 1:] @ J.T).max() < 1e-14   # Eq. 9
    G = T.copy()
    G[1:, 1:] = rng.standard_normal((3, 3)) * 100                   # garbage in the purely spatial block
    out2, _ = oracle.scj_point("ab", J, G)
    assert np.array_equal(out2[0, :], out[0, :]) and np.array_equal(out2[:, 0], out[:, 0])
    v = rng.standard_normal(4)
    o, _ = oracle.scj_point("a", J, v)
    assert o[0] == v[0] and np.abs(o[1:] - J @ v[1:]).max() < 1e-15
    T3 = rng.standard_normal((4, 4, 4))
    o3, _ = oracle.scj_point("abb", J, T3)
    assert o3[0, 0, 0] == T3[0, 0, 0]
    assert np.abs(o3[1:, 0, 0] - J @ T3[1:, 0, 0]).max() < 1e-15 and np.abs(o3[0, 0, 1:] - J @ T3[0, 0, 1:]).max() < 1e-15


def test_symmetry_is_preserved_not_assumed(oracle):
    rng = np.random.default_rng(9)
    J = rng.standard_normal((3, 3))
    o, _ = oracle.scj_point("aa", J, _rand_tensor("aa", rng))
    assert np.abs(o - o.T).max() < 1e-15
    o, _ = oracle.scj_point("abb", J, _rand_tensor("abb", rng))
    assert np.abs(o - o.swapaxes(1, 2)).max() < 1e-15
    # and an asymmetric input stays asymmetric (the evaluation does not symmetrise)
    A = rng.standard_normal((4, 4))
    o, _ = oracle.scj_point("aa", J, A)
    assert np.abs(o - _law("ab", J, A)).max() < 1e-14


def test_operation_counts_match_the_paper(oracle):
    """The instrumented count of the symmetry-free evaluation reproduces Eq. 13's printed values (15, 120); Eq. 12 enumerated
    over symmetry classes reproduces F_a, F_aa, F_ab; F_abb = 495 is the paper's printed sum 270 + F_ab + F_aa + 2 F_a."""
    g = _golden()
    rng = np.random.default_rng(1)
    J = rng.standard_normal((3, 3))
    assert oracle.scj_point("a", J, rng.standard_normal(4))[1] == g["F_a"]
    assert oracle.scj_point("ab", J, rng.standard_normal((4, 4)))[1] == g["F_ab"]
    d, r = 3, 3       # Eq. 13 for rank 3, no symmetry: (2d-1) sum_j C(r,j) d^(r-j) (r-j) = 720
    from math import comb
    assert oracle.scj_point("abb", J, rng.standard_normal((4, 4, 4)))[1] == (2 * d - 1) * sum(comb(r, j) * d ** (r - j) * (r - j) for j in range(r))
    assert oracle.scj_eq12("a") == g["F_a"] and oracle.scj_eq12("aa") == g["F_aa"] and oracle.scj_eq12("ab") == g["F_ab"]
    assert oracle.scj_eq12("abb") == g["F_abb_eq12_enumerated"]
    assert g["F_abb_purely_spatial_term"] + g["F_ab"] + g["F_aa"] + 2 * g["F_a"] == g["F_abb_printed"]
    for s in ("a", "aa", "ab"):
        assert oracle.scj_eq12(s) / g["M_" + s] == pytest.approx(g["I_" + s])
    assert g["F_abb_printed"] / g["M_abb"] == g["I_abb"]


def test_packed_arrays_and_state(oracle):
    """Packed [N_e][P] storage against the point-level law, and the 50-component state: psi, Pi as T_aa and
    Phi'_iab = J_i^k Lambda_a^c Lambda_b^d Phi_kcd."""
    rng = np.random.default_rng(3)
    P = 23
    J = rng.standard_normal((9, P))
    Lam = np.zeros((4, 4, P)); Lam[0, 0] = 1; Lam[1:, 1:] = J.reshape(3, 3, P)
    full2 = lambda t: np.array([[t[SYM.index((min(a, b), max(a, b)))] for b in range(4)] for a in range(4)])
    pack2 = lambda T: np.stack([T[a, b] for a, b in SYM])
    Ta = rng.standard_normal((4, P))
    assert np.abs(oracle.scj("a", J, Ta) - np.einsum("akp,kp->ap", Lam, Ta)).max() < 1e-14
    Tab = rng.standard_normal((16, P))
    ref = np.einsum("akp,blp,klp->abp", Lam, Lam, Tab.reshape(4, 4, P)).reshape(16, P)
    assert np.abs(oracle.scj("ab", J, Tab) - ref).max() < 1e-13
    Taa = rng.standard_normal((10, P))
    ref = pack2(np.einsum("akp,blp,klp->abp", Lam, Lam, full2(Taa)))
    assert np.abs(oracle.scj("aa", J, Taa) - ref).max() < 1e-13
    Tabb = rng.standard_normal((40, P))
    F3 = np.stack([full2(Tabb[10 * a:10 * a + 10]) for a in range(4)])
    R3 = np.einsum("akp,blp,cmp,klmp->abcp", Lam, Lam, Lam, F3)
    ref = np.concatenate([pack2(R3[a]) for a in range(4)])
    assert np.abs(oracle.scj("abb", J, Tabb) - ref).max() < 1e-13
    u = rng.standard_normal((50, P))
    out = oracle.scj_state(J, u)
    assert np.abs(out[:10] - pack2(np.einsum("akp,blp,klp->abp", Lam, Lam, full2(u[:10])))).max() < 1e-13
    assert np.abs(out[10:20] - pack2(np.einsum("akp,blp,klp->abp", Lam, Lam, full2(u[10:20])))).max() < 1e-13
    Phi = np.stack([full2(u[20 + 10 * i:30 + 10 * i]) for i in range(3)])
    Rp = np.einsum("ikp,blp,cmp,klmp->ibcp", J.reshape(3, 3, P), Lam, Lam, Phi)
    assert np.abs(out[20:] - np.concatenate([pack2(Rp[i]) for i in range(3)])).max() < 1e-13


def test_kerr_schild_is_axisymmetric(oracle):
    """A physical pin: Kerr-Schild data with the spin along z is axisymmetric, so the fields at the rotated point x' = R_z x are
    the SpatialCoordJac transform (J = R_z: covariant components, dx^k/dx'^i = R_ik) of the fields at x - for psi, Pi (T_aa)
    and Phi_iab (all three indices)."""
    rng = np.random.default_rng(5)
    x = rng.uniform(2.0, 4.0, (3, 11)) * np.sign(rng.standard_normal((3, 11)))
    R = _rot(2, 0.9)
    u = inputs.pack_fields(*inputs.kerr_schild(x, 1.0, 0.6))
    ur = inputs.pack_fields(*inputs.kerr_schild(R @ x, 1.0, 0.6))
    J = np.repeat(R.reshape(9, 1), x.shape[1], axis=1)
    out = oracle.scj_state(J, u)
    assert np.abs(out - ur).max() < 1e-13
    assert np.abs(u - ur).max() > 1e-2
