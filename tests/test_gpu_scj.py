"""GPU parity of SpatialCoordJac (NEXT-4; Eqs. 9-11) through the C ABI against oracle O13, element by element."""
import numpy as np
import pytest

from paper_1804_09101_b200 import configs, gh
from domain_util import build_case

pytestmark = pytest.mark.gpu

NE = {"a": 4, "aa": 10, "ab": 16, "abb": 40}
CODE = {"a": gh.GH_T_A, "aa": gh.GH_T_AA, "ab": gh.GH_T_AB, "abb": gh.GH_T_ABB}
TOL = 1e-11      # north_star's bar, scaled by the L-inf norm of the transformed tensor; the arithmetic is ~30 flop deep (measured ~1e-15)


def _jacobian(coords, seed):
    """a smooth, point-dependent, non-symmetric Jacobian field: rotation about z by an angle growing with r, times an
    anisotropic stretch, plus a seeded shear - the kind a rotating / expanding grid-to-inertial map gives"""
    rng = np.random.default_rng(seed)
    sh = 0.1 * rng.standard_normal((3, 3))
    out = []
    for xyz in coords:
        r = np.sqrt((xyz ** 2).sum(0))
        al = 0.3 + 0.05 * r
        c, s = np.cos(al), np.sin(al)
        J = np.zeros((3, 3, xyz.shape[1]))
        J[0, 0], J[0, 1], J[1, 0], J[1, 1], J[2, 2] = 1.1 * c, -1.1 * s, 0.9 * s, 0.9 * c, 1.0 + 0.01 * xyz[2]
        J += sh[:, :, None] * (1 + 0.1 * np.sin(xyz[0]))
        out.append(J.reshape(9, -1))
    return out


@pytest.fixture(scope="module")
def setup(oracle):
    cfg = {"id": 21, "spin": 0.3, "amplitude": 1e-3,
           "descs": [configs.shell(7, 5, 2.2, 4.0), configs.block([9, 6, 11], (3.0, -1.0, -2.0), (5.0, 1.5, 1.0)),
                     configs.shell(5, 9, 4.0, 9.0, center=(0.1, -0.2, 0.05))]}
    descs, coords, us, Hs = build_case(cfg, oracle)
    dom = gh.Domain(descs)
    Js = _jacobian(coords, 5)
    yield dom, descs, coords, us, Js
    dom.close()


@pytest.mark.parametrize("structure", ["a", "aa", "ab", "abb"])
def test_scj_parity(setup, oracle, structure):
    import torch
    dom, descs, coords, us, Js = setup
    rng = np.random.default_rng(17)
    Ts = [rng.standard_normal((NE[structure], c.shape[1])) for c in coords]
    Jp = dom.pack(Js)
    Jp[:, dom.offsets[0] + dom.sizes[0]:dom.offsets[1]] = np.nan          # padding of the Jacobian is never read
    dom.set_jacobian(Jp)
    T = dom.pack(Ts)
    out = np.full_like(T, 7.0)
    dom.spatial_coord_jac(CODE[structure], T, out)
    got = dom.unpack(out)
    for s in range(len(descs)):
        ref = oracle.scj(structure, Js[s], Ts[s])
        assert np.abs(got[s] - ref).max() <= TOL * np.abs(ref).max()
        assert np.abs(got[s] - ref).max() <= 1e-14 * np.abs(ref).max()       # what the arithmetic actually gives
        assert np.abs(ref - Ts[s]).max() > 0.1
    # device buffers, in place; padding entries are left untouched
    Td = torch.from_numpy(T).cuda()
    Td[:, dom.offsets[0] + dom.sizes[0]:dom.offsets[1]] = 5.0
    dom.spatial_coord_jac(CODE[structure], Td, Td)
    back = Td.cpu().numpy()
    for s in range(len(descs)):
        sl = slice(dom.offsets[s], dom.offsets[s] + dom.sizes[s])
        assert np.array_equal(back[:, sl], out[:, sl])
    assert np.all(back[:, dom.offsets[0] + dom.sizes[0]:dom.offsets[1]] == 5.0)


def test_scj_state_parity(setup, oracle):
    dom, descs, coords, us, Js = setup
    dom.set_jacobian(dom.pack(Js))
    dom.set_fields(dom.pack(us), 0.0)
    dom.spatial_coord_jac_state()
    got = dom.unpack(dom.get_fields())
    for s in range(len(descs)):
        ref = oracle.scj_state(Js[s], us[s])
        for sl in (slice(0, 10), slice(10, 20), slice(20, 50)):
            assert np.abs(got[s][sl] - ref[sl]).max() <= 1e-14 * np.abs(ref[sl]).max()
    # the inverse Jacobian brings the state back
    Jinv = [np.linalg.inv(J.reshape(3, 3, -1).transpose(2, 0, 1)).transpose(1, 2, 0).reshape(9, -1) for J in Js]
    dom.set_jacobian(dom.pack(Jinv))
    dom.spatial_coord_jac_state()
    back = dom.unpack(dom.get_fields())
    for s in range(len(descs)):
        assert np.abs(back[s] - us[s]).max() <= 1e-12 * np.abs(us[s]).max()


def test_scj_errors():
    dom = gh.Domain(configs.c1()["descs"])
    T = np.zeros((10, dom.S))
    with pytest.raises(gh.GHError) as e:
        dom.spatial_coord_jac(gh.GH_T_AA, T)
    assert e.value.status == gh.GH_ERR_STATE
    dom.set_jacobian(np.zeros((9, dom.S)))
    with pytest.raises(gh.GHError) as e:
        dom.spatial_coord_jac(7, T)
    assert e.value.status == gh.GH_ERR_ARG
    with pytest.raises(gh.GHError) as e:
        dom.spatial_coord_jac_state()
    assert e.value.status == gh.GH_ERR_STATE
    dmma, dfma = dom.fp64_peak()
    assert 10.0 < dfma < 60.0 and 10.0 < dmma < 60.0       # a B200 gives ~34 / ~37 TFLOP/s
    dom.close()
