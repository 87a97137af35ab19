"""GPU parity of the dual-frame right-hand side (NEXT-4; gh_set_frame_map) against oracle O14, element by element."""
import numpy as np
import pytest

from paper_1804_09101_b200 import configs, gh, inputs
from domain_util import assert_parity, build_case

pytestmark = pytest.mark.gpu
TOL = 1e-11


def _cstep(fun, xyz, h=1e-30):
    out = []
    for i in range(3):
        z = xyz.astype(complex)
        z[i] += 1j * h
        out.append(np.imag(fun(z)) / h)
    return np.stack(out)


def _map_fields(coords, seed):
    """a rotating, expanding, slightly sheared grid: Jm = d xbar / d x and the grid velocity v at the grid points"""
    rng = np.random.default_rng(seed)
    sh = 0.05 * rng.standard_normal((3, 3))
    Js, vs = [], []
    for xyz in coords:
        al = 0.2 + 0.01 * xyz[2]
        c, s = np.cos(al), np.sin(al)
        J = np.zeros((3, 3, xyz.shape[1]))
        J[0, 0], J[0, 1], J[1, 0], J[1, 1], J[2, 2] = c / 1.1, s / 1.1, -s / 1.1, c / 1.1, 1 / 1.05
        J += sh[:, :, None] * (1 + 0.1 * np.cos(xyz[1]))
        Js.append(J.reshape(9, -1))
        vs.append(np.stack([-0.3 * xyz[1] + 0.02 * xyz[0], 0.3 * xyz[0] + 0.02 * xyz[1], 0.01 * xyz[2] + 0.05]))
    return Js, vs


def test_dual_frame_parity(oracle):
    cfg = {"id": 51, "spin": 0.4, "amplitude": 1e-3,
           "descs": [configs.shell(7, 6, 2.2, 4.0, face=(0, 1), gamma=[1.0, -1.0, 1.0]),
                     configs.block([7, 6, 8], (3.0, -1.0, -2.0), (5.0, 1.0, 0.5), face=(1, 0, 0, 2, 0, 0), gamma=[1.0, -0.7, 0.5]),
                     configs.shell(5, 9, 4.0, 9.0, face=(2, 0), center=(0.1, -0.2, 0.05), gamma=[2.0, -0.4, 1.5])]}
    descs, coords, us, Hs = build_case(cfg, oracle)
    dHs = [_cstep(lambda z: inputs.kerr_schild_gauge_source(z, 1.0, cfg["spin"]), xyz).reshape(12, -1) for xyz in coords]
    Js, vs = _map_fields(coords, 6)
    dom = gh.Domain(descs)
    dom.set_gauge_source(dom.pack(Hs), dom.pack(dHs))
    dom.set_fields(dom.pack(us), 0.0)
    single = dom.unpack(dom.rhs())
    dom.set_frame_map(dom.pack(Js), dom.pack(vs))
    k = dom.unpack(dom.rhs())
    dt = 0.25 * configs.min_spacing(descs)
    dom.rk_step(dt)
    new = dom.unpack(dom.get_fields())
    dom.set_fields(dom.pack(us), 0.0)
    n_fused = dom.rk_step_norms(dt)
    assert np.array_equal(dom.get_fields(), dom.pack(new))
    dom.set_fields(dom.pack(us), 0.0)
    n_alone = dom.constraint_norms()
    floor = 1e-11 * max(np.max(np.abs(u)) for u in us)
    assert np.all(np.abs(n_fused - n_alone) <= 1e-12 * np.abs(n_alone) + floor)
    for s, d in enumerate(descs):
        ref = oracle.rhs_map(d, us[s], Hs[s], dHs[s], Js[s], vs[s])
        assert_parity(k[s], ref, state=us[s], tol=TOL, what=f"dual frame sub {s} rhs")
        assert np.max(np.abs(ref - single[s])) > 1e-3                       # the map really acts
        assert np.array_equal(k[s] == 0.0, ref == 0.0) or np.all((ref == 0.0) <= (k[s] == 0.0))      # FROZEN faces: exactly zero
        ref_u = oracle.rhs_map(d, us[s], Hs[s], dHs[s], Js[s], vs[s], dt=dt, nsteps=1)
        assert_parity(new[s], ref_u, tol=TOL, what=f"dual frame sub {s} rk3")
    # the identity map with zero velocity, and switching the map off, both give the single-frame bits back
    eye = [np.repeat(np.eye(3).reshape(9, 1), c.shape[1], axis=1) for c in coords]
    dom.set_frame_map(dom.pack(eye), dom.pack([np.zeros((3, c.shape[1])) for c in coords]))
    ident = dom.unpack(dom.rhs())
    dom.set_frame_map(None, None)
    off = dom.unpack(dom.rhs())
    for s in range(len(descs)):
        assert np.array_equal(off[s], single[s])
        assert_parity(ident[s], single[s], state=us[s], tol=1e-14, what=f"identity map sub {s}")
    with pytest.raises(gh.GHError):
        dom.set_frame_map(dom.pack(eye), None)
    dom.close()
