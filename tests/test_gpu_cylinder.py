"""GPU parity of the cylindrical-shell topology (GH_CYLINDER; reading S25) against oracle O15, element
by element: coordinates, gradient, RHS, RK3 step with fused norms, spectral filter, characteristic faces, the dual frame, and the
large-class path (an axis with N > 64, a Fourier axis with N_phi > 64) - next to shells and blocks in the same domain."""
import numpy as np
import pytest

from paper_1804_09101_b200 import configs, gh, inputs
from domain_util import assert_parity, build_case

pytestmark = pytest.mark.gpu
TOL = 1e-11


def _domain(descs, Hs, us):
    dom = gh.Domain(descs)
    dom.set_gauge_source(dom.pack(Hs))
    dom.set_fields(dom.pack(us), 0.0)
    return dom


def _frozen_mask(d):
    """points of a subdomain on a face flagged FROZEN (shells: 2 faces, cylinders: 4, blocks: 6), flat"""
    n = d["n"]
    dims = (n[0], n[1] + 1, 2 * n[1] + 2) if d["kind"] == "shell" else tuple(n)
    m = np.zeros(dims, bool)
    nf = {"shell": 2, "cylinder": 4, "block": 6}[d["kind"]]
    for f in range(nf):
        if d["face"][f] == 1:
            ix = [slice(None)] * 3
            ix[f // 2] = 0 if f % 2 == 0 else -1
            m[tuple(ix)] = True
    return m.ravel()


def _cfg(cid, faces=(0, 0, 0, 0)):
    return {"id": cid, "spin": 0.4, "amplitude": 1e-3,
            "descs": [configs.cylinder((9, 7, 12), 3.0, 6.0, -2.0, 1.5, face=faces, center=(0.2, -0.1, 0.3), gamma=[1.0, -0.6, 0.8]),
                      configs.shell(6, 7, 6.5, 9.0, face=(0, 1)),
                      configs.cylinder((5, 11, 7), 2.5, 4.0, 2.0, 5.0, face=faces),           # odd N_phi
                      configs.block([6, 5, 7], (8.0, -1.0, -1.0), (10.0, 1.0, 1.0)),
                      configs.cylinder((17, 4, 34), 4.0, 9.0, -1.0, 1.0, face=faces, gamma=[0.0, 0.0, 0.0])]}


def test_cylinder_coords_and_gradient(oracle):
    cfg = _cfg(61)
    descs, coords, us, Hs = build_case(cfg, oracle)
    dom = _domain(descs, Hs, us)
    xyz = dom.coords()
    g = dom.gradient()
    for s, d in enumerate(descs):
        sl = slice(dom.offsets[s], dom.offsets[s] + dom.sizes[s])
        assert np.max(np.abs(xyz[s] - coords[s])) < 1e-14 * 12.0, s
        ref = oracle.gradient(d, us[s])
        for k in range(3):
            err = float(np.max(np.abs(g[k][:, sl] - ref[k])))
            scale = max(float(np.max(np.abs(ref[k]))), float(np.max(np.abs(us[s]))))
            assert err <= TOL * scale, (s, k, err, scale)
    dom.close()


@pytest.mark.parametrize("faces", [(0, 0, 0, 0), (1, 0, 0, 1), (2, 2, 2, 2), (2, 1, 0, 2)])
def test_cylinder_rhs_step_and_norms(oracle, faces):
    """gh_rhs, gh_rk_step_norms and gh_constraint_norms with FREE, FROZEN and CHARACTERISTIC faces (edges where a rho face meets a
    z face included; a FROZEN face through an edge point wins)."""
    cfg = _cfg(62, faces)
    descs, coords, us, Hs = build_case(cfg, oracle)
    dom = _domain(descs, Hs, us)
    k = dom.unpack(dom.rhs())
    dt = 0.25 * configs.min_spacing(descs)
    norms = dom.rk_step_norms(dt)
    new = dom.unpack(dom.get_fields())
    for s, d in enumerate(descs):
        ref = oracle.rhs(d, us[s], Hs[s])
        assert_parity(k[s], ref, state=us[s], tol=TOL, what=f"cylinder cfg sub {s} rhs faces {faces}")
        fz = _frozen_mask(d)
        assert np.all(k[s][:, fz] == 0.0) and np.all(ref[:, fz] == 0.0)        # FROZEN faces: exactly zero
        assert fz.any() == (1 in d["face"][:4])
        assert_parity(new[s], oracle.rk3(d, us[s], Hs[s], dt, 1), tol=TOL, what=f"cylinder cfg sub {s} rk3 faces {faces}")
    ref = oracle.constraint_norms(descs, us, Hs)
    floor = 1e-11 * max(np.max(np.abs(u)) for u in us)
    assert np.all(np.abs(norms - ref) <= 1e-9 * np.abs(ref) + floor), (norms, ref)
    dom.set_fields(dom.pack(us), 0.0)
    alone = dom.constraint_norms()
    assert np.all(np.abs(alone - ref) <= 1e-9 * np.abs(ref) + floor), (alone, ref)
    dom.close()


def _sigma(f, kmax):
    k = np.arange(kmax + 1)
    if f["kind"] == "heaviside":
        return (k <= kmax - f["cut"]).astype(float)
    return np.exp(-f["alpha"] * (k / kmax) ** (2 * f["p"]))


@pytest.mark.parametrize("filt", [{"kind": "exp", "alpha": 36.0, "p": 6}, {"kind": "heaviside", "cut": 2}])
def test_cylinder_filter(oracle, filt):
    cfg = _cfg(63)
    descs, coords, us, Hs = build_case(cfg, oracle)
    dom = _domain(descs, Hs, us)
    dom.set_filter(block_axes=filt, shell_angular=filt)
    dom.apply_filter()
    got = dom.unpack(dom.get_fields())
    for s, d in enumerate(descs):
        n = d["n"]
        if d["kind"] == "shell":
            sig = [_sigma(filt, n[1])]
        elif d["kind"] == "cylinder":
            sig = [_sigma(filt, n[0] - 1), _sigma(filt, n[1] - 1), _sigma(filt, n[2] // 2)]
        else:
            sig = [_sigma(filt, m - 1) for m in n]
        ref = oracle.spectral_filter(d, us[s], sig)
        assert_parity(got[s], ref, tol=TOL, what=f"cylinder filter sub {s}")
        assert np.max(np.abs(ref - us[s])) > 0
    dom.close()


def test_cylinder_large_axes(oracle):
    """The K_gemm path on cylinders: a Chebyshev axis with N > 64 in rho and in z, and a Fourier axis with N_phi > 64 (unit stride,
    the matrix is the Fourier differentiation / filter matrix), each next to small axes; derivative, RHS, step and filter."""
    cfg = {"id": 64, "spin": 0.3, "amplitude": 1e-4,
           "descs": [configs.cylinder((80, 4, 6), 3.0, 9.0, -1.0, 1.0),
                     configs.cylinder((4, 96, 5), 3.0, 4.0, -4.0, 4.0, face=(0, 0, 1, 2)),
                     configs.cylinder((3, 4, 130), 4.0, 5.0, -1.0, 1.0),
                     configs.cylinder((5, 3, 75), 6.0, 8.0, 0.0, 1.0, face=(2, 1, 0, 0))]}
    descs, coords, us, Hs = build_case(cfg, oracle)
    dom = _domain(descs, Hs, us)
    g = dom.gradient()
    k = dom.unpack(dom.rhs())
    dt = 0.25 * configs.min_spacing(descs)
    dom.rk_step(dt)
    new = dom.unpack(dom.get_fields())

    def state_scale(got, ref, state, what):       # reading S15b: the large classes compare against the state-wide scale
        scale = max(float(np.max(np.abs(state))), float(np.max(np.abs(ref))))
        err = float(np.max(np.abs(got - ref)))
        assert err <= TOL * scale, f"{what}: max err {err:.3e} > {TOL:g} * {scale:.3e}"

    for s, d in enumerate(descs):
        sl = slice(dom.offsets[s], dom.offsets[s] + dom.sizes[s])
        ref = oracle.gradient(d, us[s])
        for a in range(3):
            state_scale(g[a][:, sl], ref[a], us[s], f"large cylinder sub {s} d_{a}")
        state_scale(k[s], oracle.rhs(d, us[s], Hs[s]), us[s], f"large cylinder sub {s} rhs")
        state_scale(new[s], oracle.rk3(d, us[s], Hs[s], dt, 1), us[s], f"large cylinder sub {s} rk3")
    filt = {"kind": "exp", "alpha": 36.0, "p": 6}
    dom.set_fields(dom.pack(us), 0.0)
    dom.set_filter(block_axes=filt)
    dom.apply_filter()
    got = dom.unpack(dom.get_fields())
    for s, d in enumerate(descs):
        n = d["n"]
        ref = oracle.spectral_filter(d, us[s], [_sigma(filt, n[0] - 1), _sigma(filt, n[1] - 1), _sigma(filt, n[2] // 2)])
        assert_parity(got[s], ref, tol=TOL, what=f"large cylinder filter sub {s}")
    dom.close()


def test_cylinder_dual_frame(oracle):
    """gh_set_frame_map on a cylinder (K_map_pre's A^-1 Jm A with the cylindrical Jacobian, K_map_post's v . A) against O14."""
    cfg = {"id": 65, "spin": 0.4, "amplitude": 1e-3,
           "descs": [configs.cylinder((7, 6, 10), 3.0, 6.0, -2.0, 1.5, face=(0, 1, 2, 0), center=(0.2, -0.1, 0.3), gamma=[1.0, -0.7, 0.5]),
                     configs.block([5, 6, 4], (7.0, -1.0, -2.0), (9.0, 1.0, 0.5))]}
    descs, coords, us, Hs = build_case(cfg, oracle)
    rng = np.random.default_rng(11)
    sh = 0.05 * rng.standard_normal((3, 3))
    Js, vs = [], []
    for xyz in coords:
        al = 0.2 + 0.01 * xyz[2]
        c, s_ = np.cos(al), np.sin(al)
        J = np.zeros((3, 3, xyz.shape[1]))
        J[0, 0], J[0, 1], J[1, 0], J[1, 1], J[2, 2] = c / 1.1, s_ / 1.1, -s_ / 1.1, c / 1.1, 1 / 1.05
        J += sh[:, :, None] * (1 + 0.1 * np.cos(xyz[1]))
        Js.append(J.reshape(9, -1))
        vs.append(np.stack([-0.3 * xyz[1] + 0.02 * xyz[0], 0.3 * xyz[0] + 0.02 * xyz[1], 0.01 * xyz[2] + 0.05]))
    dHs = [oracle.gradient(d, H).reshape(12, -1) for d, H in zip(descs, Hs)]        # [i][a], handed to both sides
    dom = gh.Domain(descs)
    dom.set_gauge_source(dom.pack(Hs), dom.pack(dHs))
    dom.set_fields(dom.pack(us), 0.0)
    single = dom.unpack(dom.rhs())
    dom.set_frame_map(dom.pack(Js), dom.pack(vs))
    k = dom.unpack(dom.rhs())
    for s, d in enumerate(descs):
        ref = oracle.rhs_map(d, us[s], Hs[s], dHs[s], Js[s], vs[s])
        assert_parity(k[s], ref, state=us[s], tol=TOL, what=f"cylinder dual frame sub {s}")
        assert np.max(np.abs(ref - single[s])) > 1e-3
    dom.close()
