"""GPU parity of the LARGE subdomain classes (Chebyshev axes with N > 64, shells with L > 47: the K_gemm path that carries the
upper two decades of the size sweep, BASELINE.json configs[4]) against the long-double oracle.  Thin subdomains keep the
oracle's cost in seconds while every tile count, the ragged tails and the class limits are exercised; the full-size members
of the sweep are compared on sampled planes and lines (test_c5_top_sampled)."""
import numpy as np
import pytest

from paper_1804_09101_b200 import configs, gh, inputs
from domain_util import assert_parity, build_case

pytestmark = pytest.mark.gpu
TOL = 1e-11


def assert_parity_state_scale(got, ref, state, what):
    """Reading S15b, large classes only: per field X in (psi, Pi, Phi), max |gpu - oracle| <= 1e-11 * max over ALL
    50 components of (|state|, |oracle result|).  d_t Pi and d_t Phi contain spectral derivatives of psi; in FP64 those carry a
    rounding floor eps ||D||inf (2/Delta) ||psi||inf, with ||D||inf ~ N^2 (N = 150: 2e4; N = 320: 1e5), which
    exceeds 1e-11 ||Pi||inf once ||Pi||inf << ||psi||inf (far from the hole: 0.02 against 0.8) - the per-field scale of S15 is
    below the rounding floor of the arithmetic at these sizes, the state-wide one is not."""
    scale = max(float(np.max(np.abs(state))), float(np.max(np.abs(ref))))
    for name, sl in (("psi", slice(0, 10)), ("Pi", slice(10, 20)), ("Phi", slice(20, 50))):
        err = float(np.max(np.abs(got[sl] - ref[sl])))
        assert err <= TOL * scale, f"{what} field {name}: max err {err:.3e} > {TOL:g} * {scale:.3e}"


def _domain(descs, Hs, us):
    dom = gh.Domain(descs)
    dom.set_gauge_source(dom.pack(Hs))
    dom.set_fields(dom.pack(us), 0.0)
    return dom


def _check_all(oracle, cfg, what, rk=True, ncomp_grad=50):
    descs, coords, us, Hs = build_case(cfg, oracle)
    dom = _domain(descs, Hs, us)
    g = dom.gradient()
    for s, d in enumerate(descs):
        ref = oracle.gradient(d, us[s][:ncomp_grad])
        got = g[:, :ncomp_grad, dom.offsets[s]:dom.offsets[s] + dom.sizes[s]]
        for k in range(3):
            assert_parity_rows(got[k], ref[k], us[s][:ncomp_grad], f"{what} sub {s} d_{k}")
    if rk:
        k = dom.unpack(dom.rhs())
        dt = 0.25 * configs.min_spacing(descs)
        norms = dom.rk_step_norms(dt)
        new = dom.unpack(dom.get_fields())
        for s, d in enumerate(descs):
            assert_parity_state_scale(k[s], oracle.rhs(d, us[s], Hs[s]), us[s], f"{what} sub {s} rhs")
            assert_parity_state_scale(new[s], oracle.rk3(d, us[s], Hs[s], dt, 1), us[s], f"{what} sub {s} rk3")
        ref = oracle.constraint_norms(descs, us, Hs)
        floor = 1e-11 * max(np.max(np.abs(u)) for u in us)
        assert np.all(np.abs(norms - ref) <= 1e-9 * np.abs(ref) + floor), (norms, ref)
    dom.close()


def assert_parity_rows(got, ref, state, what):
    """gradient rows of any subset of components: error against 1e-11 * max(||u||inf, ||d u||inf) over those components"""
    err = float(np.max(np.abs(got - ref)))
    scale = max(float(np.max(np.abs(ref))), float(np.max(np.abs(state))))
    assert err <= TOL * scale, f"{what}: max err {err:.3e} > {TOL:g} * {scale:.3e}"


def test_large_chebyshev_axes(oracle):
    """N just above the small-class limit (65), one and two M-blocks and ragged K-chunks (80, 96, 130, 150) on each of the three
    axes (strided, strided with an outer index, unit stride), next to small axes; a shell with a large radial axis."""
    cfg = {"id": 31, "spin": 0.4, "amplitude": 1e-4,
           "descs": [configs.block([80, 5, 6], (3.0, -1.0, -2.0), (6.0, 1.5, 1.0), face=(0, 1, 0, 0, 1, 0)),
                     configs.block([4, 96, 3], (-1.0, 3.0, -1.0), (1.0, 7.0, 1.0)),
                     configs.block([3, 5, 130], (3.0, 3.0, -2.0), (4.0, 4.0, 2.0), gamma=[0.5, -0.3, 0.7]),
                     configs.block([65, 2, 150], (5.0, 3.0, -2.0), (7.0, 4.0, 2.0), face=(2, 1, 0, 0, 0, 2)),
                     configs.shell(70, 4, 2.0, 9.0, face=(0, 1))]}
    _check_all(oracle, cfg, "large N")


def test_large_shells(oracle):
    """L just above the small-class limit (48: odd n_theta, ragged everything), L = 63 (n_theta = 64: exact tiles) and L = 70 with a
    large radial axis as well, next to a small shell and a block in the same domain."""
    cfg = {"id": 32, "spin": 0.3, "amplitude": 1e-4,
           "descs": [configs.shell(3, 48, 2.5, 3.5, face=(1, 0)),
                     configs.shell(5, 12, 3.5, 6.0),
                     configs.shell(2, 63, 6.0, 9.0, gamma=[2.0, -0.5, 1.5], center=(0.1, -0.2, 0.05)),
                     configs.block([6, 7, 5], (10.0, -1.0, -1.0), (12.0, 1.0, 1.0))]}
    _check_all(oracle, cfg, "large L")


def test_sweep_sizes_thin(oracle):
    """The sizes of the sweep's upper members on thin subdomains: N = 128 and 320 on each axis, L = 127 (n = 128), and a 72^3 cube
    (every axis large at once, 373 k points); gradient on every component, RHS / RK3 / fused norms on the thin ones."""
    cfg = {"id": 33, "spin": 0.5, "amplitude": 1e-4,
           "descs": [configs.block([320, 4, 4], (3.0, -1.0, -1.0), (11.0, 1.0, 1.0)),
                     configs.block([4, 128, 3], (3.0, -4.0, -1.0), (5.0, 4.0, 1.0)),
                     configs.block([3, 4, 320], (3.0, -1.0, -4.0), (5.0, 1.0, 4.0))]}
    _check_all(oracle, cfg, "sweep sizes")
    # the oracle's Y_lm quadruple loops cost ~3 s per plane at L = 127: gradient only, 16 components (one per host core)
    shell = {"id": 35, "spin": 0.5, "amplitude": 1e-4, "descs": [configs.shell(2, 127, 3.0, 4.0)]}
    _check_all(oracle, shell, "L = 127 shell", rk=False, ncomp_grad=16)
    cube = {"id": 34, "spin": 0.5, "amplitude": 1e-4, "descs": [configs.block(72, (3.0, -4.0, -4.0), (11.0, 4.0, 4.0))]}
    _check_all(oracle, cube, "72^3 cube", rk=False, ncomp_grad=8)


def test_limits_and_rejections():
    gh.Domain([configs.shell(2, 255, 3.0, 4.0)]).close()                       # GH_MAX_L
    with pytest.raises(gh.GHError):
        gh.Domain([configs.shell(4, 256, 3.0, 4.0)])
    with pytest.raises(gh.GHError):
        gh.Domain([configs.block([513, 4, 4], (0, 0, 0), (1, 1, 1))])
    dom = gh.Domain([configs.block([80, 4, 4], (3, 0, 0), (4, 1, 1))])
    with pytest.raises(gh.GHError) as e:                                        # the filter is built for the small classes only
        dom.set_filter(block_axes={"kind": "exp", "alpha": 36.0, "p": 6})
    assert e.value.status == gh.GH_ERR_ARG
    dom.close()
