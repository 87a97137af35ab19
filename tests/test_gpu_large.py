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


def _sigma(f, kmax):
    k = np.arange(kmax + 1)
    if f["kind"] == "heaviside":
        return (k <= kmax - f["cut"]).astype(float)
    return np.exp(-f["alpha"] * (k / kmax) ** (2 * f["p"]))


@pytest.mark.parametrize("filt", [{"kind": "exp", "alpha": 36.0, "p": 6}, {"kind": "heaviside", "cut": 3}])
def test_large_filter(oracle, filt):
    """gh_apply_filter on the large classes (the filter matrices through K_gemm) against the oracle's modal filter (O9): blocks
    with one large axis in each position next to small axes (the three passes share the scratch slots with the small-class
    kernel), a block with two large axes, shells with L = 48 and 63, a small shell and a shell whose radial axis alone is large
    (the filter leaves the radial direction alone)."""
    cfg = {"id": 36, "spin": 0.4, "amplitude": 1e-4,
           "descs": [configs.block([80, 5, 6], (3.0, -1.0, -2.0), (6.0, 1.5, 1.0)),
                     configs.block([4, 96, 3], (-1.0, 3.0, -1.0), (1.0, 7.0, 1.0)),
                     configs.block([3, 5, 130], (3.0, 3.0, -2.0), (4.0, 4.0, 2.0)),
                     configs.block([65, 2, 150], (5.0, 3.0, -2.0), (7.0, 4.0, 2.0)),
                     configs.block([6, 7, 5], (10.0, -1.0, -1.0), (12.0, 1.0, 1.0)),
                     configs.shell(3, 48, 2.5, 3.5, face=(1, 0)),
                     configs.shell(5, 12, 3.5, 6.0),
                     configs.shell(2, 63, 6.0, 9.0),
                     configs.shell(70, 4, 9.0, 12.0, face=(0, 1))]}
    descs, coords, us, Hs = build_case(cfg, oracle)
    dom = _domain(descs, Hs, us)
    dom.set_filter(block_axes=filt, shell_angular=filt)
    dom.apply_filter()
    got = dom.unpack(dom.get_fields())
    for s, d in enumerate(descs):
        if d["kind"] == "shell":
            ref = oracle.spectral_filter(d, us[s], [_sigma(filt, d["n"][1])])
        else:
            ref = oracle.spectral_filter(d, us[s], [_sigma(filt, n - 1) for n in d["n"]])
        assert_parity(got[s], ref, tol=TOL, what=f"large filter sub {s}")
        assert np.max(np.abs(ref - us[s])) > 0
    # one family off: its subdomains stay bit-identical; a second application after re-setting the state gives the same bits
    first = dom.get_fields().copy()
    dom.set_fields(dom.pack(us), 0.0)
    dom.apply_filter()
    assert np.array_equal(dom.get_fields(), first)
    dom.set_fields(dom.pack(us), 0.0)
    dom.set_filter(block_axes=filt, shell_angular=None)
    dom.apply_filter()
    got = dom.unpack(dom.get_fields())
    for s, d in enumerate(descs):
        if d["kind"] == "shell":
            assert np.array_equal(got[s], us[s])
    dom.close()


# ---- the sweep's large members at FULL size, on sampled outputs the oracle computes one by one --------------------------------
def _full(t10):
    """packed symmetric [10, ...] -> full [4, 4, ...]"""
    return np.array([[t10[inputs.SYM_PAIRS.index((min(a, b), max(a, b)))] for b in range(4)] for a in range(4)])


def _sampled_member(oracle, cfg, n_pts=48, comps=(0, 5, 13, 24, 37, 49)):
    """One sweep member at full size in the launch configuration bench.py --workload c5 times.  (1) The spectral Cartesian gradient
    against the oracle on sampled planes (shell: the Y_lm double sums of whole (theta,phi) planes, O2) and sampled lines (the modal
    Chebyshev derivative, O1), assembled with Eq. 8 at the sampled points.  (2) gh_rhs at sampled points against the oracle's
    pointwise RHS (O5) fed with the state and the library's own gradient there (the pointwise algebra at full size; the
    gradient itself is what (1) checks).  The gauge source's gradient is supplied to both sides (complex-step analytic)."""
    import torch
    from concurrent.futures import ThreadPoolExecutor

    d = cfg["descs"][0]
    dom = gh.Domain([d])
    P, S = dom.P, dom.S
    xyz = np.zeros((3, S)); gh.gh_domain_coords(dom.h, xyz)
    u = np.zeros((50, S)); H = np.zeros((4, S)); dH = np.zeros((12, S))
    inputs.initial_data_chunked(d, xyz[:, :P], cfg["spin"], cfg["amplitude"], cfg["id"], 0, u[:, :P], H[:, :P])
    hstep = 1e-30
    for p0 in range(0, P, 1 << 20):                     # d_i H_a analytically (complex step), chunked
        sl = slice(p0, min(P, p0 + (1 << 20)))
        for i in range(3):
            z = xyz[:, sl].astype(complex); z[i] += 1j * hstep
            dH[4 * i:4 * i + 4, sl] = np.imag(inputs.kerr_schild_gauge_source(z, 1.0, cfg["spin"])) / hstep
    dom.set_gauge_source(H, dH)
    dom.set_fields(u, 0.0)
    g = dom.empty(3, 50)
    dom.gradient(g)
    k = dom.empty(50)
    dom.rhs(k)
    torch.cuda.synchronize()
    rng = np.random.default_rng(99)
    n0, n1, n2 = (d["n"][0], d["n"][1] + 1, 2 * d["n"][1] + 2) if d["kind"] == "shell" else d["n"]
    scale_u = float(np.abs(u).max())
    worst = 0.0
    if d["kind"] == "shell":
        L = d["n"][1]
        th, _ = oracle.gl_nodes(L)
        lo, hi = d["lo"][0], d["hi"][0]
        xr = oracle.cheb_nodes(n0)
        planes = [0, n0 // 2]
        jk = [(int(j), int(kk)) for j, kk in zip(rng.integers(0, n1, n_pts), rng.integers(0, n2, n_pts))]
        with ThreadPoolExecutor(8) as ex:                # the oracle's plane transform releases the GIL (ctypes)
            ang = list(ex.map(lambda a: oracle.shell_angular(L, u[a[1], :P].reshape(n0, n1, n2)[a[0]]), [(i, c) for i in planes for c in comps]))
        it = iter(ang)
        for i in planes:
            r = lo + (hi - lo) * (xr[i] + 1) / 2
            for c in comps:
                dth, dph = next(it)
                uc = u[c, :P].reshape(n0, n1, n2)
                gg = g[:, c, :P].reshape(3, n0, n1, n2)[:, i].cpu().numpy()
                for j, kk in jk:
                    dr = oracle.cheb_derivative_line(np.ascontiguousarray(uc[:, j, kk]))[i] * 2 / (hi - lo)
                    st, ct, ph = np.sin(th[j]), np.cos(th[j]), 2 * np.pi * kk / n2
                    cp, sp = np.cos(ph), np.sin(ph)
                    ref = np.array([st * cp * dr + ct * cp / r * dth[j, kk] - sp / (r * st) * dph[j, kk],
                                    st * sp * dr + ct * sp / r * dth[j, kk] + cp / (r * st) * dph[j, kk],
                                    ct * dr - st / r * dth[j, kk]])
                    err = np.abs(gg[:, j, kk] - ref).max()
                    sc = max(scale_u, np.abs(ref).max())
                    worst = max(worst, err / sc)
                    assert err <= TOL * sc, f"{d['n']} plane {i} comp {c} point ({j},{kk}): {err:.3e} > {TOL:g} * {sc:.3e}"
    else:
        strides = (n1 * n2, n2, 1)
        for axis in range(3):
            for _ in range(n_pts // 3):
                idx = [int(rng.integers(0, n)) for n in (n0, n1, n2)]
                idx[axis] = 0
                base = idx[0] * strides[0] + idx[1] * strides[1] + idx[2] * strides[2]
                line = base + np.arange(d["n"][axis]) * strides[axis]
                for c in comps:
                    ref = oracle.cheb_derivative_line(np.ascontiguousarray(u[c, line])) * 2 / (d["hi"][axis] - d["lo"][axis])
                    got = g[axis, c, torch.from_numpy(line).cuda()].cpu().numpy()
                    err = np.abs(got - ref).max()
                    sc = max(scale_u, np.abs(ref).max())
                    worst = max(worst, err / sc)
                    assert err <= TOL * sc, f"{d['n']} axis {axis} comp {c}: {err:.3e} > {TOL:g} * {sc:.3e}"
    # (2) pointwise RHS at sampled points
    pts = rng.integers(0, P, 64)
    gs = g[:, :, torch.from_numpy(pts).cuda()].cpu().numpy()        # [3, 50, n]
    ks = k[:, torch.from_numpy(pts).cuda()].cpu().numpy()
    frozen = np.zeros(len(pts), bool)
    i0 = pts // (n1 * n2)
    if d["kind"] == "shell":
        frozen = ((i0 == 0) & (d["face"][0] == 1)) | ((i0 == n0 - 1) & (d["face"][1] == 1))
    for q, p in enumerate(pts):
        psi, Pi = _full(u[0:10, p]), _full(u[10:20, p])
        Phi = np.array([_full(u[20 + 10 * i:30 + 10 * i, p]) for i in range(3)])
        dpsi = np.array([_full(gs[kk, 0:10, q]) for kk in range(3)])
        dPi = np.array([_full(gs[kk, 10:20, q]) for kk in range(3)])
        dPhi = np.array([[_full(gs[kk, 20 + 10 * i:30 + 10 * i, q]) for i in range(3)] for kk in range(3)])
        o = oracle.rhs_point(psi, Pi, Phi, dpsi, dPi, dPhi, H[:, p], dH[:, p].reshape(3, 4), d["gamma"])
        ref = inputs.pack_fields(o[0][..., None], o[1][..., None], o[2][..., None])[:, 0]
        if frozen[q]:
            ref = np.zeros(50)
        err = np.abs(ks[:, q] - ref).max()
        sc = max(scale_u, np.abs(ref).max())
        assert err <= TOL * sc, f"{d['n']} rhs at point {p}: {err:.3e} > {TOL:g} * {sc:.3e}"
    dom.close()
    return worst


def test_c5_members_full_size_sampled(oracle):
    """c5_shell(128) (4.2 M points, L = 127) and c5_block(160) (4.1 M points): the two members in the middle of the sweep's large range."""
    for cfg in (configs.c5_shell(128), configs.c5_block(160)):
        _sampled_member(oracle, cfg)


import os


@pytest.mark.skipif(not os.environ.get("GH_LONG_TESTS"), reason="the 3.3e7-point members: ~15 minutes of input generation and oracle planes; set GH_LONG_TESTS=1")
def test_c5_top_members_full_size_sampled(oracle):
    """The top of BASELINE.json configs[4]: c5_shell(256) (L = 255, 3.36e7 points) and c5_block(320) (3.28e7 points)."""
    for cfg in (configs.c5_shell(256), configs.c5_block(320)):
        w = _sampled_member(oracle, cfg, n_pts=24, comps=(0, 13, 37))
        print(f"{cfg['descs'][0]['n']}: worst gradient gap / scale = {w:.3e}")
