"""Pins of the oracle's characteristic penalty exchange across shell interfaces (O12, NEXT-2 (iii), reading
S22).  The condition is defined on characteristic fields, so it is pinned by projecting what it adds to the right-hand side
back onto those fields (whose form and speeds test_oracle_charbc.py pins against the RHS itself)."""
import numpy as np

from paper_1804_09101_b200 import configs, inputs


def _full(v10):
    m = np.zeros(v10.shape[1:] + (4, 4)) if v10.ndim > 1 else np.zeros((4, 4))
    for s, (a, b) in enumerate(inputs.SYM_PAIRS):
        m[..., a, b] = v10[s]
        m[..., b, a] = v10[s]
    return m


def _setup(oracle, face):
    sd = configs.shell(6, 5, 2.4, 4.0, face=face, gamma=[1.5, -0.6, 2.0])
    xyz = oracle.coords(sd)
    (u,), (H,) = inputs.initial_data([sd], [xyz], 0.4, 1e-3, 21)
    return sd, xyz, u, H


def test_equal_states_on_both_sides_change_nothing(oracle):
    sd, xyz, u, H = _setup(oracle, (3, 3))
    free = dict(sd, face=[0, 0, 0, 0, 0, 0])
    pl = 6 * 12
    ref = oracle.rhs(free, u, H)
    got = oracle.rhs_ifc(sd, u, H, nbr_in=u[:, :pl].copy(), nbr_out=u[:, -pl:].copy())
    assert np.array_equal(got, ref)
    # and without neighbour data an interface face is a free face
    assert np.array_equal(oracle.rhs_ifc(sd, u, H), ref)


def test_only_incoming_fields_are_penalised_with_p_times_speed(oracle):
    sd, xyz, u, H = _setup(oracle, (0, 3))
    free = dict(sd, face=[0, 0, 0, 0, 0, 0])
    pl, P = 6 * 12, u.shape[1]
    rng = np.random.default_rng(4)
    nbr = u[:, -pl:] + 1e-3 * rng.standard_normal((50, pl))
    dk = oracle.rhs_ifc(sd, u, H, nbr_out=nbr) - oracle.rhs(free, u, H)
    assert np.max(np.abs(dk[:, :-pl])) == 0.0                       # only the outer face moves
    g1, g2 = sd["gamma"][1], sd["gamma"][2]
    pen = (6 - 1) ** 2 / (4.0 - 2.4)
    worst = 0.0
    for q in range(0, pl, 7):
        p = P - pl + q
        psi = _full(u[0:10, p])
        ginv, N, shift, _ = oracle.geometry_point(psi)
        ginv, shift = np.asarray(ginv).reshape(3, 3), np.asarray(shift)
        s = xyz[:, p] / np.linalg.norm(xyz[:, p])
        nd = s / np.sqrt(s @ ginv @ s); nu = ginv @ nd; nN = nd @ shift
        v = {"0": -(1 + g1) * nN, "1p": -nN + N, "1m": -nN - N, "2": -nN}

        def fields(x):      # x[50] -> characteristic fields
            ps, Pi = _full(x[0:10]), _full(x[10:20])
            Ph = np.stack([_full(x[20 + 10 * i:30 + 10 * i]) for i in range(3)])
            nPh = np.einsum("i,iab->ab", nu, Ph)
            return {"0": ps, "1p": Pi + nPh - g2 * ps, "1m": Pi - nPh - g2 * ps, "2": Ph - nd[:, None, None] * nPh[None]}

        du, dd = fields(u[:, p] - nbr[:, q]), fields(dk[:, p])
        for name in v:
            want = pen * v[name] * du[name] if v[name] < 0 else 0.0 * du[name]
            worst = max(worst, float(np.max(np.abs(dd[name] - want))))
        assert v["1m"] < 0 < v["1p"]
    assert worst < 1e-14


def test_every_field_is_penalised_on_exactly_one_side(oracle):
    """the neighbour sees the opposite normal: v0 -> -v0, v1+- -> -v1-+, v2 -> -v2, so what leaves one side enters the other"""
    psi = _full(inputs.pack_fields(*inputs.kerr_schild(np.array([[2.9], [0.3], [-0.8]]), 1.0, 0.5))[0:10, 0])
    z, z3 = np.zeros((4, 4)), np.zeros((3, 4, 4))
    s = np.array([2.9, 0.3, -0.8])
    _, _, _, va = oracle.char_bc_point(psi, (1.0, -0.5, 1.0), s, z, z, z3)
    _, _, _, vb = oracle.char_bc_point(psi, (1.0, -0.5, 1.0), -s, z, z, z3)
    assert np.allclose(vb, [-va[0], -va[2], -va[1], -va[3]], rtol=1e-14)


def test_analytic_data_is_continuous_across_the_interface(oracle):
    """two adjacent shells carrying the same analytic Kerr-Schild data: the face states coincide, the exchange adds nothing"""
    a = configs.shell(6, 5, 2.0, 3.0, face=(0, 3))
    b = configs.shell(7, 5, 3.0, 5.0, face=(3, 0))
    pl = 6 * 12
    ua = inputs.pack_fields(*inputs.kerr_schild(oracle.coords(a), 1.0, 0.3))
    ub = inputs.pack_fields(*inputs.kerr_schild(oracle.coords(b), 1.0, 0.3))
    assert np.max(np.abs(ua[:, -pl:] - ub[:, :pl])) < 2e-15
    Ha = inputs.kerr_schild_gauge_source(oracle.coords(a), 1.0, 0.3)
    free = dict(a, face=[0, 0, 0, 0, 0, 0])
    d = oracle.rhs_ifc(a, ua, Ha, nbr_out=ub[:, :pl]) - oracle.rhs(free, ua, Ha)
    assert np.max(np.abs(d)) < 1e-12


# ---- O12b: spectral interpolation of a face plane between grids of different band limit ------------------------------------------
def _nodes(oracle, L):
    th, _ = oracle.gl_nodes(L)
    ph = 2 * np.pi * np.arange(2 * L + 2) / (2 * L + 2)
    return np.meshgrid(th, ph, indexing="ij")


def test_interp_band_limited_fields_cross_unchanged(oracle):
    """A field band-limited to l <= min(Ls, Ld) is the same function on both grids: closed-form real harmonics up to l = 3 (and
    a seeded combination of them) sampled on the source grid come out as the same closed forms sampled on the destination
    grid, coarser or finer; Ls = Ld is the projection of O2."""
    def harmonics(th, ph):
        x, y, z = np.sin(th) * np.cos(ph), np.sin(th) * np.sin(ph), np.cos(th)
        return [np.ones_like(x), x, y, z, x * y, y * z, 3 * z * z - 1, x * z, x * x - y * y, x * y * z, z * (5 * z * z - 3), x * (x * x - 3 * y * y)]
    rng = np.random.default_rng(2)
    coef = rng.standard_normal(12)
    for Ls, Ld in ((5, 8), (8, 5), (4, 3), (3, 7), (6, 6)):
        ths, phs = _nodes(oracle, Ls)
        thd, phd = _nodes(oracle, Ld)
        hs, hd = harmonics(ths, phs), harmonics(thd, phd)
        for a, b in zip(hs, hd):
            assert np.abs(oracle.shell_interp(Ls, Ld, a) - b).max() < 1e-14 * max(1.0, np.abs(b).max())
        fs = sum(c * a for c, a in zip(coef, hs)); fd = sum(c * b for c, b in zip(coef, hd))
        assert np.abs(oracle.shell_interp(Ls, Ld, fs) - fd).max() < 2e-14 * np.abs(fd).max()
    u = rng.standard_normal((7, 14))
    assert np.abs(oracle.shell_interp(6, 6, u) - oracle.shell_project(6, u)).max() < 1e-14      # same grid: the projection


def test_interp_is_linear_and_drops_nothing_it_can_represent(oracle):
    """Linearity; coarse -> fine -> coarse is the projection on the coarse grid (the fine grid holds every coarse mode); a mode
    l = Ls (the highest the source resolves) arrives on a finer grid with its norm, and fine -> coarse of a mode above the
    coarse band limit is NOT zero at the nodes (the series is summed, not truncated: aliased point values)."""
    rng = np.random.default_rng(4)
    u, v = rng.standard_normal((5, 10)), rng.standard_normal((5, 10))
    a = oracle.shell_interp(4, 7, 2.0 * u - 3.0 * v)
    assert np.abs(a - (2.0 * oracle.shell_interp(4, 7, u) - 3.0 * oracle.shell_interp(4, 7, v))).max() < 1e-13
    back = oracle.shell_interp(7, 4, oracle.shell_interp(4, 7, u))
    assert np.abs(back - oracle.shell_project(4, u)).max() < 1e-13
    th7, ph7 = _nodes(oracle, 7)
    z = np.cos(th7)
    p6 = (231 * z ** 6 - 315 * z ** 4 + 105 * z ** 2 - 5) / 16          # Legendre P_6: l = 6 > 4
    down = oracle.shell_interp(7, 4, p6)
    th4, _ = _nodes(oracle, 4)
    z4 = np.cos(th4)
    assert np.abs(down - (231 * z4 ** 6 - 315 * z4 ** 4 + 105 * z4 ** 2 - 5) / 16).max() < 1e-13
