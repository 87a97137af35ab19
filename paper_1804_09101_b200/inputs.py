"""Seeded synthetic input generators (shared by the oracle tests and the CUDA path).

This module holds NONE of the method's arithmetic: no spectral derivative, no
generalized-harmonic right-hand side, no Runge-Kutta update, no constraint.  It
only evaluates *analytic* closed-form data at points that the caller supplies
and adds seeded smooth perturbations.  Both sides (``oracle/`` and the CUDA
library) receive exactly the same arrays produced here.

What the paper fixes about the inputs
-------------------------------------
* "analytically-computed Kerr-Schild initial data for an isolated black hole,
  defined by its mass m and its dimensionless spin-vector" (§3.1);
  the whole-code tests evolve "a stationary, single black hole with a spin of
  0.5" (§4).
* about 50 evolved variables (§2.1): psi_ab (10), Pi_ab (10),
  Phi_iab (30) of the first-order generalized-harmonic system.

Everything else (perturbation family, RNG, gauge source choice) is the recipe of
SURVEY.md §8(d) / DESIGN.md "Input recipe".

Component order (include/gh.h): s(a,b) for a<=b runs
00,01,02,03,11,12,13,22,23,33 -> 0..9;  psi: c=s;  Pi: c=10+s;
Phi_iab: c=20+10*i+s with i=0,1,2 = x,y,z.

All functions accept complex coordinates, so that tests can take exact
derivatives by the complex-step method  f'(x) = Im f(x+ih)/h.
"""
from __future__ import annotations

import numpy as np

SYM_PAIRS = [(0, 0), (0, 1), (0, 2), (0, 3), (1, 1), (1, 2), (1, 3), (2, 2), (2, 3), (3, 3)]
SYM_INDEX = np.zeros((4, 4), dtype=np.int64)
for _s, (_a, _b) in enumerate(SYM_PAIRS):
    SYM_INDEX[_a, _b] = _s
    SYM_INDEX[_b, _a] = _s

N_COMP = 50
SEED_BASE = 180409101000  # seed = SEED_BASE + 1000*config + subdomain


# --------------------------------------------------------------------------
# counter-based RNG (SplitMix64), uniform in [-1, 1)
# --------------------------------------------------------------------------
class SplitMix64:
    """SplitMix64 stream; ``uniform(n)`` returns n doubles in [-1, 1)."""

    def __init__(self, seed: int):
        self.state = np.uint64(seed & 0xFFFFFFFFFFFFFFFF)

    def next_u64(self, n: int) -> np.ndarray:
        with np.errstate(over="ignore"):
            idx = np.arange(1, n + 1, dtype=np.uint64)
            z = self.state + idx * np.uint64(0x9E3779B97F4A7C15)
            self.state = z[-1] if n > 0 else self.state
            z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
            z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
            z = z ^ (z >> np.uint64(31))
        return z

    def uniform(self, n: int) -> np.ndarray:
        u = (self.next_u64(n) >> np.uint64(11)).astype(np.float64) * (1.0 / (1 << 53))
        return 2.0 * u - 1.0

    def integers(self, lo: int, hi: int, n: int) -> np.ndarray:
        """n integers uniform in [lo, hi] inclusive."""
        span = np.uint64(hi - lo + 1)
        return (self.next_u64(n) % span).astype(np.int64) + lo


# --------------------------------------------------------------------------
# packing helpers
# --------------------------------------------------------------------------
def pack_fields(psi: np.ndarray, Pi: np.ndarray, Phi: np.ndarray) -> np.ndarray:
    """psi[4,4,P], Pi[4,4,P], Phi[3,4,4,P] -> u[50,P] (upper triangles)."""
    P = psi.shape[-1]
    u = np.empty((N_COMP, P), dtype=psi.dtype)
    for s, (a, b) in enumerate(SYM_PAIRS):
        u[s] = psi[a, b]
        u[10 + s] = Pi[a, b]
        for i in range(3):
            u[20 + 10 * i + s] = Phi[i, a, b]
    return u


def unpack_fields(u: np.ndarray):
    """u[50,P] -> psi[4,4,P], Pi[4,4,P], Phi[3,4,4,P] (symmetric fill)."""
    P = u.shape[-1]
    psi = np.empty((4, 4, P), dtype=u.dtype)
    Pi = np.empty((4, 4, P), dtype=u.dtype)
    Phi = np.empty((3, 4, 4, P), dtype=u.dtype)
    for a in range(4):
        for b in range(4):
            s = SYM_INDEX[a, b]
            psi[a, b] = u[s]
            Pi[a, b] = u[10 + s]
            for i in range(3):
                Phi[i, a, b] = u[20 + 10 * i + s]
    return psi, Pi, Phi


# --------------------------------------------------------------------------
# Kerr-Schild black hole, spin along +z, centred at the origin
# --------------------------------------------------------------------------
def _ks_scalars(xyz, M, a):
    """H, l_a[4], dH[3], dl[3,4] (analytic gradients) at points xyz[3,P]."""
    x, y, z = xyz[0], xyz[1], xyz[2]
    one = np.ones_like(x)
    zero = np.zeros_like(x)
    a2 = a * a
    rho2 = x * x + y * y + z * z
    b = rho2 - a2
    s = np.sqrt(b * b + 4.0 * a2 * z * z)
    r2 = 0.5 * (b + s)
    r = np.sqrt(r2)
    # gradient of r^2, then of r
    db = [2.0 * x, 2.0 * y, 2.0 * z]
    ds = [b * db[0] / s, b * db[1] / s, (b * db[2] + 4.0 * a2 * z) / s]
    dr = [0.5 * (db[i] + ds[i]) / (2.0 * r) for i in range(3)]
    den = r2 * r2 + a2 * z * z
    H = M * r2 * r / den
    dden = [4.0 * r2 * r * dr[0], 4.0 * r2 * r * dr[1], 4.0 * r2 * r * dr[2] + 2.0 * a2 * z]
    dH = [M * (3.0 * r2 * dr[i] * den - r2 * r * dden[i]) / (den * den) for i in range(3)]
    q = r2 + a2
    nx = r * x + a * y
    ny = r * y - a * x
    l = [one, nx / q, ny / q, z / r]
    dnx = [dr[0] * x + r, dr[1] * x + a, dr[2] * x]
    dny = [dr[0] * y - a, dr[1] * y + r, dr[2] * y]
    dl = []
    for i in range(3):
        dq = 2.0 * r * dr[i]
        dlx = (dnx[i] * q - nx * dq) / (q * q)
        dly = (dny[i] * q - ny * dq) / (q * q)
        dlz = (one if i == 2 else zero) / r - z * dr[i] / r2
        dl.append([zero, dlx, dly, dlz])
    return H, l, dH, dl


def kerr_schild(xyz: np.ndarray, M: float = 1.0, a: float = 0.0):
    """Analytic Kerr-Schild data at points xyz[3,P].

    psi_ab = eta_ab + 2 H l_a l_b,  Phi_iab = d_i psi_ab (analytic),
    Pi_ab = (N^i/N) Phi_iab (stationary: d_t psi = 0), with the closed forms
    N = (1+2H)^(-1/2), N^i = 2 H l^i / (1+2H).
    Returns psi[4,4,P], Pi[4,4,P], Phi[3,4,4,P].
    """
    xyz = np.asarray(xyz)
    H, l, dH, dl = _ks_scalars(xyz, M, a)
    P = xyz.shape[-1]
    dt = np.result_type(xyz.dtype, np.float64)
    eta = np.diag([-1.0, 1.0, 1.0, 1.0])
    psi = np.empty((4, 4, P), dtype=dt)
    Phi = np.empty((3, 4, 4, P), dtype=dt)
    for a_ in range(4):
        for b_ in range(4):
            psi[a_, b_] = eta[a_, b_] + 2.0 * H * l[a_] * l[b_]
            for i in range(3):
                Phi[i, a_, b_] = 2.0 * (dH[i] * l[a_] * l[b_] + H * dl[i][a_] * l[b_] + H * l[a_] * dl[i][b_])
    lapse = 1.0 / np.sqrt(1.0 + 2.0 * H)
    shift = [2.0 * H * l[i + 1] / (1.0 + 2.0 * H) for i in range(3)]
    Pi = np.zeros((4, 4, P), dtype=dt)
    for i in range(3):
        Pi += (shift[i] / lapse) * Phi[i]
    return psi, Pi, Phi


def kerr_schild_lapse_shift(xyz, M=1.0, a=0.0):
    """Closed-form Kerr-Schild lapse N[P] and shift N^i[3,P] (oracle pin for O4)."""
    H, l, _, _ = _ks_scalars(np.asarray(xyz), M, a)
    lapse = 1.0 / np.sqrt(1.0 + 2.0 * H)
    shift = np.stack([2.0 * H * l[i + 1] / (1.0 + 2.0 * H) for i in range(3)])
    return lapse, shift


def kerr_schild_gauge_source(xyz: np.ndarray, M: float = 1.0, a: float = 0.0) -> np.ndarray:
    """Frozen gauge source H_a = -Gamma_a of the unperturbed Kerr-Schild metric, [4,P].

    Kerr-Schild coordinates have sqrt(-g) = 1 and psi^{ab} = eta^{ab} - 2 H l^a l^b,
    so Gamma^a = -d_b psi^{ab} = 2 d_j (H l^a l^j) for stationary data, with
    l^a = (-1, l_i).  Gamma_a = psi_ab Gamma^b.  (SURVEY.md §8(c) S3.)
    """
    xyz = np.asarray(xyz)
    H, l, dH, dl = _ks_scalars(xyz, M, a)
    lup = [-l[0], l[1], l[2], l[3]]
    dlup = [[-dl[j][0], dl[j][1], dl[j][2], dl[j][3]] for j in range(3)]
    Gup = []
    for a_ in range(4):
        acc = 0.0
        for j in range(3):
            acc = acc + dH[j] * lup[a_] * lup[j + 1] + H * dlup[j][a_] * lup[j + 1] + H * lup[a_] * dlup[j][j + 1]
        Gup.append(2.0 * acc)
    eta = np.diag([-1.0, 1.0, 1.0, 1.0])
    out = np.empty((4, xyz.shape[-1]), dtype=np.result_type(xyz.dtype, np.float64))
    for a_ in range(4):
        acc = 0.0
        for b_ in range(4):
            acc = acc + (eta[a_, b_] + 2.0 * H * l[a_] * l[b_]) * Gup[b_]
        out[a_] = -acc
    return out


# --------------------------------------------------------------------------
# harmonic gauge wave: ds^2 = -H dt^2 + H dx^2 + dy^2 + dz^2, H = 1 - A sin(2 pi (x-t)/d)
# --------------------------------------------------------------------------
def gauge_wave(xyz: np.ndarray, t: float, A: float = 0.1, d: float = 2.0):
    """Returns (psi, Pi, Phi, dt_psi, dt_Pi, dt_Phi), the last three analytic.

    Harmonic coordinates: Gamma_a = 0, so the gauge source is H_a = 0.
    Pins every sign of the GH system that stationarity cannot.
    """
    xyz = np.asarray(xyz)
    x = xyz[0]
    P = x.shape[0]
    k = 2.0 * np.pi / d
    ph = k * (x - t)
    Hh = 1.0 - A * np.sin(ph)
    H1 = -A * k * np.cos(ph)        # dH/dx ; dH/dt = -H1
    H2 = A * k * k * np.sin(ph)     # d2H/dx2 ; d(H1)/dt = -H2
    rt = np.sqrt(Hh)
    dt = np.result_type(xyz.dtype, np.float64)
    psi = np.zeros((4, 4, P), dtype=dt)
    Pi = np.zeros((4, 4, P), dtype=dt)
    Phi = np.zeros((3, 4, 4, P), dtype=dt)
    dpsi = np.zeros((4, 4, P), dtype=dt)
    dPi = np.zeros((4, 4, P), dtype=dt)
    dPhi = np.zeros((3, 4, 4, P), dtype=dt)
    psi[0, 0] = -Hh
    psi[1, 1] = Hh
    psi[2, 2] = 1.0
    psi[3, 3] = 1.0
    # Pi_ab = -(1/N) d_t psi_ab, N = sqrt(H), shift = 0
    Pi[0, 0] = -H1 / rt
    Pi[1, 1] = H1 / rt
    Phi[0, 0, 0] = -H1
    Phi[0, 1, 1] = H1
    dpsi[0, 0] = H1
    dpsi[1, 1] = -H1
    # d_t(-H1/sqrt(H)) = H2/sqrt(H) + H1 * (dH/dt) / (2 H^{3/2}) = H2/sqrt(H) - H1^2/(2 H^{3/2})
    dPi[0, 0] = H2 / rt - H1 * H1 / (2.0 * Hh * rt)
    dPi[1, 1] = -dPi[0, 0]
    dPhi[0, 0, 0] = H2
    dPhi[0, 1, 1] = -H2
    return psi, Pi, Phi, dpsi, dPi, dPhi


# --------------------------------------------------------------------------
# seeded smooth perturbations
# --------------------------------------------------------------------------
def _cheb_T(kmax: int, x: np.ndarray) -> np.ndarray:
    """T_0..T_kmax at x in [-1,1] -> [kmax+1, P]."""
    th = np.arccos(np.clip(x, -1.0, 1.0))
    return np.stack([np.cos(k * th) for k in range(kmax + 1)])


def _real_ylm(lmax: int, theta: np.ndarray, phi: np.ndarray) -> np.ndarray:
    """Unnormalised real spherical harmonics l<=lmax -> [(lmax+1)^2, P] (input recipe only)."""
    from scipy.special import lpmv

    ct = np.cos(theta)
    out = []
    for l in range(lmax + 1):
        for m in range(-l, l + 1):
            plm = lpmv(abs(m), l, ct)
            sc = np.max(np.abs(plm)) if plm.size else 1.0
            plm = plm / (sc if sc > 0 else 1.0)
            out.append(plm * (np.cos(m * phi) if m >= 0 else np.sin(-m * phi)))
    return np.stack(out)


def shell_perturbation(r_lo, r_hi, center, xyz, amplitude, seed, kmax=4, lmax=4, norm=None) -> np.ndarray:
    """[50,P] perturbation: per component sum_{k<=kmax} sum_{l<=lmax,m} c_klm T_k(x(r)) Y^real_lm,
    c uniform in [-1,1) from SplitMix64(seed), each component rescaled to L-inf = amplitude.
    norm: None, or [50] maxima to normalise with instead of this call's own (chunked generation; amplitude = None returns
    the unnormalised functions)."""
    rel = np.asarray(xyz, dtype=np.float64) - np.asarray(center, dtype=np.float64)[:, None]
    r = np.sqrt((rel * rel).sum(0))
    theta = np.arccos(np.clip(rel[2] / r, -1.0, 1.0))
    phi = np.arctan2(rel[1], rel[0])
    xr = 2.0 * (r - r_lo) / (r_hi - r_lo) - 1.0
    T = _cheb_T(kmax, xr)                # [K,P]
    Y = _real_ylm(lmax, theta, phi)      # [S,P]
    rng = SplitMix64(seed)
    K, S = T.shape[0], Y.shape[0]
    out = np.empty((N_COMP, r.shape[0]))
    for c in range(N_COMP):
        coef = rng.uniform(K * S).reshape(K, S)
        f = ((coef @ Y) * T).sum(0)          # sum_k T_k(x) sum_s c_ks Y_s
        out[c] = f if amplitude is None else f * (amplitude / (np.max(np.abs(f)) if norm is None else norm[c]))
    return out


def block_perturbation(lo, hi, xyz, amplitude, seed, deg=6, norm=None) -> np.ndarray:
    """[50,P] perturbation: per component sum_{i,j,k<=deg} c_ijk T_i T_j T_k on the block's
    reference cube, rescaled to L-inf = amplitude (norm: as in shell_perturbation)."""
    xyz = np.asarray(xyz, dtype=np.float64)
    T = [_cheb_T(deg, 2.0 * (xyz[d] - lo[d]) / (hi[d] - lo[d]) - 1.0) for d in range(3)]
    rng = SplitMix64(seed)
    n = deg + 1
    out = np.empty((N_COMP, xyz.shape[1]))
    for c in range(N_COMP):
        coef = rng.uniform(n * n * n).reshape(n, n, n)
        f = (coef.reshape(n * n, n) @ T[2]).reshape(n, n, -1)   # sum over k
        f = (f * T[1][None]).sum(1)                               # sum over j
        f = (f * T[0]).sum(0)                                     # sum over i
        out[c] = f if amplitude is None else f * (amplitude / (np.max(np.abs(f)) if norm is None else norm[c]))
    return out


def initial_data(descs, coords, spin, amplitude, config_id, M=1.0):
    """Fields u[50,P_total] and gauge source H[4,P_total] for a list of subdomains.

    ``descs``: list of dicts with keys kind ('shell'|'block'|'cylinder'), lo, hi, center;
    ``coords``: list of xyz[3,P_s] arrays (from the oracle's grid or from
    ``gh_domain_coords`` — the generator never builds collocation grids itself).
    Returns lists (u_s, H_s), one entry per subdomain.
    """
    us, Hs = [], []
    for s, (d, xyz) in enumerate(zip(descs, coords)):
        psi, Pi, Phi = kerr_schild(xyz, M, spin)
        u = pack_fields(psi, Pi, Phi)
        seed = SEED_BASE + 1000 * config_id + s
        if amplitude != 0.0:
            if d["kind"] == "shell":
                u = u + shell_perturbation(d["lo"][0], d["hi"][0], d["center"], xyz, amplitude, seed)
            elif d["kind"] == "cylinder":     # the block family on the cylinder's Cartesian bounding box
                c, ro = d["center"], d["hi"][0]
                u = u + block_perturbation([c[0] - ro, c[1] - ro, c[2] + d["lo"][1]], [c[0] + ro, c[1] + ro, c[2] + d["hi"][1]],
                                           xyz, amplitude, seed)
            else:
                u = u + block_perturbation(d["lo"], d["hi"], xyz, amplitude, seed)
        us.append(np.ascontiguousarray(u))
        Hs.append(np.ascontiguousarray(kerr_schild_gauge_source(xyz, M, spin)))
    return us, Hs


def initial_data_chunked(d, xyz, spin, amplitude, config_id, s, u_out, H_out, chunk=1 << 20, M=1.0):
    """The same data as initial_data for ONE subdomain, written into u_out[50,P] / H_out[4,P] chunk by chunk (the sweep's
    largest members have 3.3e7 points: the temporaries of a single pass would be tens of GB).  Two passes over the
    perturbation: component maxima first (the L-inf normalisation is over the whole subdomain), then the data."""
    P = xyz.shape[1]
    seed = SEED_BASE + 1000 * config_id + s

    def pert(sl, amp, norm):
        if d["kind"] == "shell":
            return shell_perturbation(d["lo"][0], d["hi"][0], d["center"], xyz[:, sl], amp, seed, norm=norm)
        return block_perturbation(d["lo"], d["hi"], xyz[:, sl], amp, seed, norm=norm)

    norm = None
    if amplitude != 0.0:
        norm = np.zeros(N_COMP)
        for p0 in range(0, P, chunk):
            norm = np.maximum(norm, np.max(np.abs(pert(slice(p0, min(P, p0 + chunk)), None, None)), axis=1))
    for p0 in range(0, P, chunk):
        sl = slice(p0, min(P, p0 + chunk))
        u = pack_fields(*kerr_schild(xyz[:, sl], M, spin))
        if amplitude != 0.0:
            u = u + pert(sl, amplitude, norm)
        u_out[:, sl] = u
        H_out[:, sl] = kerr_schild_gauge_source(xyz[:, sl], M, spin)
