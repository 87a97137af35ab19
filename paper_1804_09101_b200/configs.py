"""The five BASELINE.json workloads restated as seeded synthetic domains.

Pure description: lists of subdomain descriptors (dicts) + spin / amplitude / config id.
No arithmetic of the method lives here.  The paper uses no dataset: its runs evolve
analytic Kerr-Schild data on concentric shells; the
"SingleBH" and "BBH" grid prescriptions are PAPER.md:436.

A descriptor is {'kind': 'shell'|'block', 'n': [...], 'lo': [...], 'hi': [...],
'center': [...], 'face': [...], 'gamma': [g0, g1, g2]}:
  shell: n = [N_r, L]  (N_theta = L+1 Gauss-Legendre, N_phi = 2L+2 uniform), lo[0]/hi[0] = radii,
         face = [inner, outer];   block: n = [N_x, N_y, N_z], face = [-x,+x,-y,+y,-z,+z].
face values: 0 = FREE (no boundary treatment, e.g. excision), 1 = FROZEN (RHS zeroed).
"""
from __future__ import annotations

import math

from .inputs import SEED_BASE, SplitMix64

GAMMA_DEFAULT = [1.0, -1.0, 1.0]  # SURVEY S2 (a convention; parity unpinned)


def shell(n_r, L, r_in, r_out, face=(0, 0), gamma=None, center=(0.0, 0.0, 0.0)):
    return {"kind": "shell", "n": [int(n_r), int(L), 0], "lo": [float(r_in), 0.0, 0.0], "hi": [float(r_out), 0.0, 0.0],
            "center": [float(c) for c in center], "face": list(face) + [0] * (6 - len(face)),
            "gamma": list(gamma or GAMMA_DEFAULT)}


def block(n, lo, hi, face=(0,) * 6, gamma=None):
    n = [int(n)] * 3 if isinstance(n, int) else [int(v) for v in n]
    return {"kind": "block", "n": n, "lo": [float(v) for v in lo], "hi": [float(v) for v in hi],
            "center": [0.0, 0.0, 0.0], "face": list(face), "gamma": list(gamma or GAMMA_DEFAULT)}


def cylinder(n, rho_in, rho_out, z_lo, z_hi, face=(0, 0, 0, 0), gamma=None, center=(0.0, 0.0, 0.0)):
    """Cylindrical shell (reading S25), axis along z through `center`: n = (N_rho, N_z, N_phi); z range relative to
    the centre; faces rho_in, rho_out, z_lo, z_hi."""
    return {"kind": "cylinder", "n": [int(v) for v in n], "lo": [float(rho_in), float(z_lo), 0.0],
            "hi": [float(rho_out), float(z_hi), 0.0], "center": [float(c) for c in center],
            "face": list(face) + [0] * (6 - len(face)), "gamma": list(gamma or GAMMA_DEFAULT)}


def cylinder_box(d):
    """Cartesian bounding box (lo, hi) of a cylindrical shell."""
    c, ro = d["center"], d["hi"][0]
    return [c[0] - ro, c[1] - ro, c[2] + d["lo"][1]], [c[0] + ro, c[1] + ro, c[2] + d["hi"][1]]


def num_points(d) -> int:
    if d["kind"] == "shell":
        return d["n"][0] * (d["n"][1] + 1) * (2 * d["n"][1] + 2)
    return d["n"][0] * d["n"][1] * d["n"][2]


def min_spacing(descs) -> float:
    """S14: min Euclidean distance between neighbouring nodes along any logical axis."""
    best = float("inf")
    for d in descs:
        if d["kind"] == "shell":
            n_r, L = d["n"][0], d["n"][1]
            r_in, r_out = d["lo"][0], d["hi"][0]
            best = min(best, 0.5 * (r_out - r_in) * (1.0 - math.cos(math.pi / (n_r - 1))))
            # angular neighbours on the innermost sphere: chord of the phi spacing at the first colatitude,
            # and the theta spacing near the pole (Gauss-Legendre nodes ~ pi (j+3/4)/(L+3/2))
            th0 = math.pi * 0.75 / (L + 1.5)
            best = min(best, r_in * math.sin(th0) * 2.0 * math.sin(math.pi / (2 * L + 2)))
            best = min(best, r_in * math.pi / (L + 1.5))
        elif d["kind"] == "cylinder":
            for a in range(2):
                best = min(best, 0.5 * (d["hi"][a] - d["lo"][a]) * (1.0 - math.cos(math.pi / (d["n"][a] - 1))))
            best = min(best, 2.0 * d["lo"][0] * math.sin(math.pi / d["n"][2]))
        else:
            for a in range(3):
                best = min(best, 0.5 * (d["hi"][a] - d["lo"][a]) * (1.0 - math.cos(math.pi / (d["n"][a] - 1))))
    return best


def c1():
    """C1: one shell r in [1.8,5], N_r=8, L=8, Schwarzschild, perturbation 1e-3."""
    return {"id": 1, "spin": 0.0, "amplitude": 1e-3, "descs": [shell(8, 8, 1.8, 5.0, face=(0, 1))]}


def c2():
    """C2: one 24^3 block [3,11]x[-4,4]^2 (centre (7,0,0), so r >= 3), a = 0.5, perturbation 1e-4."""
    return {"id": 2, "spin": 0.5, "amplitude": 1e-4, "descs": [block(24, (3.0, -4.0, -4.0), (11.0, 4.0, 4.0))]}


def c3():
    """C3: 8 shells, boundaries 1.9 (100/1.9)^(s/8), N_r=16, L=16, a=0.7, perturbation 1e-5.
    Innermost inner face FREE (excision), every other face FROZEN (S11)."""
    b = [1.9 * (100.0 / 1.9) ** (s / 8.0) for s in range(9)]
    descs = [shell(16, 16, b[s], b[s + 1], face=(0 if s == 0 else 1, 1)) for s in range(8)]
    return {"id": 3, "spin": 0.7, "amplitude": 1e-5, "descs": descs, "nsteps": 100, "dt": 0.25 * min_spacing(descs)}


def c4(min_points: int = 4_000_000, replicate: bool = True):
    """C4: 40 shells (N_r in [12,24], L in [12,32]) + 24 cube blocks (N in [16,32]), r = 1.9..500, a = 0.9,
    sizes drawn from SplitMix64(SEED_BASE + 4000); the subdomain set is replicated k times until
    P >= min_points (S13: subdomains are independent)."""
    rng = SplitMix64(SEED_BASE + 4000)
    nr = rng.integers(12, 24, 40)
    LL = rng.integers(12, 32, 40)
    b = [1.9 * (500.0 / 1.9) ** (s / 40.0) for s in range(41)]
    base = [shell(nr[s], LL[s], b[s], b[s + 1], face=(0 if s == 0 else 1, 1)) for s in range(40)]
    nb = rng.integers(16, 32, 24)
    hw = 2.0 + 2.0 * (rng.uniform(24) + 1.0)          # half-widths in [2,6)
    extra = 25.0 * (rng.uniform(24) + 1.0)            # extra radius in [0,50)
    cth = rng.uniform(24)
    ph = math.pi * rng.uniform(24)
    for q in range(24):
        R = 3.0 + math.sqrt(3.0) * hw[q] + extra[q]
        st = math.sqrt(max(0.0, 1.0 - cth[q] * cth[q]))
        c = (R * st * math.cos(ph[q]), R * st * math.sin(ph[q]), R * cth[q])
        base.append(block(int(nb[q]), [c[a] - hw[q] for a in range(3)], [c[a] + hw[q] for a in range(3)], face=(1,) * 6))
    P1 = sum(num_points(d) for d in base)
    k = max(1, -(-min_points // P1)) if replicate else 1
    descs = [dict(d) for _ in range(k) for d in base]
    return {"id": 4, "spin": 0.9, "amplitude": 1e-5, "descs": descs, "replicas": k, "base_subdomains": len(base),
            "dt": 0.25 * min_spacing(base)}


def c5_shell(n: int):
    """C5 shell sweep member: N_r = L+1 = n  (P = 2 n^3)."""
    return {"id": 5, "spin": 0.5, "amplitude": 1e-4, "descs": [shell(n, n - 1, 1.9, 10.0, face=(0, 1))]}


def c5_block(N: int):
    """C5 block sweep member: N^3 points."""
    return {"id": 5, "spin": 0.5, "amplitude": 1e-4, "descs": [block(N, (3.0, -4.0, -4.0), (11.0, 4.0, 4.0))]}


def single_bh(k: int):
    """PAPER.md:436 'SingleBH' shell: N_r=9+4k, N_theta=6+2k, N_phi=12+4k  (so L = 5+2k)."""
    return {"id": 5, "spin": 0.5, "amplitude": 1e-4, "descs": [shell(9 + 4 * k, 5 + 2 * k, 1.9, 10.0, face=(0, 1))]}


def bbh(k: int):
    """PAPER.md:436 'BBH' shell: N_r=4+k, N_theta=7+2k, N_phi=14+4k  (so L = 6+2k)."""
    return {"id": 5, "spin": 0.5, "amplitude": 1e-4, "descs": [shell(4 + k, 6 + 2 * k, 1.9, 10.0, face=(0, 1))]}


def paper_two_shells():
    """two shells 1.62m-6m-12m with (10,19,38) points = 2 x 7220; spin 0.5."""
    return {"id": 6, "spin": 0.5, "amplitude": 1e-5,
            "descs": [shell(10, 18, 1.62, 6.0, face=(0, 1)), shell(10, 18, 6.0, 12.0, face=(1, 1))]}
