"""The paper's operation-count models (§2.3 roofline; 271-273 DiffJac; 403-450 Deriv), used by
bench.py to quote effective rates in the paper's own convention next to the algorithmic ones.

All counts are per call; M is in memory transactions (one FP64 value = one transaction of w = 8 bytes),
F in floating-point operations, I = F / M.

The shell numbers describe the paper's DENSE formulation (one (N_theta N_phi)^2 matrix per angular derivative,
Eq. 24).  This library applies the same linear map factored axis by axis, so its executed flop count is
far lower; `shell_factored_flop` gives that count.  Reporting both, labelled, is SURVEY.md §8(d).
"""
from __future__ import annotations


def diffjac(n_x: int, n_e: int, d: int = 3):
    """M = N_x (2 N_e + d) d,  F = N_x N_e (2d - 1) d."""
    return n_x * (2 * n_e + d) * d, n_x * n_e * (2 * d - 1) * d


def diffjac_intensity(n_e: int, d: int = 3) -> float:
    m, f = diffjac(1, n_e, d)
    return f / m


def block_deriv(n_e: int, nx: int, ny: int, nz: int):
    """PAPER.md:405-423, Eqs. 25-29 (general form of Eqs. 28, 29)."""
    m = n_e * (6 * nx * ny * nz + nx * nx + nz * ny * ny + nz * nz)
    f = n_e * nx * ny * nz * (2 * (nx + ny + nz) - 3)
    return m, f


def shell_deriv_dense(n_e: int, n_r: int, n_th: int, n_ph: int):
    """PAPER.md:431-434, Eqs. 30-31 (dense angular matrices)."""
    a = n_th * n_ph
    m = n_e * (n_r * n_r + 2 * a * a + 6 * n_r * a)
    f = n_e * n_r * a * (2 * n_r + 4 * a - 3)
    return m, f


def single_bh_grid(k: int):
    """PAPER.md:436 'SingleBH': N_r = 9+4k, N_theta = 6+2k, N_phi = 12+4k."""
    return 9 + 4 * k, 6 + 2 * k, 12 + 4 * k


def bbh_grid(k: int):
    """PAPER.md:436 'BBH': N_r = 4+k, N_theta = 7+2k, N_phi = 14+4k."""
    return 4 + k, 7 + 2 * k, 14 + 4 * k


def shell_factored_flop(n_e: int, n_r: int, L: int) -> int:
    """Flop of the factored map this library executes on a shell: radial line (2 N_r - 1) plus
    8 (2L+1) per point for DFT analysis, per-m theta composites and two DFT syntheses."""
    pts = n_r * (L + 1) * (2 * L + 2)
    return n_e * pts * ((2 * n_r - 1) + 8 * (2 * L + 1))


def shell_executed_dmma_flop(n_e: int, n_r: int, L: int, nb: int = 8) -> int:
    """Flop the angular kernel K_ang actually issues on the FP64 tensor cores for one shell (512 per mma.m8n8k4), with
    both symmetry folds (phi about pi in S1/S3, theta about the equator in S2) and every tile padded to 8 x 8 x 4; planes are
    processed in groups of `nb`.  Lower than 8(2L+1) per point: the folds halve the three GEMM stages."""
    h = nt = L + 1
    hh = (nt + 1) // 2
    groups, rem = divmod(n_r, nb)
    total = 0
    for planes in [nb] * groups + ([rem] if rem else []):
        mt1 = -(-planes * nt // 8)
        s1 = mt1 * (-(-(h + 1) // 4) * -(-h // 8) + -(-L // 4) * -(-L // 8))
        s3 = mt1 * 2 * (-(-h // 4) + -(-L // 4)) * -(-(h + 1) // 8)
        ntn = -(-2 * planes // 8)
        s2 = (L + 1) * 2 * -(-2 * hh // 8) * -(-hh // 4) * ntn
        total += s1 + s2 + s3
    return n_e * total * 512


def effective_rates(m_transactions: float, flop: float, seconds: float):
    """Eqs. 3-4: BW_eff = w M / T (GB/s), P_eff = F / T (GFLOP/s)."""
    return 8.0 * m_transactions / seconds / 1e9, flop / seconds / 1e9
