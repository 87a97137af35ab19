"""Host-side checks of the C-ABI library (no GPU): it loads, exports every symbol include/gh.h declares,
plans workspaces, refuses to compute without a CUDA device, and its basis builder (A0) agrees with textbook
closed forms and with the independent oracle."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_1804_09101_b200 import build as ghbuild
from paper_1804_09101_b200 import configs, gh

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module", autouse=True)
def built():
    ghbuild.build()


def test_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "gh.h")).read()
    declared = set(re.findall(r"\b(gh_[a-z0-9_]+)\s*\(", hdr))
    assert declared == set(gh.EXPORTS)
    L = gh.lib()
    for name in declared:
        assert hasattr(L, name), name


def test_workspace_bytes_scales_with_points():
    d1 = configs.c1()["descs"]
    d2 = configs.c2()["descs"]
    b1, b2 = gh.gh_workspace_bytes(d1), gh.gh_workspace_bytes(d2)
    # store: (3*50 + 150 + 16) arrays of padded P doubles, plus tables
    assert b1 > 316 * 8 * 1296 and b2 > 316 * 8 * 13824
    assert b2 > b1


def test_invalid_descriptors_are_rejected():
    bad = configs.c1()["descs"]
    bad[0] = dict(bad[0], n=[1, 8, 0])
    with pytest.raises(gh.GHError):
        gh.gh_workspace_bytes(bad)
    bad = configs.c2()["descs"]
    bad[0] = dict(bad[0], hi=[1.0, 4.0, 4.0])   # hi < lo on x
    with pytest.raises(gh.GHError):
        gh.gh_workspace_bytes(bad)


def test_create_fails_loudly_without_a_device():
    import torch

    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    descs = configs.c1()["descs"]
    nbytes = gh.gh_workspace_bytes(descs)
    with pytest.raises(gh.GHError) as e:
        gh.gh_domain_create(descs, 256 * 4096, nbytes, 0)   # fake aligned pointer: never touched
    assert e.value.status == gh.GH_ERR_CUDA


@pytest.mark.parametrize("N", [2, 3, 8, 16, 24, 33, 64])
def test_cheb_matrix_textbook(N):
    x, D = gh.gh_basis_cheb(N)
    j = np.arange(N)
    assert np.allclose(x, -np.cos(np.pi * j / (N - 1)), atol=1e-15)
    c = np.ones(N); c[0] = c[-1] = 2
    for i in range(N):
        for k in range(N):
            if i != k:
                ref = (c[i] / c[k]) * (-1.0) ** (i + k) / (x[i] - x[k])
                assert abs(D[i, k] - ref) <= 2e-13 * abs(ref)
    assert np.max(np.abs(D.sum(axis=1))) < 1e-10 * N * N
    # exact for monomials up to degree N-1
    for p in range(N):
        ref = p * x ** max(p - 1, 0) if p > 0 else np.zeros(N)
        assert np.max(np.abs(D @ x ** p - ref)) < 1e-11 * max(1.0, p * p)


@pytest.mark.parametrize("N", [8, 24, 48])
def test_cheb_matrix_matches_oracle_tracing(N, oracle):
    """delta-function tracing: the oracle's modal derivative of e_k is column k of D."""
    _, D = gh.gh_basis_cheb(N)
    T = np.stack([oracle.cheb_derivative_line(np.eye(N)[k]) for k in range(N)], axis=1)
    assert np.max(np.abs(D - T)) < 1e-12 * np.max(np.abs(D))


@pytest.mark.parametrize("L", [1, 4, 8, 16, 31])
def test_gauss_legendre_matches_oracle(L, oracle):
    th, w = gh.gh_basis_gauss_legendre(L)
    th0, w0 = oracle.gl_nodes(L)
    assert np.max(np.abs(th - th0)) < 1e-15 * 4 and np.max(np.abs(w - w0)) < 1e-15
    assert abs(w.sum() - 2.0) < 1e-14


@pytest.mark.parametrize("L", [2, 5, 8, 12])
def test_shell_matrices_realise_the_ylm_derivatives(L, oracle):
    """Fs*Th*Fa and (d/dphi synthesis)*Pr*Fa applied to random (non band-limited) planes equal the oracle's
    explicit Y_lm double sums (Eq. 24), and Fs*Pr*Fa is the idempotent projector of PAPER.md:386."""
    Fa, Fs, Th, Pr = gh.gh_basis_shell(L)
    nt, npp = L + 1, 2 * L + 2
    rng = np.random.default_rng(L)
    u = rng.standard_normal((nt, npp))
    c = u @ Fa.T                                        # [j][q]
    m_of_q = np.array([q if q <= L else q - L for q in range(2 * L + 1)])
    a = np.stack([Th[m_of_q[q]] @ c[:, q] for q in range(2 * L + 1)], axis=1)
    b = np.stack([Pr[m_of_q[q]] @ c[:, q] for q in range(2 * L + 1)], axis=1)
    dth = a @ Fs.T
    proj = b @ Fs.T
    # d/dphi: cos(m phi) -> -m sin(m phi), sin(m phi) -> m cos(m phi)
    bp = np.zeros_like(b)
    for m in range(1, L + 1):
        bp[:, m] = m * b[:, L + m]
        bp[:, L + m] = -m * b[:, m]
    dph = bp @ Fs.T
    rth, rph = oracle.shell_angular(L, u)
    rproj = oracle.shell_project(L, u)
    sc = np.max(np.abs(rth))
    assert np.max(np.abs(dth - rth)) < 1e-12 * sc
    assert np.max(np.abs(dph - rph)) < 1e-12 * max(sc, np.max(np.abs(rph)))
    assert np.max(np.abs(proj - rproj)) < 1e-13 * np.max(np.abs(u))
    assert np.allclose(Pr[0], np.eye(nt), atol=1e-13)      # m = 0: all l <= L resolved by L+1 nodes
    for m in range(L + 1):
        assert np.linalg.matrix_rank(Pr[m], tol=1e-9) == L + 1 - m


def test_filter_sigma_reading_s20():
    """gh_filter_sigma against the formulas stated in include/gh.h (reading S20), retyped here."""
    s = gh.gh_filter_sigma({"kind": "heaviside", "cut": 3}, 9)
    assert np.array_equal(s, (np.arange(10) <= 6).astype(float))
    s = gh.gh_filter_sigma({"kind": "exp", "alpha": 36.0, "p": 4}, 12)
    assert np.allclose(s, np.exp(-36.0 * (np.arange(13) / 12.0) ** 8), rtol=1e-13, atol=0)   # long double there, double here
    assert np.array_equal(gh.gh_filter_sigma({"kind": "none"}, 5), np.ones(6))
    with pytest.raises(gh.GHError):
        gh.gh_filter_sigma({"kind": "exp", "alpha": 1.0, "p": 0}, 5)


def test_shell_basis_at_the_largest_band_limit():
    """A0 at GH_MAX_L = 255 (SURVEY.md §7 hard part 5: sin^m(theta) underflows FP64 near the poles for m >~ 200; the builder works in
    long double): quadrature orthonormality of the Pbar_lm on the 256 Gauss-Legendre nodes, read off the per-m projectors
    Pr_m = 2 pi Pbar_m^T W-weighted: idempotent with trace = rank = L + 1 - m iff sum_j 2 pi w_j Pbar_lm Pbar_l'm = delta_ll';
    Pr_0 = 1; d/dtheta composites annihilate nothing they should not: Th_m Pr_m = Th_m; the Chebyshev matrix at N = 320 still
    differentiates x^p exactly."""
    L = 255
    Fa, Fs, Th, Pr = gh.gh_basis_shell(L)
    nt = L + 1
    assert np.all(np.isfinite(Th)) and np.all(np.isfinite(Pr))
    assert np.max(np.abs(Pr[0] - np.eye(nt))) < 1e-13
    for m in (1, 2, 77, 128, 200, 254, 255):
        P = Pr[m]
        assert np.max(np.abs(P @ P - P)) < 1e-13, m
        assert abs(np.trace(P) - (L + 1 - m)) < 1e-12 * nt, m
        assert np.max(np.abs(Th[m] @ P - Th[m])) < 1e-11 * np.max(np.abs(Th[m])), m
    # the Fourier pair is the projector onto m <= L on the 512 longitudes
    F = Fs @ Fa
    assert np.max(np.abs(F @ F - F)) < 1e-13 and abs(np.trace(F) - (2 * L + 1)) < 1e-10
    x, D = gh.gh_basis_cheb(320)
    for p in (0, 1, 7, 100, 319):
        ref = p * x ** max(p - 1, 0) if p > 0 else np.zeros(320)
        assert np.max(np.abs(D @ x ** p - ref)) < 1e-9 * max(1.0, p * p), p
