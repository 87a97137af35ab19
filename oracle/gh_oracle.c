/* gh_oracle.c — CPU ORACLE.  TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * A plain, slow, obviously-correct implementation of what the hot path of
 * arXiv 1804.09101 computes: spectral derivatives on Chebyshev^3 blocks and
 * Chebyshev x Y_lm shells, the pointwise right-hand side of the first-order
 * generalized-harmonic (GH) Einstein system, the SSP-RK3 update and the
 * constraint norms.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may call it.  It shares no code with
 * paper_1804_09101_b200/csrc (no headers, tables, helpers); the CUDA path must
 * never call it.
 *
 * How it differs from the CUDA path on purpose:
 *   - derivatives are MODAL: explicit-sum transforms to Chebyshev / Y_lm
 *     coefficients, recurrence-based differentiation, explicit-sum synthesis
 *     (Eqs. 14-18; Eqs. 23-24) — never a
 *     cached differentiation matrix;
 *   - the GH right-hand side is written as index loops over FULL 4x4 and
 *     3x4x4 arrays with no symmetry exploitation;
 *   - arithmetic is `long double` (x87 80-bit) by default, because an FP64
 *     recurrence-based derivative is itself only ~1e-11 accurate at N>=32
 *     (SURVEY.md §7 hard part 1) and cannot referee a 1e-11 bar.  Compile with
 *     -DORA_DOUBLE for the timed CPU baseline (same source, Real=double).
 *
 * The paper never prints the evolved equations (it says "the Einstein equations
 * in their generalized harmonic formulation", first order in
 * "about 50 fundamental variables").  The system coded in
 * ora_rhs_point() is the standard first-order GH system of the paper's ref.
 * [34] lineage (Lindblom, Scheel, Kidder, Owen, Rinne 2006) as written out in
 * SURVEY.md §8(c) O5 / DESIGN.md "Readings" S1.
 *
 * Parity pins (tests/test_oracle_*.py): monomials, the textbook CGL matrix,
 * Gauss-Legendre exactness, Y_lm orthonormality / Unsold / closed forms,
 * Cartesian polynomials on shells, Kerr-Schild lapse/shift closed forms,
 * stationarity of exact Kerr-Schild data with analytic derivatives, the harmonic
 * gauge wave, homogeneous damping-term cases, RK3 order; spectral filter (O9):
 * single Chebyshev modes and single Y_lm scaled by sigma, sigma = 1 identity /
 * projection, Heaviside idempotence, linearity; characteristic boundary condition
 * (O10): eigenvectors of the RHS's principal part; Dormand-Prince step (O11): the
 * order conditions of the tableau and 5th-order convergence on the gauge wave;
 * interface exchange (O12): projection of what it adds onto the characteristic fields;
 * constraints (O8): C_ijab of a polynomial Phi equals its analytic curl; SpatialCoordJac
 * (O13): the tensor law with diag(1, J) by einsum, composition, Kerr-Schild axisymmetry, the
 * paper's printed operation counts.
 * PARITY UNPINNED (pure conventions, fixed by DESIGN.md): the normalisation of the
 * constraint norms (unweighted RMS over points and components), the default gamma's,
 * and the VALUE of the interface penalty factor p = (N_r-1)^2/(r_out-r_in) of O12 (its
 * structure - which fields, which sign, proportional to |v| - is pinned).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#ifdef ORA_DOUBLE
typedef double real;
#define R_SQRT sqrt
#define R_COS cos
#define R_SIN sin
#define R_ACOS acos
#define R_FABS fabs
#define R_PI 3.14159265358979323846
#else
typedef long double real;
#define R_SQRT sqrtl
#define R_COS cosl
#define R_SIN sinl
#define R_ACOS acosl
#define R_FABS fabsl
#define R_PI 3.14159265358979323846264338327950288L
#endif

typedef struct {
  int32_t kind;      /* 0 = shell (I1 x S2), 1 = block (I1^3), 2 = cylindrical shell (O15: I1 x I1 x S1, axis along z) */
  int32_t n[3];      /* shell: {N_r, L, unused}; block: {N_x, N_y, N_z}; cylinder: {N_rho, N_z, N_phi} */
  double lo[3], hi[3]; /* shell: lo[0]=r_in, hi[0]=r_out; block: corners; cylinder: [0] = rho_in / rho_out, [1] = z range (rel. to centre) */
  double center[3];  /* shell centre; cylinder: a point of the axis */
  int32_t face[6];   /* 1 = FROZEN. shell: [0]=inner,[1]=outer; block: -x,+x,-y,+y,-z,+z; cylinder: rho_in, rho_out, z_lo, z_hi */
  double gamma[3];   /* constraint damping gamma0, gamma1, gamma2 */
} ora_subdomain;

int ora_real_bytes(void) { return (int)sizeof(real); }

/* ---------------------------------------------------------------------- */
/* grid                                                                   */
/* ---------------------------------------------------------------------- */
static void dims(const ora_subdomain* sd, int* n0, int* n1, int* n2) {
  if (sd->kind == 0) { *n0 = sd->n[0]; *n1 = sd->n[1] + 1; *n2 = 2 * (sd->n[1] + 1); }
  else { *n0 = sd->n[0]; *n1 = sd->n[1]; *n2 = sd->n[2]; }
}

int64_t ora_num_points(const ora_subdomain* sd) {
  int a, b, c; dims(sd, &a, &b, &c); return (int64_t)a * b * c;
}

/* Chebyshev-Gauss-Lobatto nodes x_j = -cos(pi j/(N-1)), ascending. */
static void cgl_nodes(int N, real* x) {
  for (int j = 0; j < N; ++j) x[j] = -R_COS(R_PI * (real)j / (real)(N - 1));
}
void ora_cheb_nodes(int N, double* x) {
  real* t = malloc(sizeof(real) * N); cgl_nodes(N, t);
  for (int j = 0; j < N; ++j) x[j] = (double)t[j];
  free(t);
}

/* Legendre P_n(x) and P_n'(x) by the three-term recurrence. */
static void legendre(int n, real x, real* p, real* dp) {
  real p0 = 1, p1 = x;
  if (n == 0) { *p = 1; *dp = 0; return; }
  for (int k = 2; k <= n; ++k) { real pk = ((2 * k - 1) * x * p1 - (k - 1) * p0) / k; p0 = p1; p1 = pk; }
  *p = p1; *dp = n * (x * p1 - p0) / (x * x - 1);
}

/* Gauss-Legendre: cos(theta_j) = roots of P_{L+1} by Newton, theta ascending;
 * w_j = 2 / ((1-x_j^2) P'_{L+1}(x_j)^2). */
static void gl_nodes(int L, real* ct, real* w) {
  int n = L + 1;
  for (int j = 0; j < n; ++j) {
    real x = R_COS(R_PI * ((real)j + 0.75L) / ((real)n + 0.5L)); /* descending in x = ascending in theta */
    real p, dp;
    for (int it = 0; it < 100; ++it) { legendre(n, x, &p, &dp); real dx = p / dp; x -= dx; if (R_FABS(dx) < 1e-19L) break; }
    legendre(n, x, &p, &dp);
    ct[j] = x; w[j] = 2 / ((1 - x * x) * dp * dp);
  }
}
void ora_gl_nodes(int L, double* theta, double* w) {
  int n = L + 1; real* c = malloc(sizeof(real) * n); real* ww = malloc(sizeof(real) * n);
  gl_nodes(L, c, ww);
  for (int j = 0; j < n; ++j) { theta[j] = (double)R_ACOS(c[j]); w[j] = (double)ww[j]; }
  free(c); free(ww);
}

/* Coordinates xyz[3][P]; shells ordered (r slowest, theta, phi fastest), blocks (x,y,z). */
void ora_coords(const ora_subdomain* sd, double* xyz) {
  int n0, n1, n2; dims(sd, &n0, &n1, &n2); int64_t P = (int64_t)n0 * n1 * n2;
  if (sd->kind == 0) {
    int L = sd->n[1];
    real* xr = malloc(sizeof(real) * n0); cgl_nodes(n0, xr);
    real* ct = malloc(sizeof(real) * n1); real* w = malloc(sizeof(real) * n1); gl_nodes(L, ct, w);
    for (int i = 0; i < n0; ++i) for (int j = 0; j < n1; ++j) for (int k = 0; k < n2; ++k) {
      real r = (real)sd->lo[0] + ((real)sd->hi[0] - (real)sd->lo[0]) * (xr[i] + 1) / 2;
      real st = R_SQRT(1 - ct[j] * ct[j]); real ph = 2 * R_PI * (real)k / (real)n2;
      int64_t p = ((int64_t)i * n1 + j) * n2 + k;
      xyz[p] = (double)((real)sd->center[0] + r * st * R_COS(ph));
      xyz[P + p] = (double)((real)sd->center[1] + r * st * R_SIN(ph));
      xyz[2 * P + p] = (double)((real)sd->center[2] + r * ct[j]);
    }
    free(xr); free(ct); free(w);
  } else if (sd->kind == 2) {
    /* O15: rho on Chebyshev-Gauss-Lobatto nodes of [rho_in, rho_out], z likewise, phi_k = 2 pi k / N_phi; phi fastest */
    real* xr = malloc(sizeof(real) * n0); cgl_nodes(n0, xr);
    real* xz = malloc(sizeof(real) * n1); cgl_nodes(n1, xz);
    for (int i = 0; i < n0; ++i) for (int j = 0; j < n1; ++j) for (int k = 0; k < n2; ++k) {
      real rho = (real)sd->lo[0] + ((real)sd->hi[0] - (real)sd->lo[0]) * (xr[i] + 1) / 2;
      real z = (real)sd->lo[1] + ((real)sd->hi[1] - (real)sd->lo[1]) * (xz[j] + 1) / 2;
      real ph = 2 * R_PI * (real)k / (real)n2;
      int64_t p = ((int64_t)i * n1 + j) * n2 + k;
      xyz[p] = (double)((real)sd->center[0] + rho * R_COS(ph));
      xyz[P + p] = (double)((real)sd->center[1] + rho * R_SIN(ph));
      xyz[2 * P + p] = (double)((real)sd->center[2] + z);
    }
    free(xr); free(xz);
  } else {
    real* x[3]; int nn[3] = {n0, n1, n2};
    for (int d = 0; d < 3; ++d) { x[d] = malloc(sizeof(real) * nn[d]); cgl_nodes(nn[d], x[d]); }
    for (int i = 0; i < n0; ++i) for (int j = 0; j < n1; ++j) for (int k = 0; k < n2; ++k) {
      int64_t p = ((int64_t)i * n1 + j) * n2 + k; int idx[3] = {i, j, k};
      for (int d = 0; d < 3; ++d)
        xyz[d * P + p] = (double)((real)sd->lo[d] + ((real)sd->hi[d] - (real)sd->lo[d]) * (x[d][idx[d]] + 1) / 2);
    }
    for (int d = 0; d < 3; ++d) free(x[d]);
  }
}

/* ---------------------------------------------------------------------- */
/* O1 — Chebyshev derivative of one line (Eqs. 14-18)   */
/* ---------------------------------------------------------------------- */
/* T_k(x_j) = (-1)^k cos(pi j k/(N-1)); argument reduced in integers. */
static real cheb_T(int N, int k, int j) {
  int64_t m = ((int64_t)j * k) % (2 * (int64_t)(N - 1));
  real v = R_COS(R_PI * (real)m / (real)(N - 1));
  return (k & 1) ? -v : v;
}

/* u, du have stride `st`; derivative w.r.t. the reference coordinate x in [-1,1]. */
static void cheb_line(int N, const real* u, int64_t st, real* du, int64_t dst) {
  real* ut = malloc(sizeof(real) * N); real* dt = malloc(sizeof(real) * (N + 1));
  /* (a) PhysToSpec, Eq. 17: u~_k = (2/(N-1)) (1/c_k) sum_j (1/c_j) u_j T_k(x_j) */
  for (int k = 0; k < N; ++k) {
    real s = 0;
    for (int j = 0; j < N; ++j) { real cj = (j == 0 || j == N - 1) ? 2 : 1; s += u[j * st] * cheb_T(N, k, j) / cj; }
    real ck = (k == 0 || k == N - 1) ? 2 : 1;
    ut[k] = 2 * s / ((real)(N - 1) * ck);
  }
  /* (b) modal derivative, Eq. 18, by the downward recurrence
   *     c_{k-1} u'~_{k-1} = u'~_{k+1} + 2 k u~_k,  c_0 = 2 else 1 */
  dt[N] = 0; dt[N - 1] = 0;
  for (int k = N - 1; k >= 1; --k) { real c = (k - 1 == 0) ? 2 : 1; dt[k - 1] = (dt[k + 1] + 2 * (real)k * ut[k]) / c; }
  /* (c) SpecToPhys, Eq. 16 */
  for (int j = 0; j < N; ++j) { real s = 0; for (int k = 0; k < N; ++k) s += dt[k] * cheb_T(N, k, j); du[j * dst] = s; }
  free(ut); free(dt);
}

void ora_cheb_derivative_line(int N, const double* u, double* du) {
  real* a = malloc(sizeof(real) * N); real* b = malloc(sizeof(real) * N);
  for (int j = 0; j < N; ++j) a[j] = u[j];
  cheb_line(N, a, 1, b, 1);
  for (int j = 0; j < N; ++j) du[j] = (double)b[j];
  free(a); free(b);
}

/* ---------------------------------------------------------------------- */
/* O15 — Fourier derivative / filter of one periodic line (the S1 factor  */
/* of the cylindrical shells the paper names for binary runs,             */
/* PAPER.md:79, 564; it gives no formulas: DESIGN.md reading S25).  The   */
/* same three steps as Eqs. 14-18 with the basis e^{i m phi}:             */
/*  (a) PhysToSpec  a_m = (1/N) sum_k u_k cos(m phi_k),                   */
/*                  b_m = (1/N) sum_k u_k sin(m phi_k),  phi_k = 2 pi k/N */
/*  (b) modal step: derivative (a_m, b_m) -> (m b_m, -m a_m); filter      */
/*      (a_m, b_m) -> sigma_m (a_m, b_m)                                  */
/*  (c) SpecToPhys  u_k = a_0 + 2 sum_{0<m<N/2} (a_m cos + b_m sin)       */
/*                        [+ a_{N/2} cos(N phi_k / 2) for even N]         */
/* The derivative of the Nyquist mode of an even N vanishes at the nodes  */
/* (d/dphi cos(N phi/2) = -(N/2) sin(N phi_k/2) = 0) and is dropped.      */
/* ---------------------------------------------------------------------- */
static real four_c(int N, int m, int k) { int64_t q = ((int64_t)m * k) % N; return R_COS(2 * R_PI * (real)q / (real)N); }
static real four_s(int N, int m, int k) { int64_t q = ((int64_t)m * k) % N; return R_SIN(2 * R_PI * (real)q / (real)N); }

/* mode 0: derivative d/dphi; mode 1: filter with sigma[0 .. N/2].  u, out have strides st, dst; out may alias u. */
static void fourier_line(int N, const real* u, int64_t st, real* out, int64_t dst, int mode, const double* sigma) {
  int M = N / 2;
  real* a = malloc(sizeof(real) * (M + 1)); real* b = malloc(sizeof(real) * (M + 1)); real* o = malloc(sizeof(real) * N);
  for (int m = 0; m <= M; ++m) {
    real sa = 0, sb = 0;
    for (int k = 0; k < N; ++k) { sa += u[k * st] * four_c(N, m, k); sb += u[k * st] * four_s(N, m, k); }
    a[m] = sa / (real)N; b[m] = sb / (real)N;
  }
  for (int m = 0; m <= M; ++m) {
    if (mode == 0) { real am = a[m]; a[m] = (real)m * b[m]; b[m] = -(real)m * am; if (2 * m == N) a[m] = b[m] = 0; }
    else { a[m] *= (real)sigma[m]; b[m] *= (real)sigma[m]; }
  }
  for (int k = 0; k < N; ++k) {
    real s0 = a[0];
    for (int m = 1; m <= M; ++m) {
      if (2 * m == N) s0 += a[m] * four_c(N, m, k);
      else s0 += 2 * (a[m] * four_c(N, m, k) + b[m] * four_s(N, m, k));
    }
    o[k] = s0;
  }
  for (int k = 0; k < N; ++k) out[k * dst] = o[k];
  free(a); free(b); free(o);
}

void ora_fourier_derivative_line(int N, const double* u, double* du) {
  real* a = malloc(sizeof(real) * N); real* b = malloc(sizeof(real) * N);
  for (int j = 0; j < N; ++j) a[j] = u[j];
  fourier_line(N, a, 1, b, 1, 0, NULL);
  for (int j = 0; j < N; ++j) du[j] = (double)b[j];
  free(a); free(b);
}

/* ---------------------------------------------------------------------- */
/* O2 — shell angular derivatives through Y_lm         */
/* ---------------------------------------------------------------------- */
typedef struct {
  int L, nth, nph;
  real *ct, *w;        /* cos(theta_j), GL weights */
  real *pb, *dpb;      /* Pbar_lm(theta_j), dPbar_lm/dtheta: index [(l*(L+1)+m)*nth + j], m<=l */
  real *cs, *sn;       /* cos(m phi_k), sin(m phi_k): [m*nph + k] */
} ylm_table;

/* Orthonormalised associated Legendre functions Pbar_lm (so that Y_lm = Pbar_lm e^{i m phi}
 * is orthonormal on the sphere, Condon-Shortley phase), by the standard recurrences. */
static void pbar_all(int L, real ct, real* pb, real* dpb) {
  int n = L + 1; real st = R_SQRT(1 - ct * ct);
  for (int i = 0; i < n * n; ++i) { pb[i] = 0; dpb[i] = 0; }
  pb[0] = R_SQRT(1 / (4 * R_PI));
  for (int m = 1; m <= L; ++m) pb[m * n + m] = -R_SQRT((real)(2 * m + 1) / (real)(2 * m)) * st * pb[(m - 1) * n + (m - 1)];
  for (int m = 0; m < L; ++m) pb[(m + 1) * n + m] = R_SQRT((real)(2 * m + 3)) * ct * pb[m * n + m];
  for (int m = 0; m <= L; ++m) for (int l = m + 2; l <= L; ++l) {
    real a = R_SQRT((real)(4 * l * l - 1) / (real)(l * l - m * m));
    real b = R_SQRT((real)((l - 1) * (l - 1) - m * m) / (real)(4 * (l - 1) * (l - 1) - 1));
    pb[l * n + m] = a * (ct * pb[(l - 1) * n + m] - b * pb[(l - 2) * n + m]);
  }
  /* sin(theta) dPbar_lm/dtheta = l cos(theta) Pbar_lm - sqrt((2l+1)/(2l-1) (l^2-m^2)) Pbar_{l-1,m} */
  for (int l = 0; l <= L; ++l) for (int m = 0; m <= l; ++m) {
    real prev = (l - 1 >= m) ? pb[(l - 1) * n + m] : 0;
    real f = (l > 0) ? R_SQRT((real)(2 * l + 1) / (real)(2 * l - 1) * (real)(l * l - m * m)) : 0;
    dpb[l * n + m] = ((real)l * ct * pb[l * n + m] - f * prev) / st;
  }
}

static ylm_table* ylm_build(int L) {
  ylm_table* t = malloc(sizeof(ylm_table));
  int n = L + 1; t->L = L; t->nth = n; t->nph = 2 * n;
  t->ct = malloc(sizeof(real) * n); t->w = malloc(sizeof(real) * n); gl_nodes(L, t->ct, t->w);
  t->pb = malloc(sizeof(real) * n * n * n); t->dpb = malloc(sizeof(real) * n * n * n);
  real* a = malloc(sizeof(real) * n * n); real* b = malloc(sizeof(real) * n * n);
  for (int j = 0; j < n; ++j) {
    pbar_all(L, t->ct[j], a, b);
    for (int i = 0; i < n * n; ++i) { t->pb[(int64_t)i * n + j] = a[i]; t->dpb[(int64_t)i * n + j] = b[i]; }
  }
  free(a); free(b);
  t->cs = malloc(sizeof(real) * n * t->nph); t->sn = malloc(sizeof(real) * n * t->nph);
  for (int m = 0; m <= L; ++m) for (int k = 0; k < t->nph; ++k) {
    int64_t q = ((int64_t)m * k) % t->nph; real ang = 2 * R_PI * (real)q / (real)t->nph;
    t->cs[m * t->nph + k] = R_COS(ang); t->sn[m * t->nph + k] = R_SIN(ang);
  }
  return t;
}
static void ylm_free(ylm_table* t) { free(t->ct); free(t->w); free(t->pb); free(t->dpb); free(t->cs); free(t->sn); free(t); }

/* Pbar_lm and dPbar_lm/dtheta at one colatitude, [l*(L+1)+m] (for the pins). */
void ora_pbar(int L, double theta, double* pb, double* dpb) {
  int n = L + 1; real* a = malloc(sizeof(real) * n * n); real* b = malloc(sizeof(real) * n * n);
  pbar_all(L, R_COS((real)theta), a, b);
  for (int i = 0; i < n * n; ++i) { pb[i] = (double)a[i]; dpb[i] = (double)b[i]; }
  free(a); free(b);
}

/* One (theta,phi) plane u[nth][nph] (strides given) -> out0 = d/dtheta, out1 = d/dphi,
 * or (mode 1) out0 = the projection synthesis(analysis(u)).
 *   a_lm = sum_{j,k} w_j (2 pi/N_phi) conj(Y_lm(theta_j,phi_k)) u_jk,  0<=l<=L, 0<=m<=l
 *   real u:  u = sum_l [ a_l0 Y_l0 + 2 Re sum_{m>0} a_lm Y_lm ]  (a_{l,-m} = (-1)^m conj a_lm)
 *   d_theta u = same with dPbar/dtheta;  d_phi u = same with (i m) a_lm.
 * Explicit quadruple loops, Eq. 23-24 / SURVEY O2; both derivatives go through a_lm (S8). */
static void shell_plane(const ylm_table* t, const real* u, real* out0, real* out1, int mode) {
  int L = t->L, n = t->nth, nph = t->nph;
  real* are = calloc((size_t)n * n, sizeof(real)); real* aim = calloc((size_t)n * n, sizeof(real));
  real dphi = 2 * R_PI / (real)nph;
  for (int l = 0; l <= L; ++l) for (int m = 0; m <= l; ++m) {
    real sr = 0, si = 0; const real* pb = t->pb + (int64_t)(l * n + m) * n;
    for (int j = 0; j < n; ++j) for (int k = 0; k < nph; ++k) {
      real f = t->w[j] * dphi * pb[j] * u[j * nph + k];
      sr += f * t->cs[m * nph + k]; si -= f * t->sn[m * nph + k];
    }
    are[l * n + m] = sr; aim[l * n + m] = si;
  }
  for (int j = 0; j < n; ++j) for (int k = 0; k < nph; ++k) {
    real s0 = 0, s1 = 0;
    for (int l = 0; l <= L; ++l) for (int m = 0; m <= l; ++m) {
      real fac = (m == 0) ? 1 : 2; real ar = are[l * n + m], ai = aim[l * n + m];
      real c = t->cs[m * nph + k], s = t->sn[m * nph + k];
      real re = ar * c - ai * s;            /* Re(a e^{i m phi}) */
      real im = ar * s + ai * c;            /* Im(a e^{i m phi}) */
      if (mode == 0) {
        s0 += fac * t->dpb[(int64_t)(l * n + m) * n + j] * re;
        s1 += fac * t->pb[(int64_t)(l * n + m) * n + j] * (-(real)m * im);   /* Re(i m a e^{i m phi}) */
      } else {
        s0 += fac * t->pb[(int64_t)(l * n + m) * n + j] * re;
      }
    }
    out0[j * nph + k] = s0; if (mode == 0) out1[j * nph + k] = s1;
  }
  free(are); free(aim);
}

void ora_shell_angular(int L, const double* u, double* dth, double* dph) {
  ylm_table* t = ylm_build(L); int np = t->nth * t->nph;
  real* a = malloc(sizeof(real) * np); real* b = malloc(sizeof(real) * np); real* c = malloc(sizeof(real) * np);
  for (int i = 0; i < np; ++i) a[i] = u[i];
  shell_plane(t, a, b, c, 0);
  for (int i = 0; i < np; ++i) { dth[i] = (double)b[i]; dph[i] = (double)c[i]; }
  free(a); free(b); free(c); ylm_free(t);
}
void ora_shell_project(int L, const double* u, double* out) {
  ylm_table* t = ylm_build(L); int np = t->nth * t->nph;
  real* a = malloc(sizeof(real) * np); real* b = malloc(sizeof(real) * np);
  for (int i = 0; i < np; ++i) a[i] = u[i];
  shell_plane(t, a, b, NULL, 1);
  for (int i = 0; i < np; ++i) out[i] = (double)b[i];
  free(a); free(b); ylm_free(t);
}

/* ---------------------------------------------------------------------- */
/* O9 — spectral filter (NEXT-1).  "Spectral filtering of 1D basis        */
/* functions is similar to differentiation, the only difference being the */
/* specific form of the transformation matrix"; on     */
/* shells: PhysToSpec -> filter -> SpecToPhys, here    */
/* the scalar-in-l part; "we do not include a filter along the r-axis"    */
/* (PAPER.md:500).  The filter function sigma is an INPUT (tables).       */
/* ---------------------------------------------------------------------- */
/* one Chebyshev line in place: u~_k <- sigma[k] u~_k  (Eqs. 17, 16) */
static void cheb_filter_line(int N, real* u, int64_t st, const double* sigma) {
  real* ut = malloc(sizeof(real) * N);
  for (int k = 0; k < N; ++k) {
    real s = 0;
    for (int j = 0; j < N; ++j) { real cj = (j == 0 || j == N - 1) ? 2 : 1; s += u[j * st] * cheb_T(N, k, j) / cj; }
    real ck = (k == 0 || k == N - 1) ? 2 : 1;
    ut[k] = (real)sigma[k] * 2 * s / ((real)(N - 1) * ck);
  }
  for (int j = 0; j < N; ++j) { real s = 0; for (int k = 0; k < N; ++k) s += ut[k] * cheb_T(N, k, j); u[j * st] = s; }
  free(ut);
}

/* one (theta,phi) plane: a_lm <- sigma_l[l] a_lm, then synthesis (Eq. 23 with filtered coefficients) */
static void shell_filter_plane(const ylm_table* t, const real* u, real* out, const double* sigma_l) {
  int L = t->L, n = t->nth, nph = t->nph;
  real* are = calloc((size_t)n * n, sizeof(real)); real* aim = calloc((size_t)n * n, sizeof(real));
  real dphi = 2 * R_PI / (real)nph;
  for (int l = 0; l <= L; ++l) for (int m = 0; m <= l; ++m) {
    real sr = 0, si = 0; const real* pb = t->pb + (int64_t)(l * n + m) * n;
    for (int j = 0; j < n; ++j) for (int k = 0; k < nph; ++k) {
      real f = t->w[j] * dphi * pb[j] * u[j * nph + k];
      sr += f * t->cs[m * nph + k]; si -= f * t->sn[m * nph + k];
    }
    are[l * n + m] = (real)sigma_l[l] * sr; aim[l * n + m] = (real)sigma_l[l] * si;
  }
  for (int j = 0; j < n; ++j) for (int k = 0; k < nph; ++k) {
    real s0 = 0;
    for (int l = 0; l <= L; ++l) for (int m = 0; m <= l; ++m) {
      real fac = (m == 0) ? 1 : 2;
      real re = are[l * n + m] * t->cs[m * nph + k] - aim[l * n + m] * t->sn[m * nph + k];
      s0 += fac * t->pb[(int64_t)(l * n + m) * n + j] * re;
    }
    out[j * nph + k] = s0;
  }
  free(are); free(aim);
}

/* u[ncomp][P] in place.  blocks: sig0/sig1/sig2 = sigma_k along x/y/z ([N_x], [N_y], [N_z]);
 * shells: sig0 = sigma_l ([L+1]), sig1/sig2 unused; cylinders: sig0 / sig1 = sigma_k along rho / z ([N_rho], [N_z]),
 * sig2 = sigma_m of the Fourier modes ([N_phi/2 + 1]). */
int ora_filter_subdomain(const ora_subdomain* sd, int ncomp, double* u, const double* sig0, const double* sig1, const double* sig2) {
  int n0, n1, n2; dims(sd, &n0, &n1, &n2); int64_t P = (int64_t)n0 * n1 * n2;
  if (sd->kind == 1) {
    int nn[3] = {n0, n1, n2}; int64_t st[3] = {(int64_t)n1 * n2, n2, 1}; const double* sg[3] = {sig0, sig1, sig2};
#pragma omp parallel for schedule(dynamic)
    for (int c = 0; c < ncomp; ++c) {
      real* w = malloc(sizeof(real) * P);
      for (int64_t p = 0; p < P; ++p) w[p] = u[(int64_t)c * P + p];
      for (int d = 0; d < 3; ++d) {
        int e = (d + 1) % 3, f = (d + 2) % 3;
        for (int a = 0; a < nn[e]; ++a) for (int b = 0; b < nn[f]; ++b) cheb_filter_line(nn[d], w + a * st[e] + b * st[f], st[d], sg[d]);
      }
      for (int64_t p = 0; p < P; ++p) u[(int64_t)c * P + p] = (double)w[p];
      free(w);
    }
    return 0;
  }
  if (sd->kind == 2) {
#pragma omp parallel for schedule(dynamic)
    for (int c = 0; c < ncomp; ++c) {
      real* w = malloc(sizeof(real) * P);
      for (int64_t p = 0; p < P; ++p) w[p] = u[(int64_t)c * P + p];
      for (int j = 0; j < n1; ++j) for (int k = 0; k < n2; ++k) cheb_filter_line(n0, w + (int64_t)j * n2 + k, (int64_t)n1 * n2, sig0);
      for (int i = 0; i < n0; ++i) for (int k = 0; k < n2; ++k) cheb_filter_line(n1, w + (int64_t)i * n1 * n2 + k, n2, sig1);
      for (int i = 0; i < n0; ++i) for (int j = 0; j < n1; ++j) { real* l = w + ((int64_t)i * n1 + j) * n2; fourier_line(n2, l, 1, l, 1, 1, sig2); }
      for (int64_t p = 0; p < P; ++p) u[(int64_t)c * P + p] = (double)w[p];
      free(w);
    }
    return 0;
  }
  int L = sd->n[1]; ylm_table* t = ylm_build(L); int64_t np = (int64_t)n1 * n2;
#pragma omp parallel for schedule(dynamic)
  for (int c = 0; c < ncomp; ++c) {
    real* a = malloc(sizeof(real) * np); real* b = malloc(sizeof(real) * np);
    for (int i = 0; i < n0; ++i) {
      double* uc = u + (int64_t)c * P + i * np;
      for (int64_t q = 0; q < np; ++q) a[q] = uc[q];
      shell_filter_plane(t, a, b, sig0);
      for (int64_t q = 0; q < np; ++q) uc[q] = (double)b[q];
    }
    free(a); free(b);
  }
  ylm_free(t);
  return 0;
}

/* ---------------------------------------------------------------------- */
/* O3 — Cartesian gradient of ncomp scalar fields on one subdomain        */
/* ---------------------------------------------------------------------- */
/* u[ncomp][P] (real) -> g[3][ncomp][P] = d/dx, d/dy, d/dz. */
static void gradient_real(const ora_subdomain* sd, int ncomp, const real* u, real* g) {
  int n0, n1, n2; dims(sd, &n0, &n1, &n2); int64_t P = (int64_t)n0 * n1 * n2;
  if (sd->kind == 1) {
    /* blocks: O1 along x, y, z with the affine map factor 2/(hi-lo) (Eq. 22) */
    int nn[3] = {n0, n1, n2}; int64_t st[3] = {(int64_t)n1 * n2, n2, 1};
#pragma omp parallel for schedule(dynamic)
    for (int c = 0; c < ncomp; ++c) for (int d = 0; d < 3; ++d) {
      real sc = 2 / ((real)sd->hi[d] - (real)sd->lo[d]);
      int e = (d + 1) % 3, f = (d + 2) % 3;
      for (int a = 0; a < nn[e]; ++a) for (int b = 0; b < nn[f]; ++b) {
        int64_t off = a * st[e] + b * st[f];
        real* out = g + ((int64_t)d * ncomp + c) * P + off;
        cheb_line(nn[d], u + (int64_t)c * P + off, st[d], out, st[d]);
        for (int i = 0; i < nn[d]; ++i) out[i * st[d]] *= sc;
      }
    }
    return;
  }
  if (sd->kind == 2) {
    /* cylindrical shells (O15): O1 in rho and in z, the Fourier derivative in phi, then Eq. 8 with the cylindrical Jacobian
     *   d_x = cos(phi) d_rho - (sin(phi)/rho) d_phi,  d_y = sin(phi) d_rho + (cos(phi)/rho) d_phi,  d_z = d_z */
    real* xr = malloc(sizeof(real) * n0); cgl_nodes(n0, xr);
    real scr = 2 / ((real)sd->hi[0] - (real)sd->lo[0]), scz = 2 / ((real)sd->hi[1] - (real)sd->lo[1]);
    int64_t pl = (int64_t)n1 * n2;
#pragma omp parallel for schedule(dynamic)
    for (int c = 0; c < ncomp; ++c) {
      const real* uc = u + (int64_t)c * P;
      real* dr = malloc(sizeof(real) * P); real* dz = malloc(sizeof(real) * P); real* dph = malloc(sizeof(real) * P);
      for (int64_t q = 0; q < pl; ++q) cheb_line(n0, uc + q, pl, dr + q, pl);
      for (int i = 0; i < n0; ++i) for (int k = 0; k < n2; ++k) cheb_line(n1, uc + i * pl + k, n2, dz + i * pl + k, n2);
      for (int i = 0; i < n0; ++i) for (int j = 0; j < n1; ++j) fourier_line(n2, uc + i * pl + (int64_t)j * n2, 1, dph + i * pl + (int64_t)j * n2, 1, 0, NULL);
      for (int i = 0; i < n0; ++i) {
        real rho = (real)sd->lo[0] + ((real)sd->hi[0] - (real)sd->lo[0]) * (xr[i] + 1) / 2;
        for (int j = 0; j < n1; ++j) for (int k = 0; k < n2; ++k) {
          real ph = 2 * R_PI * (real)k / (real)n2, cp = R_COS(ph), sp = R_SIN(ph);
          int64_t p = i * pl + (int64_t)j * n2 + k;
          real a = scr * dr[p], b = scz * dz[p], e = dph[p];
          g[((int64_t)0 * ncomp + c) * P + p] = cp * a - (sp / rho) * e;
          g[((int64_t)1 * ncomp + c) * P + p] = sp * a + (cp / rho) * e;
          g[((int64_t)2 * ncomp + c) * P + p] = b;
        }
      }
      free(dr); free(dz); free(dph);
    }
    free(xr);
    return;
  }
  /* shells: O1 in r, O2 in (theta,phi), then Eq. 8 with the spherical Jacobian */
  int L = sd->n[1]; ylm_table* t = ylm_build(L); int64_t np = (int64_t)n1 * n2;
  real* xr = malloc(sizeof(real) * n0); cgl_nodes(n0, xr);
  real sc = 2 / ((real)sd->hi[0] - (real)sd->lo[0]);
#pragma omp parallel for schedule(dynamic)
  for (int c = 0; c < ncomp; ++c) {
    const real* uc = u + (int64_t)c * P;
    real* dr = malloc(sizeof(real) * P); real* dth = malloc(sizeof(real) * P); real* dph = malloc(sizeof(real) * P);
    for (int64_t q = 0; q < np; ++q) { cheb_line(n0, uc + q, np, dr + q, np); }
    for (int64_t p = 0; p < P; ++p) dr[p] *= sc;
    for (int i = 0; i < n0; ++i) shell_plane(t, uc + i * np, dth + i * np, dph + i * np, 0);
    for (int i = 0; i < n0; ++i) {
      real r = (real)sd->lo[0] + ((real)sd->hi[0] - (real)sd->lo[0]) * (xr[i] + 1) / 2;
      for (int j = 0; j < n1; ++j) for (int k = 0; k < n2; ++k) {
        real ct = t->ct[j], st = R_SQRT(1 - ct * ct); real ph = 2 * R_PI * (real)k / (real)n2;
        real cp = R_COS(ph), sp = R_SIN(ph); int64_t p = i * np + (int64_t)j * n2 + k;
        real a = dr[p], b = dth[p], e = dph[p];
        g[((int64_t)0 * ncomp + c) * P + p] = st * cp * a + (ct * cp / r) * b - (sp / (r * st)) * e;
        g[((int64_t)1 * ncomp + c) * P + p] = st * sp * a + (ct * sp / r) * b + (cp / (r * st)) * e;
        g[((int64_t)2 * ncomp + c) * P + p] = ct * a - (st / r) * b;
      }
    }
    free(dr); free(dth); free(dph);
  }
  free(xr); ylm_free(t);
}

void ora_gradient(const ora_subdomain* sd, int ncomp, const double* u, double* g) {
  int64_t P = ora_num_points(sd);
  real* a = malloc(sizeof(real) * ncomp * P); real* b = malloc(sizeof(real) * 3 * ncomp * P);
  for (int64_t i = 0; i < ncomp * P; ++i) a[i] = u[i];
  gradient_real(sd, ncomp, a, b);
  for (int64_t i = 0; i < 3 * ncomp * P; ++i) g[i] = (double)b[i];
  free(a); free(b);
}

/* ---------------------------------------------------------------------- */
/* O4 — geometry at a point                                               */
/* ---------------------------------------------------------------------- */
typedef struct { real ginv[3][3], lapse, shift[3], psiinv[4][4], tup[4], tdn[4]; } geom;

static int geometry(const real psi[4][4], geom* G) {
  real g[3][3]; for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) g[i][j] = psi[i + 1][j + 1];
  real c00 = g[1][1] * g[2][2] - g[1][2] * g[2][1], c01 = g[1][2] * g[2][0] - g[1][0] * g[2][2], c02 = g[1][0] * g[2][1] - g[1][1] * g[2][0];
  real det = g[0][0] * c00 + g[0][1] * c01 + g[0][2] * c02;
  if (!(det > 0)) return 1;
  /* g^{ij} = cofactor(j,i)/det */
  G->ginv[0][0] = c00 / det; G->ginv[1][0] = c01 / det; G->ginv[2][0] = c02 / det;
  G->ginv[0][1] = (g[0][2] * g[2][1] - g[0][1] * g[2][2]) / det;
  G->ginv[1][1] = (g[0][0] * g[2][2] - g[0][2] * g[2][0]) / det;
  G->ginv[2][1] = (g[0][1] * g[2][0] - g[0][0] * g[2][1]) / det;
  G->ginv[0][2] = (g[0][1] * g[1][2] - g[0][2] * g[1][1]) / det;
  G->ginv[1][2] = (g[0][2] * g[1][0] - g[0][0] * g[1][2]) / det;
  G->ginv[2][2] = (g[0][0] * g[1][1] - g[0][1] * g[1][0]) / det;
  real n2 = -psi[0][0];
  for (int i = 0; i < 3; ++i) { real s = 0; for (int j = 0; j < 3; ++j) s += G->ginv[i][j] * psi[0][j + 1]; G->shift[i] = s; }
  for (int i = 0; i < 3; ++i) n2 += G->shift[i] * psi[0][i + 1];
  if (!(n2 > 0)) return 1;
  G->lapse = R_SQRT(n2);
  G->psiinv[0][0] = -1 / n2;
  for (int i = 0; i < 3; ++i) { G->psiinv[0][i + 1] = G->shift[i] / n2; G->psiinv[i + 1][0] = G->shift[i] / n2; }
  for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) G->psiinv[i + 1][j + 1] = G->ginv[i][j] - G->shift[i] * G->shift[j] / n2;
  G->tup[0] = 1 / G->lapse; for (int i = 0; i < 3; ++i) G->tup[i + 1] = -G->shift[i] / G->lapse;
  G->tdn[0] = -G->lapse; G->tdn[1] = G->tdn[2] = G->tdn[3] = 0;
  return 0;
}

/* psi[16] -> ginv[9], lapse, shift[3], psiinv[16]; returns 1 if non-physical. */
int ora_geometry_point(const double* psi, double* ginv, double* lapse, double* shift, double* psiinv) {
  real p[4][4]; geom G; for (int a = 0; a < 4; ++a) for (int b = 0; b < 4; ++b) p[a][b] = psi[a * 4 + b];
  if (geometry(p, &G)) return 1;
  for (int i = 0; i < 3; ++i) { shift[i] = (double)G.shift[i]; for (int j = 0; j < 3; ++j) ginv[i * 3 + j] = (double)G.ginv[i][j]; }
  *lapse = (double)G.lapse;
  for (int a = 0; a < 4; ++a) for (int b = 0; b < 4; ++b) psiinv[a * 4 + b] = (double)G.psiinv[a][b];
  return 0;
}

/* ---------------------------------------------------------------------- */
/* O5 — GH right-hand side at a point; O8 — constraints at a point        */
/* ---------------------------------------------------------------------- */
typedef struct {
  real psi[4][4], Pi[4][4], Phi[3][4][4];
  real dpsi[3][4][4], dPi[3][4][4], dPhi[3][3][4][4]; /* spectral d_k: dPhi[k][i][a][b] = d_k Phi_iab */
  real H[4], dH[3][4];                                /* dH[i][b] = d_i H_b ; d_0 H_b = 0 */
} point_in;

/* Christoffels of the first kind from the FIRST-ORDER variables:
 * d_0 psi = -N Pi + N^i Phi_i, d_i psi = Phi_i (SURVEY O5 "two meanings of d psi"). */
static void christoffel(const point_in* in, const geom* G, real Gam[4][4][4], real Gam1[4]) {
  real D[4][4][4];
  for (int a = 0; a < 4; ++a) for (int b = 0; b < 4; ++b) {
    real s = -G->lapse * in->Pi[a][b];
    for (int i = 0; i < 3; ++i) s += G->shift[i] * in->Phi[i][a][b];
    D[0][a][b] = s;
    for (int i = 0; i < 3; ++i) D[i + 1][a][b] = in->Phi[i][a][b];
  }
  for (int a = 0; a < 4; ++a) for (int b = 0; b < 4; ++b) for (int c = 0; c < 4; ++c)
    Gam[a][b][c] = (D[b][a][c] + D[c][a][b] - D[a][b][c]) / 2;
  for (int a = 0; a < 4; ++a) { real s = 0; for (int b = 0; b < 4; ++b) for (int c = 0; c < 4; ++c) s += G->psiinv[b][c] * Gam[a][b][c]; Gam1[a] = s; }
}

static int rhs_point(const point_in* in, const real gam[3], real dtpsi[4][4], real dtPi[4][4], real dtPhi[3][4][4]) {
  geom G; if (geometry(in->psi, &G)) return 1;
  real g0 = gam[0], g1 = gam[1], g2 = gam[2], N = G.lapse;
  real Gam[4][4][4], Gam1[4], C[4]; christoffel(in, &G, Gam, Gam1);
  for (int a = 0; a < 4; ++a) C[a] = in->H[a] + Gam1[a];
  real dH4[4][4]; for (int b = 0; b < 4; ++b) { dH4[0][b] = 0; for (int i = 0; i < 3; ++i) dH4[i + 1][b] = in->dH[i][b]; }
  real tC = 0; for (int c = 0; c < 4; ++c) tC += G.tup[c] * C[c];
  real ttPi = 0; for (int c = 0; c < 4; ++c) for (int d = 0; d < 4; ++d) ttPi += G.tup[c] * G.tup[d] * in->Pi[c][d];
  for (int a = 0; a < 4; ++a) for (int b = 0; b < 4; ++b) {
    real sdpsi = 0, sPhi = 0, sdPi = 0;
    for (int k = 0; k < 3; ++k) { sdpsi += G.shift[k] * in->dpsi[k][a][b]; sPhi += G.shift[k] * in->Phi[k][a][b]; sdPi += G.shift[k] * in->dPi[k][a][b]; }
    dtpsi[a][b] = (1 + g1) * sdpsi - N * in->Pi[a][b] - g1 * sPhi;
    real gdPhi = 0; for (int k = 0; k < 3; ++k) for (int i = 0; i < 3; ++i) gdPhi += G.ginv[k][i] * in->dPhi[k][i][a][b];
    real quad = 0;
    for (int c = 0; c < 4; ++c) for (int d = 0; d < 4; ++d) {
      real t = 0;
      for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) t += G.ginv[i][j] * in->Phi[i][c][a] * in->Phi[j][d][b];
      t -= in->Pi[c][a] * in->Pi[d][b];
      for (int e = 0; e < 4; ++e) for (int f = 0; f < 4; ++f) t -= G.psiinv[e][f] * Gam[a][c][e] * Gam[b][d][f];
      quad += G.psiinv[c][d] * t;
    }
    real nabH = (dH4[a][b] + dH4[b][a]) / 2;
    for (int c = 0; c < 4; ++c) for (int d = 0; d < 4; ++d) nabH -= G.psiinv[c][d] * Gam[d][a][b] * in->H[c];
    real tPigPhi = 0;
    for (int c = 0; c < 4; ++c) for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) tPigPhi += G.tup[c] * in->Pi[c][i + 1] * G.ginv[i][j] * in->Phi[j][a][b];
    dtPi[a][b] = sdPi - N * gdPhi + g1 * g2 * sdpsi + 2 * N * quad - 2 * N * nabH - N * ttPi * in->Pi[a][b] / 2 - N * tPigPhi
               + N * g0 * (G.tdn[b] * C[a] + G.tdn[a] * C[b] - in->psi[a][b] * tC) - g1 * g2 * sPhi;
    for (int i = 0; i < 3; ++i) {
      real sdPhi = 0; for (int k = 0; k < 3; ++k) sdPhi += G.shift[k] * in->dPhi[k][i][a][b];
      real ttPhi = 0; for (int c = 0; c < 4; ++c) for (int d = 0; d < 4; ++d) ttPhi += G.tup[c] * G.tup[d] * in->Phi[i][c][d];
      real gtPP = 0;
      for (int j = 0; j < 3; ++j) for (int k = 0; k < 3; ++k) for (int c = 0; c < 4; ++c) gtPP += G.ginv[j][k] * G.tup[c] * in->Phi[i][j + 1][c] * in->Phi[k][a][b];
      dtPhi[i][a][b] = sdPhi - N * in->dPi[i][a][b] + N * g2 * in->dpsi[i][a][b] + N * ttPhi * in->Pi[a][b] / 2 + N * gtPP - N * g2 * in->Phi[i][a][b];
    }
  }
  return 0;
}

/* C_a[4], C_iab[3][4][4], C_ijab[3][3][4][4] */
static int constraints_point(const point_in* in, real Ca[4], real Ciab[3][4][4], real Cijab[3][3][4][4]) {
  geom G; if (geometry(in->psi, &G)) return 1;
  real Gam[4][4][4], Gam1[4]; christoffel(in, &G, Gam, Gam1);
  for (int a = 0; a < 4; ++a) Ca[a] = in->H[a] + Gam1[a];
  for (int i = 0; i < 3; ++i) for (int a = 0; a < 4; ++a) for (int b = 0; b < 4; ++b) Ciab[i][a][b] = in->dpsi[i][a][b] - in->Phi[i][a][b];
  for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) for (int a = 0; a < 4; ++a) for (int b = 0; b < 4; ++b)
    Cijab[i][j][a][b] = in->dPhi[i][j][a][b] - in->dPhi[j][i][a][b];
  return 0;
}

/* Flat double interface to one point, FULL (unsymmetrised) arrays, row-major:
 * psi[16], Pi[16], Phi[48], dpsi[48], dPi[48], dPhi[144] ([k][i][a][b]), H[4], dH[12] ([i][b]). */
static void load_point(point_in* in, const double* psi, const double* Pi, const double* Phi, const double* dpsi,
                       const double* dPi, const double* dPhi, const double* H, const double* dH) {
  for (int a = 0; a < 4; ++a) for (int b = 0; b < 4; ++b) { in->psi[a][b] = psi[a * 4 + b]; in->Pi[a][b] = Pi[a * 4 + b]; }
  for (int i = 0; i < 3; ++i) for (int a = 0; a < 4; ++a) for (int b = 0; b < 4; ++b) {
    in->Phi[i][a][b] = Phi[(i * 4 + a) * 4 + b]; in->dpsi[i][a][b] = dpsi[(i * 4 + a) * 4 + b]; in->dPi[i][a][b] = dPi[(i * 4 + a) * 4 + b];
    for (int k = 0; k < 3; ++k) in->dPhi[k][i][a][b] = dPhi[((k * 3 + i) * 4 + a) * 4 + b];
  }
  for (int a = 0; a < 4; ++a) in->H[a] = H[a];
  for (int i = 0; i < 3; ++i) for (int b = 0; b < 4; ++b) in->dH[i][b] = dH[i * 4 + b];
}

int ora_rhs_point(const double* psi, const double* Pi, const double* Phi, const double* dpsi, const double* dPi,
                  const double* dPhi, const double* H, const double* dH, const double* gamma,
                  double* dtpsi, double* dtPi, double* dtPhi) {
  point_in in; load_point(&in, psi, Pi, Phi, dpsi, dPi, dPhi, H, dH);
  real g[3] = {gamma[0], gamma[1], gamma[2]}, a[4][4], b[4][4], c[3][4][4];
  if (rhs_point(&in, g, a, b, c)) return 1;
  for (int x = 0; x < 4; ++x) for (int y = 0; y < 4; ++y) { dtpsi[x * 4 + y] = (double)a[x][y]; dtPi[x * 4 + y] = (double)b[x][y];
    for (int i = 0; i < 3; ++i) dtPhi[(i * 4 + x) * 4 + y] = (double)c[i][x][y]; }
  return 0;
}

/* ---------------------------------------------------------------------- */
/* O14 — dual-frame right-hand side (NEXT-4; "data is represented at        */
/* collocation points at fixed grid-coordinates ... The evolution equations, */
/* however, are formulated in asymptotic inertial coordinates.  The two      */
/* coordinate systems share the same time-coordinate, and their spatial      */
/* coordinates are related by a time-dependent coordinate transformation",   */
/* PAPER.md:87).  With grid coordinates xbar, inertial x = x(xbar, t),       */
/*   Jm_i^k = d xbar^k / d x^i   and   v^i = (d x^i / d t) at fixed xbar:    */
/*   d_i u = Jm_i^k dbar_k u          (DiffJac, Eq. 8)     */
/*   d_t u |_xbar = F[u, d_i u] + v^i d_i u                                   */
/* where F is the single-frame right-hand side O5 and the tensor components  */
/* stay inertial-frame Cartesian.                                            */
/* ---------------------------------------------------------------------- */
static void map_derivs(point_in* in, const real J[3][3]) {
  for (int a = 0; a < 4; ++a) for (int b = 0; b < 4; ++b) {
    real o[3], n[3];
    for (int k = 0; k < 3; ++k) o[k] = in->dpsi[k][a][b];
    for (int i = 0; i < 3; ++i) { n[i] = 0; for (int k = 0; k < 3; ++k) n[i] += J[i][k] * o[k]; }
    for (int i = 0; i < 3; ++i) in->dpsi[i][a][b] = n[i];
    for (int k = 0; k < 3; ++k) o[k] = in->dPi[k][a][b];
    for (int i = 0; i < 3; ++i) { n[i] = 0; for (int k = 0; k < 3; ++k) n[i] += J[i][k] * o[k]; }
    for (int i = 0; i < 3; ++i) in->dPi[i][a][b] = n[i];
    for (int j = 0; j < 3; ++j) {
      for (int k = 0; k < 3; ++k) o[k] = in->dPhi[k][j][a][b];
      for (int i = 0; i < 3; ++i) { n[i] = 0; for (int k = 0; k < 3; ++k) n[i] += J[i][k] * o[k]; }
      for (int i = 0; i < 3; ++i) in->dPhi[i][j][a][b] = n[i];
    }
  }
}
static void map_advect(const point_in* in, const real v[3], real a[4][4], real b[4][4], real c[3][4][4]) {
  for (int x = 0; x < 4; ++x) for (int y = 0; y < 4; ++y) for (int i = 0; i < 3; ++i) {
    a[x][y] += v[i] * in->dpsi[i][x][y]; b[x][y] += v[i] * in->dPi[i][x][y];
    for (int j = 0; j < 3; ++j) c[j][x][y] += v[i] * in->dPhi[i][j][x][y];
  }
}

/* one point: the derivative inputs are GRID-frame (dbar_k); Jm[9] row-major Jm[3 i + k], v[3]; dH is inertial-frame */
int ora_rhs_point_map(const double* psi, const double* Pi, const double* Phi, const double* dpsi, const double* dPi,
                      const double* dPhi, const double* H, const double* dH, const double* gamma, const double* Jm, const double* v,
                      double* dtpsi, double* dtPi, double* dtPhi) {
  point_in in; load_point(&in, psi, Pi, Phi, dpsi, dPi, dPhi, H, dH);
  real g[3] = {gamma[0], gamma[1], gamma[2]}, a[4][4], b[4][4], c[3][4][4], J[3][3], vv[3] = {v[0], v[1], v[2]};
  for (int i = 0; i < 3; ++i) for (int k = 0; k < 3; ++k) J[i][k] = Jm[3 * i + k];
  map_derivs(&in, J);
  if (rhs_point(&in, g, a, b, c)) return 1;
  map_advect(&in, vv, a, b, c);
  for (int x = 0; x < 4; ++x) for (int y = 0; y < 4; ++y) { dtpsi[x * 4 + y] = (double)a[x][y]; dtPi[x * 4 + y] = (double)b[x][y];
    for (int i = 0; i < 3; ++i) dtPhi[(i * 4 + x) * 4 + y] = (double)c[i][x][y]; }
  return 0;
}

int ora_constraints_point(const double* psi, const double* Pi, const double* Phi, const double* dpsi, const double* dPhi,
                          const double* H, double* Ca, double* Ciab, double* Cijab) {
  static const double z48[48] = {0}, z12[12] = {0};
  point_in in; load_point(&in, psi, Pi, Phi, dpsi, z48, dPhi, H, z12);
  real a[4], b[3][4][4], c[3][3][4][4];
  if (constraints_point(&in, a, b, c)) return 1;
  for (int x = 0; x < 4; ++x) Ca[x] = (double)a[x];
  for (int i = 0; i < 3; ++i) for (int x = 0; x < 4; ++x) for (int y = 0; y < 4; ++y) { Ciab[(i * 4 + x) * 4 + y] = (double)b[i][x][y];
    for (int j = 0; j < 3; ++j) Cijab[((i * 3 + j) * 4 + x) * 4 + y] = (double)c[i][j][x][y]; }
  return 0;
}

/* ---------------------------------------------------------------------- */
/* subdomain level: storage is the packed 50-component order              */
/*   s(a,b), a<=b: 00,01,02,03,11,12,13,22,23,33 -> 0..9                  */
/*   psi: c=s; Pi: c=10+s; Phi_iab: c=20+10 i+s                           */
/* (the oracle unpacks to FULL arrays before doing any tensor algebra)    */
/* ---------------------------------------------------------------------- */
static const int SYM[4][4] = {{0, 1, 2, 3}, {1, 4, 5, 6}, {2, 5, 7, 8}, {3, 6, 8, 9}};

static void fill_point(point_in* in, const real* u, const real* g, const real* H, const real* gH, int64_t P, int64_t p) {
  for (int a = 0; a < 4; ++a) for (int b = 0; b < 4; ++b) {
    int s = SYM[a][b];
    in->psi[a][b] = u[(int64_t)s * P + p]; in->Pi[a][b] = u[(int64_t)(10 + s) * P + p];
    for (int i = 0; i < 3; ++i) in->Phi[i][a][b] = u[(int64_t)(20 + 10 * i + s) * P + p];
    for (int k = 0; k < 3; ++k) {
      in->dpsi[k][a][b] = g[((int64_t)k * 50 + s) * P + p]; in->dPi[k][a][b] = g[((int64_t)k * 50 + 10 + s) * P + p];
      for (int i = 0; i < 3; ++i) in->dPhi[k][i][a][b] = g[((int64_t)k * 50 + 20 + 10 * i + s) * P + p];
    }
  }
  for (int a = 0; a < 4; ++a) { in->H[a] = H[(int64_t)a * P + p]; for (int i = 0; i < 3; ++i) in->dH[i][a] = gH[((int64_t)i * 4 + a) * P + p]; }
}

/* O6: is point p on a FROZEN face? */
static int frozen(const ora_subdomain* sd, int64_t p) {
  int n0, n1, n2; dims(sd, &n0, &n1, &n2);
  int k = (int)(p % n2), j = (int)((p / n2) % n1), i = (int)(p / ((int64_t)n1 * n2));
  if (sd->kind == 0) return (i == 0 && sd->face[0] == 1) || (i == n0 - 1 && sd->face[1] == 1);
  if (sd->kind == 2)   /* the phi direction is periodic: four faces */
    return (i == 0 && sd->face[0] == 1) || (i == n0 - 1 && sd->face[1] == 1) || (j == 0 && sd->face[2] == 1) || (j == n1 - 1 && sd->face[3] == 1);
  return (i == 0 && sd->face[0] == 1) || (i == n0 - 1 && sd->face[1] == 1) || (j == 0 && sd->face[2] == 1) ||
         (j == n1 - 1 && sd->face[3] == 1) || (k == 0 && sd->face[4] == 1) || (k == n2 - 1 && sd->face[5] == 1);
}

/* ---------------------------------------------------------------------- */
/* O10 — characteristic boundary condition, "freeze what comes in"        */
/* (NEXT-2 (i); the paper's ApplyBCs module,  */
/* which it left on the CPU).  The paper gives no formulas; these are the */
/* characteristic fields of the first-order GH system of ref. [34]'s      */
/* lineage (reading S21).  At a face point with outward unit    */
/* normal n_i = s_i / sqrt(g^{jk} s_j s_k), n^i = g^{ij} n_j:             */
/*   u0_ab   = psi_ab                              speed -(1+g1) n_k N^k  */
/*   u1+-_ab = Pi_ab +- n^i Phi_iab - g2 psi_ab     speed -n_k N^k +- N    */
/*   u2_iab  = (delta_i^k - n_i n^k) Phi_kab        speed -n_k N^k         */
/* The time derivative of every field whose speed is negative (it enters  */
/* the domain) is set to zero, the others keep the value the evolution    */
/* equations give; then back:  dt psi = dt u0,                            */
/*   dt Pi = (dt u1+ + dt u1-)/2 + g2 dt u0,                              */
/*   dt Phi_i = (dt u1+ - dt u1-)/2 n_i + dt u2_i.                        */
/* ---------------------------------------------------------------------- */
static int char_bc_point(const real psi[4][4], const real gam[3], const real s[3], real dtpsi[4][4], real dtPi[4][4],
                         real dtPhi[3][4][4]) {
  geom G; if (geometry(psi, &G)) return 1;
  real nn = 0; for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) nn += G.ginv[i][j] * s[i] * s[j];
  nn = R_SQRT(nn);
  real nd[3], nu[3], nN = 0;
  for (int i = 0; i < 3; ++i) nd[i] = s[i] / nn;
  for (int i = 0; i < 3; ++i) { nu[i] = 0; for (int j = 0; j < 3; ++j) nu[i] += G.ginv[i][j] * nd[j]; }
  for (int k = 0; k < 3; ++k) nN += nd[k] * G.shift[k];
  real v0 = -(1 + gam[1]) * nN, v1p = -nN + G.lapse, v1m = -nN - G.lapse, v2 = -nN;
  for (int a = 0; a < 4; ++a) for (int b = 0; b < 4; ++b) {
    real dpsi = dtpsi[a][b], dPi = dtPi[a][b], dPhi[3] = {dtPhi[0][a][b], dtPhi[1][a][b], dtPhi[2][a][b]};
    real nPhi = 0; for (int i = 0; i < 3; ++i) nPhi += nu[i] * dPhi[i];
    real u0 = dpsi, u1p = dPi + nPhi - gam[2] * dpsi, u1m = dPi - nPhi - gam[2] * dpsi, u2[3];
    for (int i = 0; i < 3; ++i) u2[i] = dPhi[i] - nd[i] * nPhi;
    if (v0 < 0) u0 = 0;
    if (v1p < 0) u1p = 0;
    if (v1m < 0) u1m = 0;
    if (v2 < 0) { u2[0] = u2[1] = u2[2] = 0; }
    dtpsi[a][b] = u0;
    dtPi[a][b] = (u1p + u1m) / 2 + gam[2] * u0;
    for (int i = 0; i < 3; ++i) dtPhi[i][a][b] = (u1p - u1m) / 2 * nd[i] + u2[i];
  }
  return 0;
}

/* for the pins: psi[16], gamma[3], s[3] (outward direction, any length); dtpsi[16], dtPi[16], dtPhi[48] in place;
 * speeds[4] = v0, v1+, v1-, v2 (may be NULL). */
int ora_char_bc_point(const double* psi, const double* gamma, const double* s, double* dtpsi, double* dtPi, double* dtPhi, double* speeds) {
  real p[4][4], a[4][4], b[4][4], c[3][4][4], g3[3] = {gamma[0], gamma[1], gamma[2]}, s3[3] = {s[0], s[1], s[2]};
  for (int x = 0; x < 4; ++x) for (int y = 0; y < 4; ++y) { p[x][y] = psi[4 * x + y]; a[x][y] = dtpsi[4 * x + y]; b[x][y] = dtPi[4 * x + y];
    for (int i = 0; i < 3; ++i) c[i][x][y] = dtPhi[16 * i + 4 * x + y]; }
  if (char_bc_point(p, g3, s3, a, b, c)) return 1;
  for (int x = 0; x < 4; ++x) for (int y = 0; y < 4; ++y) { dtpsi[4 * x + y] = (double)a[x][y]; dtPi[4 * x + y] = (double)b[x][y];
    for (int i = 0; i < 3; ++i) dtPhi[16 * i + 4 * x + y] = (double)c[i][x][y]; }
  if (speeds) {
    geom G; geometry(p, &G);
    real nn = 0; for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) nn += G.ginv[i][j] * s3[i] * s3[j];
    real nN = 0; for (int k = 0; k < 3; ++k) nN += s3[k] / R_SQRT(nn) * G.shift[k];
    speeds[0] = (double)(-(1 + g3[1]) * nN); speeds[1] = (double)(-nN + G.lapse); speeds[2] = (double)(-nN - G.lapse); speeds[3] = (double)(-nN);
  }
  return 0;
}

/* ---------------------------------------------------------------------- */
/* O12 — characteristic penalty exchange across an internal boundary       */
/* (NEXT-2 (iii); "internal boundaries ... characteristic"). */
/* Reading S22: with du = (own - neighbour) state at the coincident point, */
/* projected on the characteristic fields along the own outward normal,    */
/*   dt u^a  +=  - p |v_a| (u^a_own - u^a_nbr)    for every field with     */
/* v_a < 0 (it enters), p = (N_r - 1)^2 / (r_out - r_in) of the own shell  */
/* (the Chebyshev penalty bound N^2/2 of the reference interval times the  */
/* map factor 2/Delta); outgoing fields are left alone; then the same back */
/* map as O10.                                                             */
/* ---------------------------------------------------------------------- */
static int char_penalty_point(const real psi[4][4], const real gam[3], const real s[3], real pen, const real dpsi[4][4],
                              const real dPi[4][4], const real dPhi[3][4][4], real dtpsi[4][4], real dtPi[4][4], real dtPhi[3][4][4]) {
  geom G; if (geometry(psi, &G)) return 1;
  real nn = 0; for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) nn += G.ginv[i][j] * s[i] * s[j];
  nn = R_SQRT(nn);
  real nd[3], nu[3], nN = 0;
  for (int i = 0; i < 3; ++i) nd[i] = s[i] / nn;
  for (int i = 0; i < 3; ++i) { nu[i] = 0; for (int j = 0; j < 3; ++j) nu[i] += G.ginv[i][j] * nd[j]; }
  for (int k = 0; k < 3; ++k) nN += nd[k] * G.shift[k];
  real v0 = -(1 + gam[1]) * nN, v1p = -nN + G.lapse, v1m = -nN - G.lapse, v2 = -nN;
  for (int a = 0; a < 4; ++a) for (int b = 0; b < 4; ++b) {
    real e3[3] = {dPhi[0][a][b], dPhi[1][a][b], dPhi[2][a][b]};
    real nPhi = 0; for (int i = 0; i < 3; ++i) nPhi += nu[i] * e3[i];
    real u0 = dpsi[a][b], u1p = dPi[a][b] + nPhi - gam[2] * dpsi[a][b], u1m = dPi[a][b] - nPhi - gam[2] * dpsi[a][b], u2[3];
    for (int i = 0; i < 3; ++i) u2[i] = e3[i] - nd[i] * nPhi;
    real c0 = v0 < 0 ? pen * v0 * u0 : 0, c1p = v1p < 0 ? pen * v1p * u1p : 0, c1m = v1m < 0 ? pen * v1m * u1m : 0;   /* v < 0: -p|v| = p v */
    real c2[3]; for (int i = 0; i < 3; ++i) c2[i] = v2 < 0 ? pen * v2 * u2[i] : 0;
    dtpsi[a][b] += c0;
    dtPi[a][b] += (c1p + c1m) / 2 + gam[2] * c0;
    for (int i = 0; i < 3; ++i) dtPhi[i][a][b] += (c1p - c1m) / 2 * nd[i] + c2[i];
  }
  return 0;
}

/* outward directions s_i of the faces flagged CHARACTERISTIC (= 2) that contain point p, in face order; returns how many */
static int char_faces(const ora_subdomain* sd, int64_t p, const real* xyz3 /* x,y,z of the point relative to the shell centre */, real s[6][3]) {
  int n0, n1, n2; dims(sd, &n0, &n1, &n2);
  int k = (int)(p % n2), j = (int)((p / n2) % n1), i = (int)(p / ((int64_t)n1 * n2));
  int n = 0;
  if (sd->kind == 0) {
    real r = R_SQRT(xyz3[0] * xyz3[0] + xyz3[1] * xyz3[1] + xyz3[2] * xyz3[2]);
    if (i == 0 && sd->face[0] == 2) { for (int q = 0; q < 3; ++q) s[n][q] = -xyz3[q] / r; ++n; }
    if (i == n0 - 1 && sd->face[1] == 2) { for (int q = 0; q < 3; ++q) s[n][q] = xyz3[q] / r; ++n; }
    return n;
  }
  if (sd->kind == 2) {   /* rho faces: -+ rho^ = -+ (cos phi, sin phi, 0); z faces: -+ z^ */
    real rho = R_SQRT(xyz3[0] * xyz3[0] + xyz3[1] * xyz3[1]);
    if (i == 0 && sd->face[0] == 2) { s[n][0] = -xyz3[0] / rho; s[n][1] = -xyz3[1] / rho; s[n][2] = 0; ++n; }
    if (i == n0 - 1 && sd->face[1] == 2) { s[n][0] = xyz3[0] / rho; s[n][1] = xyz3[1] / rho; s[n][2] = 0; ++n; }
    if (j == 0 && sd->face[2] == 2) { s[n][0] = s[n][1] = 0; s[n][2] = -1; ++n; }
    if (j == n1 - 1 && sd->face[3] == 2) { s[n][0] = s[n][1] = 0; s[n][2] = 1; ++n; }
    return n;
  }
  int idx[3] = {i, j, k}, ext[3] = {n0, n1, n2};
  for (int a = 0; a < 3; ++a) {
    if (idx[a] == 0 && sd->face[2 * a] == 2) { s[n][0] = s[n][1] = s[n][2] = 0; s[n][a] = -1; ++n; }
    if (idx[a] == ext[a] - 1 && sd->face[2 * a + 1] == 2) { s[n][0] = s[n][1] = s[n][2] = 0; s[n][a] = 1; ++n; }
  }
  return n;
}

/* real-typed core: u[50][P], H[4][P], gH[12][P] ([i][a]) -> dtu[50][P]. Returns #non-physical points. */
static const double* g_nbr_in = NULL;    /* neighbour state on the inner / outer face of a shell, [50][n_theta n_phi], set by */
static const double* g_nbr_out = NULL;   /* ora_rhs_subdomain_ifc around its call (faces flagged INTERFACE = 3) */
static const double* g_map_J = NULL;     /* O14: frame map Jm[9][P] and grid velocity v[3][P], set by ora_rhs_subdomain_map / */
static const double* g_map_v = NULL;     /* ora_rk3_subdomain_map around their calls */

static int rhs_real(const ora_subdomain* sd, const real* u, const real* H, const real* gH, real* dtu) {
  int64_t P = ora_num_points(sd);
  real* g = malloc(sizeof(real) * 150 * P);
  gradient_real(sd, 50, u, g);
  real gam[3] = {sd->gamma[0], sd->gamma[1], sd->gamma[2]};
  int bad = 0;
  double* xyz = malloc(sizeof(double) * 3 * P); ora_coords(sd, xyz);
#pragma omp parallel for schedule(static) reduction(+ : bad)
  for (int64_t p = 0; p < P; ++p) {
    point_in in; fill_point(&in, u, g, H, gH, P, p);
    real a[4][4], b[4][4], c[3][4][4];
    if (g_map_J) {   /* O14: grid-frame derivatives -> inertial frame */
      real J[3][3]; for (int i = 0; i < 3; ++i) for (int k = 0; k < 3; ++k) J[i][k] = g_map_J[(int64_t)(3 * i + k) * P + p];
      map_derivs(&in, J);
    }
    if (rhs_point(&in, gam, a, b, c)) { bad += 1; memset(a, 0, sizeof a); memset(b, 0, sizeof b); memset(c, 0, sizeof c); }
    int fz = frozen(sd, p);
    if (!fz) {   /* O10: characteristic faces, in face order (a FROZEN face through the point wins) */
      real rel[3] = {(real)xyz[p] - (real)sd->center[0], (real)xyz[P + p] - (real)sd->center[1], (real)xyz[2 * P + p] - (real)sd->center[2]};
      real sdir[6][3]; int nf = char_faces(sd, p, rel, sdir);
      for (int f = 0; f < nf; ++f) char_bc_point(in.psi, gam, sdir[f], a, b, c);
      if (sd->kind == 0) {   /* O12: interface faces of shells */
        int n0, n1, n2; dims(sd, &n0, &n1, &n2); int64_t pl = (int64_t)n1 * n2, q = p % pl; int i0 = (int)(p / pl);
        real rr = R_SQRT(rel[0] * rel[0] + rel[1] * rel[1] + rel[2] * rel[2]);
        real pen = (real)(n0 - 1) * (real)(n0 - 1) / ((real)sd->hi[0] - (real)sd->lo[0]);
        for (int f = 0; f < 2; ++f) {
          const double* nb = f == 0 ? g_nbr_in : g_nbr_out;
          if (!(sd->face[f] == 3 && nb && i0 == (f == 0 ? 0 : n0 - 1))) continue;
          real sg = f == 0 ? -1 : 1, sv[3] = {sg * rel[0] / rr, sg * rel[1] / rr, sg * rel[2] / rr};
          real dps[4][4], dPi_[4][4], dPh[3][4][4];
          for (int x = 0; x < 4; ++x) for (int y = 0; y < 4; ++y) {
            int sxy = SYM[x][y];
            dps[x][y] = in.psi[x][y] - (real)nb[(int64_t)sxy * pl + q];
            dPi_[x][y] = in.Pi[x][y] - (real)nb[(int64_t)(10 + sxy) * pl + q];
            for (int i = 0; i < 3; ++i) dPh[i][x][y] = in.Phi[i][x][y] - (real)nb[(int64_t)(20 + 10 * i + sxy) * pl + q];
          }
          char_penalty_point(in.psi, gam, sv, pen, dps, dPi_, dPh, a, b, c);
        }
      }
    }
    if (g_map_v && !fz) {   /* O14: the time derivative at the fixed grid point (boundary treatments acted on the inertial-frame part) */
      real vv[3] = {g_map_v[p], g_map_v[P + p], g_map_v[2 * P + p]};
      map_advect(&in, vv, a, b, c);
    }
    for (int x = 0; x < 4; ++x) for (int y = x; y < 4; ++y) {
      int s = SYM[x][y];
      dtu[(int64_t)s * P + p] = fz ? 0 : a[x][y]; dtu[(int64_t)(10 + s) * P + p] = fz ? 0 : b[x][y];
      for (int i = 0; i < 3; ++i) dtu[(int64_t)(20 + 10 * i + s) * P + p] = fz ? 0 : c[i][x][y];
    }
  }
  free(g); free(xyz);
  return bad;
}

/* Full-array (16+16+48) RHS output, for the symmetry pin: out[80][P] = dtpsi[16], dtPi[16], dtPhi[48]. */
int ora_rhs_subdomain_full(const ora_subdomain* sd, const double* u, const double* H, const double* dH, double* out) {
  int64_t P = ora_num_points(sd);
  real* ur = malloc(sizeof(real) * 50 * P); real* Hr = malloc(sizeof(real) * 4 * P); real* gH = malloc(sizeof(real) * 12 * P);
  for (int64_t i = 0; i < 50 * P; ++i) ur[i] = u[i];
  for (int64_t i = 0; i < 4 * P; ++i) Hr[i] = H[i];
  if (dH) for (int64_t i = 0; i < 12 * P; ++i) gH[i] = dH[i]; else gradient_real(sd, 4, Hr, gH);
  real* g = malloc(sizeof(real) * 150 * P); gradient_real(sd, 50, ur, g);
  real gam[3] = {sd->gamma[0], sd->gamma[1], sd->gamma[2]}; int bad = 0;
  for (int64_t p = 0; p < P; ++p) {
    point_in in; fill_point(&in, ur, g, Hr, gH, P, p); real a[4][4], b[4][4], c[3][4][4];
    if (rhs_point(&in, gam, a, b, c)) { bad++; continue; }
    for (int x = 0; x < 4; ++x) for (int y = 0; y < 4; ++y) { out[(int64_t)(x * 4 + y) * P + p] = (double)a[x][y]; out[(int64_t)(16 + x * 4 + y) * P + p] = (double)b[x][y];
      for (int i = 0; i < 3; ++i) out[(int64_t)(32 + (i * 4 + x) * 4 + y) * P + p] = (double)c[i][x][y]; }
  }
  free(ur); free(Hr); free(gH); free(g); return bad;
}

/* u[50][P], H[4][P], dH[12][P] or NULL (then d_i H_a = O3 applied to H_a) -> dtu[50][P] */
int ora_rhs_subdomain(const ora_subdomain* sd, const double* u, const double* H, const double* dH, double* dtu) {
  int64_t P = ora_num_points(sd);
  real* ur = malloc(sizeof(real) * 50 * P); real* Hr = malloc(sizeof(real) * 4 * P); real* gH = malloc(sizeof(real) * 12 * P);
  real* out = malloc(sizeof(real) * 50 * P);
  for (int64_t i = 0; i < 50 * P; ++i) ur[i] = u[i];
  for (int64_t i = 0; i < 4 * P; ++i) Hr[i] = H[i];
  if (dH) for (int64_t i = 0; i < 12 * P; ++i) gH[i] = dH[i]; else gradient_real(sd, 4, Hr, gH);
  int bad = rhs_real(sd, ur, Hr, gH, out);
  for (int64_t i = 0; i < 50 * P; ++i) dtu[i] = (double)out[i];
  free(ur); free(Hr); free(gH); free(out);
  return bad;
}

/* RHS of one shell coupled to its neighbours (O12): nbr_in / nbr_out = the neighbour's state on the coincident face,
 * [50][n_theta n_phi], or NULL.  Not re-entrant (the face planes are passed through file-scope pointers). */
int ora_rhs_subdomain_ifc(const ora_subdomain* sd, const double* u, const double* H, const double* dH, const double* nbr_in,
                          const double* nbr_out, double* dtu) {
  g_nbr_in = nbr_in; g_nbr_out = nbr_out;
  int bad = ora_rhs_subdomain(sd, u, H, dH, dtu);
  g_nbr_in = NULL; g_nbr_out = NULL;
  return bad;
}

/* O7 — nsteps of Shu-Osher SSP-RK3, state kept in `real` across steps:
 *   u1 = u0 + dt k(u0); u2 = 3/4 u0 + 1/4 (u1 + dt k(u1)); u_new = 1/3 u0 + 2/3 (u2 + dt k(u2)) */
int ora_rk3_subdomain(const ora_subdomain* sd, double* u, const double* H, const double* dH, double dt, int nsteps) {
  int64_t P = ora_num_points(sd), n = 50 * P;
  real* u0 = malloc(sizeof(real) * n); real* us = malloc(sizeof(real) * n); real* k = malloc(sizeof(real) * n);
  real* Hr = malloc(sizeof(real) * 4 * P); real* gH = malloc(sizeof(real) * 12 * P);
  for (int64_t i = 0; i < n; ++i) u0[i] = u[i];
  for (int64_t i = 0; i < 4 * P; ++i) Hr[i] = H[i];
  if (dH) for (int64_t i = 0; i < 12 * P; ++i) gH[i] = dH[i]; else gradient_real(sd, 4, Hr, gH);
  real h = dt; int bad = 0;
  for (int s = 0; s < nsteps; ++s) {
    bad += rhs_real(sd, u0, Hr, gH, k);
    for (int64_t i = 0; i < n; ++i) us[i] = u0[i] + h * k[i];
    bad += rhs_real(sd, us, Hr, gH, k);
    for (int64_t i = 0; i < n; ++i) us[i] = (3 * u0[i] + (us[i] + h * k[i])) / 4;
    bad += rhs_real(sd, us, Hr, gH, k);
    for (int64_t i = 0; i < n; ++i) u0[i] = (u0[i] + 2 * (us[i] + h * k[i])) / 3;
  }
  for (int64_t i = 0; i < n; ++i) u[i] = (double)u0[i];
  free(u0); free(us); free(k); free(Hr); free(gH);
  return bad;
}

/* ---------------------------------------------------------------------- */
/* O11 — Dormand-Prince 5(4) step (NEXT-3): the stepper the paper names    */
/* ("high-order Dormand Prince").  Explicit 7-stage pair of   */
/* Dormand & Prince (1980): 5th-order solution (its weights are row 7 of   */
/* the matrix, so stage 7 is the RHS at the new state) and the embedded    */
/* 4th-order weights bh; err = dt sum_j (b_j - bh_j) k_j.                  */
/* ---------------------------------------------------------------------- */
static const real DP_C[7] = {0, (real)1 / 5, (real)3 / 10, (real)4 / 5, (real)8 / 9, 1, 1};
static const real DP_A[7][6] = {
  {0, 0, 0, 0, 0, 0},
  {(real)1 / 5, 0, 0, 0, 0, 0},
  {(real)3 / 40, (real)9 / 40, 0, 0, 0, 0},
  {(real)44 / 45, -(real)56 / 15, (real)32 / 9, 0, 0, 0},
  {(real)19372 / 6561, -(real)25360 / 2187, (real)64448 / 6561, -(real)212 / 729, 0, 0},
  {(real)9017 / 3168, -(real)355 / 33, (real)46732 / 5247, (real)49 / 176, -(real)5103 / 18656, 0},
  {(real)35 / 384, 0, (real)500 / 1113, (real)125 / 192, -(real)2187 / 6784, (real)11 / 84}};
static const real DP_BH[7] = {(real)5179 / 57600, 0, (real)7571 / 16695, (real)393 / 640, -(real)92097 / 339200, (real)187 / 2100, (real)1 / 40};

/* c[7], a[7*6] (row-major, a[i][j], j < i), b[7] (5th order = row 7 of a, b[6] = 0), bh[7] (4th order) */
void ora_dp5_tableau(double* c, double* a, double* b, double* bh) {
  for (int i = 0; i < 7; ++i) { c[i] = (double)DP_C[i]; bh[i] = (double)DP_BH[i]; b[i] = i < 6 ? (double)DP_A[6][i] : 0.0;
    for (int j = 0; j < 6; ++j) a[6 * i + j] = (double)DP_A[i][j]; }
}

/* one step of size dt: u[50][P] <- 5th-order solution, err[50][P] <- dt sum_j (b_j - bh_j) k_j.  Returns #non-physical points. */
int ora_dp5_subdomain(const ora_subdomain* sd, double* u, const double* H, const double* dH, double dt, double* err) {
  int64_t P = ora_num_points(sd), n = 50 * P;
  real* u0 = malloc(sizeof(real) * n); real* us = malloc(sizeof(real) * n); real* k[7];
  for (int q = 0; q < 7; ++q) k[q] = malloc(sizeof(real) * n);
  real* Hr = malloc(sizeof(real) * 4 * P); real* gH = malloc(sizeof(real) * 12 * P);
  for (int64_t i = 0; i < n; ++i) u0[i] = u[i];
  for (int64_t i = 0; i < 4 * P; ++i) Hr[i] = H[i];
  if (dH) for (int64_t i = 0; i < 12 * P; ++i) gH[i] = dH[i]; else gradient_real(sd, 4, Hr, gH);
  real h = dt; int bad = 0;
  for (int st = 0; st < 7; ++st) {
    for (int64_t i = 0; i < n; ++i) { real a = 0; for (int j = 0; j < st; ++j) a += DP_A[st][j] * k[j][i]; us[i] = u0[i] + h * a; }
    bad += rhs_real(sd, us, Hr, gH, k[st]);
  }
  /* us now holds the 5th-order solution (row 7 of the matrix are its weights) */
  for (int64_t i = 0; i < n; ++i) {
    real e = 0; for (int j = 0; j < 7; ++j) e += ((j < 6 ? DP_A[6][j] : 0) - DP_BH[j]) * k[j][i];
    u[i] = (double)us[i]; err[i] = (double)(h * e);
  }
  free(u0); free(us); for (int q = 0; q < 7; ++q) free(k[q]); free(Hr); free(gH);
  return bad;
}

/* O8 — constraints on one subdomain.
 * sums[3] = sum of squares over points and UNIQUE components of C_a (4), C_iab (30: a<=b),
 * C_ijab (30: i<j, a<=b); maxs[3] = max |.|.  Optional per-point fields Cfield[64][P]:
 * rows 0..3 C_a; 4+10 i+s C_iab; 34+10 q+s C_ijab with q = 0,1,2 for (i,j) = (0,1),(0,2),(1,2).
 * Domain norms: rms = sqrt(sum_over_subdomains(sums)/(P_total n_comp)). */
int ora_constraints_subdomain(const ora_subdomain* sd, const double* u, const double* H, double* sums, double* maxs, double* Cfield) {
  int64_t P = ora_num_points(sd);
  real* ur = malloc(sizeof(real) * 50 * P); real* Hr = malloc(sizeof(real) * 4 * P); real* gH = calloc(12 * P, sizeof(real));
  for (int64_t i = 0; i < 50 * P; ++i) ur[i] = u[i];
  for (int64_t i = 0; i < 4 * P; ++i) Hr[i] = H[i];
  real* g = malloc(sizeof(real) * 150 * P); gradient_real(sd, 50, ur, g);
  real S[3] = {0, 0, 0}, M[3] = {0, 0, 0}; int bad = 0;
  static const int PI_[3] = {0, 0, 1}, PJ_[3] = {1, 2, 2};
  for (int64_t p = 0; p < P; ++p) {
    point_in in; fill_point(&in, ur, g, Hr, gH, P, p); real a[4], b[3][4][4], c[3][3][4][4];
    if (constraints_point(&in, a, b, c)) { bad++; continue; }
    for (int x = 0; x < 4; ++x) { S[0] += a[x] * a[x]; if (R_FABS(a[x]) > M[0]) M[0] = R_FABS(a[x]); if (Cfield) Cfield[(int64_t)x * P + p] = (double)a[x]; }
    for (int x = 0; x < 4; ++x) for (int y = x; y < 4; ++y) {
      int s = SYM[x][y];
      for (int i = 0; i < 3; ++i) { real v = b[i][x][y]; S[1] += v * v; if (R_FABS(v) > M[1]) M[1] = R_FABS(v); if (Cfield) Cfield[(int64_t)(4 + 10 * i + s) * P + p] = (double)v; }
      for (int q = 0; q < 3; ++q) { real v = c[PI_[q]][PJ_[q]][x][y]; S[2] += v * v; if (R_FABS(v) > M[2]) M[2] = R_FABS(v); if (Cfield) Cfield[(int64_t)(34 + 10 * q + s) * P + p] = (double)v; }
    }
  }
  for (int q = 0; q < 3; ++q) { sums[q] = (double)S[q]; maxs[q] = (double)M[q]; }
  free(ur); free(Hr); free(gH); free(g);
  return bad;
}

/* ---------------------------------------------------------------------- */
/* O13 — SpatialCoordJac (NEXT-4; §3.3, Eqs. 9-11): "makes */
/* a coordinate change of a tensor's spatial indices only, by contracting   */
/* every possible combination of said spatial indices with the Jacobian.    */
/* First, one contraction per rank is performed over the purely spatial     */
/* indices.  Next, each index is respectively set to its timelike component */
/* and one contraction per remaining index is performed.  Subsequently, two */
/* indices are made timelike, ... The purely timelike component encounters  */
/* a null-op."  Rank 2:  T_ij = J_i^k J_j^l T_kl, T_0j = J_j^l T_0l,        */
/* T_i0 = J_i^k T_k0.  Written for any rank r <= 3 on FULL 4^r arrays with  */
/* no symmetry use, in exactly that order: for every set Z of indices made  */
/* timelike (|Z| = 0, 1, ..., r) the other r - |Z| indices are contracted   */
/* with J one after the other.  *flops counts 2d - 1 = 5 per element each   */
/* contraction produces (Eq. 13: 15 for rank 1, 120 for rank 2).            */
/* ---------------------------------------------------------------------- */
static void scj_full(int r, const real J[3][3], const real* Tin, real* Tout, double* flops) {
  int n = 1; for (int q = 0; q < r; ++q) n *= 4;
  double fl = 0;
  for (int Z = 0; Z < (1 << r); ++Z) {            /* bit q of Z set: index q is timelike */
    int pos[3], ns = 0;                          /* positions of the spatial indices */
    for (int q = 0; q < r; ++q) if (!((Z >> q) & 1)) pos[ns++] = q;
    int m = 1; for (int q = 0; q < ns; ++q) m *= 3;
    real W[27], V[27];
    /* gather the sub-tensor: spatial indices run over 1..3, the indices in Z are 0 */
    for (int e = 0; e < m; ++e) {
      int idx[3] = {0, 0, 0}, t = e;
      for (int q = ns - 1; q >= 0; --q) { idx[pos[q]] = 1 + t % 3; t /= 3; }
      int flat = 0; for (int q = 0; q < r; ++q) flat = flat * 4 + idx[q];
      W[e] = Tin[flat];
    }
    /* one contraction per remaining index: W'[.. i ..] = sum_k J[i][k] W[.. k ..] */
    for (int c = 0; c < ns; ++c) {
      int stride = 1; for (int q = c + 1; q < ns; ++q) stride *= 3;
      for (int e = 0; e < m; ++e) {
        int i = (e / stride) % 3, base = e - i * stride;
        real s = 0; for (int k = 0; k < 3; ++k) s += J[i][k] * W[base + k * stride];
        V[e] = s; fl += 5;
      }
      for (int e = 0; e < m; ++e) W[e] = V[e];
    }
    for (int e = 0; e < m; ++e) {
      int idx[3] = {0, 0, 0}, t = e;
      for (int q = ns - 1; q >= 0; --q) { idx[pos[q]] = 1 + t % 3; t /= 3; }
      int flat = 0; for (int q = 0; q < r; ++q) flat = flat * 4 + idx[q];
      Tout[flat] = W[e];
    }
  }
  (void)n;
  if (flops) *flops = fl;
}

/* structure: 0 = T_a (rank 1), 1 = T_aa (rank 2, symmetric), 2 = T_ab (rank 2), 3 = T_abb (rank 3, T_abc = T_acb)
 * (the four the paper's port handles). */
static int scj_rank(int structure) { return structure == 0 ? 1 : structure == 3 ? 3 : 2; }

/* one point, full arrays (4, 16, 16, 64 doubles), J[9] row-major J[3 i + k] = J_i^k; returns the flop count of the
 * symmetry-free evaluation */
double ora_scj_point(int structure, const double* J, const double* Tin, double* Tout) {
  int r = scj_rank(structure), n = 1; for (int q = 0; q < r; ++q) n *= 4;
  real Jr[3][3], a[64], b[64]; double fl = 0;
  for (int i = 0; i < 3; ++i) for (int k = 0; k < 3; ++k) Jr[i][k] = J[3 * i + k];
  for (int e = 0; e < n; ++e) a[e] = Tin[e];
  scj_full(r, Jr, a, b, &fl);
  for (int e = 0; e < n; ++e) Tout[e] = (double)b[e];
  return fl;
}

/* Eq. 12: F / N_x = (2d-1) sum_j W(r,j) S(r,j) (r-j), by brute-force enumeration: the arrangements of j
 * timelike indices and the spatial components that remain are counted ONCE per class under the tensor's symmetry. */
double ora_scj_eq12(int structure) {
  int r = scj_rank(structure);
  int sym0 = structure == 1 ? 0 : structure == 3 ? 1 : -1;   /* the symmetric pair is (sym0, sym0 + 1) */
  double F = 0;
  for (int Z = 0; Z < (1 << r) - 1; ++Z) {
    if (sym0 >= 0 && ((Z >> sym0) & 1) == 0 && ((Z >> (sym0 + 1)) & 1) == 1) continue;   /* T_..0b.. and T_..b0.. are one arrangement */
    int ns = 0; for (int q = 0; q < r; ++q) if (!((Z >> q) & 1)) ++ns;
    int m = 1; for (int q = 0; q < ns; ++q) m *= 3;
    int S = 0;
    int pairfree = sym0 >= 0 && !((Z >> sym0) & 1) && !((Z >> (sym0 + 1)) & 1);        /* both indices of the pair still spatial */
    for (int e = 0; e < m; ++e) {
      int idx[3] = {0, 0, 0}, pos[3], np_ = 0, t = e;
      for (int q = 0; q < r; ++q) if (!((Z >> q) & 1)) pos[np_++] = q;
      for (int q = ns - 1; q >= 0; --q) { idx[pos[q]] = t % 3; t /= 3; }
      if (pairfree && idx[sym0] > idx[sym0 + 1]) continue;                                 /* count (k,l) and (l,k) once */
      ++S;
    }
    F += 5.0 * S * ns;
  }
  return F;
}

/* packed storage of the four structures: T_a [4]; T_aa [10] (the order of SYM); T_ab [16] (4 a + b); T_abb [40] (10 a + SYM[b][c]) */
static int scj_ne(int structure) { return structure == 0 ? 4 : structure == 1 ? 10 : structure == 2 ? 16 : 40; }

/* whole arrays: J[9][P], T[N_e][P] -> out[N_e][P] (may alias T).  The packed symmetric storage is expanded to FULL arrays,
 * transformed without symmetry use, and the upper triangle is stored back. */
int ora_scj_subdomain(int structure, int64_t P, const double* J, const double* T, double* out) {
  int r = scj_rank(structure), ne = scj_ne(structure), n = 1; for (int q = 0; q < r; ++q) n *= 4;
#pragma omp parallel for schedule(static)
  for (int64_t p = 0; p < P; ++p) {
    real Jr[3][3], a[64], b[64];
    for (int i = 0; i < 3; ++i) for (int k = 0; k < 3; ++k) Jr[i][k] = J[(int64_t)(3 * i + k) * P + p];
    for (int e = 0; e < n; ++e) {
      int c;
      if (structure == 0 || structure == 2) c = e;
      else if (structure == 1) c = SYM[e / 4][e % 4];
      else c = 10 * (e / 16) + SYM[(e / 4) % 4][e % 4];
      a[e] = T[(int64_t)c * P + p];
    }
    scj_full(r, Jr, a, b, NULL);
    for (int e = 0; e < n; ++e) {
      int c, keep = 1;
      if (structure == 0 || structure == 2) c = e;
      else if (structure == 1) { c = SYM[e / 4][e % 4]; keep = (e / 4) <= (e % 4); }
      else { c = 10 * (e / 16) + SYM[(e / 4) % 4][e % 4]; keep = ((e / 4) % 4) <= (e % 4); }
      if (keep) out[(int64_t)c * P + p] = (double)b[e];
    }
  }
  (void)ne;
  return 0;
}

/* the evolved state u[50][P]: psi_ab and Pi_ab as T_aa, Phi_iab as the spatial-first-index part of a T_abb whose timelike
 * first index is absent (Phi has no 0ab components: the Jacobian never mixes them in, Eqs. 9-11) */
int ora_scj_state(int64_t P, const double* J, const double* u, double* out) {
  double* T = calloc((size_t)40 * P, sizeof(double)); double* R = malloc(sizeof(double) * 40 * P);
  ora_scj_subdomain(1, P, J, u, out);
  ora_scj_subdomain(1, P, J, u + 10 * P, out + 10 * P);
  memcpy(T + 10 * P, u + 20 * P, sizeof(double) * 30 * P);
  ora_scj_subdomain(3, P, J, T, R);
  memcpy(out + 20 * P, R + 10 * P, sizeof(double) * 30 * P);
  int bad = 0; for (int64_t i = 0; i < 10 * P; ++i) if (R[i] != 0) bad = 1;   /* the absent 0ab rows stay zero */
  free(T); free(R);
  return bad;
}

/* ---------------------------------------------------------------------- */
/* O12b — spectral interpolation of a face state between shells of         */
/* different band limit (NEXT-2 (iii) across non-matching grids; "at       */
/* 'internal' boundaries between neighboring domains, the characteristic   */
/* variables are computed and used as boundary conditions on the           */
/* neighboring subdomain"; interpolation "via a direct       */
/* summation of the spectral series").  One (theta,phi) plane */
/* on the Gauss-Legendre x uniform grid of band limit Ls:                  */
/*   a_lm = sum_{j,k} w_j (2 pi/N_phi) conj(Y_lm(theta_j,phi_k)) u_jk,     */
/*   0 <= l <= Ls (Eq. 23's analysis), then the series is summed at the    */
/* nodes (theta'_j', phi'_k') of the grid of band limit Ld:                */
/*   out_j'k' = sum_l [a_l0 Y_l0 + 2 Re sum_{m>0} a_lm Y_lm](theta',phi'). */
/* Explicit sums; Ls = Ld reduces to the projection of O2.                 */
/* ---------------------------------------------------------------------- */
void ora_shell_interp(int Ls, int Ld, const double* u, double* out) {
  ylm_table* t = ylm_build(Ls);
  int n = t->nth, nph = t->nph, nd = Ld + 1, npd = 2 * (Ld + 1);
  real* are = calloc((size_t)n * n, sizeof(real)); real* aim = calloc((size_t)n * n, sizeof(real));
  real dphi = 2 * R_PI / (real)nph;
  for (int l = 0; l <= Ls; ++l) for (int m = 0; m <= l; ++m) {
    real sr = 0, si = 0; const real* pb = t->pb + (int64_t)(l * n + m) * n;
    for (int j = 0; j < n; ++j) for (int k = 0; k < nph; ++k) {
      real f = t->w[j] * dphi * pb[j] * (real)u[j * nph + k];
      sr += f * t->cs[m * nph + k]; si -= f * t->sn[m * nph + k];
    }
    are[l * n + m] = sr; aim[l * n + m] = si;
  }
  real* ctd = malloc(sizeof(real) * nd); real* wd = malloc(sizeof(real) * nd); gl_nodes(Ld, ctd, wd);
  real* pb = malloc(sizeof(real) * n * n); real* dpb = malloc(sizeof(real) * n * n);
  for (int j = 0; j < nd; ++j) {
    pbar_all(Ls, ctd[j], pb, dpb);      /* Pbar_lm at the destination colatitude, l <= Ls */
    for (int k = 0; k < npd; ++k) {
      real s = 0;
      for (int l = 0; l <= Ls; ++l) for (int m = 0; m <= l; ++m) {
        int64_t q = ((int64_t)m * k) % npd; real ang = 2 * R_PI * (real)q / (real)npd;
        real c = R_COS(ang), sn = R_SIN(ang);
        real re = are[l * n + m] * c - aim[l * n + m] * sn;
        s += ((m == 0) ? 1 : 2) * pb[l * n + m] * re;
      }
      out[j * npd + k] = (double)s;
    }
  }
  free(are); free(aim); free(ctd); free(wd); free(pb); free(dpb); ylm_free(t);
}

/* O14 on one subdomain: Jm[9][P], v[3][P] (held fixed), dH[12][P] the inertial-frame gradient of H (required: the library's own
 * derivative of H would be a grid-frame one).  nsteps = 0: the right-hand side into out[50][P]; nsteps > 0: that many SSP-RK3 steps of
 * u in place with the map frozen (out unused).  Not re-entrant. */
int ora_rhs_subdomain_map(const ora_subdomain* sd, double* u, const double* H, const double* dH, const double* Jm, const double* v,
                          double dt, int nsteps, double* out) {
  g_map_J = Jm; g_map_v = v;
  int bad = nsteps > 0 ? ora_rk3_subdomain(sd, u, H, dH, dt, nsteps) : ora_rhs_subdomain(sd, u, H, dH, out);
  g_map_J = NULL; g_map_v = NULL;
  return bad;
}
