// basis.cpp — host-side basis-matrix builder (A0).  See basis.h.
#include "basis.h"

#include <cmath>

namespace ghb {

static const ld PI_L = 3.14159265358979323846264338327950288419716939937510L;

void cheb_nodes(int N, std::vector<ld>& x) {
  x.resize(N);
  for (int j = 0; j < N; ++j) x[j] = -cosl(PI_L * j / (N - 1));
  if (N & 1) x[N / 2] = 0;  // exact midpoint
}

// D_ij = (c_i/c_j) (-1)^(i+j) / (x_i - x_j), c_0 = c_{N-1} = 2, else 1; D_ii = -sum_{j != i} D_ij.
// x_i - x_j = cos(pi j/n) - cos(pi i/n) = 2 sin(pi (i+j)/(2n)) sin(pi (i-j)/(2n)), n = N-1, evaluated in that
// product form so that neighbouring nodes do not cancel.
void cheb_diff_matrix(int N, std::vector<ld>& D) {
  D.assign((size_t)N * N, 0);
  const int n = N - 1;
  for (int i = 0; i < N; ++i) {
    ld diag = 0;
    for (int j = 0; j < N; ++j) {
      if (i == j) continue;
      ld ci = (i == 0 || i == n) ? 2 : 1, cj = (j == 0 || j == n) ? 2 : 1;
      ld dx = 2 * sinl(PI_L * (i + j) / (2 * (ld)n)) * sinl(PI_L * (i - j) / (2 * (ld)n));
      ld v = (ci / cj) / dx;
      if ((i + j) & 1) v = -v;
      D[(size_t)i * N + j] = v;
      diag -= v;
    }
    D[(size_t)i * N + i] = diag;
  }
}

// Legendre P_n and P_n' at x by the Bonnet recurrence.
static void legendre_pn(int n, ld x, ld& p, ld& dp) {
  ld a = 1, b = x;
  if (n == 0) { p = 1; dp = 0; return; }
  for (int k = 1; k < n; ++k) {
    ld c = ((2 * k + 1) * x * b - k * a) / (k + 1);
    a = b; b = c;
  }
  p = b;
  dp = n * (a - x * b) / (1 - x * x);
}

void gauss_legendre(int L, std::vector<ld>& ct, std::vector<ld>& w) {
  const int n = L + 1;
  ct.resize(n); w.resize(n);
  for (int j = 0; j < (n + 1) / 2; ++j) {
    // Tricomi-type first guess, then Newton to long-double roundoff
    ld x = cosl(PI_L * (4 * j + 3) / (4 * (ld)n + 2));
    ld p, dp;
    for (int it = 0; it < 60; ++it) {
      legendre_pn(n, x, p, dp);
      ld dx = p / dp;
      x -= dx;
      if (fabsl(dx) < 4e-20L) break;
    }
    legendre_pn(n, x, p, dp);
    ld wt = 2 / ((1 - x * x) * dp * dp);
    ct[j] = x; w[j] = wt;
    ct[n - 1 - j] = -x; w[n - 1 - j] = wt;  // nodes are symmetric about the equator
  }
  if (n & 1) ct[n / 2] = 0;
}

// Orthonormalised associated Legendre functions Pb[l - m], l = m..L+1, at one colatitude and one m.
static void pbar_column(int L, int m, ld c, ld s, std::vector<ld>& Pb) {
  Pb.assign(L + 2 - m, 0);
  ld pmm = sqrtl(1 / (4 * PI_L));
  for (int k = 1; k <= m; ++k) pmm *= -sqrtl((ld)(2 * k + 1) / (ld)(2 * k)) * s;
  Pb[0] = pmm;
  if (L + 1 >= m + 1) Pb[1] = sqrtl((ld)(2 * m + 3)) * c * pmm;
  for (int l = m + 2; l <= L + 1; ++l) {
    ld a = sqrtl((ld)(4 * l * l - 1) / (ld)(l * l - m * m));
    ld b = sqrtl((ld)((l - 1) * (l - 1) - m * m) / (ld)(4 * (l - 1) * (l - 1) - 1));
    Pb[l - m] = a * (c * Pb[l - 1 - m] - b * Pb[l - 2 - m]);
  }
}

void shell_basis(int L, ShellBasis& B) {
  B.L = L; B.nt = L + 1; B.np = 2 * L + 2; B.nq = 2 * L + 1;
  const int nt = B.nt, np = B.np, nq = B.nq;
  gauss_legendre(L, B.ct, B.w);
  B.st.resize(nt);
  for (int j = 0; j < nt; ++j) B.st[j] = sqrtl((1 - B.ct[j]) * (1 + B.ct[j]));

  // real Fourier analysis / synthesis on phi_k = 2 pi k / n_p; the Nyquist mode m = L+1 is dropped, which is
  // part of the projection onto l <= L (reading S6).
  B.Fa.assign((size_t)nq * np, 0); B.Fs.assign((size_t)np * nq, 0); B.Fp.assign((size_t)np * nq, 0);
  for (int k = 0; k < np; ++k) {
    B.Fa[k] = 1 / (ld)np;
    B.Fs[(size_t)k * nq] = 1;
    for (int m = 1; m <= L; ++m) {
      int r = (int)(((long long)m * k) % np);
      ld ang = 2 * PI_L * r / np, cs = cosl(ang), sn = sinl(ang);
      B.Fa[(size_t)m * np + k] = 2 * cs / np;
      B.Fa[(size_t)(L + m) * np + k] = 2 * sn / np;
      B.Fs[(size_t)k * nq + m] = cs;
      B.Fs[(size_t)k * nq + L + m] = sn;
      B.Fp[(size_t)k * nq + m] = -m * sn;       // d/dphi cos(m phi)
      B.Fp[(size_t)k * nq + L + m] = m * cs;    // d/dphi sin(m phi)
    }
  }

  // per-m Legendre composites:  Pr_m[j'][j] = 2 pi sum_{l=m}^{L} Pbar_lm(j') w_j Pbar_lm(j),
  //                             Th_m[j'][j] = 2 pi sum_l dPbar_lm/dtheta(j') w_j Pbar_lm(j),
  // with sin(theta) dPbar_lm/dtheta = -(l+1) cos(theta) Pbar_lm + sqrt((2l+1)/(2l+3) ((l+1)^2-m^2)) Pbar_{l+1,m}.
  B.Th.assign((size_t)(L + 1) * nt * nt, 0); B.Pr.assign((size_t)(L + 1) * nt * nt, 0);
  std::vector<std::vector<ld>> P(nt), dP(nt);
  for (int m = 0; m <= L; ++m) {
    for (int j = 0; j < nt; ++j) {
      pbar_column(L, m, B.ct[j], B.st[j], P[j]);
      dP[j].assign(L + 1 - m, 0);
      for (int l = m; l <= L; ++l) {
        ld f = sqrtl((ld)(2 * l + 1) / (ld)(2 * l + 3) * (ld)((l + 1) * (l + 1) - m * m));
        dP[j][l - m] = (-(ld)(l + 1) * B.ct[j] * P[j][l - m] + f * P[j][l + 1 - m]) / B.st[j];
      }
    }
    for (int jo = 0; jo < nt; ++jo)
      for (int ji = 0; ji < nt; ++ji) {
        ld sp = 0, sd = 0;
        for (int l = m; l <= L; ++l) {
          sp += P[jo][l - m] * P[ji][l - m];
          sd += dP[jo][l - m] * P[ji][l - m];
        }
        B.Pr[((size_t)m * nt + jo) * nt + ji] = 2 * PI_L * B.w[ji] * sp;
        B.Th[((size_t)m * nt + jo) * nt + ji] = 2 * PI_L * B.w[ji] * sd;
      }
  }
}

void cheb_filter_matrix(int N, const std::vector<ld>& sigma, std::vector<ld>& F) {
  F.assign((size_t)N * N, 0);
  const int n = N - 1;
  // T_k(x_j) = (-1)^k cos(pi j k / n) for x_j = -cos(pi j / n); the argument is reduced in integers
  auto T = [&](int k, int j) {
    const long long r = ((long long)j * k) % (2LL * n);
    const ld v = cosl(PI_L * r / (ld)n);
    return (k & 1) ? -v : v;
  };
  for (int a = 0; a < N; ++a)
    for (int j = 0; j < N; ++j) {
      ld s = 0;
      const ld cj = (j == 0 || j == n) ? 2 : 1;
      for (int k = 0; k < N; ++k) {
        const ld ck = (k == 0 || k == n) ? 2 : 1;
        s += T(k, a) * sigma[k] * T(k, j) / ck;
      }
      F[(size_t)a * N + j] = 2 * s / ((ld)n * cj);
    }
}

void fourier_diff_matrix(int N, std::vector<ld>& D) {
  D.assign((size_t)N * N, 0);
  for (int j = 0; j < N; ++j)
    for (int k = 0; k < N; ++k) {
      if (j == k) continue;
      const int d = ((j - k) % N + N) % N;              // 1 .. N-1; (-1)^(j-k) cot / csc are N-periodic in j - k for the parity at hand
      const ld x = PI_L * (ld)d / (ld)N, sgn = (d & 1) ? -1 : 1;
      D[(size_t)j * N + k] = (N % 2 == 0) ? sgn * cosl(x) / (2 * sinl(x)) : sgn / (2 * sinl(x));
    }
}

void fourier_filter_matrix(int N, const std::vector<ld>& sigma, std::vector<ld>& F) {
  F.assign((size_t)N * N, 0);
  for (int j = 0; j < N; ++j)
    for (int k = 0; k < N; ++k) {
      const int d = ((j - k) % N + N) % N;
      ld s = sigma[0];
      for (int m = 1; 2 * m <= N; ++m) {
        const ld c = cosl(2 * PI_L * (ld)(((long long)m * d) % N) / (ld)N);
        s += (2 * m == N ? 1 : 2) * sigma[m] * c;
      }
      F[(size_t)j * N + k] = s / (ld)N;
    }
}

void shell_filter_composites(int L, const std::vector<ld>& sigma_l, std::vector<ld>& G) {
  const int nt = L + 1;
  std::vector<ld> ct, w, st(nt);
  gauss_legendre(L, ct, w);
  for (int j = 0; j < nt; ++j) st[j] = sqrtl((1 - ct[j]) * (1 + ct[j]));
  G.assign((size_t)(L + 1) * nt * nt, 0);
  std::vector<std::vector<ld>> P(nt);
  for (int m = 0; m <= L; ++m) {
    for (int j = 0; j < nt; ++j) pbar_column(L, m, ct[j], st[j], P[j]);
    for (int jo = 0; jo < nt; ++jo)
      for (int ji = 0; ji < nt; ++ji) {
        ld sp = 0;
        for (int l = m; l <= L; ++l) sp += sigma_l[l] * P[jo][l - m] * P[ji][l - m];
        G[((size_t)m * nt + jo) * nt + ji] = 2 * PI_L * w[ji] * sp;
      }
  }
}

void shell_interp_composites(int Ls, int Ld, std::vector<ld>& G) {
  const int ns = Ls + 1, nd = Ld + 1;
  std::vector<ld> cs, ws, cd, wd, ss(ns), sd(nd);
  gauss_legendre(Ls, cs, ws); gauss_legendre(Ld, cd, wd);
  for (int j = 0; j < ns; ++j) ss[j] = sqrtl((1 - cs[j]) * (1 + cs[j]));
  for (int j = 0; j < nd; ++j) sd[j] = sqrtl((1 - cd[j]) * (1 + cd[j]));
  G.assign((size_t)(Ls + 1) * nd * ns, 0);
  std::vector<std::vector<ld>> Ps(ns), Pd(nd);
  for (int m = 0; m <= Ls; ++m) {
    for (int j = 0; j < ns; ++j) pbar_column(Ls, m, cs[j], ss[j], Ps[j]);
    for (int j = 0; j < nd; ++j) pbar_column(Ls, m, cd[j], sd[j], Pd[j]);
    for (int jo = 0; jo < nd; ++jo)
      for (int ji = 0; ji < ns; ++ji) {
        ld sp = 0;
        for (int l = m; l <= Ls; ++l) sp += Pd[jo][l - m] * Ps[ji][l - m];
        G[((size_t)m * nd + jo) * ns + ji] = 2 * PI_L * ws[ji] * sp;
      }
  }
}

}  // namespace ghb
