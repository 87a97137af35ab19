// basis.h — host-side basis-matrix builder (step A0 of DESIGN.md).  Internal to the library.
//
// Everything here runs once per domain on the host in long double and is rounded to double at the end
// ("extra function calls needed to build the matrix ... can be ignored", §3.4).
#pragma once
#include <vector>

namespace ghb {

typedef long double ld;

// Chebyshev-Gauss-Lobatto nodes x_j = -cos(pi j/(N-1)) (ascending) and the collocation differentiation
// matrix D (row-major N x N) on [-1,1]: the "cached matrix" of PAPER.md:357-384 (Eqs. 19-22), built
// analytically instead of by delta-tracing.  Diagonal by the negative-sum trick.
void cheb_nodes(int N, std::vector<ld>& x);
void cheb_diff_matrix(int N, std::vector<ld>& D);

// Gauss-Legendre nodes: cos(theta_j) descending (theta ascending), weights; n = L+1 points.
void gauss_legendre(int L, std::vector<ld>& ct, std::vector<ld>& w);

// Shell angular matrices for band limit L (n_t = L+1, n_p = 2L+2, n_q = 2L+1), all row-major:
//   Fa [n_q][n_p]  real-Fourier analysis: rows q=0..L cos(m phi_k) (m=q), rows q=L+1..2L sin(m phi_k) (m=q-L)
//   Fs [n_p][n_q]  synthesis of u            from the (cos, sin) coefficients
//   Fp [n_p][n_q]  synthesis of d u / d phi  from the same coefficients
//   Th [L+1][n_t][n_t]  per-m:  d/dtheta of the projection onto l<=L, Th[m][j'][j]
//   Pr [L+1][n_t][n_t]  per-m:  the projection itself
// Together Fs*Th*Fa and Fp*Pr*Fa are the dense Theta and Phi matrices of Eq. 24.
struct ShellBasis {
  int L, nt, np, nq;
  std::vector<ld> ct, st, w;  // cos/sin(theta_j), GL weights
  std::vector<ld> Fa, Fs, Fp, Th, Pr;
};
void shell_basis(int L, ShellBasis& B);

// Spectral filter matrices (NEXT-1).
// Chebyshev line filter F = SpecToPhys diag(sigma) PhysToSpec on N CGL nodes (row-major N x N), Eqs. 16-17:
//   F[a][j] = sum_k T_k(x_a) sigma_k (2/(N-1)) (1/(c_k c_j)) T_k(x_j).
void cheb_filter_matrix(int N, const std::vector<ld>& sigma, std::vector<ld>& F);
// Periodic (Fourier) line on N uniform nodes phi_k = 2 pi k / N - the S1 factor of the cylindrical shells (DESIGN.md
// reading S25).  Differentiation matrix of the trigonometric interpolant (the Nyquist mode of an even N has zero derivative at
// the nodes):  D[j][k] = (1/2) (-1)^(j-k) cot(pi (j-k) / N), N even;  (1/2) (-1)^(j-k) / sin(pi (j-k) / N), N odd;  D[j][j] = 0.
void fourier_diff_matrix(int N, std::vector<ld>& D);
// Filter  F[j][k] = (1/N) sum_{|m| <= N/2} sigma_|m| e^{i m (phi_j - phi_k)}  (the Nyquist mode of an even N counted once),
// sigma[0 .. N/2].
void fourier_filter_matrix(int N, const std::vector<ld>& sigma, std::vector<ld>& F);
// Per-m filtered projectors on the Gauss-Legendre colatitudes: G[m][j'][j] = 2 pi sum_{l=m}^{L} sigma_l Pbar_lm(j') w_j Pbar_lm(j).
void shell_filter_composites(int L, const std::vector<ld>& sigma_l, std::vector<ld>& G);

// Face interpolation between shells of different band limit (NEXT-2 (iii) across non-matching grids): per m = 0..Ls the
// rectangular composite  G[m][j'][j] = 2 pi sum_{l=m}^{Ls} Pbar_lm(theta'_j') w_j Pbar_lm(theta_j)   (j' on the Gauss-Legendre grid
// of band limit Ld, j on that of Ls): analysis on the source colatitudes, the series summed at the destination ones.
void shell_interp_composites(int Ls, int Ld, std::vector<ld>& G);

}  // namespace ghb
