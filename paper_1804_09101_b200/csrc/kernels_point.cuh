// kernels_point.cuh — pointwise kernels: fused Jacobian + GH right-hand side + face mask (A4-A6),
// RK stage update (A7), constraints + reduction (A8).
//
// The evolved system is the first-order generalized-harmonic Einstein system the paper evolves
// ("the Einstein equations in their generalized harmonic formulation"; "about 50 fundamental
// variables"); the paper does not print it, reading S1 writes it out:
//   dt psi_ab  = (1+g1) N^k d_k psi_ab - N Pi_ab - g1 N^i Phi_iab
//   dt Pi_ab   = N^k d_k Pi_ab - N g^{ki} d_k Phi_iab + g1 g2 N^k (d_k psi_ab - Phi_kab)
//                + 2N psi^{cd} ( g^{ij} Phi_ica Phi_jdb - Pi_ca Pi_db - psi^{ef} Gam_ace Gam_bdf )
//                - 2N nabla_(a H_b) - 1/2 N t^c t^d Pi_cd Pi_ab - N t^c Pi_ci g^{ij} Phi_jab
//                + N g0 ( t_b C_a + t_a C_b - psi_ab t^c C_c )
//   dt Phi_iab = N^k d_k Phi_iab - N d_i Pi_ab + N g2 (d_i psi_ab - Phi_iab)
//                + 1/2 N t^c t^d Phi_icd Pi_ab + N g^{jk} t^c Phi_ijc Phi_kab
// with Gam_abc built from the first-order variables (d_0 psi = -N Pi + N^i Phi_i, d_i psi = Phi_i).
#pragma once
#include "device_types.h"
#include "kernels_deriv.cuh"

namespace ghd {

// index of the symmetric pair (a,b) in the packed order 00,01,02,03,11,12,13,22,23,33
__host__ __device__ constexpr int SI(int a, int b) {
  return a <= b ? (a * 4 - (a * (a - 1)) / 2 + b - a) : (b * 4 - (b * (b - 1)) / 2 + a - b);
}
// index of the spatial symmetric pair (i,j), i,j in 0..2, packed xx,xy,xz,yy,yz,zz
__host__ __device__ constexpr int S3(int i, int j) {
  return i <= j ? (i * 3 - (i * (i - 1)) / 2 + j - i) : (j * 3 - (j * (j - 1)) / 2 + i - j);
}

// max that PROPAGATES NaN (fmax drops a NaN operand: a NaN constraint or error estimate would report a finite maximum)
__device__ __forceinline__ double nanmax(double a, double b) { return (a != a || b != b) ? (a + b) : fmax(a, b); }

struct Geom {
  double gi[6];     // g^{ij}
  double sh[3];     // N^i
  double N;         // lapse
  double pinv[10];  // psi^{ab}
  double tu[4];     // t^a = (1/N, -N^i/N)
};

// O4 of DESIGN.md.  Returns false on non-physical data (det g_ij <= 0 or N^2 <= 0).
__device__ __forceinline__ bool geometry(const double (&psi)[10], Geom& G) {
  const double gxx = psi[SI(1, 1)], gxy = psi[SI(1, 2)], gxz = psi[SI(1, 3)];
  const double gyy = psi[SI(2, 2)], gyz = psi[SI(2, 3)], gzz = psi[SI(3, 3)];
  const double cxx = gyy * gzz - gyz * gyz, cxy = gyz * gxz - gxy * gzz, cxz = gxy * gyz - gyy * gxz;
  const double det = gxx * cxx + gxy * cxy + gxz * cxz;
  const double idet = 1.0 / det;
  G.gi[S3(0, 0)] = cxx * idet;
  G.gi[S3(0, 1)] = cxy * idet;
  G.gi[S3(0, 2)] = cxz * idet;
  G.gi[S3(1, 1)] = (gxx * gzz - gxz * gxz) * idet;
  G.gi[S3(1, 2)] = (gxy * gxz - gxx * gyz) * idet;
  G.gi[S3(2, 2)] = (gxx * gyy - gxy * gxy) * idet;
  double n2 = -psi[SI(0, 0)];
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    double s = 0.0;
#pragma unroll
    for (int j = 0; j < 3; ++j) s = fma(G.gi[S3(i, j)], psi[SI(0, j + 1)], s);
    G.sh[i] = s;
  }
#pragma unroll
  for (int i = 0; i < 3; ++i) n2 = fma(G.sh[i], psi[SI(0, i + 1)], n2);
  const bool ok = (det > 0.0) && (n2 > 0.0);
  const double in2 = 1.0 / n2;
  G.N = sqrt(n2);
  G.pinv[SI(0, 0)] = -in2;
#pragma unroll
  for (int i = 0; i < 3; ++i) G.pinv[SI(0, i + 1)] = G.sh[i] * in2;
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = i; j < 3; ++j) G.pinv[SI(i + 1, j + 1)] = G.gi[S3(i, j)] - G.sh[i] * G.sh[j] * in2;
  const double iN = 1.0 / G.N;
  G.tu[0] = iN;
#pragma unroll
  for (int i = 0; i < 3; ++i) G.tu[i + 1] = -G.sh[i] * iN;
  return ok;
}

// Phi_iab accessors: registers (K_con) or this thread's column of a shared-memory array [30][TILE_PTS] (K_rhs, where
// Phi in registers is what forces spills: the compiler fetches each value where it is used instead).
struct PhiReg {
  const double (&v)[3][10];
  __device__ __forceinline__ double operator()(int i, int s) const { return v[i][s]; }
};
struct PhiSm {
  const double* p;   // + tid
  __device__ __forceinline__ double operator()(int i, int s) const { return p[(i * 10 + s) * TILE_PTS]; }
};

// Christoffel symbols of the first kind from the first-order variables, as 4 symmetric matrices
// Gam[a][SI(b,c)] = 1/2 (D_b psi_ac + D_c psi_ab - D_a psi_bc),  D_0 = -N Pi + N^i Phi_i,  D_i = Phi_i.
template <class PI, class PH>
__device__ __forceinline__ void christoffel(const Geom& G, const PI& Pi, const PH& Phi,
                                            double (&Gam)[4][10]) {
  double D0[10];
#pragma unroll
  for (int s = 0; s < 10; ++s) {
    double v = -G.N * Pi[s];
#pragma unroll
    for (int i = 0; i < 3; ++i) v = fma(G.sh[i], Phi(i, s), v);
    D0[s] = v;
  }
#define GH_D(c, s) ((c) == 0 ? D0[s] : Phi((c) - 1, s))
#pragma unroll
  for (int a = 0; a < 4; ++a)
#pragma unroll
    for (int b = 0; b < 4; ++b)
#pragma unroll
      for (int c = b; c < 4; ++c)
        Gam[a][SI(b, c)] = 0.5 * (GH_D(b, SI(a, c)) + GH_D(c, SI(a, b)) - GH_D(a, SI(b, c)));
#undef GH_D
}

// One Christoffel matrix Gam_a[SI(b,c)] on the fly from D_0 (registers) and Phi.  K_rhs never holds all four: the 40
// values are what pushes the kernel over 255 registers; recomputing a matrix costs 30 flop.  The empty asm makes each
// recomputed value opaque, so that the compiler cannot merge the copies back into one long-lived array.
template <int a, class PH>
__device__ __forceinline__ void gam_row(const double (&D0)[10], const PH& Phi, double (&Ga)[10]) {
#define GH_D(c, s) ((c) == 0 ? D0[s] : Phi((c) - 1, s))
#pragma unroll
  for (int b = 0; b < 4; ++b)
#pragma unroll
    for (int c = b; c < 4; ++c) {
      double v = 0.5 * (GH_D(b, SI(a, c)) + GH_D(c, SI(a, b)) - GH_D(a, SI(b, c)));
      asm("" : "+d"(v));
      Ga[SI(b, c)] = v;
    }
#undef GH_D
}

// full contraction of two symmetric 4x4 matrices X^{bc} Y_bc in packed storage
__device__ __forceinline__ double symdot(const double (&X)[10], const double (&Y)[10]) {
  double s = 0.0;
#pragma unroll
  for (int b = 0; b < 4; ++b)
#pragma unroll
    for (int c = b; c < 4; ++c) s = fma((b == c ? 1.0 : 2.0) * X[SI(b, c)], Y[SI(b, c)], s);
  return s;
}

// Quantities of the algebraic part that the per-(ab) assembly needs.
struct Alg {
  double S[10];    // W_ab - (Pi psi^-1 Pi)_ab - T_ab + H^d Gam_dab
  double C[4];     // C_a = H_a + Gam_a
  double tC;       // t^c C_c
  double ttPi;     // t^c t^d Pi_cd
  double p[3];     // t^c Pi_ci
  double s[3];     // t^c t^d Phi_icd
  double w[3][3];  // w[i][j] = t^c Phi_i(j+1)c
};

template <int a, class PH>
__device__ __forceinline__ void alg_gamma(const Geom& G, const double (&D0)[10], const PH& Phi, const double (&H)[4],
                                          const double (&Hup)[4], Alg& A) {
  double Ga[10];
  gam_row<a>(D0, Phi, Ga);
  A.C[a] = H[a] + symdot(G.pinv, Ga);
#pragma unroll
  for (int s = 0; s < 10; ++s) A.S[s] = fma(Hup[a], Ga[s], A.S[s]);      // H^d Gam_dab
  double Y[4][4];  // Y[d][e] = psi^{dc} Gam_a[c][e]
#pragma unroll
  for (int d = 0; d < 4; ++d)
#pragma unroll
    for (int e = 0; e < 4; ++e) {
      double v = 0.0;
#pragma unroll
      for (int c = 0; c < 4; ++c) v = fma(G.pinv[SI(d, c)], Ga[SI(c, e)], v);
      Y[d][e] = v;
    }
  double R[10];    // R_a = psi^-1 Gam_a psi^-1
#pragma unroll
  for (int d = 0; d < 4; ++d)
#pragma unroll
    for (int f = d; f < 4; ++f) {
      double v = 0.0;
#pragma unroll
      for (int e = 0; e < 4; ++e) v = fma(Y[d][e], G.pinv[SI(e, f)], v);
      R[SI(d, f)] = v;
    }
  // T_ab = psi^{cd} psi^{ef} Gam_ace Gam_bdf = R_a : Gam_b
  A.S[SI(a, a)] -= symdot(R, Ga);
  if (a < 1) { double Gb[10]; gam_row<1>(D0, Phi, Gb); A.S[SI(a, 1)] -= symdot(R, Gb); }
  if (a < 2) { double Gb[10]; gam_row<2>(D0, Phi, Gb); A.S[SI(a, 2)] -= symdot(R, Gb); }
  if (a < 3) { double Gb[10]; gam_row<3>(D0, Phi, Gb); A.S[SI(a, 3)] -= symdot(R, Gb); }
}

template <class PI, class PH>
__device__ __forceinline__ void algebraic(const Geom& G, const PI& Pi, const PH& Phi,
                                          const double (&H)[4], Alg& A) {
  double D0[10];   // D_0 psi_ab = -N Pi_ab + N^i Phi_iab
#pragma unroll
  for (int s = 0; s < 10; ++s) {
    double v = -G.N * Pi[s];
#pragma unroll
    for (int i = 0; i < 3; ++i) v = fma(G.sh[i], Phi(i, s), v);
    D0[s] = v;
  }
  double Hup[4];
#pragma unroll
  for (int d = 0; d < 4; ++d) {
    double v = 0.0;
#pragma unroll
    for (int c = 0; c < 4; ++c) v = fma(G.pinv[SI(d, c)], H[c], v);
    Hup[d] = v;
  }
#pragma unroll
  for (int s = 0; s < 10; ++s) A.S[s] = 0.0;
  // per a: Gam_a -> C_a, H^a Gam_a, R_a = psi^-1 Gam_a psi^-1; then - T_ab = - R_a : Gam_b for b >= a
  alg_gamma<0>(G, D0, Phi, H, Hup, A);
  alg_gamma<1>(G, D0, Phi, H, Hup, A);
  alg_gamma<2>(G, D0, Phi, H, Hup, A);
  alg_gamma<3>(G, D0, Phi, H, Hup, A);
  A.tC = 0.0;
#pragma unroll
  for (int a = 0; a < 4; ++a) A.tC = fma(G.tu[a], A.C[a], A.tC);
  // - Pi_ac psi^{cd} Pi_db
  {
    double Q[4][4];  // Q[c][b] = psi^{cd} Pi_db
#pragma unroll
    for (int c = 0; c < 4; ++c)
#pragma unroll
      for (int b = 0; b < 4; ++b) {
        double v = 0.0;
#pragma unroll
        for (int d = 0; d < 4; ++d) v = fma(G.pinv[SI(c, d)], Pi[SI(d, b)], v);
        Q[c][b] = v;
      }
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
      for (int b = a; b < 4; ++b) {
        double v = 0.0;
#pragma unroll
        for (int c = 0; c < 4; ++c) v = fma(Pi[SI(a, c)], Q[c][b], v);
        A.S[SI(a, b)] -= v;
      }
  }
  // + W_ab = g^{ij} Phi_iac psi^{cd} Phi_jdb = sum_i (Phi^i psi^-1 Phi_i)_ab,  Phi^i = g^{ij} Phi_j
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    double Z[4][4];  // Z[c][b] = psi^{cd} Phi_i,db
#pragma unroll
    for (int c = 0; c < 4; ++c)
#pragma unroll
      for (int b = 0; b < 4; ++b) {
        double v = 0.0;
#pragma unroll
        for (int d = 0; d < 4; ++d) v = fma(G.pinv[SI(c, d)], Phi(i, SI(d, b)), v);
        Z[c][b] = v;
      }
#pragma unroll
    for (int a = 0; a < 4; ++a) {
      double up[4];  // Phi^i_ac, c = 0..3
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        double v = 0.0;
#pragma unroll
        for (int j = 0; j < 3; ++j) v = fma(G.gi[S3(i, j)], Phi(j, SI(a, c)), v);
        up[c] = v;
      }
#pragma unroll
      for (int b = a; b < 4; ++b) {
        double v = 0.0;
#pragma unroll
        for (int c = 0; c < 4; ++c) v = fma(up[c], Z[c][b], v);
        A.S[SI(a, b)] += v;
      }
    }
  }
  // small contractions with the normal t^a
  A.ttPi = 0.0;
#pragma unroll
  for (int c = 0; c < 4; ++c)
#pragma unroll
    for (int d = 0; d < 4; ++d) A.ttPi = fma(G.tu[c] * G.tu[d], Pi[SI(c, d)], A.ttPi);
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    double v = 0.0, u = 0.0;
#pragma unroll
    for (int c = 0; c < 4; ++c) v = fma(G.tu[c], Pi[SI(c, i + 1)], v);
    A.p[i] = v;
#pragma unroll
    for (int c = 0; c < 4; ++c)
#pragma unroll
      for (int d = 0; d < 4; ++d) u = fma(G.tu[c] * G.tu[d], Phi(i, SI(c, d)), u);
    A.s[i] = u;
#pragma unroll
    for (int j = 0; j < 3; ++j) {
      double x = 0.0;
#pragma unroll
      for (int c = 0; c < 4; ++c) x = fma(G.tu[c], Phi(i, SI(j + 1, c)), x);
      A.w[i][j] = x;
    }
  }
}


// ---------------------------------------------------------------------------------------------------------
// K_rhs.  One thread per grid point, TILE_PTS points per CTA, tiles never straddle subdomains.
// Reads 50 fields + 150 logical derivatives + 4 H_a + 12 d_iH_a once, writes 50 once (2 152 B/point).
// Stage 1: psi -> geometry; stage 2: Pi, Phi -> algebraic part (Gam, quadratic sources, C_a);
// stage 3: per symmetric pair (ab) stream in its 15 derivatives (Jacobian applied on the fly for shells),
// assemble the 5 outputs and store.  FROZEN faces get zeros (A6).
//
// A7 fused: with RK != 0 the kernel does not store d_t u but the Shu-Osher stage update
//   out = a u0 + b (u + dt d_t u)        (RK = 1: a = 0, u0 not read;  RK = 2: u0 read)
// using the field values it already holds in registers, which saves writing and re-reading d_t u and re-reading u
// (1 200 B/point/stage).  `out` may alias `u` or `u0` (in-place stages): every field of the point is in registers
// before the first store, and u / u0 / out are deliberately NOT __restrict__ so that the compiler cannot re-load them.
// ---------------------------------------------------------------------------------------------------------
struct RkArgs { const double* u0; double a, b, dt; };

// ---------------------------------------------------------------------------------------------------------
// K_face_interp (NEXT-2 (iii) between shells of different band limit; "at 'internal' boundaries between neighboring domains, the
// characteristic variables are computed and used as boundary conditions on the neighboring subdomain"; interpolation
// "via a direct summation of the spectral series"): the neighbour's face state, given on its own Gauss-Legendre x
// uniform grid of band limit Ls, is analysed there and the series is summed at the nodes of this shell's grid (band limit Ld):
//   C[j][q]  = sum_k  u[j][k] Fa_s[q][k]          real DFT on the source longitudes (q = 0: m = 0; 1..Ls: cos m; Ls+1..2Ls: sin m)
//   D[j'][q] = sum_j  G_m(q)[j'][j] C[j][q]       per m: 2 pi sum_l Pbar_lm(theta'_j') w_j Pbar_lm(theta_j)
//   out[j'][k'] = sum_q D[j'][q] Fx[k'][q]        the Fourier series at the destination longitudes (all m <= Ls, not truncated)
// grid = (faces, components); a face is a few thousand points: plain DFMA, operands staged in shared memory, the matrices stored
// transposed so that consecutive threads read consecutive addresses.
// ---------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
k_face_interp(const IfcItem* __restrict__ items, const double* __restrict__ tables, const double* __restrict__ u,
              double* __restrict__ ifc, int64_t S, int64_t Sf) {
  extern __shared__ __align__(16) double fsm[];
  const IfcItem it = items[blockIdx.x];
  const int c = blockIdx.y, tid = threadIdx.x;
  const int nts = it.Ls + 1, nps = 2 * it.Ls + 2, nqs = 2 * it.Ls + 1, ntd = it.Ld + 1, npd = 2 * it.Ld + 2;
  double* U = fsm;                       // [nts][nps]
  double* Cq = U + nts * nps;            // [nts][nqs]
  double* Dq = Cq + nts * nqs;           // [ntd][nqs]
  const double* __restrict__ src = u + (int64_t)c * S + it.src_off;
  for (int e = tid; e < nts * nps; e += 256) U[e] = src[e];
  __syncthreads();
  const double* __restrict__ FaT = tables + it.m_FaT;
  for (int e = tid; e < nts * nqs; e += 256) {
    const int j = e / nqs, q = e - j * nqs;
    double s = 0.0;
    for (int k = 0; k < nps; ++k) s = fma(U[j * nps + k], __ldg(FaT + (int64_t)k * nqs + q), s);
    Cq[e] = s;
  }
  __syncthreads();
  const double* __restrict__ GT = tables + it.m_GT;
  for (int e = tid; e < ntd * nqs; e += 256) {
    const int q = e / ntd, jd = e - q * ntd;
    const int m = q <= it.Ls ? q : q - it.Ls;
    const double* __restrict__ g = GT + (int64_t)m * nts * ntd + jd;
    double s = 0.0;
    for (int j = 0; j < nts; ++j) s = fma(__ldg(g + (int64_t)j * ntd), Cq[j * nqs + q], s);
    Dq[jd * nqs + q] = s;
  }
  __syncthreads();
  const double* __restrict__ FxT = tables + it.m_FxT;
  double* __restrict__ dst = ifc + (int64_t)c * Sf + it.dst_off;
  for (int e = tid; e < ntd * npd; e += 256) {
    const int jd = e / npd, k = e - jd * npd;
    double s = 0.0;
    for (int q = 0; q < nqs; ++q) s = fma(Dq[jd * nqs + q], __ldg(FxT + (int64_t)q * npd + k), s);
    dst[e] = s;
  }
}

// Characteristic boundary condition (NEXT-2 (i), reading S21) for one symmetric pair (ab) at a face point with outward
// direction s: with n_i = s_i / sqrt(g^{jk} s_j s_k), n^i = g^{ij} n_j,
//   u0 = psi (speed -(1+g1) n.N),  u1+- = Pi +- n^i Phi_i - g2 psi (speed -n.N +- N),  u2_i = Phi_i - n_i n^k Phi_k (speed -n.N);
// the time derivatives of the fields with negative speed (entering the domain) are set to zero, the rest kept.
__device__ __forceinline__ void char_bc_pair(const Geom& G, double g1, double g2, double sx, double sy, double sz,
                                             double& dpsi, double& dPi, double (&dPhi)[3]) {
  const double sv[3] = {sx, sy, sz};
  double gs[3], nn = 0.0;
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    double v = 0.0;
#pragma unroll
    for (int j = 0; j < 3; ++j) v = fma(G.gi[S3(i, j)], sv[j], v);
    gs[i] = v;
    nn = fma(v, sv[i], nn);
  }
  const double inv = 1.0 / sqrt(nn);
  double nd[3], nu[3], nN = 0.0, nPhi = 0.0;
#pragma unroll
  for (int i = 0; i < 3; ++i) { nd[i] = sv[i] * inv; nu[i] = gs[i] * inv; nN = fma(nd[i], G.sh[i], nN); nPhi = fma(nu[i], dPhi[i], nPhi); }
  double u0 = dpsi, u1p = dPi + nPhi - g2 * dpsi, u1m = dPi - nPhi - g2 * dpsi, u2[3];
#pragma unroll
  for (int i = 0; i < 3; ++i) u2[i] = dPhi[i] - nd[i] * nPhi;
  if (-(1.0 + g1) * nN < 0.0) u0 = 0.0;
  if (-nN + G.N < 0.0) u1p = 0.0;
  if (-nN - G.N < 0.0) u1m = 0.0;
  if (-nN < 0.0) { u2[0] = 0.0; u2[1] = 0.0; u2[2] = 0.0; }
  dpsi = u0;
  dPi = 0.5 * (u1p + u1m) + g2 * u0;
#pragma unroll
  for (int i = 0; i < 3; ++i) dPhi[i] = 0.5 * (u1p - u1m) * nd[i] + u2[i];
}

// Characteristic penalty exchange (NEXT-2 (iii), reading S22) for one symmetric pair at an INTERFACE point: e* = own minus
// neighbour state; every field entering along the outward direction s gets  d_t u^a += p v_a (u^a_own - u^a_nbr)  (v_a < 0).
__device__ __forceinline__ void char_penalty_pair(const Geom& G, double g1, double g2, double sx, double sy, double sz, double pen,
                                                  double epsi, double ePi, const double (&ePhi)[3],
                                                  double& dpsi, double& dPi, double (&dPhi)[3]) {
  const double sv[3] = {sx, sy, sz};
  double gs[3], nn = 0.0;
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    double v = 0.0;
#pragma unroll
    for (int j = 0; j < 3; ++j) v = fma(G.gi[S3(i, j)], sv[j], v);
    gs[i] = v;
    nn = fma(v, sv[i], nn);
  }
  const double inv = 1.0 / sqrt(nn);
  double nd[3], nu[3], nN = 0.0, nPhi = 0.0;
#pragma unroll
  for (int i = 0; i < 3; ++i) { nd[i] = sv[i] * inv; nu[i] = gs[i] * inv; nN = fma(nd[i], G.sh[i], nN); nPhi = fma(nu[i], ePhi[i], nPhi); }
  const double v0 = -(1.0 + g1) * nN, v1p = -nN + G.N, v1m = -nN - G.N, v2 = -nN;
  const double c0 = v0 < 0.0 ? pen * v0 * epsi : 0.0;
  const double c1p = v1p < 0.0 ? pen * v1p * (ePi + nPhi - g2 * epsi) : 0.0;
  const double c1m = v1m < 0.0 ? pen * v1m * (ePi - nPhi - g2 * epsi) : 0.0;
  dpsi += c0;
  dPi += 0.5 * (c1p + c1m) + g2 * c0;
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    const double c2 = v2 < 0.0 ? pen * v2 * (ePhi[i] - nd[i] * nPhi) : 0.0;
    dPhi[i] += 0.5 * (c1p - c1m) * nd[i] + c2;
  }
}

template <int RK>
__device__ __forceinline__ void rhs_store(double* out, const RkArgs& rk, int64_t idx, double dtu, double us, double u0v) {
  if (RK == 0) { out[idx] = dtu; return; }
  double r = rk.b * fma(rk.dt, dtu, us);
  if (RK == 2) r = fma(rk.a, u0v, r);
  out[idx] = r;
}

// Stage-3 operands of the symmetric pair s = (a,b): its 15 logical derivatives and up to 2 gauge-source gradients.
// Each thread copies ITS OWN point's values with cp.async into its own column of a shared-memory ring
// ring[slot][RHS_RING_ROWS][TILE_PTS] and later reads them back itself, so no block-level synchronisation is needed:
// the loads of pairs s .. s+RHS_RING-1 are in flight while the algebra of stage 2 and the assembly of earlier pairs
// run, which is what an HBM-bound kernel with 255 registers per thread (8 warps per SM) cannot get from the warp
// scheduler alone.
#ifndef GH_RHS_RING
#define GH_RHS_RING 3
#endif
constexpr int RHS_RING = GH_RHS_RING, RHS_RING_ROWS = 22, RHS_PHI_ROWS = 30;   // 15 derivatives + 2 gauge-source gradients + 5 u0 values (RK = 2)
constexpr size_t RHS_SMEM_BYTES = (size_t)(RHS_PHI_ROWS + RHS_RING * RHS_RING_ROWS) * TILE_PTS * sizeof(double);
// NORMS (A8 as an epilogue of A5): this thread's partials {sum C_a^2, sum C_iab^2, sum C_ijab^2, max |C_a|,
// max |C_iab|, max |C_ijab|} live in shared memory, not registers (the kernel already sits at the register limit): in rows 17..21
// of ring slot 0 and row 17 of slot 1, which only the RK = 2 prefetch uses (its u0 values) and NORMS exists for RK = 1 only -
// so the fused norms cost no shared memory (more of it would come out of the L1 that absorbs the kernel's spills).
constexpr int RHS_NORM_ROWS = 6;
__host__ __device__ constexpr int rhs_norm_row(int q) { return RHS_PHI_ROWS + (q < 5 ? 17 + q : RHS_RING_ROWS + 17); }
constexpr size_t RHS_SMEM_BYTES_NORMS = RHS_SMEM_BYTES;

template <int PAIR, int RK>
__device__ __forceinline__ void rhs_prefetch(double* __restrict__ slot /* + tid */, const double* __restrict__ du,
                                             const double* __restrict__ dHs, const double* u0, int64_t S, int64_t p) {
  constexpr int a = PAIR < 4 ? 0 : PAIR < 7 ? 1 : PAIR < 9 ? 2 : 3;
  constexpr int b = PAIR < 4 ? PAIR : PAIR < 7 ? PAIR - 3 : PAIR < 9 ? PAIR - 5 : 3;
  const int64_t DS = (int64_t)NCOMP * S;
#pragma unroll
  for (int c5 = 0; c5 < 5; ++c5)
#pragma unroll
    for (int kk = 0; kk < 3; ++kk)
      cp_async8(slot + (c5 * 3 + kk) * TILE_PTS, du + kk * DS + (int64_t)(10 * c5 + PAIR) * S + p);
  if (a > 0) cp_async8(slot + 15 * TILE_PTS, dHs + (int64_t)((a - 1) * 4 + b) * S + p);
  if (b > 0) cp_async8(slot + 16 * TILE_PTS, dHs + (int64_t)((b - 1) * 4 + a) * S + p);
  if (RK == 2) {
#pragma unroll
    for (int c5 = 0; c5 < 5; ++c5) cp_async8(slot + (17 + c5) * TILE_PTS, u0 + (int64_t)(10 * c5 + PAIR) * S + p);
  }
  cp_async_commit();
}

template <bool SHELL, int RK, bool CBC, bool NORMS>
__device__ __forceinline__ void rhs_point(const SubDev& sd, const double* __restrict__ tables, int local,
                                          const double* u, const double* __restrict__ du,
                                          const double* __restrict__ Hs, const double* __restrict__ dHs,
                                          double* k, const RkArgs& rk, int64_t S, int* __restrict__ flag,
                                          double* __restrict__ phis /* + tid */, const double* __restrict__ ifc = nullptr,
                                          int64_t Sf = 0) {
  double* __restrict__ ring = phis + RHS_PHI_ROWS * TILE_PTS;
  static_assert(!NORMS || RK == 1, "the NORMS partials sit in the ring rows of the RK = 2 prefetch");
#define GH_NACC(q) phis[rhs_norm_row(q) * TILE_PTS]    /* NORMS: this thread's six partials */
  const int64_t p = sd.off + local;
  // face mask (A6)
  bool frozen;
  int cmask = 0;   // faces flagged CHARACTERISTIC (2) through this point, bit f = face f
  {
    const int i2 = local % sd.n2, t = local / sd.n2, i1 = t % sd.n1, i0 = t / sd.n1;
    // SHELL covers shells (faces 0, 1) and cylindrical shells (kind 2: faces 0..3, the phi direction is periodic)
    const bool ax1 = !SHELL || sd.kind == 2;
    const bool on[6] = {i0 == 0, i0 == sd.n0 - 1, ax1 && i1 == 0, ax1 && i1 == sd.n1 - 1, !SHELL && i2 == 0, !SHELL && i2 == sd.n2 - 1};
    frozen = false;
#pragma unroll
    for (int f = 0; f < (SHELL ? 4 : 6); ++f) {
      frozen = frozen || (on[f] && sd.face[f] == 1);
      if (CBC && on[f] && sd.face[f] == 2) cmask |= 1 << f;
      if (CBC && SHELL && f < 2 && on[f] && sd.face[f] == 3) cmask |= 64 << f;      // INTERFACE faces: bits 6, 7
    }
  }
  constexpr int SLOT = RHS_RING_ROWS * TILE_PTS;
  // Phi_iab of this point -> shared memory (first cp.async group), then the first RHS_RING pairs of stage 3
#pragma unroll
  for (int c = 0; c < RHS_PHI_ROWS; ++c) cp_async8(phis + c * TILE_PTS, u + (int64_t)(50 - RHS_PHI_ROWS + c) * S + p);
  cp_async_commit();
  // with NORMS a frozen point takes the full path too: its constraints count, only its time derivative is zero
  const bool skip = frozen && !NORMS;
  if (!skip) {
    rhs_prefetch<0, RK>(ring + 0 * SLOT, du, dHs, rk.u0, S, p);
    rhs_prefetch<1, RK>(ring + 1 * SLOT, du, dHs, rk.u0, S, p);
    if (RHS_RING > 2) rhs_prefetch<2, RK>(ring + (RHS_RING > 2 ? 2 : 0) * SLOT, du, dHs, rk.u0, S, p);
  }
  const PhiSm Phi{phis};
  double psi[10], H[4], Pi[10];
#pragma unroll
  for (int s = 0; s < 10; ++s) Pi[s] = u[(int64_t)(10 + s) * S + p];
#pragma unroll
  for (int s = 0; s < 10; ++s) psi[s] = u[(int64_t)s * S + p];
#pragma unroll
  for (int a = 0; a < 4; ++a) H[a] = Hs[(int64_t)a * S + p];

  Geom G;
  const bool ok = geometry(psi, G);
  if (!ok) atomicOr(flag, 1);
  if (skip) cp_async_wait<0>(); else cp_async_wait<RHS_RING>();   // the Phi group has landed
  if (!ok || skip) {
    cp_async_wait<0>();   // nothing of this thread may still be landing in shared memory when the CTA retires
    // frozen points issued no prefetch: u0 comes straight from memory.  All 50 loads go out before the first store: u0 and
    // out are not __restrict__ (they may be the same array), so a load placed after a store would have to wait for it
    double z[5][10];
    if (RK == 2) {
#pragma unroll
      for (int c5 = 0; c5 < 5; ++c5)
#pragma unroll
        for (int s = 0; s < 10; ++s) z[c5][s] = rk.u0[(int64_t)(10 * c5 + s) * S + p];
    }
#pragma unroll
    for (int s = 0; s < 10; ++s) {
      rhs_store<RK>(k, rk, (int64_t)s * S + p, 0.0, psi[s], RK == 2 ? z[0][s] : 0.0);
      rhs_store<RK>(k, rk, (int64_t)(10 + s) * S + p, 0.0, Pi[s], RK == 2 ? z[1][s] : 0.0);
#pragma unroll
      for (int i = 0; i < 3; ++i)
        rhs_store<RK>(k, rk, (int64_t)(20 + 10 * i + s) * S + p, 0.0, Phi(i, s), RK == 2 ? z[2 + i][s] : 0.0);
    }
    return;
  }
  Alg A;
  algebraic(G, Pi, Phi, H, A);
  if (NORMS) {
    double s0 = 0.0, m0 = 0.0;
#pragma unroll
    for (int a = 0; a < 4; ++a) { s0 = fma(A.C[a], A.C[a], s0); m0 = nanmax(m0, fabs(A.C[a])); }
    GH_NACC(0) = s0; GH_NACC(3) = m0;
  }

  ShellJac J;
  if (SHELL) J = shell_jac(sd, tables, local);
  const double g0 = sd.gamma[0], g1 = sd.gamma[1], g2 = sd.gamma[2], N = G.N;

#pragma unroll
  for (int a = 0; a < 4; ++a)
#pragma unroll
    for (int b = a; b < 4; ++b) {
      const int s = SI(a, b);
      // groups committed so far: min(10, s + RHS_RING); group s must have landed
      if (s + RHS_RING <= 10) cp_async_wait<RHS_RING - 1>();
      else if (s == 8) cp_async_wait<1>();
      else cp_async_wait<0>();
      const double* __restrict__ slot = ring + (s % RHS_RING) * SLOT;
      // d[c5][k]: Cartesian derivative k of component (psi, Pi, Phi_x, Phi_y, Phi_z)_ab
      double d[5][3];
#pragma unroll
      for (int c5 = 0; c5 < 5; ++c5) {
        const double l0 = slot[(c5 * 3 + 0) * TILE_PTS], l1 = slot[(c5 * 3 + 1) * TILE_PTS], l2 = slot[(c5 * 3 + 2) * TILE_PTS];
        if (SHELL) {
          d[c5][0] = J.xr * l0 + J.xt * l1 + J.xp * l2;
          d[c5][1] = J.yr * l0 + J.yt * l1 + J.yp * l2;
          d[c5][2] = J.zr * l0 + J.zt * l1;
        } else {
          d[c5][0] = l0; d[c5][1] = l1; d[c5][2] = l2;
        }
      }
      if (NORMS) {   // C_iab = d_i psi_ab - Phi_iab;  C_ijab = d_i Phi_jab - d_j Phi_iab for (i,j) = (x,y), (x,z), (y,z)
        double s1 = GH_NACC(1), m1 = GH_NACC(4);
#pragma unroll
        for (int i = 0; i < 3; ++i) { const double c = d[0][i] - Phi(i, s); s1 = fma(c, c, s1); m1 = nanmax(m1, fabs(c)); }
        GH_NACC(1) = s1; GH_NACC(4) = m1;
        const double c01 = d[3][0] - d[2][1], c02 = d[4][0] - d[2][2], c12 = d[4][1] - d[3][2];
        double s2 = GH_NACC(2);
        s2 = fma(c01, c01, s2); s2 = fma(c02, c02, s2); s2 = fma(c12, c12, s2);
        GH_NACC(2) = s2;
        GH_NACC(5) = nanmax(GH_NACC(5), nanmax(fabs(c01), nanmax(fabs(c02), fabs(c12))));
      }
      double sdpsi = 0.0, sdPi = 0.0, sPhi = 0.0;
#pragma unroll
      for (int kk = 0; kk < 3; ++kk) {
        sdpsi = fma(G.sh[kk], d[0][kk], sdpsi);
        sdPi = fma(G.sh[kk], d[1][kk], sdPi);
        sPhi = fma(G.sh[kk], Phi(kk, s), sPhi);
      }
      double o_psi = (1.0 + g1) * sdpsi - N * Pi[s] - g1 * sPhi;

      double gdPhi = 0.0;   // g^{ki} d_k Phi_iab
#pragma unroll
      for (int kk = 0; kk < 3; ++kk)
#pragma unroll
        for (int i = 0; i < 3; ++i) gdPhi = fma(G.gi[S3(kk, i)], d[2 + i][kk], gdPhi);
      double up[3];         // Phi^j_ab = g^{jk} Phi_kab
#pragma unroll
      for (int j = 0; j < 3; ++j) {
        double v = 0.0;
#pragma unroll
        for (int kk = 0; kk < 3; ++kk) v = fma(G.gi[S3(j, kk)], Phi(kk, s), v);
        up[j] = v;
      }
      // 1/2 (d_a H_b + d_b H_a), d_0 H = 0 ; dHs[(i*4+b)] = d_i H_b
      double symdH = 0.0;
      if (a > 0) symdH += slot[15 * TILE_PTS];
      if (b > 0) symdH += slot[16 * TILE_PTS];
      symdH *= 0.5;
      double pup = 0.0;
#pragma unroll
      for (int i = 0; i < 3; ++i) pup = fma(A.p[i], up[i], pup);
      // t_a = (-N, 0, 0, 0)
      const double tbCa = (b == 0 ? -N * A.C[a] : 0.0), taCb = (a == 0 ? -N * A.C[b] : 0.0);
      double r = sdPi - N * gdPhi + g1 * g2 * (sdpsi - sPhi) + 2.0 * N * (A.S[s] - symdH) - 0.5 * N * A.ttPi * Pi[s] -
                 N * pup + N * g0 * (tbCa + taCb - psi[s] * A.tC);
      double o_Phi[3];
#pragma unroll
      for (int i = 0; i < 3; ++i) {
        double sdPhi = 0.0, wup = 0.0;
#pragma unroll
        for (int kk = 0; kk < 3; ++kk) sdPhi = fma(G.sh[kk], d[2 + i][kk], sdPhi);
#pragma unroll
        for (int j = 0; j < 3; ++j) wup = fma(A.w[i][j], up[j], wup);
        o_Phi[i] = sdPhi - N * d[1][i] + N * g2 * (d[0][i] - Phi(i, s)) + 0.5 * N * A.s[i] * Pi[s] + N * wup;
      }
      if (CBC && SHELL && (cmask & 192)) {   // INTERFACE faces: the neighbour's state at the coincident point, straight from u
        const int q = local % (sd.n1 * sd.n2);
#pragma unroll
        for (int f = 0; f < 2; ++f)
          if (cmask & (64 << f)) {
            // the neighbour's state at this point of the face: straight from the store where the grids coincide, else from
            // the interpolated copy K_face_interp made of it on this shell's grid
            const bool ip = sd.nbi[f] >= 0;
            const double* nb = ip ? ifc + sd.nbi[f] + q : u + sd.nbr[f] + q;
            const int64_t ns = ip ? Sf : S;
            const double sg = f ? 1.0 : -1.0;
            const double ePhi[3] = {Phi(0, s) - nb[(int64_t)(20 + s) * ns], Phi(1, s) - nb[(int64_t)(30 + s) * ns],
                                    Phi(2, s) - nb[(int64_t)(40 + s) * ns]};
            char_penalty_pair(G, g1, g2, sg * J.xr, sg * J.yr, sg * J.zr, sd.pen, psi[s] - nb[(int64_t)s * ns],
                              Pi[s] - nb[(int64_t)(10 + s) * ns], ePhi, o_psi, r, o_Phi);
          }
      }
      if (CBC && (cmask & 63)) {   // characteristic faces through this point, in face order (rare: face points only)
#pragma unroll
        for (int f = 0; f < (SHELL ? 4 : 6); ++f)
          if (cmask & (1 << f)) {
            const double sg = (f & 1) ? 1.0 : -1.0;
            // shells: +- r^ = (st cp, st sp, ct); cylindrical shells: +- rho^ = (cp, sp, 0) - the same entries - and +- z^
            if (SHELL && f < 2) char_bc_pair(G, g1, g2, sg * J.xr, sg * J.yr, sg * J.zr, o_psi, r, o_Phi);
            else if (SHELL) char_bc_pair(G, g1, g2, 0.0, 0.0, sg, o_psi, r, o_Phi);
            else char_bc_pair(G, g1, g2, f / 2 == 0 ? sg : 0.0, f / 2 == 1 ? sg : 0.0, f / 2 == 2 ? sg : 0.0, o_psi, r, o_Phi);
          }
      }
      if (NORMS && frozen) { o_psi = 0.0; r = 0.0; o_Phi[0] = o_Phi[1] = o_Phi[2] = 0.0; }      // A6
      rhs_store<RK>(k, rk, (int64_t)s * S + p, o_psi, psi[s], RK == 2 ? slot[17 * TILE_PTS] : 0.0);
      rhs_store<RK>(k, rk, (int64_t)(10 + s) * S + p, r, Pi[s], RK == 2 ? slot[18 * TILE_PTS] : 0.0);
#pragma unroll
      for (int i = 0; i < 3; ++i)
        rhs_store<RK>(k, rk, (int64_t)(20 + 10 * i + s) * S + p, o_Phi[i], Phi(i, s), RK == 2 ? slot[(19 + i) * TILE_PTS] : 0.0);
      // every value of the slot has been consumed: refill it with pair s + RHS_RING
#define GH_PF(K) if (s == K && K + RHS_RING < 10) rhs_prefetch<(K + RHS_RING < 10 ? K + RHS_RING : 9), RK>(ring + (K % RHS_RING) * SLOT, du, dHs, rk.u0, S, p);
      GH_PF(0) GH_PF(1) GH_PF(2) GH_PF(3) GH_PF(4) GH_PF(5) GH_PF(6) GH_PF(7)
#undef GH_PF

    }
#undef GH_NACC
}

// CBC: the domain has faces flagged CHARACTERISTIC (a second instantiation, so that domains without them do not pay for it).
// NORMS: the constraint norms of the INPUT state as an epilogue (A8 fused into A5: C_a, the derivatives of psi and Phi and
// Phi itself are on chip anyway; 0 extra bytes): per-tile partials part[tile][6] in the layout of K_con, folded by K_con_reduce.
#ifndef GH_RHS_CTAS
#define GH_RHS_CTAS 2      // resident CTAs per SM the register allocation aims at (3: a 170-register cap, measured slower - DESIGN.md §14)
#endif
template <int RK, bool CBC, bool NORMS = false>
__global__ void __launch_bounds__(TILE_PTS, GH_RHS_CTAS)
k_rhs(const SubDev* __restrict__ subs, const int32_t* __restrict__ tile_first, int n_sub,
      const double* __restrict__ tables, const double* u, const double* __restrict__ du,
      const double* __restrict__ Hs, const double* __restrict__ dHs, double* k, RkArgs rk, int64_t S,
      int* __restrict__ flag, double* __restrict__ part = nullptr, const double* __restrict__ ifc = nullptr, int64_t Sf = 0) {
  extern __shared__ __align__(16) double ring_s[];   // Phi [30][TILE_PTS], the ring [RHS_RING][RHS_RING_ROWS][TILE_PTS], NORMS: [6][TILE_PTS]
  __shared__ SubDev sd_s;
  __shared__ int tile0_s;
  __shared__ double red[TILE_PTS / 32][6];
  if (threadIdx.x == 0) {
    const int s = find_sub(tile_first, n_sub, blockIdx.x);
    sd_s = subs[s];
    tile0_s = tile_first[s];
  }
  double* nacc = ring_s + threadIdx.x;
  if (NORMS) {
#pragma unroll
    for (int q = 0; q < RHS_NORM_ROWS; ++q) nacc[rhs_norm_row(q) * TILE_PTS] = 0.0;      // own column: no barrier needed
  }
  __syncthreads();
  const SubDev& sd = sd_s;
  const int local = (blockIdx.x - tile0_s) * TILE_PTS + threadIdx.x;
  if (local < sd.P) {
    if (sd.kind != 1) rhs_point<true, RK, CBC, NORMS>(sd, tables, local, u, du, Hs, dHs, k, rk, S, flag, ring_s + threadIdx.x, ifc, Sf);
    else rhs_point<false, RK, CBC, NORMS>(sd, tables, local, u, du, Hs, dHs, k, rk, S, flag, ring_s + threadIdx.x);
  }
  if (NORMS) {    // the same fold as K_con: warp shuffle, then the warps in fixed order (deterministic)
    double acc[6];
#pragma unroll
    for (int q = 0; q < 6; ++q) acc[q] = nacc[rhs_norm_row(q) * TILE_PTS];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
      for (int q = 0; q < 3; ++q) acc[q] += __shfl_xor_sync(0xffffffffu, acc[q], o);
#pragma unroll
      for (int q = 3; q < 6; ++q) acc[q] = nanmax(acc[q], __shfl_xor_sync(0xffffffffu, acc[q], o));
    }
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (lane == 0)
#pragma unroll
      for (int q = 0; q < 6; ++q) red[warp][q] = acc[q];
    __syncthreads();
    if (threadIdx.x < 6) {
      const int q = threadIdx.x;
      double v = red[0][q];
      for (int w = 1; w < TILE_PTS / 32; ++w) v = (q < 3) ? v + red[w][q] : nanmax(v, red[w][q]);
      part[(int64_t)blockIdx.x * 6 + q] = v;
    }
  }
}

// ---------------------------------------------------------------------------------------------------------
// Dormand-Prince 5(4) (NEXT-3).  K_dp_stage: out = u + dt sum_{j<nk} a_j k_j over the whole store (padding is zero and
// stays zero).  K_dp_err: e = dt sum_j d_j k_j -> per-block {sum e^2, max |e|}; K_dp_err_final folds the partials in
// a fixed order.  All HBM-bound streaming kernels.
// ---------------------------------------------------------------------------------------------------------
struct DpArgs { const double2* k[7]; double a[7]; int nk; };

__global__ void __launch_bounds__(256)
k_dp_stage(const double2* __restrict__ u, DpArgs A, double dt, double2* __restrict__ out, int64_t n2) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n2; i += (int64_t)gridDim.x * blockDim.x) {
    double sx = 0.0, sy = 0.0;
#pragma unroll
    for (int j = 0; j < 7; ++j)
      if (j < A.nk) { const double2 v = A.k[j][i]; sx = fma(A.a[j], v.x, sx); sy = fma(A.a[j], v.y, sy); }
    const double2 w = u[i];
    out[i] = make_double2(fma(dt, sx, w.x), fma(dt, sy, w.y));
  }
}

__global__ void __launch_bounds__(256)
k_dp_err(DpArgs A, double dt, double* __restrict__ part, int64_t n2) {
  __shared__ double red[8][2];
  double ss = 0.0, mx = 0.0;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n2; i += (int64_t)gridDim.x * blockDim.x) {
    double sx = 0.0, sy = 0.0;
#pragma unroll
    for (int j = 0; j < 7; ++j)
      if (j < A.nk) { const double2 v = A.k[j][i]; sx = fma(A.a[j], v.x, sx); sy = fma(A.a[j], v.y, sy); }
    sx *= dt; sy *= dt;
    ss = fma(sx, sx, ss); ss = fma(sy, sy, ss);
    mx = nanmax(mx, nanmax(fabs(sx), fabs(sy)));
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) { ss += __shfl_xor_sync(0xffffffffu, ss, o); mx = nanmax(mx, __shfl_xor_sync(0xffffffffu, mx, o)); }
  if ((threadIdx.x & 31) == 0) { red[threadIdx.x >> 5][0] = ss; red[threadIdx.x >> 5][1] = mx; }
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < 8; ++w) { ss += red[w][0]; mx = nanmax(mx, red[w][1]); }
    part[2 * blockIdx.x] = ss; part[2 * blockIdx.x + 1] = mx;
  }
}

__global__ void __launch_bounds__(32)
k_dp_err_final(const double* __restrict__ part, int nblocks, double* __restrict__ out) {
  double ss = 0.0, mx = 0.0;
  for (int b = threadIdx.x; b < nblocks; b += 32) { ss += part[2 * b]; mx = nanmax(mx, part[2 * b + 1]); }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) { ss += __shfl_xor_sync(0xffffffffu, ss, o); mx = nanmax(mx, __shfl_xor_sync(0xffffffffu, mx, o)); }
  if (threadIdx.x == 0) { out[0] = ss; out[1] = mx; }
}

// ---------------------------------------------------------------------------------------------------------
// K_con (A8): constraints at a point, then warp-shuffle + block reduction to per-tile partials
// part[tile][6] = {sum C_a^2, sum C_iab^2, sum C_ijab^2, max|C_a|, max|C_iab|, max|C_ijab|};
// K_con_reduce folds the tiles of each subdomain in a fixed order (deterministic).
// ---------------------------------------------------------------------------------------------------------
template <bool SHELL>
__device__ __forceinline__ void con_point(const SubDev& sd, const double* __restrict__ tables, int local,
                                          const double* __restrict__ u, const double* __restrict__ du,
                                          const double* __restrict__ Hs, int64_t S, int* __restrict__ flag,
                                          double (&acc)[6]) {
  const int64_t p = sd.off + local;
  double psi[10], Pi[10], Phi[3][10], H[4];
#pragma unroll
  for (int s = 0; s < 10; ++s) psi[s] = u[(int64_t)s * S + p];
#pragma unroll
  for (int s = 0; s < 10; ++s) Pi[s] = u[(int64_t)(10 + s) * S + p];
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int s = 0; s < 10; ++s) Phi[i][s] = u[(int64_t)(20 + 10 * i + s) * S + p];
#pragma unroll
  for (int a = 0; a < 4; ++a) H[a] = Hs[(int64_t)a * S + p];
  Geom G;
  if (!geometry(psi, G)) { atomicOr(flag, 1); return; }
  {
    double Gam[4][10];
    christoffel(G, Pi, PhiReg{Phi}, Gam);
#pragma unroll
    for (int a = 0; a < 4; ++a) {
      const double c = H[a] + symdot(G.pinv, Gam[a]);
      acc[0] = fma(c, c, acc[0]);
      acc[3] = nanmax(acc[3], fabs(c));
    }
  }
  ShellJac J;
  if (SHELL) J = shell_jac(sd, tables, local);
  const int64_t DS = (int64_t)NCOMP * S;
#pragma unroll 1
  for (int s = 0; s < 10; ++s) {
    double d[4][3];   // Cartesian derivatives of psi_ab, Phi_xab, Phi_yab, Phi_zab
#pragma unroll
    for (int c4 = 0; c4 < 4; ++c4) {
      const int comp = (c4 == 0) ? s : 10 + 10 * c4 + s;
      const double* q = du + (int64_t)comp * S + p;
      const double l0 = q[0], l1 = q[DS], l2 = q[2 * DS];
      if (SHELL) {
        d[c4][0] = J.xr * l0 + J.xt * l1 + J.xp * l2;
        d[c4][1] = J.yr * l0 + J.yt * l1 + J.yp * l2;
        d[c4][2] = J.zr * l0 + J.zt * l1;
      } else {
        d[c4][0] = l0; d[c4][1] = l1; d[c4][2] = l2;
      }
    }
#pragma unroll
    for (int i = 0; i < 3; ++i) {
      const double c = d[0][i] - u[(int64_t)(20 + 10 * i + s) * S + p];
      acc[1] = fma(c, c, acc[1]);
      acc[4] = nanmax(acc[4], fabs(c));
    }
    // C_ijab = d_i Phi_jab - d_j Phi_iab for (i,j) = (0,1), (0,2), (1,2)
    const double c01 = d[2][0] - d[1][1], c02 = d[3][0] - d[1][2], c12 = d[3][1] - d[2][2];
    acc[2] = fma(c01, c01, acc[2]); acc[2] = fma(c02, c02, acc[2]); acc[2] = fma(c12, c12, acc[2]);
    acc[5] = nanmax(acc[5], nanmax(fabs(c01), nanmax(fabs(c02), fabs(c12))));
  }
}

__global__ void __launch_bounds__(TILE_PTS)
k_con(const SubDev* __restrict__ subs, const int32_t* __restrict__ tile_first, int n_sub,
      const double* __restrict__ tables, const double* __restrict__ u, const double* __restrict__ du,
      const double* __restrict__ Hs, int64_t S, int* __restrict__ flag, double* __restrict__ part) {
  __shared__ SubDev sd_s;
  __shared__ int tile0_s;
  __shared__ double red[TILE_PTS / 32][6];
  if (threadIdx.x == 0) {
    const int s = find_sub(tile_first, n_sub, blockIdx.x);
    sd_s = subs[s];
    tile0_s = tile_first[s];
  }
  __syncthreads();
  const SubDev& sd = sd_s;
  const int local = (blockIdx.x - tile0_s) * TILE_PTS + threadIdx.x;
  double acc[6] = {0, 0, 0, 0, 0, 0};
  if (local < sd.P) {
    if (sd.kind != 1) con_point<true>(sd, tables, local, u, du, Hs, S, flag, acc);
    else con_point<false>(sd, tables, local, u, du, Hs, S, flag, acc);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
    for (int q = 0; q < 3; ++q) acc[q] += __shfl_xor_sync(0xffffffffu, acc[q], o);
#pragma unroll
    for (int q = 3; q < 6; ++q) acc[q] = nanmax(acc[q], __shfl_xor_sync(0xffffffffu, acc[q], o));
  }
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (lane == 0)
#pragma unroll
    for (int q = 0; q < 6; ++q) red[warp][q] = acc[q];
  __syncthreads();
  if (threadIdx.x < 6) {
    const int q = threadIdx.x;
    double v = red[0][q];
    for (int w = 1; w < TILE_PTS / 32; ++w) v = (q < 3) ? v + red[w][q] : nanmax(v, red[w][q]);
    part[(int64_t)blockIdx.x * 6 + q] = v;
  }
}

// one warp per subdomain: per_sub[s][6] from its tiles, in tile order
__global__ void __launch_bounds__(32)
k_con_reduce(const int32_t* __restrict__ tile_first, const double* __restrict__ part, double* __restrict__ per_sub) {
  const int s = blockIdx.x, lane = threadIdx.x;
  const int t0 = tile_first[s], t1 = tile_first[s + 1];
  double acc[6] = {0, 0, 0, 0, 0, 0};
  for (int t = t0 + lane; t < t1; t += 32) {
#pragma unroll
    for (int q = 0; q < 3; ++q) acc[q] += part[(int64_t)t * 6 + q];
#pragma unroll
    for (int q = 3; q < 6; ++q) acc[q] = nanmax(acc[q], part[(int64_t)t * 6 + q]);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
    for (int q = 0; q < 3; ++q) acc[q] += __shfl_xor_sync(0xffffffffu, acc[q], o);
#pragma unroll
    for (int q = 3; q < 6; ++q) acc[q] = nanmax(acc[q], __shfl_xor_sync(0xffffffffu, acc[q], o));
  }
  if (lane == 0)
#pragma unroll
    for (int q = 0; q < 6; ++q) per_sub[(int64_t)s * 6 + q] = acc[q];
}

}  // namespace ghd
