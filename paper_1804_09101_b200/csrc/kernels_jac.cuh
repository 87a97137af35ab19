// kernels_jac.cuh — SpatialCoordJac (NEXT-4 of DESIGN.md; §3.3, Eqs. 9-11): "a coordinate change of a tensor's
// spatial indices only, by contracting every possible combination of said spatial indices with the Jacobian":
//   T'_ij = J_i^k J_j^l T_kl (9),  T'_0j = J_j^l T_0l (10),  T'_i0 = J_i^k T_k0 (11),  T'_00 = T_00 (null-op),
// i.e. T' = Lambda x ... x Lambda T with Lambda = diag(1, J).  The four structures the paper's port handles:
// T_a [4], T_aa [10 packed], T_ab [16], T_abb [40 = 4 x 10 packed], plus the evolved state (psi, Pi as T_aa; Phi_iab as the
// spatial-first-index rows of a T_abb).  One thread per grid point of the structure-of-arrays store: the nine Jacobian entries
// of the point sit in registers (the paper's own design note: "multiple successive contractions with the same
// Jacobian"), every component is read once and written once: (2 N_e + 9) x 8 bytes per point, HBM-bound (I = 1 ... 4.1 flop per
// transaction).  The paper's T_abb kernel spilled on the M2090; here the largest variant holds
// 30 + 9 values per thread and no variant spills.
#pragma once
#include "device_types.h"
#include "kernels_point.cuh"

namespace ghd {

// packed symmetric 4x4 (order of SI) in place:  M <- Lambda M Lambda^T
__device__ __forceinline__ void scj_sym(const double (&J)[9], double (&m)[10]) {
  double t[3];   // M'_0i = J_i^k M_0k
#pragma unroll
  for (int i = 0; i < 3; ++i) t[i] = J[3 * i] * m[SI(0, 1)] + J[3 * i + 1] * m[SI(0, 2)] + J[3 * i + 2] * m[SI(0, 3)];
  double A[3][3];   // A_il = J_i^k G_kl
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int l = 0; l < 3; ++l) A[i][l] = J[3 * i] * m[SI(1, l + 1)] + J[3 * i + 1] * m[SI(2, l + 1)] + J[3 * i + 2] * m[SI(3, l + 1)];
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    m[SI(0, i + 1)] = t[i];
#pragma unroll
    for (int j = i; j < 3; ++j) m[SI(i + 1, j + 1)] = A[i][0] * J[3 * j] + A[i][1] * J[3 * j + 1] + A[i][2] * J[3 * j + 2];
  }
}

__device__ __forceinline__ void scj_load_j(const double* __restrict__ jac, int64_t S, int64_t p, double (&J)[9]) {
#pragma unroll
  for (int e = 0; e < 9; ++e) J[e] = __ldg(jac + (int64_t)e * S + p);
}

// STRUCT: 0 T_a, 1 T_aa, 2 T_ab, 3 T_abb, 4 the 50-component state.  in / out: [N_e][S]; out may alias in (every value of the
// point is in registers before its first store; hence no __restrict__ on the two).
// Grid: the point tiles of the domain (TILE_PTS points, never straddling subdomains), so padding entries are neither read nor
// written.
template <int STRUCT>
__global__ void __launch_bounds__(TILE_PTS)
k_scj(const SubDev* __restrict__ subs, const int32_t* __restrict__ tile_first, int n_sub, const double* __restrict__ jac,
      const double* in, double* out, int64_t S) {
  const int sub = find_sub(tile_first, n_sub, blockIdx.x);
  const int local = (blockIdx.x - __ldg(tile_first + sub)) * TILE_PTS + threadIdx.x;
  if (local >= subs[sub].P) return;
  const int64_t p = subs[sub].off + local;
  double J[9];
  scj_load_j(jac, S, p, J);
  if (STRUCT == 0) {
    double v[4];
#pragma unroll
    for (int a = 0; a < 4; ++a) v[a] = in[(int64_t)a * S + p];
    out[p] = v[0];
#pragma unroll
    for (int i = 0; i < 3; ++i) out[(int64_t)(i + 1) * S + p] = J[3 * i] * v[1] + J[3 * i + 1] * v[2] + J[3 * i + 2] * v[3];
  } else if (STRUCT == 1) {
    double m[10];
#pragma unroll
    for (int s = 0; s < 10; ++s) m[s] = in[(int64_t)s * S + p];
    scj_sym(J, m);
#pragma unroll
    for (int s = 0; s < 10; ++s) out[(int64_t)s * S + p] = m[s];
  } else if (STRUCT == 2) {
    double m[4][4], w[4][4];
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
      for (int b = 0; b < 4; ++b) m[a][b] = in[(int64_t)(4 * a + b) * S + p];
    // first index, then second (Eq. 9 as two successive contractions)
#pragma unroll
    for (int b = 0; b < 4; ++b) {
      w[0][b] = m[0][b];
#pragma unroll
      for (int i = 0; i < 3; ++i) w[i + 1][b] = J[3 * i] * m[1][b] + J[3 * i + 1] * m[2][b] + J[3 * i + 2] * m[3][b];
    }
#pragma unroll
    for (int a = 0; a < 4; ++a) {
      out[(int64_t)(4 * a) * S + p] = w[a][0];
#pragma unroll
      for (int j = 0; j < 3; ++j) out[(int64_t)(4 * a + j + 1) * S + p] = J[3 * j] * w[a][1] + J[3 * j + 1] * w[a][2] + J[3 * j + 2] * w[a][3];
    }
  } else {
    // T_abb (rows 0..3) or the state (psi, Pi; Phi rows 1..3 only): the symmetric pair first, then the leading index
    if (STRUCT == 4) {
#pragma unroll
      for (int f = 0; f < 2; ++f) {
        double m[10];
#pragma unroll
        for (int s = 0; s < 10; ++s) m[s] = in[(int64_t)(10 * f + s) * S + p];
        scj_sym(J, m);
#pragma unroll
        for (int s = 0; s < 10; ++s) out[(int64_t)(10 * f + s) * S + p] = m[s];
      }
    }
    const int base = STRUCT == 4 ? 20 : 10;      // first spatial row of the leading index
    if (STRUCT == 3) {
      double m[10];
#pragma unroll
      for (int s = 0; s < 10; ++s) m[s] = in[(int64_t)s * S + p];
      scj_sym(J, m);
#pragma unroll
      for (int s = 0; s < 10; ++s) out[(int64_t)s * S + p] = m[s];
    }
    double x[3][10];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
#pragma unroll
      for (int s = 0; s < 10; ++s) x[k][s] = in[(int64_t)(base + 10 * k + s) * S + p];
      scj_sym(J, x[k]);
    }
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
      for (int s = 0; s < 10; ++s)
        out[(int64_t)(base + 10 * i + s) * S + p] = J[3 * i] * x[0][s] + J[3 * i + 1] * x[1][s] + J[3 * i + 2] * x[2][s];
  }
}

// ---------------------------------------------------------------------------------------------------------
// FP64 peak probe (profiling helper, gh_fp64_peak): register-resident kernels, MODE 0 = DFMA chains (64 independent
// accumulators per lane group), MODE 1 = DMMA mma.sync.m8n8k4 (8 independent accumulator pairs per warp).  128 flop per lane
// and iteration in both modes.  The derivative kernels report their roofline fraction against what this measures in the
// same run (bench.py), not against a nominal figure.
// ---------------------------------------------------------------------------------------------------------
template <int MODE>
__global__ void __launch_bounds__(256) k_fp64_peak(double* out, int iters, double x) {
  double f[16], c[8][2];
  const double a = x + threadIdx.x * 1e-9, b = 1.0 - x;
#pragma unroll
  for (int i = 0; i < 16; ++i) f[i] = i * x;
#pragma unroll
  for (int i = 0; i < 8; ++i) c[i][0] = c[i][1] = i * x;
  for (int it = 0; it < iters; ++it) {
    if (MODE == 0) {
#pragma unroll
      for (int r = 0; r < 4; ++r)
#pragma unroll
        for (int i = 0; i < 16; ++i) f[i] = fma(f[i], a, b);
    } else {
#pragma unroll
      for (int i = 0; i < 8; ++i)
        asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(c[i][0]), "+d"(c[i][1]) : "d"(a), "d"(b));
    }
  }
  double s = 0;
#pragma unroll
  for (int i = 0; i < 16; ++i) s += f[i];
#pragma unroll
  for (int i = 0; i < 8; ++i) s += c[i][0] + c[i][1];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

}  // namespace ghd
