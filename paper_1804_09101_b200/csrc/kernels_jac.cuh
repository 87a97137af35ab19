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
// Dual frame (NEXT-4; fields at fixed grid coordinates xbar, equations in inertial coordinates x(xbar, t) with the
// same time coordinate).  With Jm_i^k = d xbar^k / d x^i and the grid velocity v^i = d x^i / d t at fixed xbar:
//   d_i u = Jm_i^k dbar_k u   (DiffJac, Eq. 8),     d_t u |_xbar = F[u, d_i u] + v^i d_i u.
// Two passes around the unchanged fused RHS kernel, launched only while a map is set (the single-frame hot path pays nothing):
// K_map_pre rewrites the logical derivative scratch so that K_rhs / K_con, which apply the shell's spherical Jacobian A themselves,
// see inertial-frame derivatives: blocks du <- Jm du; shells du <- (A^-1 Jm A) du.  K_map_post adds coef * v^i d_i u to the output
// (coef = 1 for d_t u, b dt inside an RK stage, whose update is linear in d_t u) except on FROZEN faces, which hold their grid-frame
// value.  Both HBM-bound: 2 x 150 and 150 + 2 x 50 doubles per point.
// ---------------------------------------------------------------------------------------------------------
__device__ __forceinline__ bool point_frozen(const SubDev& sd, int local) {
  const int i2 = local % sd.n2, t = local / sd.n2, i1 = t % sd.n1, i0 = t / sd.n1;
  bool fz = (i0 == 0 && sd.face[0] == 1) || (i0 == sd.n0 - 1 && sd.face[1] == 1);
  if (sd.kind != 0) fz = fz || (i1 == 0 && sd.face[2] == 1) || (i1 == sd.n1 - 1 && sd.face[3] == 1);
  if (sd.kind == 1) fz = fz || (i2 == 0 && sd.face[4] == 1) || (i2 == sd.n2 - 1 && sd.face[5] == 1);
  return fz;
}

__global__ void __launch_bounds__(TILE_PTS)
k_map_pre(const SubDev* __restrict__ subs, const int32_t* __restrict__ tile_first, int n_sub, const double* __restrict__ tables,
          const double* __restrict__ mapJ, double* __restrict__ du, int64_t S, int ncomp) {
  const int sub = find_sub(tile_first, n_sub, blockIdx.x);
  const SubDev sd = subs[sub];
  const int local = (blockIdx.x - __ldg(tile_first + sub)) * TILE_PTS + threadIdx.x;
  if (local >= sd.P) return;
  const int64_t p = sd.off + local;
  double M[9];
  scj_load_j(mapJ, S, p, M);
  if (sd.kind != 1) {      // M <- A^-1 Jm A with A the logical -> Cartesian Jacobian of Eq. 8
    const ShellJac J = shell_jac(sd, tables, local);
    const double A[9] = {J.xr, J.xt, J.xp, J.yr, J.yt, J.yp, J.zr, J.zt, 0.0};
    double Ai[9];
    if (sd.kind == 0) {
      // A^-1 from the closed form: d_r = r^ . grad, d_theta = r theta^ . grad, d_phi = r sin(theta) phi^ . grad
      const double st = sqrt(J.xr * J.xr + J.yr * J.yr), ct = J.zr, r = -st / J.zt;
      const double cp = J.xr / st, sp = J.yr / st;
      Ai[0] = st * cp; Ai[1] = st * sp; Ai[2] = ct; Ai[3] = r * ct * cp; Ai[4] = r * ct * sp; Ai[5] = -r * st;
      Ai[6] = -r * st * sp; Ai[7] = r * st * cp; Ai[8] = 0.0;
    } else {
      // cylindrical shell: d_rho = rho^ . grad, d_z = z^ . grad, d_phi = rho phi^ . grad;  (cp, sp) = (J.xr, J.yr), 1 / rho from
      // the two phi entries (sp^2 + cp^2 = 1)
      const double cp = J.xr, sp = J.yr, rho = 1.0 / (cp * J.yp - sp * J.xp);
      Ai[0] = cp; Ai[1] = sp; Ai[2] = 0.0; Ai[3] = 0.0; Ai[4] = 0.0; Ai[5] = 1.0; Ai[6] = -rho * sp; Ai[7] = rho * cp; Ai[8] = 0.0;
    }
    double T[9];
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
      for (int k = 0; k < 3; ++k) T[3 * i + k] = M[3 * i] * A[k] + M[3 * i + 1] * A[3 + k] + M[3 * i + 2] * A[6 + k];
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
      for (int k = 0; k < 3; ++k) M[3 * i + k] = Ai[3 * i] * T[k] + Ai[3 * i + 1] * T[3 + k] + Ai[3 * i + 2] * T[6 + k];
  }
  const int64_t DS = (int64_t)ncomp * S;
  for (int c = 0; c < ncomp; ++c) {
    double* q = du + (int64_t)c * S + p;
    const double d0 = q[0], d1 = q[DS], d2 = q[2 * DS];
    q[0] = M[0] * d0 + M[1] * d1 + M[2] * d2;
    q[DS] = M[3] * d0 + M[4] * d1 + M[5] * d2;
    q[2 * DS] = M[6] * d0 + M[7] * d1 + M[8] * d2;
  }
}

__global__ void __launch_bounds__(TILE_PTS)
k_map_post(const SubDev* __restrict__ subs, const int32_t* __restrict__ tile_first, int n_sub, const double* __restrict__ tables,
           const double* __restrict__ mapv, const double* __restrict__ du, double* __restrict__ out, int64_t S, double coef) {
  const int sub = find_sub(tile_first, n_sub, blockIdx.x);
  const SubDev sd = subs[sub];
  const int local = (blockIdx.x - __ldg(tile_first + sub)) * TILE_PTS + threadIdx.x;
  if (local >= sd.P || point_frozen(sd, local)) return;
  const int64_t p = sd.off + local;
  double w0 = coef * __ldg(mapv + p), w1 = coef * __ldg(mapv + S + p), w2 = coef * __ldg(mapv + 2 * S + p);
  if (sd.kind != 1) {      // v . (A d_logical): fold A into the weights
    const ShellJac J = shell_jac(sd, tables, local);
    const double a0 = w0 * J.xr + w1 * J.yr + w2 * J.zr, a1 = w0 * J.xt + w1 * J.yt + w2 * J.zt, a2 = w0 * J.xp + w1 * J.yp;
    w0 = a0; w1 = a1; w2 = a2;
  }
  const int64_t DS = (int64_t)NCOMP * S;
  for (int c = 0; c < NCOMP; ++c) {
    const double* q = du + (int64_t)c * S + p;
    out[(int64_t)c * S + p] += w0 * q[0] + w1 * q[DS] + w2 * q[2 * DS];
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
