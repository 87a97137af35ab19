// kernels_deriv.cuh — spectral-derivative kernels (steps A2, A3 of DESIGN.md) and the stand-alone Jacobian (A4).
//
// A2: Chebyshev-line derivative, Eq. 22: du/dxi_d = (2/Delta_d) sum_i D[a,i] u[..i..].
// A3: shell angular derivatives, Eq. 24, restructured axis by axis:
//     real DFT in phi -> per-m Legendre composites along theta -> synthesis in phi.
#pragma once
#include "device_types.h"

namespace ghd {

// ---------------------------------------------------------------------------------------------------------
// K_cheb.  grid = (n_items, ncomp).  One CTA: a tile of up to TPB*CPT lines ("columns") of one component,
// staged in shared memory T[i][col] (odd pitch: conflict-free both for the transposing fill of unit-stride
// lines and for the per-column reads).  Each thread owns CPT columns and produces 8 outputs per column per
// pass: per i one broadcast read of 8 matrix entries (4 x LDS.128) and CPT x LDS.64 feed 8*CPT DFMAs, which
// keeps the shared-memory pipe under the FP64 pipe.
// ---------------------------------------------------------------------------------------------------------
template <int TPB, int CPT>
__global__ void __launch_bounds__(TPB)
k_cheb(const ChebItem* __restrict__ items, const double* __restrict__ tables, const double* __restrict__ in,
       double* __restrict__ out, int64_t S, int ncomp) {
  extern __shared__ __align__(16) double sm[];
  const ChebItem it = items[blockIdx.x];
  const int comp = blockIdx.y, tid = threadIdx.x;
  const double* __restrict__ src = in + (int64_t)comp * S + it.base;
  double* __restrict__ dst = out + ((int64_t)it.axis * ncomp + comp) * S + it.base;
  const int N = it.N, ap = it.apitch, ncols = it.ncols;
  constexpr int PITCH = TPB * CPT + 1;
  double* Dt = sm;            // [N][ap]
  double* T = sm + N * ap;    // [N][PITCH]

  for (int e = tid; e < N * ap; e += TPB) Dt[e] = tables[it.dmat + e];
  if (it.stride_i == 1) {
    // unit-stride lines (last logical axis): memory runs along i, consecutive threads take consecutive i
    for (int e = tid; e < N * ncols; e += TPB) {
      int c = e / N, i = e - c * N;
      int col = it.col0 + c;
      int64_t ca = (int64_t)(col / it.col_inner) * it.outer_stride + (col % it.col_inner);
      T[i * PITCH + c] = src[ca + i];
    }
  } else {
    for (int e = tid; e < N * ncols; e += TPB) {
      int i = e / ncols, c = e - i * ncols;
      int col = it.col0 + c;
      int64_t ca = (int64_t)(col / it.col_inner) * it.outer_stride + (col % it.col_inner);
      T[i * PITCH + c] = src[(int64_t)i * it.stride_i + ca];
    }
  }
  __syncthreads();

  int64_t caddr[CPT];
  bool valid[CPT];
#pragma unroll
  for (int q = 0; q < CPT; ++q) {
    int c = tid + q * TPB;
    valid[q] = c < ncols;
    int col = it.col0 + (valid[q] ? c : 0);
    caddr[q] = (int64_t)(col / it.col_inner) * it.outer_stride + (col % it.col_inner);
  }

  for (int a0 = 0; a0 < N; a0 += 8) {
    double acc[CPT][8];
#pragma unroll
    for (int q = 0; q < CPT; ++q)
#pragma unroll
      for (int a = 0; a < 8; ++a) acc[q][a] = 0.0;
    const double* drow = Dt + a0;
    const double* trow = T + tid;
#pragma unroll 2
    for (int i = 0; i < N; ++i) {
      const double2 d0 = *reinterpret_cast<const double2*>(drow + 0);
      const double2 d1 = *reinterpret_cast<const double2*>(drow + 2);
      const double2 d2 = *reinterpret_cast<const double2*>(drow + 4);
      const double2 d3 = *reinterpret_cast<const double2*>(drow + 6);
      const double d[8] = {d0.x, d0.y, d1.x, d1.y, d2.x, d2.y, d3.x, d3.y};
#pragma unroll
      for (int q = 0; q < CPT; ++q) {
        const double t = trow[q * TPB];
#pragma unroll
        for (int a = 0; a < 8; ++a) acc[q][a] = fma(d[a], t, acc[q][a]);
      }
      drow += ap;
      trow += PITCH;
    }
#pragma unroll
    for (int q = 0; q < CPT; ++q) {
      if (!valid[q]) continue;
#pragma unroll
      for (int a = 0; a < 8; ++a)
        if (a0 + a < N) dst[(int64_t)(a0 + a) * it.stride_i + caddr[q]] = acc[q][a];
    }
  }
}

// ---------------------------------------------------------------------------------------------------------
// K_ang.  grid = (n_items, ncomp).  One CTA: `nplanes` (theta,phi) planes of one component of one shell.
//   S1  C[b][j][q]  = sum_k U[b][j][k] Fa[q][k]                        (real DFT, Nyquist dropped)
//   S2  A[b][j'][q] = sum_j Th[m(q)][j'][j] C[b][j][q],  B likewise with Pr[m(q)]
//   S3  d_theta u[b][j'][k] = sum_q A[b][j'][q] Fs[k][q],   d_phi u[b][j'][k] = sum_q B[b][j'][q] Fp[k][q]
// Shared memory: U (reused for A after S1), C, B.
// ---------------------------------------------------------------------------------------------------------
template <int TPB>
__global__ void __launch_bounds__(TPB)
k_ang(const AngItem* __restrict__ items, const double* __restrict__ tables, const double* __restrict__ in,
      double* __restrict__ out, int64_t S, int ncomp) {
  extern __shared__ __align__(16) double sm[];
  const AngItem it = items[blockIdx.x];
  const int comp = blockIdx.y, tid = threadIdx.x;
  const int L = it.L, nt = L + 1, np = 2 * L + 2, nq = 2 * L + 1, plane = nt * np;
  const int nb = it.nplanes;
  const int64_t goff = it.off + (int64_t)it.plane0 * plane;
  const double* __restrict__ src = in + (int64_t)comp * S + goff;
  double* __restrict__ dth = out + ((int64_t)1 * ncomp + comp) * S + goff;
  double* __restrict__ dph = out + ((int64_t)2 * ncomp + comp) * S + goff;
  const double* __restrict__ Fa = tables + it.m_Fa;
  const double* __restrict__ Fs = tables + it.m_Fs;
  const double* __restrict__ Fp = tables + it.m_Fp;
  const double* __restrict__ Th = tables + it.m_Th;
  const double* __restrict__ Pr = tables + it.m_Pr;

  const int rows = nb * nt;
  double* U = sm;                       // [rows][np]   (later A: [rows][nq])
  double* Cc = U + (size_t)rows * np;    // [rows][nq]
  double* Bb = Cc + (size_t)rows * nq;   // [rows][nq]

  for (int e = tid; e < rows * np; e += TPB) U[e] = src[e];
  __syncthreads();

  // S1: analysis in phi
  for (int e = tid; e < rows * nq; e += TPB) {
    int r = e / nq, q = e - r * nq;
    const double* u = U + (size_t)r * np;
    const double* f = Fa + (size_t)q * np;
    double s = 0.0;
    for (int k = 0; k < np; ++k) s = fma(u[k], __ldg(f + k), s);
    Cc[e] = s;
  }
  __syncthreads();

  // S2: per-m Legendre composites along theta
  double* Aa = U;
  for (int e = tid; e < rows * nq; e += TPB) {
    int r = e / nq, q = e - r * nq;
    int b = r / nt, jo = r - b * nt;
    int m = (q <= L) ? q : q - L;
    const double* th = Th + ((size_t)m * nt + jo) * nt;
    const double* pr = Pr + ((size_t)m * nt + jo) * nt;
    const double* c = Cc + (size_t)b * nt * nq + q;
    double sa = 0.0, sb = 0.0;
    for (int j = 0; j < nt; ++j) {
      double v = c[(size_t)j * nq];
      sa = fma(__ldg(th + j), v, sa);
      sb = fma(__ldg(pr + j), v, sb);
    }
    Aa[e] = sa;
    Bb[e] = sb;
  }
  __syncthreads();

  // S3: synthesis in phi
  for (int e = tid; e < rows * np; e += TPB) {
    int r = e / np, k = e - r * np;
    const double* a = Aa + (size_t)r * nq;
    const double* b = Bb + (size_t)r * nq;
    const double* fs = Fs + (size_t)k * nq;
    const double* fp = Fp + (size_t)k * nq;
    double s0 = 0.0, s1 = 0.0;
    for (int q = 0; q < nq; ++q) {
      s0 = fma(a[q], __ldg(fs + q), s0);
      s1 = fma(b[q], __ldg(fp + q), s1);
    }
    dth[e] = s0;
    dph[e] = s1;
  }
}

// binary search: largest s with first[s] <= tile  (first has n+1 entries, first[n] = total)
__device__ __forceinline__ int find_sub(const int32_t* __restrict__ first, int n, int tile) {
  int lo = 0, hi = n;
  while (hi - lo > 1) {
    int mid = (lo + hi) >> 1;
    if (__ldg(first + mid) <= tile) lo = mid; else hi = mid;
  }
  return lo;
}

// Spherical -> Cartesian Jacobian of Eq. 8 for a shell point (i, j, k):
//   d_x = st cp d_r + (ct cp / r) d_th - (sp / (r st)) d_ph
//   d_y = st sp d_r + (ct sp / r) d_th + (cp / (r st)) d_ph
//   d_z = ct    d_r - (st / r)    d_th
struct ShellJac { double xr, xt, xp, yr, yt, yp, zr, zt; };

__device__ __forceinline__ ShellJac shell_jac(const SubDev& sd, const double* __restrict__ tables, int local) {
  const int k = local % sd.n2, t = local / sd.n2, j = t % sd.n1, i = t / sd.n1;
  const double ri = __ldg(tables + sd.t_rinv + i);
  const double ct = __ldg(tables + sd.t_ct + j), st = __ldg(tables + sd.t_st + j);
  const double cp = __ldg(tables + sd.t_cp + k), sp = __ldg(tables + sd.t_sp + k);
  ShellJac J;
  J.xr = st * cp; J.xt = ct * cp * ri; J.xp = -sp * ri / st;
  J.yr = st * sp; J.yt = ct * sp * ri; J.yp = cp * ri / st;
  J.zr = ct;      J.zt = -st * ri;
  return J;
}

// K_jac: in-place logical -> Cartesian on shells for a gradient array g[3][ncomp][S] (debug / gauge-source path;
// inside gh_rhs the same transform is fused into K_rhs).
__global__ void __launch_bounds__(TILE_PTS)
k_jac(const SubDev* __restrict__ subs, const int32_t* __restrict__ tile_first, int n_sub,
      const double* __restrict__ tables, double* __restrict__ g, int64_t S, int ncomp) {
  const int s = find_sub(tile_first, n_sub, blockIdx.x);
  const SubDev sd = subs[s];
  if (sd.kind != 0) return;
  const int local = (blockIdx.x - tile_first[s]) * TILE_PTS + threadIdx.x;
  if (local >= sd.P) return;
  const ShellJac J = shell_jac(sd, tables, local);
  const int64_t p = sd.off + local;
  for (int c = 0; c < ncomp; ++c) {
    double* a = g + (int64_t)c * S + p;
    const int64_t st = (int64_t)ncomp * S;
    const double dr = a[0], dt = a[st], dp = a[2 * st];
    a[0] = J.xr * dr + J.xt * dt + J.xp * dp;
    a[st] = J.yr * dr + J.yt * dt + J.yp * dp;
    a[2 * st] = J.zr * dr + J.zt * dt;
  }
}

}  // namespace ghd
