// kernels_deriv.cuh — spectral-derivative kernels (steps A2, A3 of DESIGN.md) and the stand-alone Jacobian (A4).
//
// A2: Chebyshev-line derivative, Eq. 22: du/dxi_d = (2/Delta_d) sum_i D[a,i] u[..i..].
// A3: shell angular derivatives, Eq. 24, restructured axis by axis:
//     real DFT in phi -> per-m Legendre composites along theta -> synthesis in phi.
#pragma once
#include "device_types.h"

namespace ghd {

// ---------------------------------------------------------------------------------------------------------
// K_cheb.  grid = (n_items, ncomp), TPB threads.  out[a, col] = sum_i D[a][i] u[i, col] as a GEMM on the FP64 tensor
// cores (mma.sync.m8n8k4, DMMA: 37.1 TFLOP/s measured against 33.9 for DFMA, profiles/r01_fp64_peak.md), M = a,
// K = i, N = col.  One warp owns 8*NTW columns of one component and ALL of M and K, so every input element is
// loaded exactly once, straight from global memory into its B-fragment register (lane (g, tl) of k-step ks holds
// u[i = 4 ks + tl][col = 8 n + g]: per request 4 rows x 64 B for the strided axes, 8 lines x 32 B for the
// unit-stride axis - whole 32-byte sectors either way), and every output leaves from its accumulator fragment
// (row a = 8 mt + g, columns 8 n + 2 tl, +1).  No shared-memory staging of the data and no transposes; shared memory
// only holds the differentiation matrix in A-fragment order (one conflict-free LDS.64 per fragment).  All K-steps of
// a warp tile are loaded before the first DMMA, which keeps KS*NTW*256 B per warp in flight.
// MTM / KSM: compile-time bounds on the m-tiles (N <= 8 MTM) and k-steps (N <= 4 KSM) of the class.
// ---------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
  asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
      : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

template <int TPB, int MTM, int KSM, int NTW>
__global__ void __launch_bounds__(TPB)
k_cheb(const ChebItem* __restrict__ items, const double* __restrict__ tables, const double* __restrict__ in,
       double* __restrict__ out, int64_t S, int ncomp) {
  extern __shared__ __align__(16) double sm[];   // D in fragment order [mt][ks][32]
  const ChebItem it = items[blockIdx.x];
  const int comp = blockIdx.y, tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int g = lane >> 2, tl = lane & 3;
  const double* __restrict__ src = in + (int64_t)comp * S + it.base;
  double* __restrict__ dst = out + ((int64_t)it.axis * ncomp + comp) * S + it.base;
  const int N = it.N, MTn = (N + 7) >> 3, KS = (N + 3) >> 2, ncols = it.ncols;
  const int64_t si = it.stride_i;

  for (int e = tid; e < MTn * KS * 32; e += TPB) sm[e] = __ldg(tables + it.dmat + e);

  // B fragments of the whole warp tile (independent of shared memory: issued before the barrier)
  const int wc0 = warp * (8 * NTW);
  int64_t caddr[NTW];
  bool cok[NTW];
#pragma unroll
  for (int n = 0; n < NTW; ++n) {
    const int c = wc0 + n * 8 + g;
    cok[n] = c < ncols;
    const int col = it.col0 + (cok[n] ? c : 0);
    const int q = col / it.col_inner;
    caddr[n] = (int64_t)q * it.outer_stride + (col - q * it.col_inner);
  }
  double b[KSM][NTW];
#pragma unroll
  for (int ks = 0; ks < KSM; ++ks)
    if (ks < KS) {
      const int i = ks * 4 + tl;
#pragma unroll
      for (int n = 0; n < NTW; ++n) b[ks][n] = (cok[n] && i < N) ? src[caddr[n] + (int64_t)i * si] : 0.0;
    }
  __syncthreads();
  if (wc0 >= ncols) return;

  double acc[MTM][NTW][2];
#pragma unroll
  for (int mt = 0; mt < MTM; ++mt)
#pragma unroll
    for (int n = 0; n < NTW; ++n) acc[mt][n][0] = acc[mt][n][1] = 0.0;
#pragma unroll
  for (int ks = 0; ks < KSM; ++ks)
    if (ks < KS) {
#pragma unroll
      for (int mt = 0; mt < MTM; ++mt)
        if (mt < MTn) {
          const double a = sm[(mt * KS + ks) * 32 + lane];
#pragma unroll
          for (int n = 0; n < NTW; ++n) dmma884(acc[mt][n][0], acc[mt][n][1], a, b[ks][n]);
        }
    }

  // C fragments: row a = 8 mt + g, columns 8 n + 2 tl and + 1; their addresses come from the lanes that loaded them
  const bool pair = (si != 1) && ((it.col_inner & 1) == 0);
#pragma unroll
  for (int n = 0; n < NTW; ++n) {
    const int64_t c0a = __shfl_sync(0xffffffffu, caddr[n], (2 * tl) * 4);
    const int64_t c1a = __shfl_sync(0xffffffffu, caddr[n], (2 * tl + 1) * 4);
    const int c = wc0 + n * 8 + 2 * tl;
    const bool ok0 = c < ncols, ok1 = c + 1 < ncols;
#pragma unroll
    for (int mt = 0; mt < MTM; ++mt) {
      const int a = mt * 8 + g;
      if (mt < MTn && a < N) {
        if (pair && ok1) {
          *reinterpret_cast<double2*>(dst + c0a + (int64_t)a * si) = make_double2(acc[mt][n][0], acc[mt][n][1]);
        } else {
          if (ok0) dst[c0a + (int64_t)a * si] = acc[mt][n][0];
          if (ok1) dst[c1a + (int64_t)a * si] = acc[mt][n][1];
        }
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------------------
// K_ang.  grid = (n_items, ncomp), TPB = 256 (8 warps).  One CTA: `nb` (theta,phi) planes of one component of
// one shell, kept in shared memory through three stages, each a small GEMM executed by warps with the FP64
// tensor-core instruction mma.sync.m8n8k4 (DMMA: measured 37.1 TFLOP/s on B200 against 33.8 for register-
// resident DFMA, at 1/8 of the issue slots; profiles/fp64_peak_r01.md):
//   S1  C[r][q]       = sum_k  U[r][k] Fa[q][k]            rows r = (plane b, theta j); real DFT, Nyquist dropped
//   S2  A[b][j'][q]   = sum_j  Th_m[j'][j] C[b][j][q]      m = m(q);  in place over C
//       B'[b][j'][q~] = +-sum_j (m Pr_m)[j'][j] C[b][j][q]  q~ = the cos<->sin partner of q:  d/dphi in coefficient space
//   S3  d_theta u[r][k] = sum_q A[r][q] Fs[k][q],   d_phi u[r][k] = sum_q B'[r][q] Fs[k][q]
// Shared memory: X (U, later B'), Y (C, later A), F (Fa, later Fs).  Row (b, j) of X / Y starts at b*ps + j*pitch
// doubles; pitch = 4 mod 8 and ps = 1 mod 16 make every fragment load conflict-free.
// The per-m matrices [Th_m ; m Pr_m] are read from global memory (L2) in fragment order: one coalesced 256-byte
// load per 8x4 fragment, prefetched one k-step ahead.
// ---------------------------------------------------------------------------------------------------------
__host__ __device__ inline int ang_pitch(int L) {   // row pitch (doubles): >= n_phi rounded to 4, and = 4 mod 8
  int p = (2 * L + 2 + 3) / 4 * 4;
  return (p % 8 == 0) ? p + 4 : p;
}
__host__ __device__ inline int ang_plane_stride(int L) {   // plane stride (doubles): = 1 mod 16
  return ((L + 1) * ang_pitch(L) + 15) / 16 * 16 + 1;
}

constexpr int ANG_NTC = 6;   // n-tiles per warp unit in S1 / S3

template <int TPB>
__global__ void __launch_bounds__(TPB)
k_ang(const AngItem* __restrict__ items, const double* __restrict__ tables, const double* __restrict__ in,
      double* __restrict__ out, int64_t S, int ncomp) {
  extern __shared__ __align__(16) double sm[];
  constexpr int NW = TPB / 32;
  const AngItem it = items[blockIdx.x];
  const int comp = blockIdx.y, tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int g = lane >> 2, tl = lane & 3;
  const int L = it.L, nt = L + 1, np = 2 * L + 2, nq = 2 * L + 1, plane = nt * np;
  const int nb = it.nplanes, R = nb * nt;
  const int pitch = ang_pitch(L), ps = ang_plane_stride(L);
  const int NP8 = (np + 7) & ~7, NQ8 = (nq + 7) & ~7;
  const int64_t goff = it.off + (int64_t)it.plane0 * plane;
  const double* __restrict__ src = in + (int64_t)comp * S + goff;
  double* __restrict__ dth = out + ((int64_t)1 * ncomp + comp) * S + goff;
  double* __restrict__ dph = out + ((int64_t)2 * ncomp + comp) * S + goff;

  double* X = sm;                          // [nb][ps]
  double* Y = X + (size_t)it.nb_alloc * ps;   // [nb][ps]
  double* F = Y + (size_t)it.nb_alloc * ps;   // [NP8][pitch]

  // ---- stage 0: U -> X (pad columns zero), Fa -> F (pad rows / columns zero) ----
  {
    const int hp = pitch >> 1;
    for (int e = tid; e < R * hp; e += TPB) {
      const int r = e / hp, k = (e - r * hp) * 2;
      const int b = r / nt, j = r - b * nt;
      double2 v = make_double2(0.0, 0.0);
      if (k < np) v = *reinterpret_cast<const double2*>(src + (size_t)r * np + k);
      double* d = X + (size_t)b * ps + j * pitch + k;
      d[0] = v.x; d[1] = v.y;
    }
    const double* __restrict__ Fa = tables + it.m_Fa;
    for (int e = tid; e < NQ8 * pitch; e += TPB) {
      const int q = e / pitch, k = e - q * pitch;
      F[e] = (q < nq && k < np) ? __ldg(Fa + (size_t)q * np + k) : 0.0;
    }
  }
  __syncthreads();

  const int MT1 = (R + 7) >> 3;
  // ---- S1: C = U Fa^T ----
  {
    const int KS = (np + 3) >> 2, NT = NQ8 >> 3;
    const int nch = (NT + ANG_NTC - 1) / ANG_NTC, per = (NT + nch - 1) / nch;
    for (int u = warp; u < MT1 * nch; u += NW) {
      const int mt = u / nch, ch = u - mt * nch;
      const int n0 = ch * per, nn = min(per, NT - n0);
      const int r = mt * 8 + g;
      const bool rok = r < R;
      const int rb = rok ? (r / nt) : 0, rj = rok ? (r - rb * nt) : 0;
      const double* ap = X + (size_t)rb * ps + rj * pitch + tl;
      const double* bp = F + (size_t)(n0 * 8 + g) * pitch + tl;
      double acc[ANG_NTC][2];
#pragma unroll
      for (int n = 0; n < ANG_NTC; ++n) acc[n][0] = acc[n][1] = 0.0;
      for (int ks = 0; ks < KS; ++ks) {
        const double a = rok ? ap[ks * 4] : 0.0;
#pragma unroll
        for (int n = 0; n < ANG_NTC; ++n)
          if (n < nn) dmma884(acc[n][0], acc[n][1], a, bp[(size_t)n * 8 * pitch + ks * 4]);
      }
      // C fragment: row g, columns 2 tl, 2 tl + 1 of each n-tile
      const int r2 = mt * 8 + g;
      if (r2 < R) {
        double* yp = Y + (size_t)rb * ps + rj * pitch;
#pragma unroll
        for (int n = 0; n < ANG_NTC; ++n)
          if (n < nn) {
            const int c = (n0 + n) * 8 + 2 * tl;
            if (c < pitch) yp[c] = acc[n][0];
            if (c + 1 < pitch) yp[c + 1] = acc[n][1];
          }
      }
    }
  }
  __syncthreads();

  // ---- Fs -> F (the buffer is free once S1 is done; S2 does not touch it) ----
  {
    const double* __restrict__ Fs = tables + it.m_Fs;
    for (int e = tid; e < NP8 * pitch; e += TPB) {
      const int k = e / pitch, q = e - k * pitch;
      F[e] = (k < np && q < nq) ? __ldg(Fs + (size_t)k * nq + q) : 0.0;
    }
  }
  // ---- S2: per m, [A ; B'] = [Th_m ; m Pr_m] C_m over the columns (t, b), t = cos / sin, b = plane ----
  {
    const int MTn = (nt + 7) >> 3, KS = (nt + 3) >> 2;        // <= 6, <= 12
    const double* __restrict__ TP = tables + it.m_TP;
    for (int m = warp; m <= L; m += NW) {
      const int ncols = (m == 0) ? nb : 2 * nb;               // <= 16
      const int NTn = (ncols + 7) >> 3;                       // 1 or 2
      // B fragment columns of this lane: n = 8 n_tile + g  ->  (t, b)
      int boff[2]; bool bok[2];
#pragma unroll
      for (int n = 0; n < 2; ++n) {
        const int c = n * 8 + g;
        bok[n] = c < ncols;
        const int t = bok[n] ? c / nb : 0, b = bok[n] ? c - t * nb : 0;
        boff[n] = b * ps + (t ? L + m : m);
      }
      // part 1 first (m Pr_m -> X), then part 0 (Th_m -> Y, in place over the C_m it has just been read from)
#pragma unroll 1
      for (int p = 1; p >= 0; --p) {
        double acc[6][2][2];
#pragma unroll
        for (int mt = 0; mt < 6; ++mt)
#pragma unroll
          for (int n = 0; n < 2; ++n) acc[mt][n][0] = acc[mt][n][1] = 0.0;
        const double* __restrict__ tp = TP + ((size_t)(m * 2 + p) * MTn * KS) * 32 + lane;   // [mt][ks][32]
        double an[6];
#pragma unroll
        for (int mt = 0; mt < 6; ++mt) an[mt] = (mt < MTn) ? __ldg(tp + (size_t)(mt * KS) * 32) : 0.0;
        for (int ks = 0; ks < KS; ++ks) {
          double a[6];
#pragma unroll
          for (int mt = 0; mt < 6; ++mt) a[mt] = an[mt];
          if (ks + 1 < KS) {
#pragma unroll
            for (int mt = 0; mt < 6; ++mt)
              if (mt < MTn) an[mt] = __ldg(tp + (size_t)(mt * KS + ks + 1) * 32);
          }
          const int j = ks * 4 + tl;
          double bf[2];
#pragma unroll
          for (int n = 0; n < 2; ++n) bf[n] = (bok[n] && j < nt) ? Y[boff[n] + j * pitch] : 0.0;
#pragma unroll
          for (int mt = 0; mt < 6; ++mt)
            if (mt < MTn) {
              dmma884(acc[mt][0][0], acc[mt][0][1], a[mt], bf[0]);
              if (NTn > 1) dmma884(acc[mt][1][0], acc[mt][1][1], a[mt], bf[1]);
            }
        }
        __syncwarp();   // every lane has read its C_m entries before any lane overwrites them
#pragma unroll
        for (int mt = 0; mt < 6; ++mt) {
          const int jo = mt * 8 + g;
          if (mt < MTn && jo < nt) {
#pragma unroll
            for (int n = 0; n < 2; ++n)
#pragma unroll
              for (int e = 0; e < 2; ++e) {
                const int c = n * 8 + 2 * tl + e;
                if (c < ncols) {
                  const int t = c / nb, b = c - t * nb;
                  const int row = b * ps + jo * pitch;
                  const double v = acc[mt][n][e];
                  if (p == 0) Y[row + (t ? L + m : m)] = v;          // A: same coefficient slot
                  else if (m == 0) X[row] = 0.0;                      // d/dphi of the m = 0 mode
                  else if (t == 0) X[row + L + m] = -v;               // sin slot <- -m (Pr C_cos)
                  else X[row + m] = v;                                // cos slot <- +m (Pr C_sin)
                }
              }
          }
        }
      }
    }
  }
  __syncthreads();

  // ---- S3: [d_theta u ; d_phi u] = [A ; B'] Fs^T, stored straight from the accumulator fragments ----
  {
    const int KS = (nq + 3) >> 2, NT = NP8 >> 3;
    const int nch = (NT + ANG_NTC - 1) / ANG_NTC, per = (NT + nch - 1) / nch;
    for (int u = warp; u < 2 * MT1 * nch; u += NW) {
      const int mt2 = u / nch, ch = u - mt2 * nch;
      const int part = mt2 >= MT1, mt = part ? mt2 - MT1 : mt2;
      const int n0 = ch * per, nn = min(per, NT - n0);
      const int r = mt * 8 + g;
      const bool rok = r < R;
      const int rb = rok ? (r / nt) : 0, rj = rok ? (r - rb * nt) : 0;
      const double* ap = (part ? X : Y) + (size_t)rb * ps + rj * pitch;
      const double* bp = F + (size_t)(n0 * 8 + g) * pitch + tl;
      double acc[ANG_NTC][2];
#pragma unroll
      for (int n = 0; n < ANG_NTC; ++n) acc[n][0] = acc[n][1] = 0.0;
      for (int ks = 0; ks < KS; ++ks) {
        const int q = ks * 4 + tl;
        const double a = (rok && q < nq) ? ap[q] : 0.0;
#pragma unroll
        for (int n = 0; n < ANG_NTC; ++n)
          if (n < nn) dmma884(acc[n][0], acc[n][1], a, bp[(size_t)n * 8 * pitch + ks * 4]);
      }
      if (rok) {
        double* gp = (part ? dph : dth) + (size_t)r * np;
#pragma unroll
        for (int n = 0; n < ANG_NTC; ++n)
          if (n < nn) {
            const int c = (n0 + n) * 8 + 2 * tl;
            if (c < np) *reinterpret_cast<double2*>(gp + c) = make_double2(acc[n][0], acc[n][1]);
          }
      }
    }
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
