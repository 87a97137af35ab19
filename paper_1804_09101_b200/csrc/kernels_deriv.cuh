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

// The derivative kernels run over `ncomp` components of an array with `total` components, skipping `skip_n` of them from
// `skip_lo` on (gh_constraint_norms needs no derivative of Pi): launch index c -> component c (< skip_lo) or c + skip_n.
struct CompMap {
  int total, skip_lo, skip_n;
  __device__ __forceinline__ int map(int c) const { return c < skip_lo ? c : c + skip_n; }
};

template <int TPB, int MTM, int KSM, int NTW>
__global__ void __launch_bounds__(TPB, (MTM * NTW >= 16) ? 3 : (MTM * NTW >= 12) ? 4 : (MTM * NTW >= 8) ? 5 : 7)
k_cheb(const ChebItem* __restrict__ items, const double* __restrict__ tables, const double* __restrict__ in,
       double* __restrict__ out, int64_t S, int ncomp, CompMap cm) {
  extern __shared__ __align__(16) double sm[];   // D in fragment order [mt][ks][32]
  const ChebItem it = items[blockIdx.x];
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int g = lane >> 2, tl = lane & 3;
  const int N = it.N, MTn = (N + 7) >> 3, KS = (N + 3) >> 2, ncols = it.ncols;
  const int si0 = (int)it.stride_i;   // offsets inside a subdomain fit 32 bits (P_s <= 2^30)

  for (int e = tid; e < MTn * KS * 32; e += TPB) sm[e] = __ldg(tables + it.dmat + e);

  // column addresses of this lane's B fragments (loads) and C fragments (stores)
  const int wc0 = warp * (8 * NTW);
  int caddr[NTW];
  bool cok[NTW];
#pragma unroll
  for (int n = 0; n < NTW; ++n) {
    const int c = wc0 + n * 8 + g;
    cok[n] = c < ncols;
    const int col = it.col0 + (cok[n] ? c : 0);
    const int q = col / it.col_inner;
    caddr[n] = q * (int)it.outer_stride + (col - q * it.col_inner);
  }
  const bool pair = (si0 != 1) && ((it.col_inner & 1) == 0);
  int c0a[NTW], c1a[NTW];
#pragma unroll
  for (int n = 0; n < NTW; ++n) {
    c0a[n] = __shfl_sync(0xffffffffu, caddr[n], (2 * tl) * 4);
    c1a[n] = __shfl_sync(0xffffffffu, caddr[n], (2 * tl + 1) * 4);
  }

  __syncthreads();
  if (wc0 >= ncols) return;

  // the CTA walks over components blockIdx.y, blockIdx.y + gridDim.y, ... (one launch and one matrix load for all of them)
#pragma unroll 1
  for (int cw = blockIdx.y; cw < ncomp; cw += gridDim.y) {
    const int comp = cm.map(cw);
    // B fragments of the whole warp tile.  (si is laundered so that the compiler recomputes the 2 x KS x NTW element
    // offsets per component instead of keeping them all live across the loop: that costs 40 registers and a CTA per SM)
    int si = si0;
    asm volatile("" : "+r"(si));
    double b[KSM][NTW];
    {
      const double* __restrict__ src = in + (int64_t)comp * S + it.base;
#pragma unroll
      for (int ks = 0; ks < KSM; ++ks)
        if (ks < KS) {
          const int i = ks * 4 + tl;
#pragma unroll
          for (int n = 0; n < NTW; ++n) b[ks][n] = (cok[n] && i < N) ? src[caddr[n] + i * si] : 0.0;
        }
    }
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
    // C fragments: row a = 8 mt + g, columns 8 n + 2 tl and + 1
    double* __restrict__ dst = out + ((int64_t)it.axis * cm.total + comp) * S + it.base;
#pragma unroll
    for (int n = 0; n < NTW; ++n) {
      const int c = wc0 + n * 8 + 2 * tl;
      const bool ok0 = c < ncols, ok1 = c + 1 < ncols;
#pragma unroll
      for (int mt = 0; mt < MTM; ++mt) {
        const int a = mt * 8 + g;
        if (mt < MTn && a < N) {
          if (pair && ok1) {
            *reinterpret_cast<double2*>(dst + c0a[n] + a * si) = make_double2(acc[mt][n][0], acc[mt][n][1]);
          } else {
            if (ok0) dst[c0a[n] + a * si] = acc[mt][n][0];
            if (ok1) dst[c1a[n] + a * si] = acc[mt][n][1];
          }
        }
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------------------
// K_ang.  grid = (n_items, ncomp).  One CTA: `nb` (theta,phi) planes of one component of one shell, kept in shared
// memory through three GEMM stages on the FP64 tensor cores (mma.sync.m8n8k4).  With h = L+1 = n_phi/2:
//   fold        E_k = U_k + U_{n_phi-k}, O_k = U_k - U_{n_phi-k} (k = 1..L), E_0 = U_0, E_h = U_h: cos(m phi) is even and
//               sin(m phi) odd about phi = pi, so the real DFT splits into two half-length ones (half the flop of S1,
//               S3).  The fold happens in the A-operand load of S1 (two LDS and one add per fragment; the raw row
//               carries a zero at column n_phi and the k = h row of Fa_c is halved, so no lane needs a predicate)
//   S1  Cc[r][m] = sum_{k=0..h} E[r][k] Fa_c[m][k]  (m = 0..L),   Cs[r][m] = sum_{k=1..L} O[r][k] Fa_s[m][k]  (m = 1..L)
//   S2  [A ; B'](m) = [Th_m ; m Pr_m] C_m   per m, columns (t = cos/sin, plane b); A in place over C, B' into the
//               cos<->sin partner slot with sign (d/dphi in coefficient space); folded about the equator (see S2 unit)
//   S3  e[r][k] = sum_m Ac[r][m] Fs_c[k][m],  o[r][k] = sum_m As[r][m] Fs_s[k][m]  (k = 0..h), same for B';
//               d u[r][k] = e + o,  d u[r][n_phi-k] = e - o, stored straight from the accumulators
// Every matrix operand is stored in DMMA fragment order, zero padded to whole tiles ([k_step][tile][32 lanes]: one
// conflict-free LDS.64 / coalesced 256-byte LDG per fragment, tile offsets are immediates), so the inner loops carry
// no bounds predicate.  Fa / Fs fragments live in shared memory; the per-m stacked matrices [Th_m ; m Pr_m] stream
// from L2 two k-steps ahead.  Planes: X (raw U, later B') and Y (C, later A), row (b, j) at b*ps + j*pitch
// doubles; coefficient rows hold cos m at column m and sin m at column kc + m - 1 (kc = 4 ceil(h/4)).
// pitch = 4 mod 8 and ps = 1 mod 16 keep the data-fragment loads conflict-free.  Rows beyond the tile range read a
// zeroed row.
// ---------------------------------------------------------------------------------------------------------
struct AngDims {
  int h, KSe1, NTc, KSo1, NTs, kc, KSe3, KSo3, NT3;
};
__host__ __device__ inline AngDims ang_dims(int L) {
  AngDims d;
  d.h = L + 1;
  d.KSe1 = (d.h + 1 + 3) / 4; d.NTc = (d.h + 7) / 8;      // S1 even: K = h+1 (k = 0..h),  N = h   (m = 0..L)
  d.KSo1 = (L + 3) / 4;       d.NTs = (L + 7) / 8;        // S1 odd:  K = L   (k = 1..L),  N = L   (m = 1..L)
  d.KSe3 = (d.h + 3) / 4; d.KSo3 = (L + 3) / 4;           // S3: K = h (m = 0..L) / L (m = 1..L)
  d.kc = 4 * d.KSe3;                                      // coefficient rows: cos m at m, sin m at kc + m - 1
  d.NT3 = (d.h + 1 + 7) / 8;                              //     N = h+1 (k = 0..h) for both
  return d;
}
__host__ __device__ inline int ang_pitch(int L) {   // row pitch (doubles), = 4 mod 8
  const AngDims d = ang_dims(L);
  const int a = d.kc + 4 * d.KSo3, b = 2 * L + 2 + 1;     // coefficient rows; raw rows need n_phi + 1 (a zero at column n_phi)
  int p = ((a > b ? a : b) + 3) / 4 * 4;
  return (p % 8 == 0) ? p + 4 : p;
}
__host__ __device__ inline int ang_plane_stride(int L) {   // plane stride (doubles), = 1 mod 16
  return ((L + 1) * ang_pitch(L) + 15) / 16 * 16 + 1;
}
__host__ __device__ inline size_t ang_fa_doubles(int L) { const AngDims d = ang_dims(L); return (size_t)(d.KSe1 * d.NTc + d.KSo1 * d.NTs) * 32; }
__host__ __device__ inline size_t ang_fs_doubles(int L) { const AngDims d = ang_dims(L); return (size_t)(d.KSe3 + d.KSo3) * d.NT3 * 32; }
__host__ __device__ inline size_t ang_f_doubles(int L) {
  const size_t fa = ang_fa_doubles(L), fs = ang_fs_doubles(L);
  return fa > fs ? fa : fs;
}
// shared memory (doubles) of K_ang for nb planes: X, Y, one zero row, F fragments, row-offset table (ints)
__host__ __device__ inline size_t ang_smem_doubles(int L, int nb) {
  const size_t rows = (size_t)nb * (L + 1);
  return 2 * (size_t)nb * ang_plane_stride(L) + ang_pitch(L) + 16 + ang_f_doubles(L) + ((rows + 8) * sizeof(int) + 7) / 8;
}

__device__ __forceinline__ void cp_async8(double* smem_dst, const double* gsrc) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async16(double* smem_dst, const double* gsrc) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// S1 unit: one m-tile (8 rows) x NTC n-tiles.  The A operand is folded on the fly from the raw row: element k is
// U[k] + sg U[n_phi - k]; ap / am: this lane's first element and its mirror; bp: F fragments of the first n-tile (+ lane)
template <int NTC>
__device__ __forceinline__ void ang_s1_unit(const double* __restrict__ ap, const double* __restrict__ am, double sg,
                                            const double* __restrict__ bp, int KS, int NT,
                                            double* __restrict__ yrow, int c0, int climit, bool rok) {
  double acc[NTC][2];
#pragma unroll
  for (int n = 0; n < NTC; ++n) acc[n][0] = acc[n][1] = 0.0;
  const int bstep = NT * 32;
#pragma unroll 2
  for (int ks = 0; ks < KS; ++ks) {
    const double a = fma(sg, am[0], ap[0]);
#pragma unroll
    for (int n = 0; n < NTC; ++n) dmma884(acc[n][0], acc[n][1], a, bp[n * 32]);
    ap += 4; am -= 4; bp += bstep;
  }
  if (rok) {
#pragma unroll
    for (int n = 0; n < NTC; ++n) {
      const int c = c0 + n * 8;
      if (c < climit) { yrow[c] = acc[n][0]; yrow[c + 1] = acc[n][1]; }     // climit: end of the cos / sin region (multiple of 4)
    }
  }
}

// S3 unit: one m-tile x NTC n-tiles (columns k = 0..h), both parts (theta from Y, phi from X), even and odd GEMMs;
// a0p / a1p: this lane's rows (+ tl) of Y / X at the cos region; the sin region starts kc doubles further.
// PARTS = 1 (spectral filter): only the Y part, stored to g0.
template <int NTC, int PARTS>
__device__ __forceinline__ void ang_s3_unit(const double* __restrict__ a0p, const double* __restrict__ a1p, int kc,
                                            const double* __restrict__ bpe, const double* __restrict__ bpo, int KSe,
                                            int KSo, int NT, double* __restrict__ g0, double* __restrict__ g1, int c0,
                                            int h, int np, bool rok) {
  double e0[NTC][2], e1[NTC][2], o0[NTC][2], o1[NTC][2];
#pragma unroll
  for (int n = 0; n < NTC; ++n) {
    e0[n][0] = e0[n][1] = e1[n][0] = e1[n][1] = 0.0;
    o0[n][0] = o0[n][1] = o1[n][0] = o1[n][1] = 0.0;
  }
  const int bstep = NT * 32;
  {
    const double* p0 = a0p; const double* p1 = a1p;
#pragma unroll 2
    for (int ks = 0; ks < KSe; ++ks) {
      const double a0 = p0[0], a1 = PARTS == 2 ? p1[0] : 0.0;
#pragma unroll
      for (int n = 0; n < NTC; ++n) {
        const double b = bpe[n * 32];
        dmma884(e0[n][0], e0[n][1], a0, b);
        if (PARTS == 2) dmma884(e1[n][0], e1[n][1], a1, b);
      }
      p0 += 4; p1 += 4; bpe += bstep;
    }
  }
  {
    const double* p0 = a0p + kc; const double* p1 = a1p + kc;
#pragma unroll 2
    for (int ks = 0; ks < KSo; ++ks) {
      const double a0 = p0[0], a1 = PARTS == 2 ? p1[0] : 0.0;
#pragma unroll
      for (int n = 0; n < NTC; ++n) {
        const double b = bpo[n * 32];
        dmma884(o0[n][0], o0[n][1], a0, b);
        if (PARTS == 2) dmma884(o1[n][0], o1[n][1], a1, b);
      }
      p0 += 4; p1 += 4; bpo += bstep;
    }
  }
  if (rok) {
#pragma unroll
    for (int n = 0; n < NTC; ++n) {
      const int k = c0 + n * 8;             // even; this lane holds columns k and k + 1
      if (k + 1 <= h) {
        *reinterpret_cast<double2*>(g0 + k) = make_double2(e0[n][0] + o0[n][0], e0[n][1] + o0[n][1]);
        if (PARTS == 2) *reinterpret_cast<double2*>(g1 + k) = make_double2(e1[n][0] + o1[n][0], e1[n][1] + o1[n][1]);
      } else if (k <= h) {
        g0[k] = e0[n][0] + o0[n][0];
        if (PARTS == 2) g1[k] = e1[n][0] + o1[n][0];
      }
      // mirror columns n_phi - k (k = 1..L)
      if (k >= 1 && k < h) { g0[np - k] = e0[n][0] - o0[n][0]; if (PARTS == 2) g1[np - k] = e1[n][0] - o1[n][0]; }
      if (k + 1 < h) { g0[np - k - 1] = e0[n][1] - o0[n][1]; if (PARTS == 2) g1[np - k - 1] = e1[n][1] - o1[n][1]; }
    }
  }
}

// S2 unit: mode m, n-tile `ntile` of its columns.  The Gauss-Legendre nodes are symmetric about the equator
// (theta_{nt-1-j} = pi - theta_j), the projector Pr_m commutes with that reflection and d/dtheta anticommutes, so with
// p_j = C_j + C_jbar, q_j = C_j - C_jbar (j < hh = ceil(nt/2), jbar = nt-1-j) folded on the fly in the B-operand load,
//   [alpha ; gamma] = ME_m p,  [beta ; delta] = MO_m q      (two stacked (2 hh x hh) matrices instead of one (2 nt x nt))
//   A_j = alpha + beta, A_jbar = beta - alpha;   B_j = gamma + delta, B_jbar = gamma - delta:      half the flop of S2.
// MTH m-tiles of each stacked matrix; fragments [ks][which][mt][32] stream from L2 one k-step ahead.
// FILTER: the stacked matrix is only the filtered projector G_m (hh rows, commutes with the reflection like Pr_m): the
// filtered coefficients gamma +- delta replace C in Y; X is not written.
// np_ / nq_: the fragments of this unit's first k-step, already loaded; on return they hold those of the NEXT unit's first
// k-step (tnext, or untouched if tnext == nullptr), fetched during this unit's last k-step so that the L2 latency hides
// behind its DMMAs and epilogue: the units are only 3-5 k-steps long.
template <int MTH, bool FILTER>
__device__ __forceinline__ void ang_s2_unit(const double* __restrict__ tp /* T_m fragments + lane */,
                                            const double* __restrict__ tnext, double (&np_)[MTH], double (&nq_)[MTH], int KSh,
                                            double* __restrict__ X, double* __restrict__ Y, int m, int ntile, int nb,
                                            int L, int kc, int pitch, int ps, int g, int tl) {
  const int nt = L + 1, hh = (nt + 1) >> 1, ncols = (m == 0) ? nb : 2 * nb;
  const int slot_c = m, slot_s = kc + m - 1;      // coefficient columns of cos m / sin m
  // B fragment column of this lane
  const int cb = ntile * 8 + g;
  const bool bok = cb < ncols;
  const int tb = (bok && cb >= nb) ? 1 : 0, bb = bok ? cb - tb * nb : 0;
  const double* __restrict__ ycol = Y + bb * ps + (tb ? slot_s : slot_c);
  double ap_[MTH][2], aq_[MTH][2];
#pragma unroll
  for (int mt = 0; mt < MTH; ++mt) ap_[mt][0] = ap_[mt][1] = aq_[mt][0] = aq_[mt][1] = 0.0;
#pragma unroll 1
  for (int ks = 0; ks < KSh; ++ks) {
    double fp[MTH], fq[MTH];
#pragma unroll
    for (int mt = 0; mt < MTH; ++mt) { fp[mt] = np_[mt]; fq[mt] = nq_[mt]; }
    tp += 2 * MTH * 32;
    const double* __restrict__ tn = (ks + 1 < KSh) ? tp : tnext;
    if (tn) {
#pragma unroll
      for (int mt = 0; mt < MTH; ++mt) { np_[mt] = __ldg(tn + mt * 32); nq_[mt] = __ldg(tn + (MTH + mt) * 32); }
    }
    const int j = ks * 4 + tl;
    const bool jok = bok && j < hh;
    const int jc = jok ? j : 0;
    const double y0 = ycol[jc * pitch], y1 = ycol[(nt - 1 - jc) * pitch];
    const double bp = jok ? y0 + y1 : 0.0, bq = jok ? y0 - y1 : 0.0;
#pragma unroll
    for (int mt = 0; mt < MTH; ++mt) {
      dmma884(ap_[mt][0], ap_[mt][1], fp[mt], bp);
      dmma884(aq_[mt][0], aq_[mt][1], fq[mt], bq);
    }
  }
  __syncwarp();   // every lane has read its C_m entries before any lane overwrites them
  // C fragments: stacked row 8 mt + g (rows [0, hh): theta part, [hh, 2 hh): phi part), columns 8 ntile + 2 tl + e.
  // A -> Y at the same slot; B' -> X at the partner slot with sign (cos input -> sin slot, negated; sin -> cos); m = 0 -> 0
  double* ydst[2]; double* xdst[2]; double sgn[2]; bool cok[2];
#pragma unroll
  for (int e = 0; e < 2; ++e) {
    const int c = ntile * 8 + 2 * tl + e;
    cok[e] = c < ncols;
    const int t = (cok[e] && c >= nb) ? 1 : 0, bq = cok[e] ? c - t * nb : 0;
    ydst[e] = Y + bq * ps + (t ? slot_s : slot_c);
    xdst[e] = X + bq * ps + ((t || m == 0) ? slot_c : slot_s);
    sgn[e] = (m == 0) ? 0.0 : (t ? 1.0 : -1.0);
  }
#pragma unroll
  for (int mt = 0; mt < MTH; ++mt) {
    const int rr = mt * 8 + g;
    if (rr < hh) {
      const int jb = nt - 1 - rr;
#pragma unroll
      for (int e = 0; e < 2; ++e)
        if (cok[e]) {
          ydst[e][rr * pitch] = ap_[mt][e] + aq_[mt][e];
          if (jb != rr) ydst[e][jb * pitch] = FILTER ? ap_[mt][e] - aq_[mt][e] : aq_[mt][e] - ap_[mt][e];
        }
    } else if (!FILTER && rr < 2 * hh) {
      const int j = rr - hh, jb = nt - 1 - j;
#pragma unroll
      for (int e = 0; e < 2; ++e)
        if (cok[e]) {
          xdst[e][j * pitch] = sgn[e] * (ap_[mt][e] + aq_[mt][e]);
          if (jb != j) xdst[e][jb * pitch] = sgn[e] * (ap_[mt][e] - aq_[mt][e]);
        }
    }
  }
}

// all S2 units of one warp: u = warp, warp + NW, ... over (m, n-tile)
template <int MTH, bool FILTER>
__device__ __forceinline__ void ang_s2_loop(const double* __restrict__ T /* + lane */, int KSh, double* __restrict__ X,
                                            double* __restrict__ Y, int nb, int L, int kc, int pitch, int ps, int g, int tl,
                                            int warp, int NW) {
  const int NTn = (2 * nb + 7) >> 3, nunits = (L + 1) * NTn;
  const size_t mstride = (size_t)KSh * 2 * MTH * 32;
  auto skip = [&](int u) { return u < NTn && u * 8 >= nb; };       // m = 0 has only the nb cos columns
  int u = warp;
  while (u < nunits && skip(u)) u += NW;
  if (u >= nunits) return;
  double np_[MTH], nq_[MTH];
  {
    const double* __restrict__ tp = T + (size_t)(u / NTn) * mstride;
#pragma unroll
    for (int mt = 0; mt < MTH; ++mt) { np_[mt] = __ldg(tp + mt * 32); nq_[mt] = __ldg(tp + (MTH + mt) * 32); }
  }
  while (u < nunits) {
    int un = u + NW;
    while (un < nunits && skip(un)) un += NW;
    const int m = u / NTn, ntile = u - m * NTn;
    const double* tnext = un < nunits ? T + (size_t)(un / NTn) * mstride : nullptr;
    ang_s2_unit<MTH, FILTER>(T + (size_t)m * mstride, tnext, np_, nq_, KSh, X, Y, m, ntile, nb, L, kc, pitch, ps, g, tl);
    u = un;
  }
}

#define GH_NTC_SWITCH(nn, CALL)                       \
  switch (nn) {                                        \
    case 1: CALL(1); break;                            \
    case 2: CALL(2); break;                            \
    case 3: CALL(3); break;                            \
    case 4: CALL(4); break;                            \
    default: CALL(5); break;                           \
  }
#define GH_NTC3_SWITCH(nn, CALL)                      \
  switch (nn) {                                        \
    case 1: CALL(1); break;                            \
    case 2: CALL(2); break;                            \
    default: CALL(3); break;                           \
  }

constexpr int ANG_NTC = 5;    // most n-tiles per warp unit in S1
constexpr int ANG_NTC3 = 3;   // most n-tiles per warp unit in S3 (four accumulator sets)

template <int TPB, bool FILTER>
__global__ void __launch_bounds__(TPB, TPB <= 256 ? 2 : 1)
k_ang(const AngItem* __restrict__ items, const double* __restrict__ tables, const double* in,
      double* out, int64_t S, CompMap cm) {
  extern __shared__ __align__(16) double sm[];
  constexpr int NW = TPB / 32;
  const AngItem it = items[blockIdx.x];
  const int comp = cm.map(blockIdx.y), ncomp = cm.total, tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int g = lane >> 2, tl = lane & 3;
  const int L = it.L, nt = L + 1, np = 2 * L + 2, plane = nt * np;
  const AngDims D = ang_dims(L);
  const int h = D.h, kc = D.kc;
  const int nb = it.nplanes, R = nb * nt;
  const int pitch = ang_pitch(L), ps = ang_plane_stride(L);
  const int64_t goff = it.off + (int64_t)it.plane0 * plane;
  const double* src = in + (int64_t)comp * S + goff;
  // derivative slots 1 (theta) and 2 (phi) of `out`; FILTER: the filtered planes, over the input when out == in (every plane
  // of this CTA is in shared memory before the first store)
  double* dth = FILTER ? out + (int64_t)comp * S + goff : out + ((int64_t)1 * ncomp + comp) * S + goff;
  double* dph = out + ((int64_t)2 * ncomp + comp) * S + goff;

  double* X = sm;                               // [nb][ps]
  double* Y = X + (size_t)it.nb_alloc * ps;     // [nb][ps]
  double* Z = Y + (size_t)it.nb_alloc * ps;     // zero row [pitch + 16]
  double* F = Z + pitch + 16;                   // Fa fragments (even | odd), later Fs fragments (even | odd)
  int* rowoff = reinterpret_cast<int*>(F + ang_f_doubles(L));   // [R rounded up to 8]: offset of row r in X / Y; pad rows -> Z
  const int zoff = (int)(Z - X);

  // ---- stage 0: raw U -> X and Fa fragments -> F by cp.async (all loads in flight at once); tables; padding ----
  {
    const int padc = pitch - np;
    int b = warp / nt, j = warp - b * nt;
    for (int r = warp; r < R; r += NW) {
      const double* __restrict__ urow = src + (size_t)r * np;
      double* xrow = X + (size_t)b * ps + j * pitch;
      for (int c = lane; c < np; c += 32) cp_async8(xrow + c, urow + c);
      if (lane < padc) xrow[np + lane] = 0.0;      // column n_phi = 0 (mirror of k = 0); the rest finite for S3
      j += NW;
      while (j >= nt) { j -= nt; ++b; }
    }
    const double* __restrict__ Fa = tables + it.m_Fa;
    const int nfa = (int)ang_fa_doubles(L);
    for (int e = tid * 2; e < nfa; e += TPB * 2) cp_async16(F + e, Fa + e);
    cp_async_commit();
    const int R8 = (R + 7) & ~7;
    for (int r = tid; r < R8; r += TPB) {
      const int b = r / nt, j = r - b * nt;
      rowoff[r] = (r < R) ? b * ps + j * pitch : zoff;
    }
    for (int e = tid; e < pitch + 16; e += TPB) Z[e] = 0.0;
    cp_async_wait<0>();
  }
  __syncthreads();

  const int MT1 = (R + 7) >> 3;
  // ---- S1: Cc = E Fa_c^T (columns 0..), Cs = O Fa_s^T (columns kc..) ----
  {
    const int nche = it.nch1e, pere = (D.NTc + nche - 1) / nche;
    const int ncho = it.nch1o, pero = (D.NTs + ncho - 1) / ncho;
    const int upm = nche + ncho;                       // units per m-tile
    const double* __restrict__ Fo = F + D.KSe1 * D.NTc * 32;
    for (int u = warp; u < MT1 * upm; u += NW) {
      const int mt = u / upm, ch = u - mt * upm;
      const int r = mt * 8 + g;
      const int ro = rowoff[r];
      if (ch < nche) {
        const int n0 = ch * pere, nn = min(pere, D.NTc - n0);
        const double* ap = X + ro + tl;                  // k = 4 ks + tl, mirror n_phi - k
        const double* am = X + ro + np - tl;
        const double* bp = F + n0 * 32 + lane;
        double* yrow = Y + ro;
        const int c0 = n0 * 8 + 2 * tl;
#define GH_CALL(K) ang_s1_unit<K>(ap, am, 1.0, bp, D.KSe1, D.NTc, yrow, c0, kc, r < R)
        GH_NTC_SWITCH(nn, GH_CALL)
#undef GH_CALL
      } else {
        const int n0 = (ch - nche) * pero, nn = min(pero, D.NTs - n0);
        const double* ap = X + ro + 1 + tl;              // k = 4 ks + tl + 1, mirror n_phi - k
        const double* am = X + ro + np - 1 - tl;
        const double* bp = Fo + n0 * 32 + lane;
        double* yrow = Y + ro + kc;
        const int c0 = n0 * 8 + 2 * tl;
#define GH_CALL(K) ang_s1_unit<K>(ap, am, -1.0, bp, D.KSo1, D.NTs, yrow, c0, 4 * D.KSo3, r < R)
        GH_NTC_SWITCH(nn, GH_CALL)
#undef GH_CALL
      }
    }
  }
  __syncthreads();

  // ---- Fs fragments -> F (free once S1 is done; S2 does not touch it) ----
  {
    const double* __restrict__ Fs = tables + it.m_Fs;
    const int nfs = (int)ang_fs_doubles(L);
    for (int e = tid * 2; e < nfs; e += TPB * 2) cp_async16(F + e, Fs + e);
    cp_async_commit();
  }
  // ---- S2: per m and n-tile of its columns ----
  {
    const int hh = (nt + 1) >> 1, MTH = ((FILTER ? hh : 2 * hh) + 7) >> 3, KSh = (hh + 3) >> 2;
    const double* __restrict__ T = tables + (FILTER ? it.m_G : it.m_T) + lane;
#define GH_S2(K) ang_s2_loop<K, FILTER>(T, KSh, X, Y, nb, L, kc, pitch, ps, g, tl, warp, NW)
    switch (MTH) {
      case 1: GH_S2(1); break;
      case 2: GH_S2(2); break;
      case 3: GH_S2(3); break;
      case 4: GH_S2(4); break;
      case 5: GH_S2(5); break;
      default: GH_S2(6); break;
    }
#undef GH_S2
  }
  cp_async_wait<0>();
  __syncthreads();

  // ---- S3: even / odd syntheses of A (Y) and B' (X), unfolded in the epilogue ----
  {
    const int nch = it.nch3, per = (D.NT3 + nch - 1) / nch;
    const int yx = (int)(Y - X);
    const double* __restrict__ Fo = F + D.KSe3 * D.NT3 * 32;
    for (int u = warp; u < MT1 * nch; u += NW) {
      const int mt = u / nch, ch = u - mt * nch;
      const int n0 = ch * per, nn = min(per, D.NT3 - n0);
      const int r = mt * 8 + g;
      const bool rok = r < R;
      const int ro = rowoff[r];
      const double* a1p = X + ro + tl;                             // B'
      const double* a0p = rok ? a1p + yx : a1p;                     // A (pad rows: the zero row for both)
      const int kcr = rok ? kc : 0;                                 // the zero row is only pitch + 16 long
      const double* bpe = F + n0 * 32 + lane;
      const double* bpo = Fo + n0 * 32 + lane;
      const int c0 = n0 * 8 + 2 * tl;
      double* g0 = dth + (size_t)r * np;
      double* g1 = dph + (size_t)r * np;
#define GH_CALL(K) ang_s3_unit<K, FILTER ? 1 : 2>(a0p, a1p, kcr, bpe, bpo, D.KSe3, D.KSo3, D.NT3, g0, g1, c0, h, np, rok)
      GH_NTC3_SWITCH(nn, GH_CALL)
#undef GH_CALL
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
