// kernels_ang.cuh — K_ang: shell angular derivatives through the l <= L projection (step A3 of DESIGN.md; Eq. 24),
// restructured axis by axis: real DFT in phi -> per-m Legendre composites along theta -> synthesis in phi.
//
// grid = (n_items, ncomp).  One CTA: `nb` (theta,phi) planes of one component of one shell, kept in shared memory through three
// GEMM stages on the FP64 tensor cores (mma.sync.m8n8k4).  With h = L+1 = n_phi/2:
//   fold   E_k = U_k + U_{n_phi-k}, O_k = U_k - U_{n_phi-k} (k = 1..L), E_0 = U_0, E_h = U_h: cos(m phi) is even and sin(m phi)
//          odd about phi = pi, so the real DFT splits into two half-length ones (half the flop of S1, S3).  The fold happens in
//          the A-operand load of S1 (two LDS and one add per fragment; the raw row carries a zero at column n_phi and the k = h
//          row of Fa_c is halved, so no lane needs a predicate)
//   S1  Cc[r][m] = sum_{k=0..h} E[r][k] Fa_c[m][k]  (m = 0..L),   Cs[r][m] = sum_{k=1..L} O[r][k] Fa_s[m][k]  (m = 1..L)
//   S2  [A ; B'](m) = [Th_m ; m Pr_m] C_m   per m, columns (t = cos/sin, plane b); A in place over C, B' into the cos<->sin
//          partner slot with sign (d/dphi in coefficient space); folded about the equator (see ang_s2_unit)
//   S3  e[r][k] = sum_m Ac[r][m] Fs_c[k][m],  o[r][k] = sum_m As[r][m] Fs_s[k][m]  (k = 0..h), same for B';
//          d u[r][k] = e + o,  d u[r][n_phi-k] = e - o, stored straight from the accumulators
//
// Round 2: the round-1 kernel kept its FP64 tensor pipe 37-42 % busy because it was bound by INSTRUCTION ISSUE, not by the pipe:
// ncu counted 21.4 issued instructions per DMMA (IMAD 22 %, ISETP 10 %, BRA 7 %, integer divisions in every unit prologue; DMMA
// itself 4.7 % of the instructions; profiles/r02_ncu_k_ang.md), and one DMMA per 16 cycles and scheduler leaves only 16 issue slots
// per DMMA.  This version makes every tile count a COMPILE-TIME constant of the shell's class NT = ceil((L+1)/8) (one
// instantiation per NT = 1..6 behind a switch; matrices are laid out and zero padded for the class on the host), so that the
// inner loops are fully unrolled with immediate shared-memory offsets, and it runs fewer, fatter warp units: S1 one (m-tile,
// parity) with all its n-tiles, S2 one mode m with all its column tiles, S3 one (m-tile, n-chunk); no integer division anywhere.
//
// Every matrix operand is stored in DMMA fragment order ([k_step][tile][32 lanes]: one conflict-free LDS.64 / coalesced 256-byte
// LDG per fragment).  Fa / Fs fragments live in shared memory; the per-m stacked matrices stream from L2 one k-step ahead.
// Planes: X (later B') and Y (C, later A), row (b, j) at b*ps + j*pitch doubles; coefficient rows hold cos m at column m
// and sin m at column kc + m - 1, kc = 8 NT.  pitch = 4 mod 8 and ps = 1 mod 16 keep the data-fragment loads conflict-free.  Rows
// beyond the tile range read a zeroed row.  The RAW planes are staged into the X region in a layout of their own (row r at
// r * raw_pitch, 16-byte aligned, dead after S1), one TMA bulk copy per row onto an mbarrier: the round-1 kernel issued one 8-byte
// LDGSTS per element, and its first warp spent 13 % of the CTA's time just issuing them (clock64 probe, profiles/r02_ncu_k_ang.md).
#pragma once
#include "device_types.h"
#include "kernels_deriv.cuh"
#include "kernels_gemm.cuh"     // mbarrier / TMA bulk-copy helpers

namespace ghd {

__host__ __device__ constexpr int ang_nt_class(int L) { return (L + 1 + 7) / 8; }      // NT = ceil(h / 8), 1..6 for L <= 47
// class constants (c_ prefix: compile-time in the kernel; the host uses the same functions to lay the matrices out)
__host__ __device__ constexpr int c_kse1(int NT) { return 2 * NT + 1; }   // S1 even: K = h+1 <= 8 NT + 1
__host__ __device__ constexpr int c_kso1(int NT) { return 2 * NT; }       // S1 odd:  K = L
__host__ __device__ constexpr int c_ks3(int NT) { return 2 * NT; }        // S3: K = h (cos m) / L (sin m)
__host__ __device__ constexpr int c_nt3(int NT) { return NT + 1; }        // S3: N = h+1 columns k = 0..h
__host__ __device__ constexpr int c_kc(int NT) { return 8 * NT; }         // coefficient rows: sin m at kc + m - 1
__host__ __device__ constexpr int c_mtf(int NT) { return (NT + 1) / 2; }  // filter: m-tiles of the hh-row projector
__host__ __device__ constexpr int c_fa_e(int NT) { return c_kse1(NT) * NT * 32; }
__host__ __device__ constexpr int c_fa(int NT) { return c_fa_e(NT) + c_kso1(NT) * NT * 32; }
__host__ __device__ constexpr int c_fs_e(int NT) { return c_ks3(NT) * c_nt3(NT) * 32; }
__host__ __device__ constexpr int c_fs(int NT) { return 2 * c_fs_e(NT); }
__host__ __device__ constexpr int c_tm(int NT) { return NT * 2 * NT * 32; }            // one mode of T: [ks < NT][p|q][mt < NT][32]
__host__ __device__ constexpr int c_gm(int NT) { return NT * 2 * c_mtf(NT) * 32; }     // one mode of G (filter)

__host__ __device__ inline int ang_pitch(int L) {   // row pitch (doubles), = 4 mod 8
  const int NT = ang_nt_class(L);
  const int a = c_kc(NT) + 4 * ((L + 3) / 4), b = 2 * L + 2 + 1;     // coefficient rows; raw rows need n_phi + 1 (a zero at column n_phi)
  int p = ((a > b ? a : b) + 3) / 4 * 4;
  return (p % 8 == 0) ? p + 4 : p;
}
__host__ __device__ inline int ang_raw_pitch(int L) {   // pitch (doubles) of the raw rows as staged (n_phi + a zero), = 4 mod 8
  const int p = (2 * L + 2 + 1 + 3) / 4 * 4;
  return (p % 8 == 0) ? p + 4 : p;
}
__host__ __device__ inline int ang_plane_stride(int L) {   // plane stride (doubles), = 1 mod 16
  return ((L + 1) * ang_pitch(L) + 15) / 16 * 16 + 1;
}
__host__ __device__ inline size_t ang_fa_doubles(int L) { return (size_t)c_fa(ang_nt_class(L)); }
__host__ __device__ inline size_t ang_fs_doubles(int L) { return (size_t)c_fs(ang_nt_class(L)); }
__host__ __device__ inline size_t ang_f_doubles(int L) {
  const size_t fa = ang_fa_doubles(L), fs = ang_fs_doubles(L);
  return fa > fs ? fa : fs;
}
// shared memory (doubles) of K_ang for nb planes: X, Y, one zero row, F fragments, the staging mbarrier, row-offset table (ints)
__host__ __device__ inline size_t ang_smem_doubles(int L, int nb) {
  const size_t rows = (size_t)nb * (L + 1);
  return 2 * (size_t)nb * ang_plane_stride(L) + ang_pitch(L) + 16 + ang_f_doubles(L) + 2 + ((rows + 8) * sizeof(int) + 7) / 8;
}

// ---- S1 unit: one m-tile (8 rows) x all NN n-tiles of one parity (NN = NT, or NT - 1 for the sin part when L = 0 mod 8: an exact
// compile-time count - guards inside unrolled loops become predicated-off DMMAs that still take their issue slots).  The A operand
// is folded on the fly from the raw row: element k is U[k] + sg U[n_phi - k]; ap / am: this lane's first element and its
// mirror; F: fragments [ks][NT][32] (+ lane).  The k loop is a real loop (KS is a run-time count).
template <int NT, int NN>
__device__ __forceinline__ void ang_s1_unit(const double* __restrict__ ap, const double* __restrict__ am, double sg,
                                            const double* __restrict__ F, int KS, double* __restrict__ yrow /* + 2 tl */,
                                            int climit, bool rok) {
  double acc[NN][2];
#pragma unroll
  for (int n = 0; n < NN; ++n) acc[n][0] = acc[n][1] = 0.0;
#pragma unroll 2
  for (int ks = 0; ks < KS; ++ks) {
    const double a = fma(sg, am[0], ap[0]);
#pragma unroll
    for (int n = 0; n < NN; ++n) dmma884(acc[n][0], acc[n][1], a, F[n * 32]);
    ap += 4; am -= 4; F += NT * 32;
  }
  if (rok) {
#pragma unroll
    for (int n = 0; n < NN; ++n)
      if (n * 8 + 2 * (int)(threadIdx.x & 3) < climit) {   // climit: end of the cos / sin region (a multiple of 4); this lane's pair starts at 8 n + 2 tl
        yrow[n * 8] = acc[n][0]; yrow[n * 8 + 1] = acc[n][1];     // (rows of odd planes are not 16-byte aligned: ps = 1 mod 16)
      }
  }
}

// ---- S3 unit: one m-tile x NN n-tiles from n0 on (columns k = 0..h), both parts (theta from Y, phi from X), even and odd GEMMs.
// a0p / a1p: this lane's rows (+ tl) of Y / X at the cos region; the sin region starts kc doubles further.
// PARTS = 1 (spectral filter): only the Y part, stored to g0.  NN: exact compile-time tile count (1..3).
template <int NT, int NN, int PARTS>
__device__ __forceinline__ void ang_s3_unit(const double* __restrict__ a0p, const double* __restrict__ a1p, int kcr,
                                            const double* __restrict__ Fe /* + lane + n0 * 32 */, int KSe, int KSo,
                                            double* __restrict__ g0, double* __restrict__ g1, int c0 /* 8 n0 + 2 tl */,
                                            int h, int np, bool rok) {
  constexpr int NT3 = c_nt3(NT);
  const double* __restrict__ Fo = Fe + c_fs_e(NT);
  double e0[NN][2], e1[NN][2], o0[NN][2], o1[NN][2];
#pragma unroll
  for (int n = 0; n < NN; ++n) {
    e0[n][0] = e0[n][1] = e1[n][0] = e1[n][1] = 0.0;
    o0[n][0] = o0[n][1] = o1[n][0] = o1[n][1] = 0.0;
  }
  {
    const double* p0 = a0p; const double* p1 = a1p;
#pragma unroll 2
    for (int ks = 0; ks < KSe; ++ks) {
      const double a0 = p0[0], a1 = PARTS == 2 ? p1[0] : 0.0;
#pragma unroll
      for (int n = 0; n < NN; ++n) {
        const double b = Fe[n * 32];
        dmma884(e0[n][0], e0[n][1], a0, b);
        if (PARTS == 2) dmma884(e1[n][0], e1[n][1], a1, b);
      }
      p0 += 4; p1 += 4; Fe += NT3 * 32;
    }
  }
  {
    const double* p0 = a0p + kcr; const double* p1 = a1p + kcr;
#pragma unroll 2
    for (int ks = 0; ks < KSo; ++ks) {
      const double a0 = p0[0], a1 = PARTS == 2 ? p1[0] : 0.0;
#pragma unroll
      for (int n = 0; n < NN; ++n) {
        const double b = Fo[n * 32];
        dmma884(o0[n][0], o0[n][1], a0, b);
        if (PARTS == 2) dmma884(o1[n][0], o1[n][1], a1, b);
      }
      p0 += 4; p1 += 4; Fo += NT3 * 32;
    }
  }
  if (rok) {
#pragma unroll
    for (int n = 0; n < NN; ++n) {
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

// ---- S2 unit: mode m, column tiles [t0, t0 + NTN) of its columns (column c < nb: the cos coefficient of plane c; c >= nb: the sin
// coefficient of plane c - nb; m = 0 has only the nb cos columns).  The Gauss-Legendre nodes are symmetric about the equator
// (theta_{nt-1-j} = pi - theta_j), the projector Pr_m commutes with that reflection and d/dtheta anticommutes, so with
// p_j = C_j + C_jbar, q_j = C_j - C_jbar (j < hh = ceil(nt/2), jbar = nt-1-j) folded on the fly in the B-operand load,
//   [alpha ; gamma] = ME_m p,  [beta ; delta] = MO_m q      (two stacked (2 hh x hh) matrices instead of one (2 nt x nt))
//   A_j = alpha + beta, A_jbar = beta - alpha;   B_j = gamma + delta, B_jbar = gamma - delta:      half the flop of S2.
// Fragments [ks < NT][p | q][mt < MT][32] of the mode stream from L2 (the whole mode is contiguous) through a register ring
// of D = c_s2d(NT) k-steps: `fr` holds the unit's first D k-steps on entry (loaded by the previous unit of this warp before ITS
// epilogue, so that the L2 latency hides behind the scatter stores) and the next unit's on return (tm_next, or untouched).
// FILTER: the stacked matrix is only the filtered projector G_m (hh rows, MT = ceil(NT/2) m-tiles; commutes with the
// reflection like Pr_m): the filtered coefficients gamma +- delta replace C in Y; X is not written.
// NTN: exact compile-time number of column tiles of this unit.  The k-steps and m-tiles need no run-time count: with nt = L+1,
// hh = ceil(nt/2): ceil(hh/4) = ceil(nt/8) = NT k-steps, ceil(2 hh/8) = NT m-tiles (FILTER: ceil(hh/8) = ceil(NT/2)), always.
#ifndef GH_ANG_S2D4
#define GH_ANG_S2D4 2      // depth 4 for NT = 4 (the whole mode ahead) spills 32 B at 168 registers: 2.839 against 2.769 ms per call on C4
#endif
__host__ __device__ constexpr int c_s2d(int NT) { return NT <= 3 ? NT : NT == 4 ? GH_ANG_S2D4 : (NT % 2 == 0 ? 2 : 1); }   // ring depth: divides NT

template <int NT, int NTN, bool FILTER>
__device__ __forceinline__ void ang_s2_unit(const double* __restrict__ tm /* fragments of mode m + lane */,
                                            const double* __restrict__ tm_next,
                                            double (&fr)[c_s2d(NT)][2 * (FILTER ? c_mtf(NT) : NT)],
                                            double* __restrict__ X, double* __restrict__ Y, int m, int t0, int nb, int nt,
                                            int pitch, int ps, int g, int tl) {
  constexpr int MT = FILTER ? c_mtf(NT) : NT, KC = c_kc(NT), D = c_s2d(NT);
  const int hh = (nt + 1) >> 1, ncols = (m == 0) ? nb : 2 * nb;
  const int slot_c = m, slot_s = KC + m - 1;      // coefficient columns of cos m / sin m
  // B fragment columns of this lane
  const double* ycol[NTN];
  bool bok[NTN];
#pragma unroll
  for (int n = 0; n < NTN; ++n) {
    const int cb = (t0 + n) * 8 + g;
    bok[n] = cb < ncols;
    const int tb = (bok[n] && cb >= nb) ? 1 : 0, bb = bok[n] ? cb - tb * nb : 0;
    ycol[n] = Y + bb * ps + (tb ? slot_s : slot_c);
  }
  double ap_[MT][NTN][2], aq_[MT][NTN][2];
#pragma unroll
  for (int mt = 0; mt < MT; ++mt)
#pragma unroll
    for (int n = 0; n < NTN; ++n) ap_[mt][n][0] = ap_[mt][n][1] = aq_[mt][n][0] = aq_[mt][n][1] = 0.0;
#pragma unroll
  for (int ks = 0; ks < NT; ++ks) {
    double cp[MT], cq[MT];
#pragma unroll
    for (int mt = 0; mt < MT; ++mt) { cp[mt] = fr[ks % D][mt]; cq[mt] = fr[ks % D][MT + mt]; }
    // the slot is free: refill it with k-step ks + D of this unit, or (NT is a multiple of D) with k-step ks + D - NT of the next
    if (ks + D < NT) {
#pragma unroll
      for (int q = 0; q < 2 * MT; ++q) fr[ks % D][q] = __ldg(tm + ((ks + D) * 2 * MT + q) * 32);
    } else if (tm_next) {
#pragma unroll
      for (int q = 0; q < 2 * MT; ++q) fr[ks % D][q] = __ldg(tm_next + ((ks + D - NT) * 2 * MT + q) * 32);
    }
    const int j = ks * 4 + tl;
    const bool jin = j < hh;
    const int jo = (jin ? j : 0) * pitch, jbo = (nt - 1 - (jin ? j : 0)) * pitch;
#pragma unroll
    for (int n = 0; n < NTN; ++n) {
      const double y0 = ycol[n][jo], y1 = ycol[n][jbo];
      const bool ok = jin && bok[n];
      const double bp = ok ? y0 + y1 : 0.0, bq = ok ? y0 - y1 : 0.0;
#pragma unroll
      for (int mt = 0; mt < MT; ++mt) {
        dmma884(ap_[mt][n][0], ap_[mt][n][1], cp[mt], bp);
        dmma884(aq_[mt][n][0], aq_[mt][n][1], cq[mt], bq);
      }
    }
  }
  __syncwarp();   // every lane has read its C_m entries before any lane overwrites them
  // C fragments: stacked row 8 mt + g (rows [0, hh): theta part, [hh, 2 hh): phi part), columns 8 (t0 + n) + 2 tl + e.
  // A -> Y at the same slot; B' -> X at the partner slot with sign (cos input -> sin slot, negated; sin -> cos); m = 0 -> 0
#pragma unroll
  for (int n = 0; n < NTN; ++n) {
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        const int c = (t0 + n) * 8 + 2 * tl + e;
        if (c < ncols) {
          const int t = c >= nb ? 1 : 0, bq = c - t * nb;
          double* ydst = Y + bq * ps + (t ? slot_s : slot_c);
          double* xdst = X + bq * ps + ((t || m == 0) ? slot_c : slot_s);
          const double sgn = (m == 0) ? 0.0 : (t ? 1.0 : -1.0);
#pragma unroll
          for (int mt = 0; mt < MT; ++mt) {
              const int rr = mt * 8 + g;
              const double s = ap_[mt][n][e] + aq_[mt][n][e], df = ap_[mt][n][e] - aq_[mt][n][e];
              if (rr < hh) {
                const int jb = nt - 1 - rr;
                ydst[rr * pitch] = s;
                if (jb != rr) ydst[jb * pitch] = FILTER ? df : -df;
              } else if (!FILTER && rr < 2 * hh) {
                const int j = rr - hh, jb = nt - 1 - j;
                xdst[j * pitch] = sgn * s;
                if (jb != j) xdst[jb * pitch] = sgn * df;
              }
            }
        }
      }
    }
}

// n-tiles of S2 one unit takes: the accumulators are 4 NT NTN doubles
#ifndef GH_ANG_NTN45
#define GH_ANG_NTN45 1      // two column tiles per S2 unit for NT = 4, 5 measured no gain (2.783 against 2.775 ms per call on C4)
#endif
__host__ __device__ constexpr int c_ntn(int NT) { return NT == 1 ? 6 : NT == 2 ? 3 : NT == 3 ? 2 : NT <= 5 ? GH_ANG_NTN45 : 1; }

// the three stages for a shell of class NT (everything that depends on NT at compile time)
template <int NT, int NW, bool FILTER>
__device__ __forceinline__ void ang_body(const AngItem& it, const double* __restrict__ tables, double* __restrict__ X,
                                         double* __restrict__ Y, double* __restrict__ F, const int* __restrict__ rowoff,
                                         double* dth, double* dph, int nb, int R, int pitch, int ps, int warp, int lane) {
  const int g = lane >> 2, tl = lane & 3;
  const int L = it.L, nt = L + 1, np = 2 * L + 2, h = nt;
  constexpr int KC = c_kc(NT);
  const int KSe1 = (h + 1 + 3) >> 2, KSo1 = (L + 3) >> 2, KSe3 = (h + 3) >> 2, KSo3 = (L + 3) >> 2;
  const int MT1 = (R + 7) >> 3;
  // ---- S1: Cc = E Fa_c^T (columns 0..), Cs = O Fa_s^T (columns kc..): unit = (m-tile, parity) ----
  {
    const double* __restrict__ Fe = F + lane;
    const double* __restrict__ Fo = F + c_fa_e(NT) + lane;
    const int par = warp & 1;
    const int pr = ang_raw_pitch(L);
    for (int mt = (warp >> 1); mt < MT1; mt += NW / 2) {
      const int r = mt * 8 + g;
      const int ro = rowoff[r];
      const double* __restrict__ xr = X + r * pr;       // raw row (pad rows of the last m-tile read whatever follows: their results are dropped)
      if (par == 0)
        ang_s1_unit<NT, NT>(xr + tl, xr + np - tl, 1.0, Fe, KSe1, Y + ro + 2 * tl, KC, r < R);
      else if (NT == 1 || ((L + 7) >> 3) == NT)          // n-tiles of the sin part: ceil(L / 8) = NT or NT - 1
        ang_s1_unit<NT, NT>(xr + 1 + tl, xr + np - 1 - tl, -1.0, Fo, KSo1, Y + ro + KC + 2 * tl, 4 * KSo3, r < R);
      else
        ang_s1_unit<NT, (NT > 1 ? NT - 1 : 1)>(xr + 1 + tl, xr + np - 1 - tl, -1.0, Fo, KSo1, Y + ro + KC + 2 * tl, 4 * KSo3, r < R);
    }
  }
  __syncthreads();

  // ---- Fs fragments -> F (free once S1 is done; S2 does not touch it) ----
  {
    const double* __restrict__ Fs = tables + it.m_Fs;
    for (int e = (warp * 32 + lane) * 2; e < c_fs(NT); e += NW * 64) cp_async16(F + e, Fs + e);
    cp_async_commit();
  }
  // ---- S2: per m, its column tiles in chunks of c_ntn(NT): unit = (m, chunk) ----
  {
    constexpr int NTN = c_ntn(NT);
    const int ntn_all = (2 * nb + 7) >> 3, ntn0 = (nb + 7) >> 3;      // column tiles of a mode m > 0 / of m = 0
    const int nchunk = (ntn_all + NTN - 1) / NTN;
    const double* __restrict__ T = tables + (FILTER ? it.m_G : it.m_T) + lane;
    constexpr int TM = FILTER ? c_gm(NT) : c_tm(NT);
    constexpr int D = c_s2d(NT), MT2 = 2 * (FILTER ? c_mtf(NT) : NT);
    // this warp's units (m, chunk): warp, warp + NW, ... in (m, chunk) order; a chunk beyond the tiles of m = 0 is skipped
    auto advance = [&](int& m, int& ch, int by) {
      do {
        ch += by; by = NW;      // a unit that does not exist (m = 0 has fewer tiles) is passed over with the same stride
        while (ch >= nchunk) { ch -= nchunk; ++m; }
      } while (m <= L && ch * NTN >= (m == 0 ? ntn0 : ntn_all));
    };
    int m = 0, ch = -1;
    advance(m, ch, warp + 1);
    double fr[D][MT2];
    if (m <= L) {
      const double* __restrict__ tm = T + (size_t)m * TM;
#pragma unroll
      for (int k = 0; k < D; ++k)
#pragma unroll
        for (int q = 0; q < MT2; ++q) fr[k][q] = __ldg(tm + (k * MT2 + q) * 32);
    }
    while (m <= L) {
      int mn = m, chn = ch;
      advance(mn, chn, NW);
      const int t0 = ch * NTN, tiles = (m == 0 ? ntn0 : ntn_all) - t0;
      const double* __restrict__ tm = T + (size_t)m * TM;
      const double* __restrict__ tmn = mn <= L ? T + (size_t)mn * TM : nullptr;
      const int ntn = tiles < NTN ? tiles : NTN;
#define GH_S2(K) ang_s2_unit<NT, (K <= NTN ? K : 1), FILTER>(tm, tmn, fr, X, Y, m, t0, nb, nt, pitch, ps, g, tl)
      switch (ntn) {
        case 1: GH_S2(1); break;
        case 2: GH_S2(2); break;
        case 3: GH_S2(3); break;
        case 4: GH_S2(4); break;
        case 5: GH_S2(5); break;
        default: GH_S2(6); break;
      }
#undef GH_S2
      m = mn; ch = chn;
    }
  }
  cp_async_wait<0>();
  __syncthreads();

  // ---- S3: even / odd syntheses of A (Y) and B' (X), unfolded in the epilogue: unit = (m-tile, n-chunk) ----
  {
    constexpr int NT3 = c_nt3(NT), NCH = NT3 < 3 ? NT3 : 3;
    const int nt3 = (h + 1 + 7) >> 3;                 // n-tiles that exist (NT or NT + 1)
    const int nch = it.nch3, per = (nt3 + nch - 1) / nch;      // host-chosen chunking (per <= 3)
    const int yx = (int)(Y - X);
    int mt = 0, ch = warp;
    while (ch >= nch) { ch -= nch; ++mt; }
    while (mt < MT1) {
      const int n0 = ch * per, nn = min(per, nt3 - n0);
      const int r = mt * 8 + g;
      const bool rok = r < R;
      const int ro = rowoff[r];
      const double* a1p = X + ro + tl;                             // B'
      const double* a0p = rok ? a1p + yx : a1p;                     // A (pad rows: the zero row for both)
      const int kcr = rok ? KC : 0;                                 // the zero row is only pitch + 16 long
#define GH_S3(K) ang_s3_unit<NT, (K <= NCH ? K : 1), FILTER ? 1 : 2>(a0p, a1p, kcr, F + n0 * 32 + lane, KSe3, KSo3, dth + (size_t)r * np, \
                                                                     dph + (size_t)r * np, n0 * 8 + 2 * tl, h, np, rok)
      switch (nn) {
        case 1: GH_S3(1); break;
        case 2: GH_S3(2); break;
        default: GH_S3(3); break;
      }
#undef GH_S3
      ch += NW;
      while (ch >= nch) { ch -= nch; ++mt; }
    }
  }
}

#ifndef GH_ANG_CTAS
#define GH_ANG_CTAS 2
#endif
template <int TPB, bool FILTER>
__global__ void __launch_bounds__(TPB, TPB <= 256 ? GH_ANG_CTAS : 1)
k_ang(const AngItem* __restrict__ items, const double* __restrict__ tables, const double* in,
      double* out, int64_t S, CompMap cm) {
  extern __shared__ __align__(16) double sm[];
  constexpr int NW = TPB / 32;
  const AngItem it = items[blockIdx.x];
  const int comp = cm.map(blockIdx.y), ncomp = cm.total, tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int L = it.L, nt = L + 1, np = 2 * L + 2, plane = nt * np;
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
  uint64_t& bar = *reinterpret_cast<uint64_t*>(F + ang_f_doubles(L));   // mbarrier of the raw-plane bulk copies (8-byte aligned: all offsets are in doubles)
  int* rowoff = reinterpret_cast<int*>(F + ang_f_doubles(L) + 2);   // [R + 8]: offset of row r in X / Y; pad rows -> Z
  const int zoff = (int)(Z - X);

  // ---- stage 0: raw U -> X (one TMA bulk copy per row, raw layout) and Fa fragments -> F by cp.async, all in flight at once;
  // row table; padding.  Every global row starts 16-byte aligned (offsets are multiples of 16 doubles, n_phi is even).
  {
    const int pr = ang_raw_pitch(L);
    if (tid == 0) {
      mbar_init(&bar, 1);
      asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
      mbar_expect_tx(&bar, (unsigned)(R * np * 8));
    }
    __syncthreads();
    for (int r = tid; r < R; r += TPB) {
      double* xrow = X + r * pr;
      bulk_g2s(xrow, src + (size_t)r * np, (unsigned)(np * 8), &bar);
      for (int c = np; c < pr; ++c) xrow[c] = 0.0;     // column n_phi = 0 (the mirror of k = 0)
    }
    const double* __restrict__ Fa = tables + it.m_Fa;
    const int nfa = (int)ang_fa_doubles(L);
    for (int e = tid * 2; e < nfa; e += TPB * 2) cp_async16(F + e, Fa + e);
    cp_async_commit();
    {
      int b = 0, j = tid;
      while (j >= nt) { j -= nt; ++b; }
      for (int r = tid; r < R; r += TPB) {
        rowoff[r] = b * ps + j * pitch;
        j += TPB;
        while (j >= nt) { j -= nt; ++b; }
      }
    }
    // S3 reads whole k-steps of the B' rows in X, padding columns included (times zero rows of Fs): what S2 does not write there must
    // be finite.  Inside the raw layout it is raw data or zeros; the tail of the X region behind the raw layout is cleared here.
    for (int e = R * pr + tid; e < nb * ps; e += TPB) X[e] = 0.0;
    if (tid < 8) rowoff[R + tid] = zoff;           // the pad rows of the last m-tile (R + 8 entries are allocated)
    for (int e = tid; e < pitch + 16; e += TPB) Z[e] = 0.0;
    cp_async_wait<0>();
    mbar_wait(&bar, 0);
  }
  __syncthreads();

#define GH_ANG_BODY(K) ang_body<K, NW, FILTER>(it, tables, X, Y, F, rowoff, dth, dph, nb, R, pitch, ps, warp, lane)
  switch (ang_nt_class(L)) {
    case 1: GH_ANG_BODY(1); break;
    case 2: GH_ANG_BODY(2); break;
    case 3: GH_ANG_BODY(3); break;
    case 4: GH_ANG_BODY(4); break;
    case 5: GH_ANG_BODY(5); break;
    default: GH_ANG_BODY(6); break;
  }
#undef GH_ANG_BODY
}

}  // namespace ghd
