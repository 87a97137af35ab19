// kernels_gemm.cuh — K_gemm: the derivative contractions of the LARGE subdomains (Chebyshev axes with N > 64, shells with
// L > 47; the upper two decades of the size sweep, BASELINE.json configs[4]).  Same linear maps as K_cheb / K_ang (Eq. 22,
// PAPER.md:379-384; Eq. 24), restructured as one generic FP64 tensor-core GEMM
//     Out[a, col] = sum_k A[a, k] X[k, col],      a < M, k < K, col < ncols
// with A a cached constant matrix (D; the real-Fourier analysis / synthesis matrices; per m the Legendre composites Theta_m,
// Pr_m) and X / Out strided views of the field store (contraction index stride sk, output row stride sa, columns
// (c / inner) * outer + (c % inner) * cs).  At these sizes the matrices no longer fit shared memory (N = 320: 819 KB;
// L = 255: 268 MB for all m) and an accumulator for every output row no longer fits the register file, so:
//   - A is stored in DMMA A-fragment order, blocked [m_block][k_chunk][mbs <= MB m-tiles][KB k-steps][32 lanes], zero padded: one
//     (m_block, k_chunk) tile is ONE contiguous 16 / 32 KB piece, fetched by a single TMA bulk copy (cp.async.bulk, completion
//     on an mbarrier) into a 3-deep shared-memory ring by one elected thread and shared by the CTA's 8 warps;
//   - a warp owns 16 columns, walks the M-blocks with MB x 2 accumulator tiles, and streams its X fragments straight from
//     global memory (L2) into registers one k-chunk ahead of the DMMAs (the same sector-exact access patterns as K_cheb).
// A CTA walks over several components so that the pipeline is filled once.  FP64-bound (N = 320: 40 flop per byte).
#pragma once
#include <type_traits>

#include "device_types.h"
#include "kernels_deriv.cuh"

namespace ghd {

struct GemmItem {
  int64_t in_base, out_base;     // offsets (doubles) inside a component of the input / output array
  int64_t in_sk, out_sa;         // stride of the contraction index in X, of the output row index in Out
  int64_t in_outer, out_outer;   // column c lives at (c / inner) * outer + (c % inner) * cs
  int32_t in_inner, out_inner;
  int32_t in_cs, out_cs;
  int32_t M, K;
  int32_t col0, ncols;
  int64_t amat;                  // offset (doubles, even) of the blocked fragment matrix in the table memory
  int32_t in_slot, out_slot;     // -1: the kernel's `in` array (as output: the spectral filter writes the state back); 0..2: slot of the derivative scratch [3][total][S]
  int32_t pair;                  // 1: Out columns are contiguous and 16-byte aligned in pairs (double2 stores)
  int32_t mbs;                   // m-tiles per M-block (<= MB): the m-tiles are spread evenly over the fewest blocks
};

// 8 warps x 2 n-tiles.  Measured alternative, not kept: 16 warps x 1 n-tile (128 registers, four warps per scheduler to cover the
// fixed DMMA issue waits) is 5 % slower on 160^3 / n = 128 - twice the shared-memory fragment loads per DMMA.
#ifndef GH_GEMM_NST
#define GH_GEMM_NST 3
#endif
constexpr int GEMM_TPB = 256, GEMM_KB = 8, GEMM_NST = GH_GEMM_NST, GEMM_NTW = 2;
constexpr int GEMM_CT = (GEMM_TPB / 32) * 8 * GEMM_NTW;     // 128 columns per CTA
__host__ __device__ constexpr size_t gemm_stage_doubles(int MB) { return (size_t)MB * GEMM_KB * 32; }
__host__ __device__ constexpr size_t gemm_smem_bytes(int MB) { return GEMM_NST * gemm_stage_doubles(MB) * sizeof(double); }
// m-tiles per M-block for an M-row matrix: the fewest blocks of at most MB m-tiles, evenly filled (20 m-tiles: 10 + 10, not 16 + 4)
inline int gemm_mbs(int M, int MB) { const int MT = (M + 7) / 8, nMB = (MT + MB - 1) / MB; return (MT + nMB - 1) / nMB; }
// doubles of the blocked fragment matrix for an (M x K) matrix
inline size_t gemm_amat_doubles(int M, int K, int MB) {
  const int MT = (M + 7) / 8, KS = (K + 3) / 4, mbs = gemm_mbs(M, MB);
  return (size_t)((MT + mbs - 1) / mbs) * ((KS + GEMM_KB - 1) / GEMM_KB) * gemm_stage_doubles(mbs);
}

__device__ __forceinline__ void mbar_init(uint64_t* bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"((unsigned)__cvta_generic_to_shared(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, unsigned parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}\n" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(parity) : "memory");
}
// TMA bulk copy global -> shared, completion counted in bytes on the mbarrier (SASS: UBLKCP)
__device__ __forceinline__ void bulk_g2s(double* smem_dst, const double* gsrc, unsigned bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::
               "r"((unsigned)__cvta_generic_to_shared(smem_dst)), "l"(gsrc), "r"(bytes), "r"((unsigned)__cvta_generic_to_shared(bar)) : "memory");
}

template <int MB>
__global__ void __launch_bounds__(GEMM_TPB, 1)
k_gemm(const GemmItem* __restrict__ items, const double* __restrict__ tables, const double* in, double* dub, int64_t S,
       int ncomp, CompMap cm) {
  extern __shared__ __align__(16) double sm[];      // GEMM_NST stages of MB x KB fragments (bulk copies need 16-byte alignment)
  __shared__ __align__(8) uint64_t full[GEMM_NST], empty[GEMM_NST];
  constexpr int KB = GEMM_KB, NST = GEMM_NST, NTW = GEMM_NTW;
  constexpr int STAGE_MAX = MB * KB * 32;
  const GemmItem it = items[blockIdx.x];
  const int mbs = it.mbs, STAGE = mbs * KB * 32;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, g = lane >> 2, tl = lane & 3;
  const int MT = (it.M + 7) >> 3, KS = (it.K + 3) >> 2;
  const int nMB = (MT + mbs - 1) / mbs, nKC = (KS + KB - 1) / KB;
  // components this CTA walks over: blockIdx.y, + gridDim.y, ...
  const int ncw = (ncomp - (int)blockIdx.y + (int)gridDim.y - 1) / (int)gridDim.y;
  const int per = nMB * nKC, total = ncw * per;
  const double* __restrict__ amat = tables + it.amat;

  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < NST; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], GEMM_TPB / 32); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  auto issue = [&](int t) {       // stage t: the (m_block, k_chunk) tile of its position inside the component
    const int r = t % per;
    mbar_expect_tx(&full[t % NST], STAGE * 8);
    bulk_g2s(sm + (size_t)(t % NST) * STAGE_MAX, amat + (size_t)r * STAGE, STAGE * 8, &full[t % NST]);
  };
  if (tid == 0)
    for (int t = 0; t < NST - 1 && t < total; ++t) issue(t);

  // columns of this lane: B fragments (loads, column 8 n + g) and C fragments (stores, columns 8 n + 2 tl, + 1)
  const int wc0 = warp * (8 * NTW);
  int64_t cin[NTW], cout0[NTW], cout1[NTW];
  bool cok[NTW], ok0[NTW], ok1[NTW];
#pragma unroll
  for (int n = 0; n < NTW; ++n) {
    const int c = wc0 + n * 8 + g;
    cok[n] = c < it.ncols;
    const int col = it.col0 + (cok[n] ? c : 0);
    cin[n] = (int64_t)(col / it.in_inner) * it.in_outer + (int64_t)(col % it.in_inner) * it.in_cs;
    const int c0 = wc0 + n * 8 + 2 * tl;
    ok0[n] = c0 < it.ncols; ok1[n] = c0 + 1 < it.ncols;
    const int q0 = it.col0 + (ok0[n] ? c0 : 0), q1 = it.col0 + (ok1[n] ? c0 + 1 : 0);
    cout0[n] = (int64_t)(q0 / it.out_inner) * it.out_outer + (int64_t)(q0 % it.out_inner) * it.out_cs;
    cout1[n] = (int64_t)(q1 / it.out_inner) * it.out_outer + (int64_t)(q1 % it.out_inner) * it.out_cs;
  }
  const bool active = wc0 < it.ncols;      // idle warps still take part in the block barriers
  const int64_t slot_stride = (int64_t)cm.total * S;
  auto in_ptr = [&](int cw) {
    const int comp = cm.map((int)blockIdx.y + cw * (int)gridDim.y);
    return (it.in_slot < 0 ? in : dub + it.in_slot * slot_stride) + (int64_t)comp * S + it.in_base;
  };
  auto out_ptr = [&](int cw) {
    const int comp = cm.map((int)blockIdx.y + cw * (int)gridDim.y);
    return (it.out_slot < 0 ? const_cast<double*>(in) : dub + it.out_slot * slot_stride) + (int64_t)comp * S + it.out_base;
  };
  auto load_b = [&](int t, double (&b)[KB][NTW]) {
    const int cw = t / per, kc = (t % per) % nKC;
    const double* src = in_ptr(cw);
#pragma unroll
    for (int ks = 0; ks < KB; ++ks) {
      const int k = (kc * KB + ks) * 4 + tl;
#pragma unroll
      for (int n = 0; n < NTW; ++n) b[ks][n] = (active && cok[n] && k < it.K) ? src[cin[n] + (int64_t)k * it.in_sk] : 0.0;
    }
  };

  // The stage loop, instantiated for the item's EXACT m-tiles per block (MBS <= MB): a run-time bound inside the unrolled m loop
  // becomes predicated DMMAs that keep their issue and pipe slots when off (N = 160: 10 of 16 tiles exist; measured 17 TFLOP/s).
  auto run = [&](auto mbs_c) {
  constexpr int MBS = decltype(mbs_c)::value;
  double acc[MBS][NTW][2];
  double bn[KB][NTW];
  if (total > 0) load_b(0, bn);
#pragma unroll 1
  for (int t = 0; t < total; ++t) {
    const int r = t % per, mb = r / nKC, kc = r - mb * nKC;
    // Producer / consumer ring without a block barrier: the slot of stage t + NST - 1 is the one stage t - 1 used; the elected
    // thread refills it once every warp has arrived on its `empty` barrier.  Only warp 0 waits for the slowest warp here; the
    // others run up to NST - 1 stages apart, so their B-fragment loads, waits and epilogues no longer fall on the same cycles
    // (with a __syncthreads per stage the pipe idled through them: 69 % busy, profiles/r02_ncu_k_gemm.md).
    if (tid == 0 && t + NST - 1 < total) {
      if (t >= 1) mbar_wait(&empty[(t - 1) % NST], (unsigned)(((t - 1) / NST) & 1));
      issue(t + NST - 1);
    }
    __syncwarp();
    if (kc == 0) {
#pragma unroll
      for (int mt = 0; mt < MBS; ++mt)
#pragma unroll
        for (int n = 0; n < NTW; ++n) acc[mt][n][0] = acc[mt][n][1] = 0.0;
    }
    double b[KB][NTW];
#pragma unroll
    for (int ks = 0; ks < KB; ++ks)
#pragma unroll
      for (int n = 0; n < NTW; ++n) b[ks][n] = bn[ks][n];
    if (t + 1 < total) load_b(t + 1, bn);
    mbar_wait(&full[t % NST], (unsigned)((t / NST) & 1));
    if (active) {
      const double* __restrict__ a_s = sm + (size_t)(t % NST) * STAGE_MAX + lane;
      const int mtn = min(mbs, MT - mb * mbs);    // m-tiles of this block that exist
      // mtn < MBS only in the last block of a matrix whose m-tiles do not divide evenly (N = 320: 14 + 14 + 12).  The two cases
      // are separate loops: a per-tile guard inside the unrolled loop costs a branch and a WARPSYNC per DMMA pair in EVERY block
      // (ncu: 8 % of the issued instructions; 2.5 % of the kernel time on 160^3 and n = 128)
      if (mtn == MBS) {
#pragma unroll
        for (int ks = 0; ks < KB; ++ks)
#pragma unroll
          for (int mt = 0; mt < MBS; ++mt) {
            const double a = a_s[(mt * KB + ks) * 32];
#pragma unroll
            for (int n = 0; n < NTW; ++n) dmma884(acc[mt][n][0], acc[mt][n][1], a, b[ks][n]);
          }
      } else {
#pragma unroll
        for (int ks = 0; ks < KB; ++ks)
#pragma unroll
          for (int mt = 0; mt < MBS; ++mt)
            if (mt < mtn) {
              const double a = a_s[(mt * KB + ks) * 32];
#pragma unroll
              for (int n = 0; n < NTW; ++n) dmma884(acc[mt][n][0], acc[mt][n][1], a, b[ks][n]);
            }
      }
      if (kc == nKC - 1) {
        double* dst = out_ptr(t / per);
#pragma unroll
        for (int mt = 0; mt < MBS; ++mt) {
          const int a = (mb * mbs + mt) * 8 + g;
          if (mt < mtn && a < it.M) {
            const int64_t ao = (int64_t)a * it.out_sa;
#pragma unroll
            for (int n = 0; n < NTW; ++n) {
              if (it.pair && ok1[n]) {
                *reinterpret_cast<double2*>(dst + cout0[n] + ao) = make_double2(acc[mt][n][0], acc[mt][n][1]);
              } else {
                if (ok0[n]) dst[cout0[n] + ao] = acc[mt][n][0];
                if (ok1[n]) dst[cout1[n] + ao] = acc[mt][n][1];
              }
            }
          }
        }
      }
    }
    __syncwarp();                                   // every lane has its A fragments of this slot in registers
    if (lane == 0) mbar_arrive(&empty[t % NST]);
  }
  };
#define GH_GEMM_RUN(K) case K: run(std::integral_constant<int, (K <= MB ? K : MB)>{}); break;
  switch (mbs) {
    GH_GEMM_RUN(1) GH_GEMM_RUN(2) GH_GEMM_RUN(3) GH_GEMM_RUN(4) GH_GEMM_RUN(5) GH_GEMM_RUN(6) GH_GEMM_RUN(7) GH_GEMM_RUN(8)
    GH_GEMM_RUN(9) GH_GEMM_RUN(10) GH_GEMM_RUN(11) GH_GEMM_RUN(12) GH_GEMM_RUN(13) GH_GEMM_RUN(14) GH_GEMM_RUN(15)
    default: run(std::integral_constant<int, MB>{}); break;
  }
#undef GH_GEMM_RUN
}

}  // namespace ghd
