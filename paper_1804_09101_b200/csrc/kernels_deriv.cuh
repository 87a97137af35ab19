// kernels_deriv.cuh — Chebyshev-line derivative kernel (step A2 of DESIGN.md), the stand-alone Jacobian (A4) and helpers shared
// by the derivative kernels (K_ang: kernels_ang.cuh; the large classes: kernels_gemm.cuh).
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

// The component walk of one warp with EXACT compile-time tile counts MT = ceil(N/8), KS = ceil(N/4) (KS = 2 MT - 1 or 2 MT): guards
// inside unrolled loops (`if (ks < KS)`) compile to predicated DMMAs, which still take their issue and pipe slots when switched
// off - for N = 16 in the N <= 24 class that was 10 of 18 DMMAs per k-sweep (ncu / cuobjdump, profiles/r02_ncu_k_ang.md §2 a).
template <int MT, int KS, int NTW>
__device__ __forceinline__ void cheb_body(const ChebItem& it, const double* __restrict__ sm, const double* __restrict__ in,
                                          double* __restrict__ out, int64_t S, int ncomp, const CompMap& cm, int si0,
                                          const int (&caddr)[NTW], const bool (&cok)[NTW], const int (&c0a)[NTW],
                                          const int (&c1a)[NTW], bool pair, int wc0, int lane) {
  const int g = lane >> 2, tl = lane & 3, N = it.N, ncols = it.ncols;
  // the CTA walks over components blockIdx.y, blockIdx.y + gridDim.y, ... (one launch and one matrix load for all of them)
#pragma unroll 1
  for (int cw = blockIdx.y; cw < ncomp; cw += gridDim.y) {
    const int comp = cm.map(cw);
    // B fragments of the whole warp tile.  (si is laundered so that the compiler recomputes the 2 x KS x NTW element
    // offsets per component instead of keeping them all live across the loop: that costs 40 registers and a CTA per SM)
    int si = si0;
    asm volatile("" : "+r"(si));
    double b[KS][NTW];
    {
      const double* __restrict__ src = in + (int64_t)comp * S + it.base;
#pragma unroll
      for (int ks = 0; ks < KS; ++ks) {
        const int i = ks * 4 + tl;
#pragma unroll
        for (int n = 0; n < NTW; ++n) b[ks][n] = (cok[n] && i < N) ? src[caddr[n] + i * si] : 0.0;
      }
    }
    double acc[MT][NTW][2];
#pragma unroll
    for (int mt = 0; mt < MT; ++mt)
#pragma unroll
      for (int n = 0; n < NTW; ++n) acc[mt][n][0] = acc[mt][n][1] = 0.0;
#pragma unroll
    for (int ks = 0; ks < KS; ++ks)
#pragma unroll
      for (int mt = 0; mt < MT; ++mt) {
        const double a = sm[(mt * KS + ks) * 32 + lane];
#pragma unroll
        for (int n = 0; n < NTW; ++n) dmma884(acc[mt][n][0], acc[mt][n][1], a, b[ks][n]);
      }
    // C fragments: row a = 8 mt + g, columns 8 n + 2 tl and + 1
    double* __restrict__ dst = out + ((int64_t)it.axis * cm.total + comp) * S + it.base;
#pragma unroll
    for (int n = 0; n < NTW; ++n) {
      const int c = wc0 + n * 8 + 2 * tl;
      const bool ok0 = c < ncols, ok1 = c + 1 < ncols;
#pragma unroll
      for (int mt = 0; mt < MT; ++mt) {
        const int a = mt * 8 + g;
        if (a < N) {
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

// MTM / KSM: the largest tile counts of the launch's register class (they size the registers: launch bounds); the body runs with the
// item's exact counts.
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
  // exact tile counts of this item: KS = KSM - d, MT = ceil(KS / 2), for the (at most six) counts of the class
#define GH_CHEB_BODY(K) cheb_body<((K) + 1) / 2, (K), NTW>(it, sm, in, out, S, ncomp, cm, si0, caddr, cok, c0a, c1a, pair, wc0, lane)
  constexpr int KLO = KSM == 6 ? 1 : KSM == 8 ? 7 : KSM == 12 ? 9 : 13;     // smallest KS of the class (N <= 24 | 32 | 48 | 64)
  if (KS == KSM) GH_CHEB_BODY(KSM);
  else if (KSM - 1 >= KLO && KS == KSM - 1) GH_CHEB_BODY(KSM - 1 >= 1 ? KSM - 1 : 1);
  else if (KSM - 2 >= KLO && KS == KSM - 2) GH_CHEB_BODY(KSM - 2 >= 1 ? KSM - 2 : 1);
  else if (KSM - 3 >= KLO && KS == KSM - 3) GH_CHEB_BODY(KSM - 3 >= 1 ? KSM - 3 : 1);
  else if (KSM - 4 >= KLO && KS == KSM - 4) GH_CHEB_BODY(KSM - 4 >= 1 ? KSM - 4 : 1);
  else GH_CHEB_BODY(KSM - 5 >= 1 ? KSM - 5 : 1);
#undef GH_CHEB_BODY
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
  // cylindrical shell (kind 2), logical (rho, z, phi): its tables hold 1 / rho, st = 1, ct = 0, so the six entries above are
  // already  d_x = cp d_rho - (sp / rho) d_phi,  d_y = sp d_rho + (cp / rho) d_phi;  only  d_z = d_z (the second slot)  differs
  if (sd.kind == 2) J.zt = 1.0;
  return J;
}

// K_jac: in-place logical -> Cartesian on shells for a gradient array g[3][ncomp][S] (debug / gauge-source path;
// inside gh_rhs the same transform is fused into K_rhs).
__global__ void __launch_bounds__(TILE_PTS)
k_jac(const SubDev* __restrict__ subs, const int32_t* __restrict__ tile_first, int n_sub,
      const double* __restrict__ tables, double* __restrict__ g, int64_t S, int ncomp) {
  const int s = find_sub(tile_first, n_sub, blockIdx.x);
  const SubDev sd = subs[s];
  if (sd.kind == 1) return;
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
