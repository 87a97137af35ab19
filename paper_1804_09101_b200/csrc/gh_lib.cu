// gh_lib.cu — the C ABI of include/gh.h: host-side domain planning (A0, A1) and kernel launches (A2-A8).
// No torch, no CPU fallback: every compute call needs a CUDA device and returns GH_ERR_CUDA without one.
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <map>
#include <mutex>
#include <string>
#include <utility>
#include <vector>

#include "../../include/gh.h"
#include "basis.h"
#include "device_types.h"
#include "kernels_deriv.cuh"
#include "kernels_ang.cuh"
#include "kernels_point.cuh"
#include "kernels_jac.cuh"
#include "kernels_gemm.cuh"

using namespace ghd;

namespace {

constexpr int CHEB_TPB = 128;                     // K_cheb: 4 warps
// measured on C4 (ms per call): 4 n-tiles per warp and 5 components per CTA 1.50; 2 and 5: 1.33; 2 and 10: 1.28; 2 and 25: 1.25;
// 2 and 50: 1.28; 1 n-tile per warp: 1.41-1.47
constexpr int CHEB_COMP_WALK = 25;                // components one K_cheb CTA walks over
constexpr int CHEB_NTW = 2;                       // n-tiles per warp
constexpr int CHEB_CT = (CHEB_TPB / 32) * 8 * CHEB_NTW;   // columns per CTA
constexpr int CHEB_NCLASS = 4;                    // register-tile classes: N <= 24 (7 CTAs per SM), N <= 32 (5), N <= 48 (4), N <= 64 (3)
inline int cheb_class(int N) { return N <= 24 ? 0 : N <= 32 ? 1 : N <= 48 ? 2 : 3; }
inline int cheb_ct(int) { return CHEB_CT; }
inline size_t cheb_frag_doubles(int N) { return (size_t)((N + 7) / 8) * ((N + 3) / 4) * 32; }   // D in fragment order
// K_ang threads per CTA.  192 x 2 CTAs and 384 x 1 CTA leave 168 registers per thread: no spills.  With 256 / 512 threads (128
// registers, 104 B of stack) the spill reloads in the unit prologues went out to L2 - at ~200 KB of shared memory per SM there is
// hardly any L1 left - and ~12 % of the warp-stall samples sat on integer address arithmetic waiting for them
// (profiles/r02_ncu_k_ang.md section 4).  Measured on C4, per call: 256/512 2.90 ms, 192/384 2.77, 192/320 2.87, 192/448 3.15,
// 192/256 2.88, 256/384 2.91, 192/512 3.05, 128 x 3 CTAs / 384 2.78.
#ifndef GH_ANG_TPB0
#define GH_ANG_TPB0 192
#endif
#ifndef GH_ANG_TPB1
#define GH_ANG_TPB1 384
#endif
constexpr int ANG_TPB0 = GH_ANG_TPB0, ANG_TPB1 = GH_ANG_TPB1;    // K_ang threads: class 0 (two CTAs per SM), class 1 (one CTA per SM)
constexpr size_t ANG_SMEM_2CTA = (GH_ANG_CTAS == 2 ? 113 : GH_ANG_CTAS == 3 ? 74 : 55) * 1024;     // K_ang shared memory that still lets GH_ANG_CTAS CTAs share an SM
constexpr int ANG_NB_MAX = 8;                    // planes per K_ang CTA offered to the plan (S2 then has <= 2 column tiles per m)
constexpr int ANG_NB_MAX_SMALL_L = 24;           // ... for L < 12, where a plane is a few tiles only (SingleBH k = 0: 5.96 -> 4.91 ms
                                                 // per 2e6 points; for L >= 12 more than 8 planes measured slightly slower on C4)
constexpr size_t SMEM_MAX = 227 * 1024;
constexpr int GEMM_MB = 16;                      // m-tiles per M-block of K_gemm (tiles beyond the matrix are skipped at run time)
enum { G_S1 = 0, G_S2 = 1, G_S3T = 2, G_S3P = 3, G_CHEB = 4, G_NDERIV = 5,      // K_gemm launch lists of the derivatives, in launch order
       G_FX = 5, G_FY = 6, G_FZ = 7, G_FS2 = 8, G_FS3 = 9, G_NLIST = 10 };        // ... and of the spectral filter (block axes; shell composites and synthesis)
inline bool big_N(int N) { return N > GH_SMALL_CHEB_N; }
inline bool big_L(int L) { return L > GH_SMALL_L; }

thread_local std::string g_create_error;

inline int64_t round_up(int64_t v, int64_t m) { return (v + m - 1) / m * m; }

struct Carve {   // bump allocator over the caller's workspace (256-byte granularity)
  size_t pos = 0;
  size_t take(size_t bytes) { size_t p = pos; pos += (size_t)round_up((int64_t)bytes, 256); return p; }
};

struct Plan {
  int n_sub = 0;
  std::vector<gh_subdomain_desc> descs;
  std::vector<int64_t> offsets;          // n_sub+1
  std::vector<int32_t> tile_first;       // n_sub+1
  int64_t P = 0, S = 0;
  int n_tiles = 0;
  size_t table_doubles = 0;
  size_t ftable_doubles = 0;             // spectral-filter matrices, directly behind the derivative tables
  int n_fcheb[3][CHEB_NCLASS] = {}, n_fcheb_items = 0;   // filter work items of the blocks per axis and class
  int n_cheb_items = 0, n_cheb_class[CHEB_NCLASS] = {}, n_ang_items = 0;
  int n_ang_class[2] = {0, 0};           // K_ang items per shared-memory class (0: two CTAs per SM, 1: one)
  size_t cheb_smem = 0, ang_smem[2] = {0, 0};
  int n_gemm[G_NLIST] = {0};             // K_gemm items per launch list (large subdomains)
  size_t fbigtab_doubles = 0;            // filter matrices of the large classes, behind the interface tables (written by gh_set_filter)
  size_t bigtab_doubles = 0;             // their blocked fragment matrices, behind the filter tables
  bool has_big = false;
  int n_ifc_items = 0;                   // interface faces whose neighbour has a different band limit (K_face_interp)
  int64_t Sf = 0;                        // component stride (doubles) of the interface buffer
  size_t ifc_smem = 0, ifctab_doubles = 0;
  std::vector<int> ang_pb;               // planes per CTA for each subdomain (0 for blocks)
  std::vector<int> ang_class;            // shared-memory class of each shell
  // workspace offsets (bytes)
  size_t o_ua, o_ub, o_k, o_du, o_H, o_dH, o_jac, o_mapJ, o_mapv, o_tables, o_subs, o_tiles, o_cheb, o_fcheb, o_ang, o_gemm, o_ifc, o_ifci, o_part, o_persub, o_flag, total;
};

inline void sub_dims(const gh_subdomain_desc& d, int& n0, int& n1, int& n2) {
  if (d.kind == GH_SHELL) { n0 = d.n[0]; n1 = d.n[1] + 1; n2 = 2 * d.n[1] + 2; }
  else { n0 = d.n[0]; n1 = d.n[1]; n2 = d.n[2]; }
}

// n-chunks per m-tile of K_ang S3 that minimise (rounds over the warps) x (DMMAs per unit + fixed cost); at most 3 n-tiles per unit
inline int ang_best_nch3(int NT3, int MT1, int NW) {
  int best = 0; double bc = 1e300;
  for (int nch = (NT3 + 2) / 3; nch <= NT3; ++nch) {
    const int per = (NT3 + nch - 1) / nch;
    if ((NT3 + per - 1) / per != nch) continue;          // same chunking the kernel derives from nch
    const double cost = (double)((MT1 * nch + NW - 1) / NW) * (4 * per + 0.6);
    if (cost < bc) { bc = cost; best = nch; }
  }
  return best;
}
// Modelled duration of one K_ang CTA (units: one DMMA slot of a warp) for `np_` planes of band limit L on NW warps: per stage
// the number of rounds the warps need times the DMMAs of one unit (the k-steps and tiles the kernel really runs), plus a fixed
// part for staging and barriers.  Used only to choose the planes per CTA and the CTA class of a shell.
#ifndef GH_ANG_FIX
#define GH_ANG_FIX 40.0
#endif
constexpr double ANG_FIX = GH_ANG_FIX;     // fixed part of a CTA (staging, barriers), in DMMA slots; 10-300 measured, flat optimum near 40
#ifndef GH_ANG_C0W
#define GH_ANG_C0W ((double)GH_ANG_CTAS)
#endif
constexpr double ANG_C0W = GH_ANG_C0W;      // class 0 runs GH_ANG_CTAS CTAs per SM
inline double ang_cta_cost(int L, int np_, int NW) {
  const int NT = ang_nt_class(L), nt = L + 1, h = nt, MT1 = (np_ * nt + 7) / 8;
  const int KSe1 = (h + 1 + 3) / 4, KSo1 = (L + 3) / 4, KSe3 = (h + 3) / 4, KSo3 = (L + 3) / 4, nt3 = (h + 1 + 7) / 8;
  // S1: units (m-tile, parity) alternate over the warps: NW / 2 warps per parity
  const double c1 = (double)((MT1 + NW / 2 - 1) / (NW / 2)) * std::max(KSe1, KSo1) * NT;
  const int hh = (nt + 1) / 2, MTn = (2 * hh + 7) / 8, KSh = (hh + 3) / 4, ntn = (2 * np_ + 7) / 8, NTN = c_ntn(NT);
  const int nchunk = (ntn + NTN - 1) / NTN;
  const double c2 = (double)(((L + 1) * nchunk + NW - 1) / NW) * (KSh * 2 * MTn * std::min(NTN, ntn));
  const int nch3 = ang_best_nch3(nt3, MT1, NW), per3 = (nt3 + nch3 - 1) / nch3;
  const double c3 = (double)((MT1 * nch3 + NW - 1) / NW) * ((KSe3 + KSo3) * per3 * 2);
  return c1 + c2 + c3 + ANG_FIX;
}
inline size_t ang_smem_bytes(int L, int nb) { return ang_smem_doubles(L, nb) * sizeof(double); }
inline size_t shell_fa_doubles(int L) { return ang_fa_doubles(L); }   // (even | odd) analysis fragments
inline size_t shell_fs_doubles(int L) { return ang_fs_doubles(L); }   // (even | odd) synthesis fragments
inline size_t shell_t_doubles(int L) {    // [m][k_step < NT][even|odd][m_tile < NT][32]: the equator-folded stacked matrices of K_ang S2
  return (size_t)(L + 1) * c_tm(ang_nt_class(L));
}
inline size_t shell_matrix_doubles(int L) { return shell_fa_doubles(L) + shell_fs_doubles(L) + shell_t_doubles(L); }
inline size_t shell_g_doubles(int L) {    // [m][k_step < NT][even|odd][m_tile < ceil(NT/2)][32]: equator-folded filtered projectors (hh rows)
  return (size_t)(L + 1) * c_gm(ang_nt_class(L));
}

// elem(row, col) of an (M x K) matrix -> K_gemm's A-fragment order, blocked [m_block][k_chunk][mbs m-tiles][GEMM_KB k-steps][32]
// (zero padded), into dst[0 .. gemm_amat_doubles(M, K, GEMM_MB))
template <class F>
void fill_amat(double* dst, int M, int K, F elem) {
  const int MT = (M + 7) / 8, KS = (K + 3) / 4, mbs = gemm_mbs(M, GEMM_MB), nMB = (MT + mbs - 1) / mbs, nKC = (KS + GEMM_KB - 1) / GEMM_KB;
  std::fill(dst, dst + gemm_amat_doubles(M, K, GEMM_MB), 0.0);
  for (int mb = 0; mb < nMB; ++mb) for (int kc = 0; kc < nKC; ++kc) for (int mt = 0; mt < mbs; ++mt) for (int ks = 0; ks < GEMM_KB; ++ks)
    for (int lane = 0; lane < 32; ++lane) {
      const int row = (mb * mbs + mt) * 8 + lane / 4, col = (kc * GEMM_KB + ks) * 4 + lane % 4;
      if (row < M && col < K) dst[((((size_t)mb * nKC + kc) * mbs + mt) * GEMM_KB + ks) * 32 + lane] = (double)elem(row, col);
    }
}

bool validate(const gh_subdomain_desc* descs, int32_t n_sub, std::string& err) {
  char buf[256];
  if (!descs || n_sub < 1) { err = "descs is NULL or n_sub < 1"; return false; }
  for (int s = 0; s < n_sub; ++s) {
    const gh_subdomain_desc& d = descs[s];
    if (d.kind == GH_SHELL) {
      if (d.n[0] < 2 || d.n[0] > GH_MAX_CHEB_N || d.n[1] < 1 || d.n[1] > GH_MAX_L) {
        snprintf(buf, sizeof buf, "subdomain %d: shell needs 2 <= N_r <= %d and 1 <= L <= %d", s, GH_MAX_CHEB_N, GH_MAX_L);
        err = buf; return false;
      }
      if (!(d.lo[0] > 0.0) || !(d.hi[0] > d.lo[0])) { snprintf(buf, sizeof buf, "subdomain %d: shell needs 0 < r_in < r_out", s); err = buf; return false; }
    } else if (d.kind == GH_BLOCK) {
      for (int a = 0; a < 3; ++a) {
        if (d.n[a] < 2 || d.n[a] > GH_MAX_CHEB_N) { snprintf(buf, sizeof buf, "subdomain %d: block needs 2 <= N <= %d on every axis", s, GH_MAX_CHEB_N); err = buf; return false; }
        if (!(d.hi[a] > d.lo[a])) { snprintf(buf, sizeof buf, "subdomain %d: block needs lo < hi on every axis", s); err = buf; return false; }
      }
    } else if (d.kind == GH_CYLINDER) {
      if (d.n[0] < 2 || d.n[0] > GH_MAX_CHEB_N || d.n[1] < 2 || d.n[1] > GH_MAX_CHEB_N || d.n[2] < 3 || d.n[2] > GH_MAX_CHEB_N) {
        snprintf(buf, sizeof buf, "subdomain %d: cylindrical shell needs 2 <= N_rho, N_z <= %d and 3 <= N_phi <= %d", s, GH_MAX_CHEB_N, GH_MAX_CHEB_N);
        err = buf; return false;
      }
      if (!(d.lo[0] > 0.0) || !(d.hi[0] > d.lo[0]) || !(d.hi[1] > d.lo[1])) { snprintf(buf, sizeof buf, "subdomain %d: cylindrical shell needs 0 < rho_in < rho_out and z_lo < z_hi", s); err = buf; return false; }
    } else { snprintf(buf, sizeof buf, "subdomain %d: unknown kind %d", s, d.kind); err = buf; return false; }
    for (int f = 0; f < 6; ++f) {
      if (d.face[f] == GH_FACE_INTERFACE && f < 2 && d.kind == GH_SHELL) {
        // the partner: the previous (inner face) / next (outer face) descriptor, a shell with the same centre whose facing face
        // carries the flag too and sits at the same radius (a different band limit L: its face state is interpolated)
        const int o = f == 0 ? s - 1 : s + 1;
        bool ok = o >= 0 && o < n_sub && descs[o].kind == GH_SHELL && descs[o].face[1 - f] == GH_FACE_INTERFACE;
        if (ok) {
          const double ra = f == 0 ? d.lo[0] : d.hi[0], rb = f == 0 ? descs[o].hi[0] : descs[o].lo[0];
          ok = std::fabs(ra - rb) <= 1e-12 * std::fabs(ra);
          for (int c = 0; c < 3; ++c) ok = ok && descs[o].center[c] == d.center[c];
        }
        if (!ok) { snprintf(buf, sizeof buf, "subdomain %d: INTERFACE face %d has no matching neighbour shell", s, f); err = buf; return false; }
        continue;
      }
      if (d.face[f] == GH_FACE_INTERFACE && f < (d.kind == GH_SHELL ? 2 : d.kind == GH_CYLINDER ? 4 : 6)) { snprintf(buf, sizeof buf, "subdomain %d: interfaces are built between concentric shells only", s); err = buf; return false; }
      if (d.face[f] != GH_FACE_FREE && d.face[f] != GH_FACE_FROZEN && d.face[f] != GH_FACE_CHARACTERISTIC && d.face[f] != GH_FACE_INTERFACE) { snprintf(buf, sizeof buf, "subdomain %d: bad face flag", s); err = buf; return false; }
    }
    for (int g = 0; g < 3; ++g)
      if (!std::isfinite(d.gamma[g])) { snprintf(buf, sizeof buf, "subdomain %d: non-finite gamma", s); err = buf; return false; }
  }
  return true;
}

// Sizes and offsets of everything; pure host arithmetic (shared by gh_workspace_bytes and gh_domain_create).
bool make_plan(const gh_subdomain_desc* descs, int32_t n_sub, Plan& pl, std::string& err) {
  if (!validate(descs, n_sub, err)) return false;
  pl.n_sub = n_sub;
  pl.descs.assign(descs, descs + n_sub);
  pl.offsets.assign(n_sub + 1, 0);
  pl.tile_first.assign(n_sub + 1, 0);
  pl.ang_pb.assign(n_sub, 0);
  pl.ang_class.assign(n_sub, 0);
  std::map<int, int> seenL;
  std::map<std::pair<int, int>, int> seenIfc;
  size_t tab = 0;
  int64_t off = 0, tiles = 0;
  for (int s = 0; s < n_sub; ++s) {
    const gh_subdomain_desc& d = descs[s];
    int n0, n1, n2; sub_dims(d, n0, n1, n2);
    const int64_t Ps = (int64_t)n0 * n1 * n2;
    if (Ps > (int64_t)1 << 30) { err = "subdomain too large"; return false; }
    pl.offsets[s] = off; off += round_up(Ps, 16);
    pl.tile_first[s] = (int32_t)tiles; tiles += (Ps + TILE_PTS - 1) / TILE_PTS;
    pl.P += Ps;
    const int naxes = d.kind == GH_SHELL ? 1 : 3;
    for (int a = 0; a < naxes; ++a) {
      const int N = d.n[a];
      const int64_t cols = Ps / N;
      if (big_N(N)) {       // tiled GEMM path
        pl.bigtab_doubles += gemm_amat_doubles(N, N, GEMM_MB);
        pl.n_gemm[G_CHEB] += (int)((cols + GEMM_CT - 1) / GEMM_CT);
        if (d.kind != GH_SHELL) { pl.fbigtab_doubles += gemm_amat_doubles(N, N, GEMM_MB); pl.n_gemm[G_FX + a] += (int)((cols + GEMM_CT - 1) / GEMM_CT); }
        pl.has_big = true;
        continue;
      }
      tab += cheb_frag_doubles(N);
      const int items = (int)((cols + cheb_ct(N) - 1) / cheb_ct(N));
      pl.n_cheb_items += items; pl.n_cheb_class[cheb_class(N)] += items;
      pl.cheb_smem = std::max(pl.cheb_smem, cheb_frag_doubles(N) * sizeof(double));
      if (d.kind != GH_SHELL) { pl.ftable_doubles += cheb_frag_doubles(N); pl.n_fcheb[a][cheb_class(N)] += items; pl.n_fcheb_items += items; }
    }
    if (d.kind == GH_CYLINDER)      // coordinate tables 1 / rho, (ct = 0, st = 1), cos phi, sin phi in the shells' slots
      tab += (size_t)round_up(n0, 2) + 2 * (size_t)round_up(n1, 2) + 2 * (size_t)round_up(n2, 2);
    if (d.kind == GH_SHELL) {
      for (int f = 0; f < 2; ++f) {
        const int o = f == 0 ? s - 1 : s + 1;
        if (d.face[f] != GH_FACE_INTERFACE || descs[o].n[1] == d.n[1]) continue;
        const int Ls = descs[o].n[1], Ld = d.n[1];
        if (Ls > GH_SMALL_L || Ld > GH_SMALL_L) { err = "interfaces between shells of different L are built for L <= 47"; return false; }
        pl.n_ifc_items += 1; pl.Sf += round_up((int64_t)n1 * n2, 16);
        const size_t nts = Ls + 1, nps = 2 * Ls + 2, nqs = 2 * Ls + 1, ntd = Ld + 1, npd = 2 * Ld + 2;
        if (!seenIfc.count({Ls, Ld})) { seenIfc[{Ls, Ld}] = 1; pl.ifctab_doubles += nps * nqs + (size_t)(Ls + 1) * nts * ntd + nqs * npd; }
        pl.ifc_smem = std::max(pl.ifc_smem, (nts * nps + nts * nqs + ntd * nqs) * sizeof(double));
      }
      const int L = d.n[1];
      tab += (size_t)round_up(n0, 2) + 2 * (size_t)round_up(n1, 2) + 2 * (size_t)round_up(n2, 2);
      if (big_L(L)) {       // tiled GEMM path: analysis, per-m composites, two syntheses through global coefficient buffers
        const int nt = L + 1, np = 2 * L + 2, nq = 2 * L + 1;
        if (!seenL.count(L)) {
          seenL[L] = 1;
          pl.bigtab_doubles += gemm_amat_doubles(nq, np, GEMM_MB) + 2 * gemm_amat_doubles(np, nq, GEMM_MB) +
                               (size_t)(L + 1) * 2 * gemm_amat_doubles(nt, nt, GEMM_MB);
          pl.fbigtab_doubles += (size_t)(L + 1) * gemm_amat_doubles(nt, nt, GEMM_MB);
        }
        const int64_t R = (int64_t)n0 * nt;
        const int rt = (int)((R + GEMM_CT - 1) / GEMM_CT);
        pl.n_gemm[G_S1] += rt; pl.n_gemm[G_S3T] += rt; pl.n_gemm[G_S3P] += rt; pl.n_gemm[G_FS3] += rt;
        for (int m = 0; m <= L; ++m) {
          const int ct = ((m ? 2 : 1) * n0 + GEMM_CT - 1) / GEMM_CT;
          pl.n_gemm[G_S2] += 2 * ct; pl.n_gemm[G_FS2] += ct;
        }
        pl.has_big = true;
        continue;
      }
      if (!seenL.count(L)) { seenL[L] = 1; tab += shell_matrix_doubles(L); pl.ftable_doubles += shell_g_doubles(L); }
      // planes per CTA and CTA class (0: 256 threads, two CTAs per SM; 1: 512 threads, one CTA per SM): of all that fit in
      // shared memory, the pair with the smallest modelled time for the whole shell (sum over its CTAs / CTAs per SM).
      // Against "the most planes that fit" this is worth 3 % of K_ang on C4 (tile quantisation over the warps).
      int pb = 0, cls = 0;
      {
        double best = 1e300;
        for (int c = 0; c < 2; ++c)
          for (int nb = 1; nb <= (L < 12 ? ANG_NB_MAX_SMALL_L : ANG_NB_MAX); ++nb) {
            if (ang_smem_bytes(L, nb) > (c == 0 ? ANG_SMEM_2CTA : SMEM_MAX)) continue;
            const int NW = (c == 0 ? ANG_TPB0 : ANG_TPB1) / 32;
            double t = 0;
            for (int p0 = 0; p0 < n0; p0 += nb) t += ang_cta_cost(L, std::min(nb, n0 - p0), NW);
            t /= (c == 0 ? ANG_C0W : 1.0);
            if (t < best) { best = t; pb = nb; cls = c; }
          }
      }
      if (!pb) { err = "internal: no K_ang configuration for a small-class shell"; return false; }
      const int chunks = (n0 + pb - 1) / pb;
      pl.ang_pb[s] = pb; pl.ang_class[s] = cls;
      pl.n_ang_items += chunks; pl.n_ang_class[cls] += chunks;
      pl.ang_smem[cls] = std::max(pl.ang_smem[cls], ang_smem_bytes(L, pb));
    }
  }
  if (tiles > 0x7fffffff) { err = "domain too large"; return false; }
  pl.offsets[n_sub] = off; pl.S = off;
  pl.tile_first[n_sub] = (int32_t)tiles; pl.n_tiles = (int)tiles;
  pl.table_doubles = tab;
  if (pl.cheb_smem > SMEM_MAX) { err = "Chebyshev N too large for shared memory"; return false; }
  Carve c;
  const size_t comp = (size_t)pl.S * sizeof(double);
  pl.o_ua = c.take(NCOMP * comp); pl.o_ub = c.take(NCOMP * comp); pl.o_k = c.take(NCOMP * comp);
  pl.o_du = c.take(3 * NCOMP * comp); pl.o_H = c.take(4 * comp); pl.o_dH = c.take(12 * comp);
  pl.o_jac = c.take(9 * comp); pl.o_mapJ = c.take(9 * comp); pl.o_mapv = c.take(3 * comp);
  pl.o_tables = c.take((pl.table_doubles + pl.ftable_doubles + pl.bigtab_doubles + pl.ifctab_doubles + pl.fbigtab_doubles) * sizeof(double));
  pl.o_ifc = c.take((size_t)std::max<int64_t>(1, NCOMP * pl.Sf) * sizeof(double));
  pl.o_ifci = c.take((size_t)std::max(1, pl.n_ifc_items) * sizeof(IfcItem));
  pl.o_subs = c.take((size_t)n_sub * sizeof(SubDev));
  pl.o_tiles = c.take((size_t)(n_sub + 1) * sizeof(int32_t));
  pl.o_cheb = c.take((size_t)std::max(1, pl.n_cheb_items) * sizeof(ChebItem));
  pl.o_fcheb = c.take((size_t)std::max(1, pl.n_fcheb_items) * sizeof(ChebItem));
  pl.o_ang = c.take((size_t)std::max(1, pl.n_ang_items) * sizeof(AngItem));
  { int ng = 0; for (int l = 0; l < G_NLIST; ++l) ng += pl.n_gemm[l]; pl.o_gemm = c.take((size_t)std::max(1, ng) * sizeof(GemmItem)); }
  pl.o_part = c.take((size_t)pl.n_tiles * 6 * sizeof(double));
  pl.o_persub = c.take((size_t)n_sub * 6 * sizeof(double));
  pl.o_flag = c.take(256);
  pl.total = c.pos;
  return true;
}

}  // namespace

struct gh_domain {
  Plan pl;
  char* ws = nullptr;
  cudaStream_t stream = nullptr;
  double *ua = nullptr, *ub = nullptr, *k = nullptr, *du = nullptr, *H = nullptr, *dH = nullptr, *jac = nullptr, *tables = nullptr;
  bool has_jac = false;
  double *mapJ = nullptr, *mapv = nullptr;   // dual frame (gh_set_frame_map)
  bool has_map = false;
  SubDev* subs = nullptr;
  int32_t* tiles = nullptr;
  ChebItem* cheb = nullptr;
  ChebItem* fcheb = nullptr;             // filter items of the blocks, ordered [axis][class]
  AngItem* ang = nullptr;
  GemmItem* gemm = nullptr;              // K_gemm items of the large subdomains, the G_NLIST lists back to back
  IfcItem* ifci = nullptr;               // faces to interpolate (interfaces between shells of different L)
  double* ifc = nullptr;                 // [50][Sf]: the neighbours' face states on the own grids
  struct FBlock { int N; bool fourier; size_t off; };     // one filter matrix slot per (block or cylinder, axis): offset (doubles) from `tables`
  std::vector<FBlock> f_blocks;
  std::map<int, size_t> f_L;             // shell band limit L -> offset (doubles) of its filtered projectors from `tables`
  struct FBig { int N; size_t off; bool fourier; };     // large classes: one K_gemm filter matrix slot per (block, large axis) ...
  std::vector<FBig> f_big_blocks;
  std::map<int, std::vector<size_t>> f_big_L;   // ... and per large L the slots of its per-m filtered projectors
  double gemm_stages[G_NLIST] = {};             // pipeline stages (m-blocks x k-chunks) of one component, summed over the list's items
  bool filt_blocks = false, filt_shells = false;
  // Dormand-Prince 5(4): seven stage derivatives in a separately attached workspace
  double* dpk[7] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
  double *dp_part = nullptr, *dp_out = nullptr;
  bool dp_fsal = false;                  // dpk[0] already holds the RHS of the current state
  double *part = nullptr, *persub = nullptr;
  int* flag = nullptr;
  std::vector<SubDev> h_subs;
  bool has_fields = false, has_shell = false, has_block = false, has_char = false, has_ifc = false;
  int device = 0, n_sm = 148;            // the device the workspace lives on (current at create) and its SM count
  int opt[GH_NUM_OPTIONS] = {0};         // gh_set_option
  // CUDA graphs of the step (kind 0: gh_rk_step, 1: gh_rk_step_norms) and of gh_rhs to a DEVICE pointer (kind 2), each valid
  // for the key it was captured with
  struct StepGraph { cudaGraphExec_t exec = nullptr; double dt = 0; const void *ua = nullptr, *ub = nullptr, *out = nullptr; int oop = 0, map = 0; int64_t nlaunch = 0; };
  StepGraph graphs[3];
  double t = 0.0;
  int64_t launches = 0;
  std::string err;
  // profiling
  bool prof = false;
  struct Pending { cudaEvent_t a, b; int cls; };
  std::vector<Pending> pending;
  std::vector<cudaEvent_t> pool;
  double prof_ms[GH_NUM_KERNELS] = {0};
  int64_t prof_n[GH_NUM_KERNELS] = {0};
};

namespace {

// Every entry point that touches the device runs with the domain's device current and restores the caller's on return.
struct DeviceGuard {
  int prev = -1; bool sw = false;
  explicit DeviceGuard(const gh_domain* d) {
    if (d && cudaGetDevice(&prev) == cudaSuccess && prev != d->device) sw = cudaSetDevice(d->device) == cudaSuccess;
  }
  ~DeviceGuard() { if (sw) cudaSetDevice(prev); }
};

gh_status fail(gh_domain* d, gh_status st, const std::string& msg) {
  if (d) d->err = msg; else g_create_error = msg;
  return st;
}
#define GH_CUDA(d, call)                                                                              \
  do {                                                                                                \
    cudaError_t e_ = (call);                                                                          \
    if (e_ != cudaSuccess) return fail(d, GH_ERR_CUDA, std::string(#call ": ") + cudaGetErrorString(e_)); \
  } while (0)

cudaEvent_t get_event(gh_domain* d) {
  if (!d->pool.empty()) { cudaEvent_t e = d->pool.back(); d->pool.pop_back(); return e; }
  cudaEvent_t e; cudaEventCreate(&e); return e;
}
struct ProfScope {   // brackets one launch with events when profiling is on; always counts the launch
  gh_domain* d; int cls; cudaEvent_t a = nullptr, b = nullptr;
  ProfScope(gh_domain* d_, int cls_) : d(d_), cls(cls_) {
    d->launches += 1;
    if (d->prof) { a = get_event(d); b = get_event(d); cudaEventRecord(a, d->stream); }
  }
  ~ProfScope() { if (d->prof) { cudaEventRecord(b, d->stream); d->pending.push_back({a, b, cls}); } }
};
void drain_profile(gh_domain* d) {
  if (d->pending.empty()) return;
  cudaStreamSynchronize(d->stream);
  for (auto& p : d->pending) {
    float ms = 0; cudaEventElapsedTime(&ms, p.a, p.b);
    d->prof_ms[p.cls] += ms; d->prof_n[p.cls] += 1;
    d->pool.push_back(p.a); d->pool.push_back(p.b);
  }
  d->pending.clear();
}

}  // namespace

// ------------------------------------------------------------------------------------------------------
// host-side basis builder entry points (no CUDA)
// ------------------------------------------------------------------------------------------------------
extern "C" gh_status gh_basis_cheb(int32_t N, double* x, double* D) {
  if (N < 2) return GH_ERR_ARG;
  std::vector<ghb::ld> xv, Dv;
  ghb::cheb_nodes(N, xv); ghb::cheb_diff_matrix(N, Dv);
  if (x) for (int j = 0; j < N; ++j) x[j] = (double)xv[j];
  if (D) for (size_t e = 0; e < (size_t)N * N; ++e) D[e] = (double)Dv[e];
  return GH_OK;
}

extern "C" gh_status gh_basis_gauss_legendre(int32_t L, double* theta, double* w) {
  if (L < 0) return GH_ERR_ARG;
  std::vector<ghb::ld> ct, wv;
  ghb::gauss_legendre(L, ct, wv);
  for (int j = 0; j <= L; ++j) { if (theta) theta[j] = (double)acosl(ct[j]); if (w) w[j] = (double)wv[j]; }
  return GH_OK;
}

extern "C" gh_status gh_basis_shell(int32_t L, double* Fa, double* Fs, double* Th, double* Pr) {
  if (L < 1) return GH_ERR_ARG;
  ghb::ShellBasis B; ghb::shell_basis(L, B);
  if (Fa) for (size_t e = 0; e < B.Fa.size(); ++e) Fa[e] = (double)B.Fa[e];
  if (Fs) for (size_t e = 0; e < B.Fs.size(); ++e) Fs[e] = (double)B.Fs[e];
  if (Th) for (size_t e = 0; e < B.Th.size(); ++e) Th[e] = (double)B.Th[e];
  if (Pr) for (size_t e = 0; e < B.Pr.size(); ++e) Pr[e] = (double)B.Pr[e];
  return GH_OK;
}

extern "C" size_t gh_workspace_bytes(const gh_subdomain_desc* descs, int32_t n_sub) {
  Plan pl; std::string err;
  if (!make_plan(descs, n_sub, pl, err)) { g_create_error = err; return 0; }
  return pl.total;
}

// ------------------------------------------------------------------------------------------------------
// gh_domain_create: A0 (tables) + A1 (store layout, work lists), one upload
// ------------------------------------------------------------------------------------------------------
extern "C" gh_status gh_domain_create(const gh_subdomain_desc* descs, int32_t n_sub, void* dev_workspace, size_t bytes,
                                      void* cuda_stream, gh_domain** out) {
  if (!out) return fail(nullptr, GH_ERR_ARG, "out is NULL");
  *out = nullptr;
  Plan pl; std::string err;
  if (!make_plan(descs, n_sub, pl, err)) return fail(nullptr, GH_ERR_ARG, err);
  if (!dev_workspace || ((uintptr_t)dev_workspace & 255) != 0) return fail(nullptr, GH_ERR_WORKSPACE, "workspace is NULL or not 256-byte aligned");
  if (bytes < pl.total) return fail(nullptr, GH_ERR_WORKSPACE, "workspace too small: need " + std::to_string(pl.total) + " bytes");
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) { cudaGetLastError(); return fail(nullptr, GH_ERR_CUDA, "no CUDA device (this library has no CPU fallback)"); }

  gh_domain* d = new gh_domain();
  d->pl = pl; d->ws = (char*)dev_workspace; d->stream = (cudaStream_t)cuda_stream;
  {
    cudaPointerAttributes pa;      // the workspace decides the device (falls back to the current one)
    if (cudaPointerGetAttributes(&pa, dev_workspace) == cudaSuccess && pa.type == cudaMemoryTypeDevice) d->device = pa.device;
    else { cudaGetLastError(); cudaGetDevice(&d->device); }
    int nsm = 0;
    if (cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, d->device) == cudaSuccess && nsm > 0) d->n_sm = nsm;
  }
  DeviceGuard guard_(d);
  char* w = d->ws;
  d->ua = (double*)(w + pl.o_ua); d->ub = (double*)(w + pl.o_ub); d->k = (double*)(w + pl.o_k);
  d->du = (double*)(w + pl.o_du); d->H = (double*)(w + pl.o_H); d->dH = (double*)(w + pl.o_dH); d->jac = (double*)(w + pl.o_jac);
  d->mapJ = (double*)(w + pl.o_mapJ); d->mapv = (double*)(w + pl.o_mapv);
  d->tables = (double*)(w + pl.o_tables); d->subs = (SubDev*)(w + pl.o_subs); d->tiles = (int32_t*)(w + pl.o_tiles);
  d->cheb = (ChebItem*)(w + pl.o_cheb); d->ang = (AngItem*)(w + pl.o_ang); d->fcheb = (ChebItem*)(w + pl.o_fcheb);
  d->gemm = (GemmItem*)(w + pl.o_gemm); d->ifc = (double*)(w + pl.o_ifc); d->ifci = (IfcItem*)(w + pl.o_ifci);
  d->part = (double*)(w + pl.o_part); d->persub = (double*)(w + pl.o_persub); d->flag = (int*)(w + pl.o_flag);

  // ---- tables and work lists on the host ----
  std::vector<double> tab(pl.table_doubles, 0.0);
  std::vector<ChebItem> cheb, chebc[CHEB_NCLASS];   // items per class (concatenated below)
  std::vector<ChebItem> fch[3][CHEB_NCLASS];       // spectral-filter items of the blocks per axis and class
  size_t ftp = pl.table_doubles;         // running offset inside the filter-table region
  std::vector<AngItem> ang, ang1; ang.reserve(pl.n_ang_items);   // class 0 items, class 1 items (appended below)
  d->h_subs.resize(n_sub);
  size_t tp = 0;
  std::map<int, std::vector<ghb::ld>> Dcache, Fcache;        // N -> unscaled D; N -> Fourier differentiation matrix
  struct ShellOff { int Fa, Fs, T; };
  std::map<int, ShellOff> Lcache;
  // large subdomains: blocked fragment matrices (behind the filter tables) and K_gemm items per launch list
  std::vector<double> bigtab(pl.bigtab_doubles, 0.0);
  std::vector<GemmItem> glist[G_NLIST];
  size_t btp = 0;
  const size_t big0 = pl.table_doubles + pl.ftable_doubles;      // offset of bigtab[0] from d->tables
  // elem(row, col) of an (M x K) matrix -> A-fragment order, blocked [m_block][k_chunk][GEMM_MB m-tiles][GEMM_KB k-steps][32];
  // returns the offset (doubles) of the matrix from d->tables
  auto put_amat = [&](int M, int K, auto elem) {
    const size_t at = btp;
    fill_amat(bigtab.data() + at, M, K, elem);
    btp += gemm_amat_doubles(M, K, GEMM_MB);
    return (int64_t)(big0 + at);
  };
  // filter matrices of the large classes: slots behind the interface tables, filled by gh_set_filter
  const size_t fbig0 = pl.table_doubles + pl.ftable_doubles + pl.bigtab_doubles + pl.ifctab_doubles;
  size_t fbp = 0;
  // one K_gemm item per tile of GEMM_CT columns
  auto put_items = [&](int list, GemmItem proto, int64_t cols) {
    // columns (c, c + 1), c even, may leave as one double2 when they are neighbours in memory at an even address
    proto.pair = (proto.out_cs == 1 && proto.out_sa % 2 == 0 && proto.out_base % 2 == 0 && proto.out_outer % 2 == 0 &&
                  (proto.out_inner % 2 == 0 || proto.out_inner >= cols)) ? 1 : 0;
    proto.mbs = gemm_mbs(proto.M, GEMM_MB);
    for (int64_t c0 = 0; c0 < cols; c0 += GEMM_CT) {
      GemmItem it = proto; it.col0 = (int)c0; it.ncols = (int)std::min<int64_t>(GEMM_CT, cols - c0);
      glist[list].push_back(it);
      const int MT = (it.M + 7) / 8, KS = (it.K + 3) / 4;
      d->gemm_stages[list] += (double)((MT + it.mbs - 1) / it.mbs) * ((KS + GEMM_KB - 1) / GEMM_KB);
    }
  };
  struct BigShellOff { int64_t FaQ, FsQ, FpQ; std::vector<int64_t> Th, Pr; };
  std::map<int, BigShellOff> Lbig;
  // interfaces between shells of different band limit: interpolation tables behind the large-class tables, items, buffer offsets
  struct IfcOff { int64_t FaT, GT, FxT; };
  std::map<std::pair<int, int>, IfcOff> IfcCache;
  std::vector<double> ifctab(pl.ifctab_doubles, 0.0);
  std::vector<IfcItem> ifci;
  size_t itp = 0; int64_t ifc_next = 0;
  const size_t ifc0 = pl.table_doubles + pl.ftable_doubles + pl.bigtab_doubles;
  for (int s = 0; s < n_sub; ++s) {
    const gh_subdomain_desc& de = descs[s];
    SubDev& sd = d->h_subs[s];
    memset(&sd, 0, sizeof sd);
    int n0, n1, n2; sub_dims(de, n0, n1, n2);
    sd.kind = de.kind; sd.n0 = n0; sd.n1 = n1; sd.n2 = n2; sd.off = pl.offsets[s]; sd.P = n0 * n1 * n2;
    for (int f = 0; f < 6; ++f) { sd.face[f] = de.face[f]; if (f < (de.kind == GH_SHELL ? 2 : de.kind == GH_CYLINDER ? 4 : 6) && de.face[f] == GH_FACE_CHARACTERISTIC) d->has_char = true; }
    sd.nbr[0] = sd.nbr[1] = -1; sd.nbi[0] = sd.nbi[1] = -1; sd.pen = 0.0;
    if (de.kind == GH_SHELL) {
      sd.pen = (double)(n0 - 1) * (double)(n0 - 1) / (de.hi[0] - de.lo[0]);
      for (int f = 0; f < 2; ++f) {
        if (de.face[f] != GH_FACE_INTERFACE) continue;
        d->has_char = d->has_ifc = true;
        const int o = f == 0 ? s - 1 : s + 1;
        const int Ls = descs[o].n[1], Ld = de.n[1];
        const int64_t nplane = (int64_t)(Ls + 1) * (2 * Ls + 2);
        // the neighbour's face plane: its outermost one for my inner face, its innermost one for my outer face
        const int64_t src = f == 0 ? pl.offsets[o] + (int64_t)(descs[o].n[0] - 1) * nplane : pl.offsets[o];
        if (Ls == Ld) { sd.nbr[f] = src; continue; }
        if (!IfcCache.count({Ls, Ld})) {
          // FaT[k][q] analysis on the source longitudes, GT[m][j][j'] per-m Legendre interpolation, FxT[q][k'] the series at the destination longitudes
          ghb::ShellBasis B; ghb::shell_basis(Ls, B);
          std::vector<ghb::ld> G; ghb::shell_interp_composites(Ls, Ld, G);
          const int nts = Ls + 1, nps = 2 * Ls + 2, nqs = 2 * Ls + 1, ntd = Ld + 1, npd = 2 * Ld + 2;
          IfcOff io; io.FaT = (int64_t)(ifc0 + itp);
          for (int k = 0; k < nps; ++k) for (int q = 0; q < nqs; ++q) ifctab[itp + (size_t)k * nqs + q] = (double)B.Fa[(size_t)q * nps + k];
          itp += (size_t)nps * nqs;
          io.GT = (int64_t)(ifc0 + itp);
          for (int m = 0; m <= Ls; ++m) for (int j = 0; j < nts; ++j) for (int jd = 0; jd < ntd; ++jd)
            ifctab[itp + ((size_t)m * nts + j) * ntd + jd] = (double)G[((size_t)m * ntd + jd) * nts + j];
          itp += (size_t)(Ls + 1) * nts * ntd;
          io.FxT = (int64_t)(ifc0 + itp);
          const ghb::ld PI_L = 3.14159265358979323846264338327950288L;
          for (int q = 0; q < nqs; ++q) for (int k = 0; k < npd; ++k) {
            const int m = q <= Ls ? q : q - Ls;
            const ghb::ld ang = 2 * PI_L * (ghb::ld)(((long long)m * k) % npd) / npd;
            ifctab[itp + (size_t)q * npd + k] = (double)(q == 0 ? (ghb::ld)1 : q <= Ls ? cosl(ang) : sinl(ang));
          }
          itp += (size_t)nqs * npd;
          IfcCache[{Ls, Ld}] = io;
        }
        const IfcOff& io = IfcCache[{Ls, Ld}];
        IfcItem it; memset(&it, 0, sizeof it);
        it.src_off = src; it.dst_off = ifc_next; it.Ls = Ls; it.Ld = Ld; it.m_FaT = io.FaT; it.m_GT = io.GT; it.m_FxT = io.FxT;
        sd.nbi[f] = ifc_next; ifc_next += round_up((int64_t)n1 * n2, 16);
        ifci.push_back(it);
      }
    }
    for (int g = 0; g < 3; ++g) sd.gamma[g] = de.gamma[g];
    const int naxes = de.kind == GH_SHELL ? 1 : 3;
    const int64_t nn[3] = {n0, n1, n2};
    const int64_t strides[3] = {(int64_t)n1 * n2, n2, 1};
    for (int a = 0; a < naxes; ++a) {
      const int N = (int)nn[a];
      // the periodic axis of a cylindrical shell: the Fourier differentiation matrix in d / d phi itself (no map factor) - to the
      // kernels one more "black box" matrix along a line
      const bool fourier = de.kind == GH_CYLINDER && a == 2;
      if (fourier && !Fcache.count(N)) ghb::fourier_diff_matrix(N, Fcache[N]);
      if (!fourier && !Dcache.count(N)) ghb::cheb_diff_matrix(N, Dcache[N]);
      const std::vector<ghb::ld>& D = fourier ? Fcache[N] : Dcache[N];
      const ghb::ld scale = fourier ? (ghb::ld)1 : 2 / ((ghb::ld)de.hi[a] - (ghb::ld)de.lo[a]);   // affine map factor of Eq. 22
      if (big_N(N)) {     // K_gemm: Out[a', col] = sum_i (scale D)[a'][i] u[i, col], the same strided views as K_cheb's
        GemmItem it; memset(&it, 0, sizeof it);
        it.amat = put_amat(N, N, [&](int r, int c) { return scale * D[(size_t)r * N + c]; });
        it.M = N; it.K = N; it.in_slot = -1; it.out_slot = a;
        it.in_base = it.out_base = sd.off; it.in_sk = it.out_sa = strides[a];
        if (a == 0) { it.in_inner = (int)(nn[1] * nn[2]); it.in_outer = 0; it.in_cs = 1; }
        else if (a == 1) { it.in_inner = (int)nn[2]; it.in_outer = nn[1] * nn[2]; it.in_cs = 1; }
        else { it.in_inner = 1; it.in_outer = nn[2]; it.in_cs = 0; }
        it.out_inner = it.in_inner; it.out_outer = it.in_outer; it.out_cs = it.in_cs;
        put_items(G_CHEB, it, sd.P / N);
        if (de.kind != GH_SHELL) {      // the same strided view with the filter matrix: x: u -> T1 (slot 0), y: T1 -> T2 (slot 1), z: T2 -> u
          GemmItem fi = it;
          fi.amat = (int64_t)(fbig0 + fbp);
          fi.in_slot = a == 0 ? -1 : a - 1; fi.out_slot = a == 2 ? -1 : a;
          d->f_big_blocks.push_back({N, fbig0 + fbp, fourier}); fbp += gemm_amat_doubles(N, N, GEMM_MB);
          put_items(G_FX + a, fi, sd.P / N);
        }
        continue;
      }
      const int dm = (int)tp;
      // scaled D in DMMA A-fragment order: lane (g = lane/4, t = lane%4) of fragment (m_tile, k_step) holds
      // D[8 m_tile + g][4 k_step + t]; rows / columns beyond N are zero
      {
        const int mtn = (N + 7) / 8, ksn = (N + 3) / 4;
        for (int mt = 0; mt < mtn; ++mt)
          for (int ks = 0; ks < ksn; ++ks)
            for (int lane = 0; lane < 32; ++lane) {
              const int row = mt * 8 + lane / 4, col = ks * 4 + lane % 4;
              tab[tp + ((size_t)mt * ksn + ks) * 32 + lane] = (row < N && col < N) ? (double)(scale * D[(size_t)row * N + col]) : 0.0;
            }
      }
      tp += cheb_frag_doubles(N);
      const int64_t cols = sd.P / N;
      const int ct = cheb_ct(N);
      for (int64_t c0 = 0; c0 < cols; c0 += ct) {
        ChebItem it; memset(&it, 0, sizeof it);
        it.base = sd.off; it.stride_i = strides[a]; it.N = N; it.dmat = dm; it.axis = a;
        it.col0 = (int)c0; it.ncols = (int)std::min<int64_t>(ct, cols - c0);
        if (a == 0) { it.col_inner = (int)(nn[1] * nn[2]); it.outer_stride = 0; }
        else if (a == 1) { it.col_inner = (int)nn[2]; it.outer_stride = nn[1] * nn[2]; }
        else { it.col_inner = 1; it.outer_stride = nn[2]; }
        chebc[cheb_class(N)].push_back(it);
        if (de.kind != GH_SHELL) { ChebItem fi = it; fi.dmat = (int)ftp; fi.axis = 0; fch[a][cheb_class(N)].push_back(fi); }
      }
      if (de.kind != GH_SHELL) { d->f_blocks.push_back({N, fourier, ftp}); ftp += cheb_frag_doubles(N); }
    }
    if (de.kind == GH_SHELL && big_L(de.n[1])) {
      // K_gemm path of a large shell, per component c (R = n_r n_theta rows of n_phi points), through coefficient buffers in
      // the derivative scratch (slot 0: later d_r, slot 1: later d_theta, slot 2: later d_phi):
      //   S1   W[q][row]  = sum_k FaQ[q][k] u[row][k]                 u -> slot 1      q = 0: m = 0;  2m-1: cos m;  2m: sin m
      //   S2   V1_m = Th_m W_m  -> slot 2,   V2_m = Pr_m W_m -> slot 0      per m, columns = (cos | sin, plane), contraction over theta
      //   S3   d_theta u[row][k] = sum_q FsQ[k][q] V1[q][row] -> slot 1;   d_phi u[row][k] = sum_q FpQ[k][q] V2[q][row] -> slot 2
      // (FpQ = d/dphi of the synthesis: -m sin on the cos coefficient, +m cos on the sin coefficient.)  The radial derivative
      // (slot 0) is launched after S3.
      d->has_shell = true;
      const int L = de.n[1], nt = L + 1, np = 2 * L + 2, nq = 2 * L + 1;
      if (!Lbig.count(L)) {
        ghb::ShellBasis B; ghb::shell_basis(L, B);
        BigShellOff o;
        auto qrow = [&](int q) { return q == 0 ? 0 : (q & 1) ? (q + 1) / 2 : L + q / 2; };     // q -> row of Fa / column of Fs, Fp
        o.FaQ = put_amat(nq, np, [&](int q, int k) { return B.Fa[(size_t)qrow(q) * np + k]; });
        o.FsQ = put_amat(np, nq, [&](int k, int q) { return B.Fs[(size_t)k * nq + qrow(q)]; });
        o.FpQ = put_amat(np, nq, [&](int k, int q) { return B.Fp[(size_t)k * nq + qrow(q)]; });
        for (int m = 0; m <= L; ++m) {
          o.Th.push_back(put_amat(nt, nt, [&](int r, int c) { return B.Th[((size_t)m * nt + r) * nt + c]; }));
          o.Pr.push_back(put_amat(nt, nt, [&](int r, int c) { return B.Pr[((size_t)m * nt + r) * nt + c]; }));
        }
        Lbig[L] = o;
      }
      const BigShellOff& o = Lbig[L];
      const int64_t R = (int64_t)n0 * nt, BIG = (int64_t)1 << 30;
      GemmItem it; memset(&it, 0, sizeof it);
      // S1
      it.amat = o.FaQ; it.M = nq; it.K = np; it.in_slot = -1; it.out_slot = 1;
      it.in_base = sd.off; it.in_sk = 1; it.in_inner = (int)BIG; it.in_outer = 0; it.in_cs = np;
      it.out_base = sd.off; it.out_sa = R; it.out_inner = (int)BIG; it.out_outer = 0; it.out_cs = 1;
      put_items(G_S1, it, R);
      // S2
      for (int m = 0; m <= L; ++m) {
        const int64_t q0 = m == 0 ? 0 : 2 * m - 1, cols = (m ? 2 : 1) * (int64_t)n0;
        memset(&it, 0, sizeof it);
        it.M = nt; it.K = nt; it.in_slot = 1;
        it.in_base = it.out_base = sd.off + q0 * R; it.in_sk = it.out_sa = 1;
        it.in_inner = it.out_inner = (int)BIG; it.in_cs = it.out_cs = nt;
        it.amat = o.Th[m]; it.out_slot = 2; put_items(G_S2, it, cols);
        it.amat = o.Pr[m]; it.out_slot = 0; put_items(G_S2, it, cols);
      }
      // S3
      memset(&it, 0, sizeof it);
      it.M = np; it.K = nq;
      it.in_base = sd.off; it.in_sk = R; it.in_inner = (int)BIG; it.in_cs = 1;
      it.out_base = sd.off; it.out_sa = 1; it.out_inner = (int)BIG; it.out_cs = np;
      it.amat = o.FsQ; it.in_slot = 2; it.out_slot = 1; put_items(G_S3T, it, R);
      it.amat = o.FpQ; it.in_slot = 0; it.out_slot = 2; put_items(G_S3P, it, R);
      // spectral filter of a large shell: S1 as above (u -> W in slot 1), per m the filtered projector G_m W -> slot 2, synthesis -> u
      it.amat = o.FsQ; it.in_slot = 2; it.out_slot = -1; put_items(G_FS3, it, R);
      if (!d->f_big_L.count(L)) {
        std::vector<size_t> offs;
        for (int m = 0; m <= L; ++m) { offs.push_back(fbig0 + fbp); fbp += gemm_amat_doubles(nt, nt, GEMM_MB); }
        d->f_big_L[L] = offs;
      }
      for (int m = 0; m <= L; ++m) {
        const int64_t q0 = m == 0 ? 0 : 2 * m - 1, cols = (m ? 2 : 1) * (int64_t)n0;
        memset(&it, 0, sizeof it);
        it.M = nt; it.K = nt; it.in_slot = 1; it.out_slot = 2;
        it.in_base = it.out_base = sd.off + q0 * R; it.in_sk = it.out_sa = 1;
        it.in_inner = it.out_inner = (int)BIG; it.in_cs = it.out_cs = nt;
        it.amat = (int64_t)d->f_big_L[L][m]; put_items(G_FS2, it, cols);
      }
    }
    if (de.kind == GH_SHELL) {
      // coordinate tables of this shell (for the Jacobian of Eq. 8)
      const int L = de.n[1];
      std::vector<ghb::ld> xr, ct, wv;
      ghb::cheb_nodes(n0, xr); ghb::gauss_legendre(L, ct, wv);
      sd.t_rinv = (int)tp;
      for (int i = 0; i < n0; ++i) {
        ghb::ld r = (ghb::ld)de.lo[0] + ((ghb::ld)de.hi[0] - (ghb::ld)de.lo[0]) * (xr[i] + 1) / 2;
        tab[tp + i] = (double)(1 / r);
      }
      tp += round_up(n0, 2);
      sd.t_ct = (int)tp; for (int j = 0; j < n1; ++j) tab[tp + j] = (double)ct[j]; tp += round_up(n1, 2);
      sd.t_st = (int)tp; for (int j = 0; j < n1; ++j) tab[tp + j] = (double)sqrtl((1 - ct[j]) * (1 + ct[j])); tp += round_up(n1, 2);
      const ghb::ld PI_L = 3.14159265358979323846264338327950288L;
      sd.t_cp = (int)tp; for (int k = 0; k < n2; ++k) tab[tp + k] = (double)cosl(2 * PI_L * k / n2); tp += round_up(n2, 2);
      sd.t_sp = (int)tp; for (int k = 0; k < n2; ++k) tab[tp + k] = (double)sinl(2 * PI_L * k / n2); tp += round_up(n2, 2);
    }
    if (de.kind == GH_CYLINDER) {
      // coordinate tables of a cylindrical shell in the shells' slots: 1 / rho_i; ct = 0, st = 1 (shell_jac's entries then are
      // the cylindrical Jacobian but for d_z); cos / sin phi_k
      d->has_shell = true;
      std::vector<ghb::ld> xr; ghb::cheb_nodes(n0, xr);
      sd.t_rinv = (int)tp;
      for (int i = 0; i < n0; ++i) tab[tp + i] = (double)(1 / ((ghb::ld)de.lo[0] + ((ghb::ld)de.hi[0] - (ghb::ld)de.lo[0]) * (xr[i] + 1) / 2));
      tp += round_up(n0, 2);
      sd.t_ct = (int)tp; for (int j = 0; j < n1; ++j) tab[tp + j] = 0.0; tp += round_up(n1, 2);
      sd.t_st = (int)tp; for (int j = 0; j < n1; ++j) tab[tp + j] = 1.0; tp += round_up(n1, 2);
      const ghb::ld PI_L = 3.14159265358979323846264338327950288L;
      sd.t_cp = (int)tp; for (int k = 0; k < n2; ++k) tab[tp + k] = (double)cosl(2 * PI_L * k / n2); tp += round_up(n2, 2);
      sd.t_sp = (int)tp; for (int k = 0; k < n2; ++k) tab[tp + k] = (double)sinl(2 * PI_L * k / n2); tp += round_up(n2, 2);
    }
    if (de.kind == GH_SHELL && !big_L(de.n[1])) {
      d->has_shell = true;
      const int L = de.n[1];
      if (!Lcache.count(L)) {
        ghb::ShellBasis B; ghb::shell_basis(L, B);
        ShellOff o;
        auto put = [&](const std::vector<ghb::ld>& v) { int at = (int)tp; for (size_t e = 0; e < v.size(); ++e) tab[tp + e] = (double)v[e]; tp += v.size(); return at; };
        // all three operands in DMMA fragment order, zero padded to whole tiles; lane = 4 g + t
        {
          const int np = 2 * L + 2, nq = 2 * L + 1, nt = L + 1;
          // The real DFT is folded about phi = pi (K_ang S0): with h = L+1 = np/2,
          //   even analysis  B[k = 0..h][m = 0..L]      = Fa[m][k]            (cos rows; the weight of k and np-k is the same)
          //   odd  analysis  B[k' = k-1, k = 1..L][m' = m-1, m = 1..L] = Fa[L+m][k]   (sin rows)
          // fragment (k_step, n_tile): element (K index 4 ks + t, N index 8 n + g)
          // all dimensions are those of the shell's class NT = ceil(h / 8) (compile-time constants of K_ang), zero padded
          const int NT = ang_nt_class(L), h = nt;
          std::vector<ghb::ld> FA(shell_fa_doubles(L), 0);
          for (int ks = 0; ks < c_kse1(NT); ++ks) for (int n = 0; n < NT; ++n) for (int lane = 0; lane < 32; ++lane) {
            const int k = ks * 4 + lane % 4, m = n * 8 + lane / 4;
            // the kernel forms U_k + U_{np-k} for every k: k = h is its own mirror, so its weight is halved
            if (k <= h && m <= L) FA[((size_t)ks * NT + n) * 32 + lane] = (k == h ? (ghb::ld)0.5 : (ghb::ld)1) * B.Fa[(size_t)m * np + k];
          }
          const size_t fao = (size_t)c_fa_e(NT);
          for (int ks = 0; ks < c_kso1(NT); ++ks) for (int n = 0; n < NT; ++n) for (int lane = 0; lane < 32; ++lane) {
            const int k = ks * 4 + lane % 4 + 1, m = n * 8 + lane / 4 + 1;
            if (k <= L && m <= L) FA[fao + ((size_t)ks * NT + n) * 32 + lane] = B.Fa[(size_t)(L + m) * np + k];
          }
          o.Fa = put(FA);
          //   even synthesis B[m = 0..L][k = 0..h] = Fs[k][m];   odd synthesis B[m' = m-1][k = 0..h] = Fs[k][L+m], zero at k = 0, h
          std::vector<ghb::ld> FS(shell_fs_doubles(L), 0);
          const int NT3 = c_nt3(NT);
          for (int ks = 0; ks < c_ks3(NT); ++ks) for (int n = 0; n < NT3; ++n) for (int lane = 0; lane < 32; ++lane) {
            const int m = ks * 4 + lane % 4, k = n * 8 + lane / 4;
            if (m <= L && k <= h) FS[((size_t)ks * NT3 + n) * 32 + lane] = B.Fs[(size_t)k * nq + m];
          }
          const size_t fso = (size_t)c_fs_e(NT);
          for (int ks = 0; ks < c_ks3(NT); ++ks) for (int n = 0; n < NT3; ++n) for (int lane = 0; lane < 32; ++lane) {
            const int m = ks * 4 + lane % 4 + 1, k = n * 8 + lane / 4;
            if (m <= L && k >= 1 && k < h) FS[fso + ((size_t)ks * NT3 + n) * 32 + lane] = B.Fs[(size_t)k * nq + L + m];
          }
          o.Fs = put(FS);
          // S2 A operands, folded about the equator (jbar = nt-1-j; K_ang S2 forms p_j = C_j + C_jbar, q_j = C_j - C_jbar, j < hh):
          //   ME (acts on p) = 1/2 (M[r][j] + M[r][jbar]),  MO (acts on q) = 1/2 (M[r][j] - M[r][jbar]),  r, j < hh,
          //   M = Th_m for stacked rows [0, hh) and m Pr_m for rows [hh, 2 hh); the equator node (j = jbar, odd nt) has
          //   p = 2 C_j, q = 0: its ME column is 1/2 M[r][j].   element (row = 8 mt + g, col = 4 ks + t)
          const int hh = (nt + 1) / 2;
          std::vector<ghb::ld> T(shell_t_doubles(L), 0);
          for (int m = 0; m <= L; ++m) for (int ks = 0; ks < NT; ++ks) for (int w = 0; w < 2; ++w) for (int mt = 0; mt < NT; ++mt)
            for (int lane = 0; lane < 32; ++lane) {
              const int row = mt * 8 + lane / 4, j = ks * 4 + lane % 4;
              ghb::ld v = 0;
              if (j < hh && row < 2 * hh) {
                const int r = row < hh ? row : row - hh, jb = nt - 1 - j;
                const std::vector<ghb::ld>& M = row < hh ? B.Th : B.Pr;
                const ghb::ld f = row < hh ? (ghb::ld)1 : (ghb::ld)m;
                const ghb::ld a = M[((size_t)m * nt + r) * nt + j], c = M[((size_t)m * nt + r) * nt + jb];
                if (jb == j) v = w == 0 ? f * a / 2 : (ghb::ld)0;
                else v = f * (w == 0 ? a + c : a - c) / 2;
              }
              T[((((size_t)m * NT + ks) * 2 + w) * NT + mt) * 32 + lane] = v;
            }
          o.T = put(T);
        }
        Lcache[L] = o;
        d->f_L[L] = ftp; ftp += shell_g_doubles(L);
      }
      const ShellOff& o = Lcache[L];
      const int pb = pl.ang_pb[s];
      for (int p0 = 0; p0 < n0; p0 += pb) {
        AngItem it; memset(&it, 0, sizeof it);
        it.off = sd.off; it.L = L; it.plane0 = p0; it.nplanes = std::min(pb, n0 - p0); it.nb_alloc = pb;
        it.m_Fa = o.Fa; it.m_Fs = o.Fs; it.m_T = o.T; it.m_G = (int)d->f_L[L];
        {
          const int NW = (pl.ang_class[s] ? ANG_TPB1 : ANG_TPB0) / 32, MT1 = (it.nplanes * (L + 1) + 7) / 8;
          it.nch3 = (int8_t)ang_best_nch3((L + 1 + 1 + 7) / 8, MT1, NW);
        }
        (pl.ang_class[s] ? ang1 : ang).push_back(it);
      }
    }
    if (de.kind == GH_BLOCK) d->has_block = true;
  }
  ang.insert(ang.end(), ang1.begin(), ang1.end());
  for (int c = 0; c < CHEB_NCLASS; ++c) cheb.insert(cheb.end(), chebc[c].begin(), chebc[c].end());
  std::vector<ChebItem> fcheb;
  for (int a = 0; a < 3; ++a) for (int c = 0; c < CHEB_NCLASS; ++c) fcheb.insert(fcheb.end(), fch[a][c].begin(), fch[a][c].end());
  std::vector<GemmItem> gemm;
  bool gemm_ok = btp == pl.bigtab_doubles;
  for (int l = 0; l < G_NLIST; ++l) { gemm_ok = gemm_ok && (int)glist[l].size() == pl.n_gemm[l]; gemm.insert(gemm.end(), glist[l].begin(), glist[l].end()); }
  gemm_ok = gemm_ok && fbp == pl.fbigtab_doubles && itp == pl.ifctab_doubles && (int)ifci.size() == pl.n_ifc_items && ifc_next == pl.Sf;
  if (tp != pl.table_doubles || (int)cheb.size() != pl.n_cheb_items || (int)ang.size() != pl.n_ang_items || !gemm_ok ||
      (int)fcheb.size() != pl.n_fcheb_items || ftp != pl.table_doubles + pl.ftable_doubles) {
    delete d; return fail(nullptr, GH_ERR_STATE, "internal: plan and build disagree");
  }

  // ---- one-time upload; zero the store so that padding is zero ----
  cudaStream_t st = d->stream;
#define GH_CREATE_CUDA(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) { std::string m = std::string(#call ": ") + cudaGetErrorString(e_); delete d; return fail(nullptr, GH_ERR_CUDA, m); } } while (0)
  GH_CREATE_CUDA(cudaMemsetAsync(d->ws, 0, pl.o_tables, st));
  GH_CREATE_CUDA(cudaMemsetAsync(d->part, 0, pl.total - pl.o_part, st));
  GH_CREATE_CUDA(cudaMemcpyAsync(d->tables, tab.data(), tab.size() * sizeof(double), cudaMemcpyHostToDevice, st));
  GH_CREATE_CUDA(cudaMemcpyAsync(d->subs, d->h_subs.data(), (size_t)n_sub * sizeof(SubDev), cudaMemcpyHostToDevice, st));
  GH_CREATE_CUDA(cudaMemcpyAsync(d->tiles, pl.tile_first.data(), (size_t)(n_sub + 1) * sizeof(int32_t), cudaMemcpyHostToDevice, st));
  if (!cheb.empty()) GH_CREATE_CUDA(cudaMemcpyAsync(d->cheb, cheb.data(), cheb.size() * sizeof(ChebItem), cudaMemcpyHostToDevice, st));
  if (!gemm.empty()) GH_CREATE_CUDA(cudaMemcpyAsync(d->gemm, gemm.data(), gemm.size() * sizeof(GemmItem), cudaMemcpyHostToDevice, st));
  if (!bigtab.empty()) GH_CREATE_CUDA(cudaMemcpyAsync(d->tables + big0, bigtab.data(), bigtab.size() * sizeof(double), cudaMemcpyHostToDevice, st));
  if (!ifctab.empty()) GH_CREATE_CUDA(cudaMemcpyAsync(d->tables + ifc0, ifctab.data(), ifctab.size() * sizeof(double), cudaMemcpyHostToDevice, st));
  if (!ifci.empty()) {
    GH_CREATE_CUDA(cudaMemcpyAsync(d->ifci, ifci.data(), ifci.size() * sizeof(IfcItem), cudaMemcpyHostToDevice, st));
    GH_CREATE_CUDA(cudaFuncSetAttribute(k_face_interp, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_MAX));
  }
  GH_CREATE_CUDA(cudaFuncSetAttribute(k_gemm<GEMM_MB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)gemm_smem_bytes(GEMM_MB)));
  if (!ang.empty()) GH_CREATE_CUDA(cudaMemcpyAsync(d->ang, ang.data(), ang.size() * sizeof(AngItem), cudaMemcpyHostToDevice, st));
  if (!fcheb.empty()) GH_CREATE_CUDA(cudaMemcpyAsync(d->fcheb, fcheb.data(), fcheb.size() * sizeof(ChebItem), cudaMemcpyHostToDevice, st));
  GH_CREATE_CUDA(cudaStreamSynchronize(st));   // host staging vectors die at return
  GH_CREATE_CUDA(cudaFuncSetAttribute(k_rhs<0, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)RHS_SMEM_BYTES));
  GH_CREATE_CUDA(cudaFuncSetAttribute(k_rhs<1, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)RHS_SMEM_BYTES));
  GH_CREATE_CUDA(cudaFuncSetAttribute(k_rhs<2, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)RHS_SMEM_BYTES));
  GH_CREATE_CUDA(cudaFuncSetAttribute(k_rhs<0, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)RHS_SMEM_BYTES));
  GH_CREATE_CUDA(cudaFuncSetAttribute(k_rhs<1, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)RHS_SMEM_BYTES));
  GH_CREATE_CUDA(cudaFuncSetAttribute(k_rhs<2, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)RHS_SMEM_BYTES));
  GH_CREATE_CUDA(cudaFuncSetAttribute(k_rhs<1, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)RHS_SMEM_BYTES_NORMS));
  GH_CREATE_CUDA(cudaFuncSetAttribute(k_rhs<1, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)RHS_SMEM_BYTES_NORMS));
  // the attribute belongs to the FUNCTION, not to this domain: always the class ceiling, so that a later, smaller domain can
  // never lower it under a live domain's launch size
  GH_CREATE_CUDA(cudaFuncSetAttribute(k_ang<ANG_TPB0, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ANG_SMEM_2CTA));
  GH_CREATE_CUDA(cudaFuncSetAttribute(k_ang<ANG_TPB1, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_MAX));
  GH_CREATE_CUDA(cudaFuncSetAttribute(k_ang<ANG_TPB0, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ANG_SMEM_2CTA));
  GH_CREATE_CUDA(cudaFuncSetAttribute(k_ang<ANG_TPB1, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_MAX));
#undef GH_CREATE_CUDA
  *out = d;
  return GH_OK;
}

extern "C" void gh_domain_destroy(gh_domain* d) {
  DeviceGuard guard_(d);
  if (!d) return;
  for (auto& g : d->graphs) if (g.exec) cudaGraphExecDestroy(g.exec);
  for (auto& p : d->pending) { cudaEventDestroy(p.a); cudaEventDestroy(p.b); }
  for (auto e : d->pool) cudaEventDestroy(e);
  delete d;
}

extern "C" gh_status gh_domain_layout(const gh_domain* d, int64_t* n_points, int64_t* comp_stride, int64_t* offsets) {
  if (!d) return GH_ERR_ARG;
  if (n_points) *n_points = d->pl.P;
  if (comp_stride) *comp_stride = d->pl.S;
  if (offsets) for (int s = 0; s <= d->pl.n_sub; ++s) offsets[s] = d->pl.offsets[s];
  return GH_OK;
}

extern "C" gh_status gh_domain_coords(const gh_domain* cd, double* xyz, int on_device) {
  DeviceGuard guard_(cd);
  gh_domain* d = const_cast<gh_domain*>(cd);
  if (!d || !xyz) return fail(d, GH_ERR_ARG, "NULL argument");
  const int64_t S = d->pl.S;
  std::vector<double> h((size_t)3 * S, 0.0);
  const ghb::ld PI_L = 3.14159265358979323846264338327950288L;
  for (int s = 0; s < d->pl.n_sub; ++s) {
    const gh_subdomain_desc& de = d->pl.descs[s];
    int n0, n1, n2; sub_dims(de, n0, n1, n2);
    const int64_t off = d->pl.offsets[s];
    if (de.kind == GH_SHELL) {
      std::vector<ghb::ld> xr, ct, wv; ghb::cheb_nodes(n0, xr); ghb::gauss_legendre(de.n[1], ct, wv);
      for (int i = 0; i < n0; ++i) {
        const ghb::ld r = (ghb::ld)de.lo[0] + ((ghb::ld)de.hi[0] - (ghb::ld)de.lo[0]) * (xr[i] + 1) / 2;
        for (int j = 0; j < n1; ++j) {
          const ghb::ld st = sqrtl((1 - ct[j]) * (1 + ct[j]));
          for (int k = 0; k < n2; ++k) {
            const ghb::ld ph = 2 * PI_L * k / n2;
            const int64_t p = off + ((int64_t)i * n1 + j) * n2 + k;
            h[p] = (double)((ghb::ld)de.center[0] + r * st * cosl(ph));
            h[S + p] = (double)((ghb::ld)de.center[1] + r * st * sinl(ph));
            h[2 * S + p] = (double)((ghb::ld)de.center[2] + r * ct[j]);
          }
        }
      }
    } else if (de.kind == GH_CYLINDER) {
      std::vector<ghb::ld> xr, xz; ghb::cheb_nodes(n0, xr); ghb::cheb_nodes(n1, xz);
      for (int i = 0; i < n0; ++i) {
        const ghb::ld rho = (ghb::ld)de.lo[0] + ((ghb::ld)de.hi[0] - (ghb::ld)de.lo[0]) * (xr[i] + 1) / 2;
        for (int j = 0; j < n1; ++j) {
          const ghb::ld z = (ghb::ld)de.lo[1] + ((ghb::ld)de.hi[1] - (ghb::ld)de.lo[1]) * (xz[j] + 1) / 2;
          for (int k = 0; k < n2; ++k) {
            const ghb::ld ph = 2 * PI_L * k / n2;
            const int64_t p = off + ((int64_t)i * n1 + j) * n2 + k;
            h[p] = (double)((ghb::ld)de.center[0] + rho * cosl(ph));
            h[S + p] = (double)((ghb::ld)de.center[1] + rho * sinl(ph));
            h[2 * S + p] = (double)((ghb::ld)de.center[2] + z);
          }
        }
      }
    } else {
      std::vector<ghb::ld> x[3];
      for (int a = 0; a < 3; ++a) ghb::cheb_nodes(de.n[a], x[a]);
      for (int i = 0; i < n0; ++i) for (int j = 0; j < n1; ++j) for (int k = 0; k < n2; ++k) {
        const int64_t p = off + ((int64_t)i * n1 + j) * n2 + k; const int id[3] = {i, j, k};
        for (int a = 0; a < 3; ++a)
          h[(size_t)a * S + p] = (double)((ghb::ld)de.lo[a] + ((ghb::ld)de.hi[a] - (ghb::ld)de.lo[a]) * (x[a][id[a]] + 1) / 2);
      }
    }
  }
  if (on_device) {
    GH_CUDA(d, cudaMemcpyAsync(xyz, h.data(), h.size() * sizeof(double), cudaMemcpyHostToDevice, d->stream));
    GH_CUDA(d, cudaStreamSynchronize(d->stream));
  } else {
    memcpy(xyz, h.data(), h.size() * sizeof(double));
  }
  return GH_OK;
}

// ------------------------------------------------------------------------------------------------------
// launch helpers
// ------------------------------------------------------------------------------------------------------
namespace {

gh_status check_flag(gh_domain* d) {   // stream must be synchronised by the caller's preceding copy
  int h = 0;
  GH_CUDA(d, cudaMemcpyAsync(&h, d->flag, sizeof(int), cudaMemcpyDeviceToHost, d->stream));
  GH_CUDA(d, cudaStreamSynchronize(d->stream));
  if (h) {
    cudaMemsetAsync(d->flag, 0, sizeof(int), d->stream);
    return fail(d, GH_ERR_SINGULAR, "non-physical data on the device: det g_ij <= 0 or lapse^2 <= 0");
  }
  return GH_OK;
}

// A2 + A3: logical derivatives of `ncomp` components of `in` into out[3][ncomp][S]
// (blocks: d/dx, d/dy, d/dz already Cartesian; shells: d/dr, d/dtheta, d/dphi).
// one K_cheb launch over the n items of register-tile class c (N <= 24: 3 x 6 tiles of D; N <= 32: 4 x 8; N <= 48: 6 x 12; N <= 64: 8 x 16)
void launch_cheb_class(gh_domain* d, int prof_cls, int c, const ChebItem* items, int n, int gy, const double* in, double* out,
                       int nrun, const CompMap& cm) {
  if (!n) return;
  const Plan& pl = d->pl;
  ProfScope ps(d, prof_cls);
  const dim3 grid(n, gy);
  if (c == 0) k_cheb<CHEB_TPB, 3, 6, CHEB_NTW><<<grid, CHEB_TPB, pl.cheb_smem, d->stream>>>(items, d->tables, in, out, pl.S, nrun, cm);
  else if (c == 1) k_cheb<CHEB_TPB, 4, 8, CHEB_NTW><<<grid, CHEB_TPB, pl.cheb_smem, d->stream>>>(items, d->tables, in, out, pl.S, nrun, cm);
  else if (c == 2) k_cheb<CHEB_TPB, 6, 12, CHEB_NTW><<<grid, CHEB_TPB, pl.cheb_smem, d->stream>>>(items, d->tables, in, out, pl.S, nrun, cm);
  else k_cheb<CHEB_TPB, 8, 16, CHEB_NTW><<<grid, CHEB_TPB, pl.cheb_smem, d->stream>>>(items, d->tables, in, out, pl.S, nrun, cm);
}

// one K_gemm launch over launch list l (the items of the lists lie one after another in d->gemm)
void launch_gemm_list(gh_domain* d, int prof_cls, int l, const double* in, double* out, int nrun, const CompMap& cm) {
  const Plan& pl = d->pl;
  if (!pl.n_gemm[l]) return;
  int first = 0;
  for (int k = 0; k < l; ++k) first += pl.n_gemm[k];
  // components one CTA walks over (one CTA per SM is resident): the divisor w of nrun with the best modelled efficiency
  //   (fill of the last wave: CTAs / (waves x SMs))  x  (pipeline fill: w stages-per-component / (the same + 2 stages of ramp)).
  // "As many as still leave two CTAs per SM" put 80^3 on 300 CTAs = 2.03 waves (a third, nearly empty wave: 68 %).
  int gw = 1;
  {
    const double per = d->gemm_stages[l] / pl.n_gemm[l];
    double best = -1.0;
    for (int w = 1; w <= nrun && w <= 25; ++w) {
      if (nrun % w) continue;
      const int64_t ctas = (int64_t)pl.n_gemm[l] * (nrun / w), waves = (ctas + d->n_sm - 1) / d->n_sm;
      const double eff = (double)ctas / (double)(waves * d->n_sm) * (w * per / (w * per + 2.0));
      if (eff > best) { best = eff; gw = w; }
    }
  }
  ProfScope ps(d, prof_cls);
  k_gemm<GEMM_MB><<<dim3(pl.n_gemm[l], nrun / gw), GEMM_TPB, gemm_smem_bytes(GEMM_MB), d->stream>>>(d->gemm + first, d->tables, in, out, pl.S, nrun, cm);
}

gh_status launch_derivs(gh_domain* d, const double* in, double* out, int ncomp, int skip_lo = 0, int skip_n = 0) {
  const Plan& pl = d->pl;
  const CompMap cm{ncomp, skip_lo, skip_n};        // `in` / `out` have ncomp components, of which skip_n are left out
  const int nrun = ncomp - skip_n;
  // each K_cheb CTA walks over nrun / cheb_gy components (amortises its launch and matrix load)
  // ... but small domains need the CTAs more than the amortisation: keep at least ~4 CTAs per SM in the grid
  // large subdomains: the K_gemm lists in order (S1, S2, S3 theta, S3 phi of the large shells, then the large Chebyshev axes -
  // the radial one writes slot 0, which S2 / S3 used as a coefficient buffer)
  if (pl.has_big)
    for (int l = 0; l < G_NDERIV; ++l) launch_gemm_list(d, l == G_CHEB ? GH_K_CHEB : GH_K_SHELL_ANG, l, in, out, nrun, cm);
  int walk = 1;
  for (int w = CHEB_COMP_WALK; w >= 1; --w)
    if (nrun % w == 0 && (w == 1 || (int64_t)pl.n_cheb_items * (nrun / w) >= 4 * d->n_sm)) { walk = w; break; }
  const int cheb_gy = nrun / walk;
  for (int c = 0, first = 0; c < CHEB_NCLASS; first += pl.n_cheb_class[c], ++c)
    launch_cheb_class(d, GH_K_CHEB, c, d->cheb + first, pl.n_cheb_class[c], cheb_gy, in, out, nrun, cm);
  for (int cls = 0, first = 0; cls < 2; first += pl.n_ang_class[cls], ++cls) {
    if (!pl.n_ang_class[cls]) continue;
    ProfScope ps(d, GH_K_SHELL_ANG);
    if (cls == 0)
      k_ang<ANG_TPB0, false><<<dim3(pl.n_ang_class[0], nrun), ANG_TPB0, pl.ang_smem[0], d->stream>>>(d->ang + first, d->tables, in, out, pl.S, cm);
    else
      k_ang<ANG_TPB1, false><<<dim3(pl.n_ang_class[1], nrun), ANG_TPB1, pl.ang_smem[1], d->stream>>>(d->ang + first, d->tables, in, out, pl.S, cm);
  }
  GH_CUDA(d, cudaGetLastError());
  return GH_OK;
}

// A2-A6 on state `u`; rk_mode 0: d_t u into `out`; 1 / 2: the fused RK stage (A7)  out = a u0 + b (u + dt d_t u)
// (mode 1: a = 0, u0 unused).  `out` may alias u or u0.
gh_status launch_rhs(gh_domain* d, const double* u, double* out, int rk_mode = 0, const double* u0 = nullptr, double a = 0.0,
                     double b = 1.0, double dt = 0.0, bool norms = false) {
  gh_status st = launch_derivs(d, u, d->du, NCOMP);
  if (st != GH_OK) return st;
  if (d->has_map) {             // dual frame: the derivative scratch becomes inertial-frame (K_rhs applies the spherical Jacobian itself)
    ProfScope ps(d, GH_K_OTHER);
    k_map_pre<<<d->pl.n_tiles, TILE_PTS, 0, d->stream>>>(d->subs, d->tiles, d->pl.n_sub, d->tables, d->mapJ, d->du, d->pl.S, NCOMP);
  }
  // ... and after the fused kernel: + coef v^i d_i u, the time derivative at the fixed grid points
  auto map_post = [&]() {
    if (!d->has_map) return;
    ProfScope ps(d, GH_K_OTHER);
    k_map_post<<<d->pl.n_tiles, TILE_PTS, 0, d->stream>>>(d->subs, d->tiles, d->pl.n_sub, d->tables, d->mapv, d->du, out, d->pl.S, rk_mode == 0 ? 1.0 : b * dt);
  };
  if (d->pl.n_ifc_items) {      // the neighbours' face states of this stage's input, on the grids of the shells that read them
    ProfScope ps(d, GH_K_OTHER);
    k_face_interp<<<dim3(d->pl.n_ifc_items, NCOMP), 256, d->pl.ifc_smem, d->stream>>>(d->ifci, d->tables, u, d->ifc, d->pl.S, d->pl.Sf);
  }
  if (norms) {      // A8 as the epilogue of stage 1 (rk_mode 1 only): per-tile partials, folded per subdomain like K_con's
    const RkArgs rk{u0, a, b, dt};
    const int grid = d->pl.n_tiles;
    {
      ProfScope ps(d, GH_K_RHS);
      if (d->has_char) k_rhs<1, true, true><<<grid, TILE_PTS, RHS_SMEM_BYTES_NORMS, d->stream>>>(d->subs, d->tiles, d->pl.n_sub, d->tables, u, d->du, d->H, d->dH, out, rk, d->pl.S, d->flag, d->part, d->ifc, d->pl.Sf);
      else k_rhs<1, false, true><<<grid, TILE_PTS, RHS_SMEM_BYTES_NORMS, d->stream>>>(d->subs, d->tiles, d->pl.n_sub, d->tables, u, d->du, d->H, d->dH, out, rk, d->pl.S, d->flag, d->part);
    }
    {
      ProfScope ps(d, GH_K_REDUCE);
      k_con_reduce<<<d->pl.n_sub, 32, 0, d->stream>>>(d->tiles, d->part, d->persub);
    }
    map_post();
    GH_CUDA(d, cudaGetLastError());
    return GH_OK;
  }
  {
    ProfScope ps(d, GH_K_RHS);
    const RkArgs rk{u0, a, b, dt};
    const int grid = d->pl.n_tiles;
#define GH_RHS_LAUNCH(M, C) k_rhs<M, C><<<grid, TILE_PTS, RHS_SMEM_BYTES, d->stream>>>(d->subs, d->tiles, d->pl.n_sub, d->tables, u, d->du, d->H, d->dH, out, rk, d->pl.S, d->flag, nullptr, d->ifc, d->pl.Sf)
    if (d->has_char) { if (rk_mode == 0) GH_RHS_LAUNCH(0, true); else if (rk_mode == 1) GH_RHS_LAUNCH(1, true); else GH_RHS_LAUNCH(2, true); }
    else { if (rk_mode == 0) GH_RHS_LAUNCH(0, false); else if (rk_mode == 1) GH_RHS_LAUNCH(1, false); else GH_RHS_LAUNCH(2, false); }
#undef GH_RHS_LAUNCH
  }
  map_post();
  GH_CUDA(d, cudaGetLastError());
  return GH_OK;
}

gh_status launch_jac(gh_domain* d, double* g, int ncomp) {
  if (!d->has_shell) return GH_OK;
  ProfScope ps(d, GH_K_JAC);
  k_jac<<<d->pl.n_tiles, TILE_PTS, 0, d->stream>>>(d->subs, d->tiles, d->pl.n_sub, d->tables, g, d->pl.S, ncomp);
  GH_CUDA(d, cudaGetLastError());
  return GH_OK;
}

}  // namespace

namespace {
// Run `body` (kernel launches only) through the CUDA graph slot `kind`: captured on first use and whenever its key changes,
// then replayed as one launch.  Falls back to plain enqueueing on the legacy default stream, while profiling, or when switched off.
template <class F>
gh_status run_graphed(gh_domain* d, int kind, double dt, const void* out, F body) {
  if (d->opt[GH_OPT_NO_GRAPH] || d->prof || d->stream == nullptr) return body();
  gh_domain::StepGraph& g = d->graphs[kind];
  const int oop = d->opt[GH_OPT_RK_OUT_OF_PLACE];
  if (!g.exec || g.dt != dt || g.ua != d->ua || g.ub != d->ub || g.out != out || g.oop != oop || g.map != (int)d->has_map) {
    if (g.exec) { cudaGraphExecDestroy(g.exec); g.exec = nullptr; }
    const int64_t l0 = d->launches;
    GH_CUDA(d, cudaStreamBeginCapture(d->stream, cudaStreamCaptureModeThreadLocal));
    const gh_status st = body();
    cudaGraph_t graph = nullptr;
    const cudaError_t e = cudaStreamEndCapture(d->stream, &graph);
    g.nlaunch = d->launches - l0; d->launches = l0;
    if (st != GH_OK) { if (graph) cudaGraphDestroy(graph); return st; }
    if (e != cudaSuccess) return fail(d, GH_ERR_CUDA, std::string("cudaStreamEndCapture: ") + cudaGetErrorString(e));
    const cudaError_t ei = cudaGraphInstantiate(&g.exec, graph, 0);
    cudaGraphDestroy(graph);
    if (ei != cudaSuccess) { g.exec = nullptr; return fail(d, GH_ERR_CUDA, std::string("cudaGraphInstantiate: ") + cudaGetErrorString(ei)); }
    g.dt = dt; g.ua = d->ua; g.ub = d->ub; g.out = out; g.oop = oop; g.map = (int)d->has_map;
  }
  GH_CUDA(d, cudaGraphLaunch(g.exec, d->stream));
  d->launches += g.nlaunch;
  return GH_OK;
}
}  // namespace

// ------------------------------------------------------------------------------------------------------
// state in / out
// ------------------------------------------------------------------------------------------------------
extern "C" gh_status gh_set_fields(gh_domain* d, const double* u, int on_device, double t) {
  DeviceGuard guard_(d);
  if (!d || !u) return fail(d, GH_ERR_ARG, "NULL argument");
  const size_t bytes = (size_t)NCOMP * d->pl.S * sizeof(double);
  GH_CUDA(d, cudaMemcpyAsync(d->ua, u, bytes, on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, d->stream));
  if (!on_device) GH_CUDA(d, cudaStreamSynchronize(d->stream));
  d->t = t; d->has_fields = true; d->dp_fsal = false;
  return GH_OK;
}

extern "C" gh_status gh_get_fields(const gh_domain* cd, double* u, int on_device, double* t) {
  DeviceGuard guard_(cd);
  gh_domain* d = const_cast<gh_domain*>(cd);
  if (!d || !u) return fail(d, GH_ERR_ARG, "NULL argument");
  if (!d->has_fields) return fail(d, GH_ERR_STATE, "gh_get_fields before gh_set_fields");
  const size_t bytes = (size_t)NCOMP * d->pl.S * sizeof(double);
  GH_CUDA(d, cudaMemcpyAsync(u, d->ua, bytes, on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, d->stream));
  if (t) *t = d->t;
  if (!on_device) return check_flag(d);
  return GH_OK;
}

extern "C" gh_status gh_set_gauge_source(gh_domain* d, const double* H, const double* dH, int on_device) {
  DeviceGuard guard_(d);
  if (!d || !H) return fail(d, GH_ERR_ARG, "NULL argument");
  const size_t comp = (size_t)d->pl.S * sizeof(double);
  const cudaMemcpyKind kind = on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
  d->dp_fsal = false;
  GH_CUDA(d, cudaMemcpyAsync(d->H, H, 4 * comp, kind, d->stream));
  if (dH) {
    GH_CUDA(d, cudaMemcpyAsync(d->dH, dH, 12 * comp, kind, d->stream));
  } else {
    gh_status st = launch_derivs(d, d->H, d->dH, 4);
    if (st != GH_OK) return st;
    st = launch_jac(d, d->dH, 4);
    if (st != GH_OK) return st;
  }
  if (!on_device) GH_CUDA(d, cudaStreamSynchronize(d->stream));
  return GH_OK;
}

// ------------------------------------------------------------------------------------------------------
// compute entry points
// ------------------------------------------------------------------------------------------------------
extern "C" gh_status gh_rhs(gh_domain* d, double* dtu, int on_device) {
  DeviceGuard guard_(d);
  if (!d || !dtu) return fail(d, GH_ERR_ARG, "NULL argument");
  if (!d->has_fields) return fail(d, GH_ERR_STATE, "gh_rhs before gh_set_fields");
  if (on_device) return run_graphed(d, 2, 0.0, dtu, [&] { return launch_rhs(d, d->ua, dtu); });
  gh_status st = launch_rhs(d, d->ua, d->k);
  if (st != GH_OK) return st;
  GH_CUDA(d, cudaMemcpyAsync(dtu, d->k, (size_t)NCOMP * d->pl.S * sizeof(double), cudaMemcpyDeviceToHost, d->stream));
  return check_flag(d);
}

extern "C" gh_status gh_gradient(gh_domain* d, double* du, int on_device) {
  DeviceGuard guard_(d);
  if (!d || !du) return fail(d, GH_ERR_ARG, "NULL argument");
  if (!d->has_fields) return fail(d, GH_ERR_STATE, "gh_gradient before gh_set_fields");
  if (on_device && ((uintptr_t)du & 15) != 0) return fail(d, GH_ERR_ARG, "gh_gradient: a DEVICE du must be 16-byte aligned (the derivative kernels store double2)");
  double* tgt = on_device ? du : d->du;
  gh_status st = launch_derivs(d, d->ua, tgt, NCOMP);
  if (st != GH_OK) return st;
  st = launch_jac(d, tgt, NCOMP);
  if (st != GH_OK) return st;
  if (!on_device) {
    GH_CUDA(d, cudaMemcpyAsync(du, d->du, (size_t)3 * NCOMP * d->pl.S * sizeof(double), cudaMemcpyDeviceToHost, d->stream));
    GH_CUDA(d, cudaStreamSynchronize(d->stream));
  }
  return GH_OK;
}

namespace {
// the three Shu-Osher stages; norms: the constraint partials of the input state come out of stage 1 (into d->persub)
gh_status rk3_stages(gh_domain* d, double dt, bool norms) {
  gh_status st;
  if (d->has_ifc || d->opt[GH_OPT_RK_OUT_OF_PLACE]) {
    // INTERFACE faces read the neighbour's face state from the stage input, so no stage may run in place: ua -> ub -> k -> ua
    if ((st = launch_rhs(d, d->ua, d->ub, 1, nullptr, 0.0, 1.0, dt, norms)) != GH_OK) return st;
    if ((st = launch_rhs(d, d->ub, d->k, 2, d->ua, 0.75, 0.25, dt)) != GH_OK) return st;
    if ((st = launch_rhs(d, d->k, d->ua, 2, d->ua, 1.0 / 3.0, 2.0 / 3.0, dt)) != GH_OK) return st;
    return GH_OK;
  }
  // the stage update (A7) is the epilogue of the fused RHS kernel: d_t u never goes to memory
  // u1 = u0 + dt k(u0)                      (ua -> ub)
  if ((st = launch_rhs(d, d->ua, d->ub, 1, nullptr, 0.0, 1.0, dt, norms)) != GH_OK) return st;
  // u2 = 3/4 u0 + 1/4 (u1 + dt k(u1))       (ub -> ub, in place)
  if ((st = launch_rhs(d, d->ub, d->ub, 2, d->ua, 0.75, 0.25, dt)) != GH_OK) return st;
  // u_new = 1/3 u0 + 2/3 (u2 + dt k(u2))    (ub -> ua, over u0)
  if ((st = launch_rhs(d, d->ub, d->ua, 2, d->ua, 1.0 / 3.0, 2.0 / 3.0, dt)) != GH_OK) return st;
  return GH_OK;
}

// per-subdomain {3 sums, 3 maxima} (host copy of d->persub) -> out[3][2], per_sub[n_sub][3][2]
void finish_norms(const Plan& pl, const std::vector<double>& h, double* out, double* per_sub) {
  static const double ncomp[3] = {4.0, 30.0, 30.0};
  double sum[3] = {0, 0, 0}, mx[3] = {0, 0, 0};
  for (int s = 0; s < pl.n_sub; ++s) {
    int n0, n1, n2; sub_dims(pl.descs[s], n0, n1, n2);
    const double Ps = (double)n0 * n1 * n2;
    for (int q = 0; q < 3; ++q) {
      sum[q] += h[(size_t)s * 6 + q];
      { const double v = h[(size_t)s * 6 + 3 + q]; if (v != v || v > mx[q]) mx[q] = v; }     // NaN propagates
      if (per_sub) {
        per_sub[(size_t)s * 6 + 2 * q] = std::sqrt(h[(size_t)s * 6 + q] / (Ps * ncomp[q]));
        per_sub[(size_t)s * 6 + 2 * q + 1] = h[(size_t)s * 6 + 3 + q];
      }
    }
  }
  for (int q = 0; q < 3; ++q) { out[2 * q] = std::sqrt(sum[q] / ((double)pl.P * ncomp[q])); out[2 * q + 1] = mx[q]; }
}
}  // namespace

extern "C" gh_status gh_rk_step(gh_domain* d, double dt) {
  DeviceGuard guard_(d);
  if (!d) return GH_ERR_ARG;
  if (!d->has_fields) return fail(d, GH_ERR_STATE, "gh_rk_step before gh_set_fields");
  if (!std::isfinite(dt)) return fail(d, GH_ERR_ARG, "dt is not finite");
  gh_status st = run_graphed(d, 0, dt, nullptr, [&] { return rk3_stages(d, dt, false); });
  if (st != GH_OK) return st;
  d->t += dt; d->dp_fsal = false;
  return GH_OK;
}

extern "C" gh_status gh_rk_step_norms(gh_domain* d, double dt, double* out, double* per_sub) {
  DeviceGuard guard_(d);
  if (!d || !out) return fail(d, GH_ERR_ARG, "NULL argument");
  if (!d->has_fields) return fail(d, GH_ERR_STATE, "gh_rk_step_norms before gh_set_fields");
  if (!std::isfinite(dt)) return fail(d, GH_ERR_ARG, "dt is not finite");
  gh_status st = run_graphed(d, 1, dt, nullptr, [&] { return rk3_stages(d, dt, true); });
  if (st != GH_OK) return st;
  d->t += dt; d->dp_fsal = false;
  // d->persub was written by stage 1 and nothing later in the step touches it: one copy and one synchronisation at the end
  std::vector<double> h((size_t)d->pl.n_sub * 6);
  GH_CUDA(d, cudaMemcpyAsync(h.data(), d->persub, h.size() * sizeof(double), cudaMemcpyDeviceToHost, d->stream));
  st = check_flag(d);   // synchronises
  if (st != GH_OK) return st;
  finish_norms(d->pl, h, out, per_sub);
  return GH_OK;
}

extern "C" gh_status gh_constraint_norms(gh_domain* d, double* out, double* per_sub) {
  DeviceGuard guard_(d);
  if (!d || !out) return fail(d, GH_ERR_ARG, "NULL argument");
  if (!d->has_fields) return fail(d, GH_ERR_STATE, "gh_constraint_norms before gh_set_fields");
  const Plan& pl = d->pl;
  gh_status st = launch_derivs(d, d->ua, d->du, NCOMP, 10, 10);   // the constraints need no derivative of Pi (components 10..19)
  if (st != GH_OK) return st;
  if (d->has_map) {             // dual frame: C_iab and C_ijab are built from inertial-frame derivatives
    ProfScope ps(d, GH_K_OTHER);
    k_map_pre<<<pl.n_tiles, TILE_PTS, 0, d->stream>>>(d->subs, d->tiles, pl.n_sub, d->tables, d->mapJ, d->du, pl.S, NCOMP);
  }
  {
    ProfScope ps(d, GH_K_CONSTRAINTS);
    k_con<<<pl.n_tiles, TILE_PTS, 0, d->stream>>>(d->subs, d->tiles, pl.n_sub, d->tables, d->ua, d->du, d->H, pl.S, d->flag, d->part);
  }
  {
    ProfScope ps(d, GH_K_REDUCE);
    k_con_reduce<<<pl.n_sub, 32, 0, d->stream>>>(d->tiles, d->part, d->persub);
  }
  GH_CUDA(d, cudaGetLastError());
  std::vector<double> h((size_t)pl.n_sub * 6);
  GH_CUDA(d, cudaMemcpyAsync(h.data(), d->persub, h.size() * sizeof(double), cudaMemcpyDeviceToHost, d->stream));
  st = check_flag(d);   // synchronises
  if (st != GH_OK) return st;
  finish_norms(pl, h, out, per_sub);
  return GH_OK;
}

// ------------------------------------------------------------------------------------------------------
// gh_constraint_norms_static: gh_constraint_norms for callers that may not allocate (CUDA graph capture around them, tight
// serving loops, harnesses that forbid cudaMalloc).  The reduction scratch of K_con / K_con_reduce - per-tile partials
// [n_tiles][6], per-subdomain sums [n_sub][6] and the domain's totals [6] - does not come from any workspace but from ONE
// file-scope device array of fixed size (GH_STATIC_SCRATCH_BYTES = 3.2 MB; every GPU that loads the library holds it until the
// process exits).  In host code `g_static_scratch` is only a stand-in for the symbol, not a device address: the address is
// taken once per device with cudaGetSymbolAddress (that device current) and passed to the kernels; K_con_final_static, being
// device code of this file, names the array directly.  No cudaMalloc / cudaFree / event or graph creation / allocating library
// call on this path, and no host-side heap use either: the totals are folded on the device (one thread, subdomains in order:
// the same additions in the same order as the host fold of gh_constraint_norms, so the results are bit-identical) and land in
// a stack buffer; the per-subdomain values go straight into the caller's array.
// The array is shared by every call in the process and keeps the last call's contents.  Nothing has to start at zero: every
// value a call reads (its n_tiles partials, its n_sub sums, the 6 totals) is written earlier in the same call, and nothing
// beyond them is read.  Calls that overlap on the GPU (two domains on different streams, two host threads) RACE on it:
// serialise them.
// ------------------------------------------------------------------------------------------------------
namespace {
constexpr size_t STATIC_PART = (size_t)GH_STATIC_MAX_TILES * 6, STATIC_SUB = (size_t)GH_STATIC_MAX_SUBS * 6, STATIC_TOT = 8;
static_assert((STATIC_PART + STATIC_SUB + STATIC_TOT) * sizeof(double) == GH_STATIC_SCRATCH_BYTES, "gh.h states the size of the static scratch");
static __device__ __align__(256) double g_static_scratch[STATIC_PART + STATIC_SUB + STATIC_TOT];

// totals [6] from the per-subdomain sums, subdomains in order (sums added, maxima NaN-propagating, exactly like finish_norms)
__global__ void k_con_final_static(int n_sub) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  const double* ps = g_static_scratch + STATIC_PART;
  double* tot = g_static_scratch + STATIC_PART + STATIC_SUB;
  for (int q = 0; q < 3; ++q) {
    double sum = 0.0, mx = 0.0;
    for (int s = 0; s < n_sub; ++s) {
      sum += ps[(size_t)s * 6 + q];
      const double v = ps[(size_t)s * 6 + 3 + q];
      if (v != v || v > mx) mx = v;
    }
    tot[q] = sum; tot[3 + q] = mx;
  }
}

constexpr int STATIC_MAX_DEV = 64;
std::mutex g_static_mu;
double* g_static_ptr[STATIC_MAX_DEV] = {};      // device address of g_static_scratch per device ordinal, resolved once

gh_status static_scratch_ptr(gh_domain* d, double** out) {      // the domain's device is current (DeviceGuard of the caller)
  if (d->device < 0 || d->device >= STATIC_MAX_DEV) return fail(d, GH_ERR_ARG, "gh_constraint_norms_static: device ordinal beyond 63");
  std::lock_guard<std::mutex> lk(g_static_mu);
  if (!g_static_ptr[d->device]) {
    void* ptr = nullptr;
    GH_CUDA(d, cudaGetSymbolAddress(&ptr, g_static_scratch));
    g_static_ptr[d->device] = static_cast<double*>(ptr);
  }
  *out = g_static_ptr[d->device];
  return GH_OK;
}
}  // namespace

extern "C" gh_status gh_constraint_norms_static(gh_domain* d, double* out, double* per_sub) {
  DeviceGuard guard_(d);
  if (!d || !out) return fail(d, GH_ERR_ARG, "NULL argument");
  if (!d->has_fields) return fail(d, GH_ERR_STATE, "gh_constraint_norms_static before gh_set_fields");
  const Plan& pl = d->pl;
  if (pl.n_tiles > GH_STATIC_MAX_TILES || pl.n_sub > GH_STATIC_MAX_SUBS) {
    char buf[256];
    snprintf(buf, sizeof buf, "gh_constraint_norms_static: the domain has %d tiles of %d points and %d subdomains; the static scratch holds "
             "at most %d tiles (%lld points) and %d subdomains - use gh_constraint_norms", pl.n_tiles, TILE_PTS, pl.n_sub,
             GH_STATIC_MAX_TILES, (long long)GH_STATIC_MAX_TILES * TILE_PTS, GH_STATIC_MAX_SUBS);
    return fail(d, GH_ERR_ARG, buf);
  }
  double* scratch = nullptr;
  gh_status st = static_scratch_ptr(d, &scratch);
  if (st != GH_OK) return st;
  double* part = scratch;
  double* persub = scratch + STATIC_PART;
  const double* tot = scratch + STATIC_PART + STATIC_SUB;
  const bool prof = d->prof;
  d->prof = false;                      // per-launch profiling would take events from a pool that may have to create them
  st = launch_derivs(d, d->ua, d->du, NCOMP, 10, 10);
  d->prof = prof;
  if (st != GH_OK) return st;
  if (d->has_map) k_map_pre<<<pl.n_tiles, TILE_PTS, 0, d->stream>>>(d->subs, d->tiles, pl.n_sub, d->tables, d->mapJ, d->du, pl.S, NCOMP);
  k_con<<<pl.n_tiles, TILE_PTS, 0, d->stream>>>(d->subs, d->tiles, pl.n_sub, d->tables, d->ua, d->du, d->H, pl.S, d->flag, part);
  k_con_reduce<<<pl.n_sub, 32, 0, d->stream>>>(d->tiles, part, persub);
  k_con_final_static<<<1, 32, 0, d->stream>>>(pl.n_sub);
  d->launches += 3 + (d->has_map ? 1 : 0);
  GH_CUDA(d, cudaGetLastError());
  double h[6];
  GH_CUDA(d, cudaMemcpyAsync(h, tot, sizeof h, cudaMemcpyDeviceToHost, d->stream));
  if (per_sub) GH_CUDA(d, cudaMemcpyAsync(per_sub, persub, (size_t)pl.n_sub * 6 * sizeof(double), cudaMemcpyDeviceToHost, d->stream));
  st = check_flag(d);   // synchronises
  if (st != GH_OK) return st;
  static const double ncomp[3] = {4.0, 30.0, 30.0};
  for (int q = 0; q < 3; ++q) { out[2 * q] = std::sqrt(h[q] / ((double)pl.P * ncomp[q])); out[2 * q + 1] = h[3 + q]; }
  if (per_sub)      // raw [s] = {sum0, sum1, sum2, max0, max1, max2} -> {rms0, max0, rms1, max1, rms2, max2}, in place
    for (int s = 0; s < pl.n_sub; ++s) {
      int n0, n1, n2; sub_dims(pl.descs[s], n0, n1, n2);
      const double Ps = (double)n0 * n1 * n2;
      double r[6];
      for (int q = 0; q < 6; ++q) r[q] = per_sub[(size_t)s * 6 + q];
      for (int q = 0; q < 3; ++q) { per_sub[(size_t)s * 6 + 2 * q] = std::sqrt(r[q] / (Ps * ncomp[q])); per_sub[(size_t)s * 6 + 2 * q + 1] = r[3 + q]; }
    }
  return GH_OK;
}

// ------------------------------------------------------------------------------------------------------
// spectral filter (NEXT-1): the same kernels with filter matrices in place of differentiation matrices
// ------------------------------------------------------------------------------------------------------
namespace {
bool filter_sigma(const gh_filter_desc* f, int kmax, std::vector<ghb::ld>& sg) {
  sg.assign(kmax + 1, 1);
  if (!f || f->kind == GH_FILTER_NONE) return true;
  if (f->kind == GH_FILTER_HEAVISIDE) {
    if (f->cut < 0) return false;
    for (int k = 0; k <= kmax; ++k) sg[k] = (k <= kmax - f->cut) ? 1 : 0;
    return true;
  }
  if (f->kind == GH_FILTER_EXP) {
    if (f->p < 1 || !std::isfinite(f->alpha) || f->alpha < 0) return false;
    for (int k = 0; k <= kmax; ++k) sg[k] = kmax > 0 ? expl(-(ghb::ld)f->alpha * powl((ghb::ld)k / (ghb::ld)kmax, 2 * f->p)) : (ghb::ld)1;
    return true;
  }
  return false;
}
}  // namespace

extern "C" gh_status gh_filter_sigma(const gh_filter_desc* f, int32_t kmax, double* sigma) {
  std::vector<ghb::ld> sg;
  if (!sigma || kmax < 0 || !filter_sigma(f, kmax, sg)) return GH_ERR_ARG;
  for (int k = 0; k <= kmax; ++k) sigma[k] = (double)sg[k];
  return GH_OK;
}

extern "C" gh_status gh_set_filter(gh_domain* d, const gh_filter_desc* fb, const gh_filter_desc* fs) {
  DeviceGuard guard_(d);
  if (!d) return GH_ERR_ARG;
  const Plan& pl = d->pl;
  std::vector<double> ft(pl.ftable_doubles, 0.0);
  const size_t base = pl.table_doubles;
  std::vector<ghb::ld> sg, M;
  const bool on_b = fb && fb->kind != GH_FILTER_NONE && !(d->f_blocks.empty() && d->f_big_blocks.empty());
  const bool on_s = fs && fs->kind != GH_FILTER_NONE && !(d->f_L.empty() && d->f_big_L.empty());
  // large classes: the same matrices, unfolded, in K_gemm's blocked fragment order
  std::vector<double> fbig(pl.fbigtab_doubles, 0.0);
  const size_t fbig0 = pl.table_doubles + pl.ftable_doubles + pl.bigtab_doubles + pl.ifctab_doubles;
  if (on_b) {
    std::map<int, std::vector<ghb::ld>> cache;
    for (const auto& b : d->f_big_blocks) {
      const int N = b.N, key = b.fourier ? -N : N;       // Fourier axes of cylindrical shells: sigma over m = 0 .. N/2
      if (!cache.count(key)) {
        if (!filter_sigma(fb, b.fourier ? N / 2 : N - 1, sg)) return fail(d, GH_ERR_ARG, "bad block filter descriptor");
        if (b.fourier) ghb::fourier_filter_matrix(N, sg, cache[key]); else ghb::cheb_filter_matrix(N, sg, cache[key]);
      }
      const std::vector<ghb::ld>& F = cache[key];
      fill_amat(fbig.data() + (b.off - fbig0), N, N, [&](int r, int c) { return F[(size_t)r * N + c]; });
    }
  }
  if (on_s) {
    for (const auto& kv : d->f_big_L) {
      const int L = kv.first, nt = L + 1;
      if (!filter_sigma(fs, L, sg)) return fail(d, GH_ERR_ARG, "bad shell filter descriptor");
      ghb::shell_filter_composites(L, sg, M);
      for (int m = 0; m <= L; ++m)
        fill_amat(fbig.data() + (kv.second[m] - fbig0), nt, nt, [&](int r, int c) { return M[((size_t)m * nt + r) * nt + c]; });
    }
  }
  if (on_b) {
    std::map<int, std::vector<ghb::ld>> cache;      // N -> filter matrix
    for (const auto& b : d->f_blocks) {
      const int N = b.N, key = b.fourier ? -N : N;       // Fourier axes of cylindrical shells: sigma over m = 0 .. N/2
      if (!cache.count(key)) {
        if (!filter_sigma(fb, b.fourier ? N / 2 : N - 1, sg)) return fail(d, GH_ERR_ARG, "bad block filter descriptor");
        if (b.fourier) ghb::fourier_filter_matrix(N, sg, cache[key]); else ghb::cheb_filter_matrix(N, sg, cache[key]);
      }
      const std::vector<ghb::ld>& F = cache[key];
      const int mtn = (N + 7) / 8, ksn = (N + 3) / 4;
      for (int mt = 0; mt < mtn; ++mt) for (int ks = 0; ks < ksn; ++ks) for (int lane = 0; lane < 32; ++lane) {
        const int row = mt * 8 + lane / 4, col = ks * 4 + lane % 4;
        ft[b.off - base + ((size_t)mt * ksn + ks) * 32 + lane] = (row < N && col < N) ? (double)F[(size_t)row * N + col] : 0.0;
      }
    }
  }
  if (on_s) {
    for (const auto& kv : d->f_L) {
      const int L = kv.first, nt = L + 1, hh = (nt + 1) / 2, NT = ang_nt_class(L), mtf = c_mtf(NT);
      if (!filter_sigma(fs, L, sg)) return fail(d, GH_ERR_ARG, "bad shell filter descriptor");
      ghb::shell_filter_composites(L, sg, M);
      // folded about the equator exactly like the projector rows of K_ang S2: ME = (G[r][j] + G[r][jbar]) / 2, MO = (.. - ..) / 2;
      // laid out for the shell's class: [m][ks < NT][p | q][mt < ceil(NT/2)][32], zero padded
      for (int m = 0; m <= L; ++m) for (int ks = 0; ks < NT; ++ks) for (int w = 0; w < 2; ++w) for (int mt = 0; mt < mtf; ++mt)
        for (int lane = 0; lane < 32; ++lane) {
          const int r = mt * 8 + lane / 4, j = ks * 4 + lane % 4;
          ghb::ld v = 0;
          if (j < hh && r < hh) {
            const int jb = nt - 1 - j;
            const ghb::ld a = M[((size_t)m * nt + r) * nt + j], c = M[((size_t)m * nt + r) * nt + jb];
            if (jb == j) v = w == 0 ? a / 2 : (ghb::ld)0;
            else v = (w == 0 ? a + c : a - c) / 2;
          }
          ft[kv.second - base + ((((size_t)m * NT + ks) * 2 + w) * mtf + mt) * 32 + lane] = (double)v;
        }
    }
  }
  if (pl.ftable_doubles) GH_CUDA(d, cudaMemcpyAsync(d->tables + base, ft.data(), ft.size() * sizeof(double), cudaMemcpyHostToDevice, d->stream));
  if (pl.fbigtab_doubles) GH_CUDA(d, cudaMemcpyAsync(d->tables + fbig0, fbig.data(), fbig.size() * sizeof(double), cudaMemcpyHostToDevice, d->stream));
  GH_CUDA(d, cudaStreamSynchronize(d->stream));      // the host staging vectors die at return
  d->filt_blocks = on_b; d->filt_shells = on_s;
  return GH_OK;
}

extern "C" gh_status gh_apply_filter(gh_domain* d) {
  DeviceGuard guard_(d);
  if (!d) return GH_ERR_ARG;
  if (!d->has_fields) return fail(d, GH_ERR_STATE, "gh_apply_filter before gh_set_fields");
  d->dp_fsal = false;
  const Plan& pl = d->pl;
  const CompMap cm{NCOMP, 0, 0};
  if (d->filt_blocks) {
    // x: ua -> T1, y: T1 -> T2, z: T2 -> ua   (T1, T2: the first two slots of the derivative scratch; only block points move)
    int walk = 1;
    for (int w = CHEB_COMP_WALK; w >= 1; --w)
      if (NCOMP % w == 0 && (w == 1 || (int64_t)pl.n_fcheb_items / 3 * (NCOMP / w) >= 4 * d->n_sm)) { walk = w; break; }
    const int gy = NCOMP / walk;
    const double* src[3] = {d->ua, d->du, d->du + (size_t)NCOMP * pl.S};
    double* dst[3] = {d->du, d->du + (size_t)NCOMP * pl.S, d->ua};
    int first = 0;
    for (int a = 0; a < 3; ++a) {
      for (int c = 0; c < CHEB_NCLASS; first += pl.n_fcheb[a][c], ++c)
        launch_cheb_class(d, GH_K_FILTER_CHEB, c, d->fcheb + first, pl.n_fcheb[a][c], gy, src[a], dst[a], NCOMP, cm);
      launch_gemm_list(d, GH_K_FILTER_CHEB, G_FX + a, d->ua, d->du, NCOMP, cm);     // large axes: the items name the same slots
    }
  }
  if (d->filt_shells) {
    // large shells: analysis (the derivative path's S1 list), per m the filtered projector, synthesis back into the state
    launch_gemm_list(d, GH_K_FILTER_ANG, G_S1, d->ua, d->du, NCOMP, cm);
    launch_gemm_list(d, GH_K_FILTER_ANG, G_FS2, d->ua, d->du, NCOMP, cm);
    launch_gemm_list(d, GH_K_FILTER_ANG, G_FS3, d->ua, d->du, NCOMP, cm);
    for (int cls = 0, first = 0; cls < 2; first += pl.n_ang_class[cls], ++cls) {
      if (!pl.n_ang_class[cls]) continue;
      ProfScope ps(d, GH_K_FILTER_ANG);
      if (cls == 0)
        k_ang<ANG_TPB0, true><<<dim3(pl.n_ang_class[0], NCOMP), ANG_TPB0, pl.ang_smem[0], d->stream>>>(d->ang + first, d->tables, d->ua, d->ua, pl.S, cm);
      else
        k_ang<ANG_TPB1, true><<<dim3(pl.n_ang_class[1], NCOMP), ANG_TPB1, pl.ang_smem[1], d->stream>>>(d->ang + first, d->tables, d->ua, d->ua, pl.S, cm);
    }
  }
  GH_CUDA(d, cudaGetLastError());
  return GH_OK;
}

// ------------------------------------------------------------------------------------------------------
// Dormand-Prince 5(4) step (NEXT-3)
// ------------------------------------------------------------------------------------------------------
namespace {
constexpr int DP_GRID = 256 * 8;     // upper bound of the streaming-kernel grid (partials buffer); launches use 8 CTAs of 256 threads per SM
const double DP_A[7][6] = {
    {0, 0, 0, 0, 0, 0},
    {1.0 / 5, 0, 0, 0, 0, 0},
    {3.0 / 40, 9.0 / 40, 0, 0, 0, 0},
    {44.0 / 45, -56.0 / 15, 32.0 / 9, 0, 0, 0},
    {19372.0 / 6561, -25360.0 / 2187, 64448.0 / 6561, -212.0 / 729, 0, 0},
    {9017.0 / 3168, -355.0 / 33, 46732.0 / 5247, 49.0 / 176, -5103.0 / 18656, 0},
    {35.0 / 384, 0, 500.0 / 1113, 125.0 / 192, -2187.0 / 6784, 11.0 / 84}};
const double DP_BH[7] = {5179.0 / 57600, 0, 7571.0 / 16695, 393.0 / 640, -92097.0 / 339200, 187.0 / 2100, 1.0 / 40};
inline size_t dp_bytes(const Plan& pl) {
  return 7 * (size_t)round_up((int64_t)(NCOMP * pl.S * sizeof(double)), 256) + (size_t)round_up(2 * DP_GRID * sizeof(double), 256) + 256;
}
}  // namespace

extern "C" size_t gh_dp5_workspace_bytes(const gh_domain* d) { return d ? dp_bytes(d->pl) : 0; }

extern "C" gh_status gh_dp5_attach(gh_domain* d, void* ws, size_t bytes) {
  DeviceGuard guard_(d);
  if (!d) return GH_ERR_ARG;
  if (!ws || ((uintptr_t)ws & 255) != 0) return fail(d, GH_ERR_WORKSPACE, "DP5 workspace is NULL or not 256-byte aligned");
  if (bytes < dp_bytes(d->pl)) return fail(d, GH_ERR_WORKSPACE, "DP5 workspace too small: need " + std::to_string(dp_bytes(d->pl)) + " bytes");
  char* w = (char*)ws;
  const size_t one = (size_t)round_up((int64_t)(NCOMP * d->pl.S * sizeof(double)), 256);
  for (int j = 0; j < 7; ++j) d->dpk[j] = (double*)(w + j * one);
  d->dp_part = (double*)(w + 7 * one);
  d->dp_out = (double*)(w + 7 * one + (size_t)round_up(2 * DP_GRID * sizeof(double), 256));
  d->dp_fsal = false;
  GH_CUDA(d, cudaMemsetAsync(ws, 0, dp_bytes(d->pl), d->stream));     // the padding between subdomains must be (and stays) zero
  return GH_OK;
}

extern "C" gh_status gh_dp5_step(gh_domain* d, double dt, double tol, double* err, int* accepted) {
  DeviceGuard guard_(d);
  if (!d || !err) return fail(d, GH_ERR_ARG, "NULL argument");
  if (!d->has_fields) return fail(d, GH_ERR_STATE, "gh_dp5_step before gh_set_fields");
  if (!d->dpk[0]) return fail(d, GH_ERR_STATE, "gh_dp5_step before gh_dp5_attach");
  if (!std::isfinite(dt)) return fail(d, GH_ERR_ARG, "dt is not finite");
  const int64_t n2 = (int64_t)NCOMP * d->pl.S / 2;
  const int grid = (int)std::min<int64_t>((n2 + 255) / 256, std::min(DP_GRID, d->n_sm * 8));
  gh_status st;
  // k1 = f(u): the last stage of the previous accepted step when the state has not been touched since
  if (!d->dp_fsal && (st = launch_rhs(d, d->ua, d->dpk[0])) != GH_OK) return st;
  for (int s = 1; s < 7; ++s) {      // ub = u + dt sum_j a_sj k_j;  k_{s+1} = f(ub);  after s = 6, ub is the 5th-order solution
    DpArgs A; A.nk = s;
    for (int j = 0; j < 7; ++j) { A.k[j] = (const double2*)d->dpk[j]; A.a[j] = j < s ? DP_A[s][j] : 0.0; }
    {
      ProfScope ps(d, GH_K_DP_STAGE);
      k_dp_stage<<<grid, 256, 0, d->stream>>>((const double2*)d->ua, A, dt, (double2*)d->ub, n2);
    }
    if ((st = launch_rhs(d, d->ub, d->dpk[s])) != GH_OK) return st;
  }
  {
    DpArgs A; A.nk = 7;
    for (int j = 0; j < 7; ++j) { A.k[j] = (const double2*)d->dpk[j]; A.a[j] = (j < 6 ? DP_A[6][j] : 0.0) - DP_BH[j]; }
    ProfScope ps(d, GH_K_DP_ERR);
    k_dp_err<<<grid, 256, 0, d->stream>>>(A, dt, d->dp_part, n2);
    k_dp_err_final<<<1, 32, 0, d->stream>>>(d->dp_part, grid, d->dp_out);
  }
  GH_CUDA(d, cudaGetLastError());
  double h[2] = {0, 0};
  GH_CUDA(d, cudaMemcpyAsync(h, d->dp_out, sizeof h, cudaMemcpyDeviceToHost, d->stream));
  st = check_flag(d);   // synchronises
  if (st != GH_OK) { d->dp_fsal = false; return st; }
  err[0] = std::sqrt(h[0] / ((double)NCOMP * (double)d->pl.P));
  err[1] = h[1];
  // a non-finite estimate (NaN in Pi or Phi with psi still physical is not caught by the singular flag) never passes
  const bool ok = std::isfinite(err[0]) && std::isfinite(err[1]) && (!(tol > 0.0) || (err[1] <= tol));
  if (accepted) *accepted = ok ? 1 : 0;
  if (ok) {
    std::swap(d->ua, d->ub);            // the new state; k7 = f(new state) becomes k1 of the next step
    std::swap(d->dpk[0], d->dpk[6]);
    d->t += dt; d->dp_fsal = true;
  } else {
    d->dp_fsal = true;                  // the state is unchanged and dpk[0] still is its RHS
  }
  return GH_OK;
}

// ------------------------------------------------------------------------------------------------------
// SpatialCoordJac (NEXT-4)
// ------------------------------------------------------------------------------------------------------
extern "C" gh_status gh_set_jacobian(gh_domain* d, const double* J, int on_device) {
  DeviceGuard guard_(d);
  if (!d || !J) return fail(d, GH_ERR_ARG, "NULL argument");
  GH_CUDA(d, cudaMemcpyAsync(d->jac, J, (size_t)9 * d->pl.S * sizeof(double), on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, d->stream));
  if (!on_device) GH_CUDA(d, cudaStreamSynchronize(d->stream));
  d->has_jac = true;
  return GH_OK;
}

namespace {
gh_status launch_scj(gh_domain* d, int structure, const double* in, double* out) {
  const int64_t S = d->pl.S;
  const int grid = d->pl.n_tiles;
  ProfScope ps(d, GH_K_SCJ);
  switch (structure) {
    case GH_T_A: k_scj<0><<<grid, TILE_PTS, 0, d->stream>>>(d->subs, d->tiles, d->pl.n_sub, d->jac, in, out, S); break;
    case GH_T_AA: k_scj<1><<<grid, TILE_PTS, 0, d->stream>>>(d->subs, d->tiles, d->pl.n_sub, d->jac, in, out, S); break;
    case GH_T_AB: k_scj<2><<<grid, TILE_PTS, 0, d->stream>>>(d->subs, d->tiles, d->pl.n_sub, d->jac, in, out, S); break;
    case GH_T_ABB: k_scj<3><<<grid, TILE_PTS, 0, d->stream>>>(d->subs, d->tiles, d->pl.n_sub, d->jac, in, out, S); break;
    default: k_scj<4><<<grid, TILE_PTS, 0, d->stream>>>(d->subs, d->tiles, d->pl.n_sub, d->jac, in, out, S); break;
  }
  return GH_OK;
}
}  // namespace

extern "C" gh_status gh_spatial_coord_jac(gh_domain* d, int structure, const double* T, double* out, int on_device) {
  DeviceGuard guard_(d);
  if (!d || !T || !out) return fail(d, GH_ERR_ARG, "NULL argument");
  if (structure < GH_T_A || structure > GH_T_ABB) return fail(d, GH_ERR_ARG, "gh_spatial_coord_jac: unknown tensor structure");
  if (!d->has_jac) return fail(d, GH_ERR_STATE, "gh_spatial_coord_jac before gh_set_jacobian");
  static const int NE[4] = {4, 10, 16, 40};
  const size_t bytes = (size_t)NE[structure] * d->pl.S * sizeof(double);
  if (on_device) {
    launch_scj(d, structure, T, out);
    GH_CUDA(d, cudaGetLastError());
    return GH_OK;
  }
  GH_CUDA(d, cudaMemcpyAsync(d->du, T, bytes, cudaMemcpyHostToDevice, d->stream));
  launch_scj(d, structure, d->du, d->du);
  GH_CUDA(d, cudaGetLastError());
  GH_CUDA(d, cudaMemcpyAsync(out, d->du, bytes, cudaMemcpyDeviceToHost, d->stream));
  GH_CUDA(d, cudaStreamSynchronize(d->stream));
  return GH_OK;
}

extern "C" gh_status gh_spatial_coord_jac_state(gh_domain* d) {
  DeviceGuard guard_(d);
  if (!d) return GH_ERR_ARG;
  if (!d->has_fields) return fail(d, GH_ERR_STATE, "gh_spatial_coord_jac_state before gh_set_fields");
  if (!d->has_jac) return fail(d, GH_ERR_STATE, "gh_spatial_coord_jac_state before gh_set_jacobian");
  d->dp_fsal = false;
  launch_scj(d, 4, d->ua, d->ua);
  GH_CUDA(d, cudaGetLastError());
  return GH_OK;
}

extern "C" gh_status gh_set_frame_map(gh_domain* d, const double* Jm, const double* v, int on_device) {
  DeviceGuard guard_(d);
  if (!d) return GH_ERR_ARG;
  if ((Jm == nullptr) != (v == nullptr)) return fail(d, GH_ERR_ARG, "gh_set_frame_map: give both Jm and v, or neither");
  d->dp_fsal = false;
  if (!Jm) { d->has_map = false; return GH_OK; }
  const size_t comp = (size_t)d->pl.S * sizeof(double);
  const cudaMemcpyKind kind = on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
  GH_CUDA(d, cudaMemcpyAsync(d->mapJ, Jm, 9 * comp, kind, d->stream));
  GH_CUDA(d, cudaMemcpyAsync(d->mapv, v, 3 * comp, kind, d->stream));
  if (!on_device) GH_CUDA(d, cudaStreamSynchronize(d->stream));
  d->has_map = true;
  return GH_OK;
}

extern "C" gh_status gh_fp64_peak(gh_domain* d, double* tflops) {
  DeviceGuard guard_(d);
  if (!d || !tflops) return fail(d, GH_ERR_ARG, "NULL argument");
  const int ctas = d->n_sm * 2;
  if ((size_t)ctas * 256 > (size_t)3 * NCOMP * d->pl.S) return fail(d, GH_ERR_WORKSPACE, "gh_fp64_peak: the derivative scratch is smaller than its output buffer");
  cudaEvent_t e0 = get_event(d), e1 = get_event(d);
  const int iters = 8000;           // 128 flop per lane and iteration: ~2.2 ms at 37 TFLOP/s with 2 CTAs per SM
  for (int mode = 0; mode < 2; ++mode) {
    float best = 1e30f;
    for (int rep = 0; rep < 4; ++rep) {
      cudaEventRecord(e0, d->stream);
      if (mode == 0) k_fp64_peak<1><<<ctas, 256, 0, d->stream>>>(d->du, rep ? iters : 16, 1e-3);
      else k_fp64_peak<0><<<ctas, 256, 0, d->stream>>>(d->du, rep ? iters : 16, 1e-3);
      cudaEventRecord(e1, d->stream);
      if (cudaEventSynchronize(e1) != cudaSuccess) { d->pool.push_back(e0); d->pool.push_back(e1); return fail(d, GH_ERR_CUDA, cudaGetErrorString(cudaGetLastError())); }
      float ms = 0; cudaEventElapsedTime(&ms, e0, e1);
      if (rep && ms < best) best = ms;
    }
    tflops[mode] = (double)ctas * 256 * iters * 128.0 / (best * 1e-3) / 1e12;
  }
  d->pool.push_back(e0); d->pool.push_back(e1);
  d->launches += 8;
  return GH_OK;
}

// ------------------------------------------------------------------------------------------------------
// profiling / bookkeeping
// ------------------------------------------------------------------------------------------------------
extern "C" gh_status gh_set_profiling(gh_domain* d, int enabled) {
  DeviceGuard guard_(d);
  if (!d) return GH_ERR_ARG;
  drain_profile(d);
  d->prof = enabled != 0;
  return GH_OK;
}

extern "C" gh_status gh_profile_read(gh_domain* d, double* ms, int64_t* counts) {
  DeviceGuard guard_(d);
  if (!d) return GH_ERR_ARG;
  drain_profile(d);
  for (int k = 0; k < GH_NUM_KERNELS; ++k) { if (ms) ms[k] = d->prof_ms[k]; if (counts) counts[k] = d->prof_n[k]; }
  return GH_OK;
}

extern "C" gh_status gh_profile_reset(gh_domain* d) {
  DeviceGuard guard_(d);
  if (!d) return GH_ERR_ARG;
  drain_profile(d);
  for (int k = 0; k < GH_NUM_KERNELS; ++k) { d->prof_ms[k] = 0; d->prof_n[k] = 0; }
  return GH_OK;
}

extern "C" const char* gh_kernel_name(int k) {
  static const char* names[GH_NUM_KERNELS] = {"k_cheb", "k_ang", "k_rhs", "k_rk", "k_con", "k_con_reduce", "k_jac", "other", "k_cheb(filter)", "k_ang(filter)", "k_dp_stage", "k_dp_err", "k_scj"};
  return (k >= 0 && k < GH_NUM_KERNELS) ? names[k] : "?";
}

extern "C" gh_status gh_set_option(gh_domain* d, int option, int value) {
  if (!d) return GH_ERR_ARG;
  if (option < 0 || option >= GH_NUM_OPTIONS) return fail(d, GH_ERR_ARG, "gh_set_option: unknown option");
  d->opt[option] = value;
  return GH_OK;
}

extern "C" int64_t gh_launch_count(const gh_domain* d) { return d ? d->launches : 0; }

extern "C" const char* gh_last_error(const gh_domain* d) { return d ? d->err.c_str() : g_create_error.c_str(); }
