// device_types.h — plain structs shared by the host API (gh_lib.cu) and the kernels (kernels.cuh).
#pragma once
#include <stdint.h>

namespace ghd {

constexpr int NCOMP = 50;
constexpr int TILE_PTS = 128;   // points per CTA of the pointwise kernels (K_rhs, K_con, K_jac)

// One spectral subdomain as the kernels see it.
struct SubDev {
  int32_t kind;            // 0 shell, 1 block, 2 cylindrical shell (logical axes rho, z, phi; the pointwise kernels treat it as a
                           // "shell": curvilinear, Jacobian from tables)
  int32_t n0, n1, n2;      // logical extents, n2 fastest (shell: N_r, L+1, 2L+2)
  int64_t off;             // start inside a component (multiple of 16 doubles)
  int32_t P;               // n0*n1*n2
  int32_t face[6];         // 1 = FROZEN
  double gamma[3];
  // shells only: offsets (in doubles) into the table memory
  int32_t t_rinv;          // 1/r_i               [n0]
  int32_t t_ct, t_st;      // cos/sin(theta_j)     [n1]
  int32_t t_cp, t_sp;      // cos/sin(phi_k)       [n2]
  int32_t pad_;
  // shells with INTERFACE faces: start (inside a component) of the neighbour's coincident (theta,phi) plane for the inner /
  // outer face (-1: none) and the penalty factor (N_r - 1)^2 / (r_out - r_in)
  int64_t nbr[2];
  double pen;
  // ... when the neighbour has a different band limit its face state is interpolated to this shell's grid first (K_face_interp):
  // start (inside a component) of that copy in the interface buffer, -1: the grids coincide and nbr[] is used
  int64_t nbi[2];
};

// One face plane to interpolate (NEXT-2 (iii) between shells of different L): the neighbour's (theta,phi) plane at src_off of
// every component of the state -> dst_off of every component of the interface buffer, on this shell's grid.
struct IfcItem {
  int64_t src_off, dst_off;
  int32_t Ls, Ld;
  int64_t m_FaT, m_GT, m_FxT;   // offsets (doubles) in the table memory: FaT[k][q] (n_phi_s x n_q_s), GT[m][j][j'] (per m: n_theta_s x n_theta_d), FxT[q][k'] (n_q_s x n_phi_d)
};

// One tile of Chebyshev lines: out[a, col] = sum_i D[a][i] in[i, col] for `ncols` columns (A2, Eq. 22).
// Element (i, col) lives at  base + i*stride_i + (col / col_inner)*outer_stride + (col % col_inner).
struct ChebItem {
  int64_t base;
  int64_t stride_i;
  int64_t outer_stride;
  int32_t N;
  int32_t col_inner;
  int32_t col0;
  int32_t ncols;
  int32_t dmat;     // offset (doubles) of D, multiplied by 2/(hi-lo), in DMMA A-fragment order [m_tile][k_step][32]
  int32_t pad0_;
  int32_t axis;     // which logical-derivative slot the result goes to
  int32_t pad_;
};

// One batch of angular planes of one shell (A3, Eq. 24): planes [plane0, plane0+nplanes) of component
// `blockIdx.y`; plane ir starts at off + ir * n1*n2.
struct AngItem {
  int64_t off;
  int32_t L;
  int32_t plane0;
  int32_t nplanes;
  int32_t nb_alloc;              // planes the shared-memory layout is sized for (>= nplanes)
  int32_t m_Fa, m_Fs, m_T;       // offsets (doubles) in the table memory, all in DMMA fragment order [k_step][n_tile][32]:
                                 // Fa = (even | odd) analysis, Fs = (even | odd) synthesis (see K_ang); stacked per-m
                                 // matrices [Th_m ; m Pr_m] as [m][k_step][m_tile][32]
  int32_t m_G;                   // spectral filter: per-m folded filtered projectors [m][k_step][even|odd][m_tile][32] (gh_set_filter)
  int8_t nch1e, nch1o, nch3, pad8_;   // n-chunks per m-tile in S1 (even, odd GEMM) / S3 (host-chosen for balance over the warps)
};

}  // namespace ghd
