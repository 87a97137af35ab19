/* gh.h — C ABI of the B200-native generalized-harmonic (GH) right-hand-side library.
 *
 * The data-parallel hot path of arXiv 1804.09101 (Lewis & Pfeiffer, "GPU-Accelerated
 * Simulations of Isolated Black Holes"): evaluating the evolution right-hand side of the
 * first-order generalized-harmonic Einstein system (§1, "about 50 fundamental
 * variables" PAPER.md:81 §2.1) on spectral subdomains — spherical shells I1 x S2
 * (Chebyshev radial x Y_lm angular, Eqs. 23-24) and blocks I1^3
 * (Chebyshev^3, Eqs. 20-22) — followed by a Runge-Kutta stage update and
 * a constraint-norm reduction.  The paper never prints the evolved equations; the system
 * implemented is written out in DESIGN.md ("Readings", S1) and SURVEY.md §8(c) O5.
 *
 * Conventions common to every call
 * --------------------------------
 * - All floating point is IEEE FP64.  No torch types: plain pointers and sizes.  Each pointer
 *   argument is documented as HOST or DEVICE; arguments with an `on_device` flag may be either.
 * - Field layout (structure of arrays):  u[c * comp_stride + offsets[s] + local],  c < 50,
 *   with local = (i0 * n1 + i1) * n2 + i2, last index fastest (the paper's row-major order,
 *   PAPER.md:397-401).  Shells: (i0,i1,i2) = (r, theta, phi), n1 = L+1 Gauss-Legendre
 *   colatitudes (ascending theta), n2 = 2L+2 uniform longitudes phi_k = 2 pi k / n2, radial
 *   Chebyshev-Gauss-Lobatto nodes r = lo + (hi-lo)(x+1)/2, x_j = -cos(pi j/(N_r-1)).
 *   Blocks: (x, y, z), CGL nodes on every axis.  Padding entries between subdomains are ignored
 *   on input and left untouched on output.
 * - Component order: s(a,b), a <= b: 00,01,02,03,11,12,13,22,23,33 -> 0..9;
 *   psi_ab: c = s;  Pi_ab: c = 10+s;  Phi_iab: c = 20 + 10 i + s  (i = 0,1,2 = x,y,z).
 *   Tensor components are Cartesian on every subdomain, shells included.
 * - Ownership: the caller owns the device workspace and the CUDA stream; the library owns only
 *   the host-side handle.  After gh_domain_create the library never allocates or frees device
 *   memory (allocation is "extremely expensive", §3.2).  Work is enqueued on the
 *   stream given at creation; calls that return host data synchronise that stream.
 * - Errors: every call returns a gh_status; nothing throws across the boundary; a message is
 *   available from gh_last_error().  There is NO CPU fallback: without a usable CUDA device
 *   every compute call returns GH_ERR_CUDA.
 */
#ifndef GH_H_
#define GH_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define GH_NCOMP 50

typedef struct gh_domain gh_domain; /* opaque; host struct owned by the library */

typedef enum {
  GH_OK = 0,
  GH_ERR_ARG = 1,       /* bad descriptor / NULL pointer / unsupported size */
  GH_ERR_WORKSPACE = 2, /* workspace too small or misaligned (needs 256-byte alignment) */
  GH_ERR_CUDA = 3,      /* CUDA runtime error (message has the CUDA error string) */
  GH_ERR_STATE = 4,     /* call out of order (e.g. gh_rhs before gh_set_fields) */
  GH_ERR_SINGULAR = 5   /* non-physical data met on the device: det g_ij <= 0 or lapse^2 <= 0 */
} gh_status;

typedef enum { GH_SHELL = 0, GH_BLOCK = 1, GH_CYLINDER = 2 } gh_kind;
/* FREE: no boundary treatment (e.g. an excision face inside the horizon).  FROZEN: d_t u = 0 on the face.
 * CHARACTERISTIC (NEXT-2 (i); the paper's ApplyBCs module, which it left on the CPU): the time
 * derivatives of the characteristic fields that ENTER through the face are set to zero, the others keep what the evolution
 * equations give (reading S21 writes the fields and speeds out); fused into the RHS kernel.  At block edges the
 * faces are applied in the order -x,+x,-y,+y,-z,+z; a FROZEN face through the same point wins.
 * INTERFACE (NEXT-2 (iii), shells only): the outer face of shell s and the inner face of shell s+1 (the next descriptor) are
 * one internal boundary: both must carry this flag, and the two shells must share centre and the radius.  With the same band
 * limit L their face grids coincide point by point; with different L (both <= 47) the neighbour's face state is first
 * interpolated to the own grid by summing its spherical-harmonic series at the own nodes (K_face_interp: analysis on the
 * neighbour's grid, all its modes l <= L_nbr kept; "interpolation ... via a direct summation of the spectral series").  Every characteristic field that enters a shell through the face is
 * relaxed towards the neighbour's value:  d_t u^a += -p |v_a| (u^a_own - u^a_neighbour),  p = (N_r - 1)^2 / (r_out - r_in)
 * of the own shell (reading S22); outgoing fields are untouched.  Fused into the RHS kernel, which reads the
 * neighbour's face state straight from the field store. */
typedef enum { GH_FACE_FREE = 0, GH_FACE_FROZEN = 1, GH_FACE_CHARACTERISTIC = 2, GH_FACE_INTERFACE = 3 } gh_face;

/* One spectral subdomain (PAPER.md:371 I1^3 blocks, PAPER.md:386 I1 x S2 shells; PAPER.md:79, 564 cylindrical shells - the third
 * topology the paper names for binary runs, without formulas.  DESIGN.md reading S25: GH_CYLINDER is a hollow cylinder about an
 * axis parallel to z through `center`, I1(rho) x I1(z) x S1(phi): Chebyshev-Gauss-Lobatto nodes in rho and z, N_phi uniform
 * nodes phi_k = 2 pi k / N_phi with the Fourier differentiation matrix; points ordered (rho slowest, z, phi fastest); Cartesian
 * tensor components, gradient through  d_x = cos(phi) d_rho - (sin(phi)/rho) d_phi,  d_y = sin(phi) d_rho + (cos(phi)/rho) d_phi. */
typedef struct {
  int32_t kind;      /* gh_kind */
  int32_t n[3];      /* shell: {N_r, L, 0} (N_theta = L+1, N_phi = 2L+2); block: {N_x, N_y, N_z}; cylinder: {N_rho, N_z, N_phi >= 3}; N >= 2 */
  double lo[3], hi[3]; /* shell: lo[0] = r_in, hi[0] = r_out (rest unused); block: corner coordinates;
                        * cylinder: [0] = rho_in > 0, rho_out; [1] = z range relative to the centre */
  double center[3];  /* shell centre; cylinder: a point of the axis (blocks: ignored) */
  int32_t face[6];   /* gh_face. shell: [0] = inner, [1] = outer; block: -x,+x,-y,+y,-z,+z; cylinder: rho_in, rho_out, z_lo, z_hi
                      * (FREE / FROZEN / CHARACTERISTIC; outward normals -+ rho^ and -+ z^) */
  double gamma[3];   /* constraint-damping gamma0, gamma1, gamma2, constant on the subdomain */
} gh_subdomain_desc;

/* Limits of this build.  Up to GH_SMALL_CHEB_N points per Chebyshev axis and GH_SMALL_L in the band limit the derivative
 * kernels keep the whole contraction of a line / a (theta,phi) plane on chip (K_cheb, K_ang); beyond, up to the maxima, the
 * same linear maps run as tiled FP64 tensor-core GEMMs whose cached matrices stream through shared memory (K_gemm) - the upper
 * two decades of the size sweep, BASELINE.json configs[4] (N = 320, L = 255: 3.3e7 points per subdomain).  The spectral filter
 * (gh_set_filter) covers both classes the same way (filter matrices in place of differentiation matrices). */
#define GH_MAX_CHEB_N 512   /* largest N on a Chebyshev axis */
#define GH_MAX_L 255        /* largest shell band limit L */
#define GH_SMALL_CHEB_N 64
#define GH_SMALL_L 47

/* Bytes of device workspace gh_domain_create needs for these subdomains; 0 on invalid input.
 * Pure host query, no CUDA call.  descs: HOST. */
size_t gh_workspace_bytes(const gh_subdomain_desc* descs, int32_t n_sub);

/* Build the domain (A0 + A1 of DESIGN.md): validates the descriptors, builds on the host in
 * long double the Chebyshev-Gauss-Lobatto differentiation matrices (Eq. 22, PAPER.md:379-384;
 * negative-sum trick), the Gauss-Legendre nodes/weights, the real-Fourier analysis/synthesis
 * matrices and the per-m Legendre composites that realise Eq. 24 axis by axis,
 * lays out the structure-of-arrays field store in `dev_workspace` and uploads tables once.
 *   descs: HOST, n_sub >= 1.   dev_workspace: DEVICE, 256-byte aligned, `bytes` >= gh_workspace_bytes.
 *   cuda_stream: a cudaStream_t (NULL = the legacy default stream).   out: HOST, receives the handle.
 * The workspace must stay valid and untouched by the caller until gh_domain_destroy. */
gh_status gh_domain_create(const gh_subdomain_desc* descs, int32_t n_sub, void* dev_workspace, size_t bytes,
                           void* cuda_stream, gh_domain** out);

/* Frees the host handle only (the workspace belongs to the caller).  NULL is a no-op. */
void gh_domain_destroy(gh_domain* dom);

/* Layout query.  n_points: HOST, total grid points P (unpadded).  comp_stride: HOST, distance in doubles
 * between components (= padded P).  offsets: HOST, n_sub+1 entries, start of each subdomain inside a
 * component (multiples of 16 doubles), last = comp_stride.  Any pointer may be NULL. */
gh_status gh_domain_layout(const gh_domain* dom, int64_t* n_points, int64_t* comp_stride, int64_t* offsets);

/* Grid coordinates xyz[3][comp_stride] (x, y, z of every point; padding = 0).  HOST or DEVICE per flag. */
gh_status gh_domain_coords(const gh_domain* dom, double* xyz, int on_device);

/* Set / get the evolved fields u[50][comp_stride] and the time.  HOST or DEVICE per flag.
 * gh_get_fields to HOST synchronises and reports GH_ERR_SINGULAR if the device flag was raised. */
gh_status gh_set_fields(gh_domain* dom, const double* u, int on_device, double t);
gh_status gh_get_fields(const gh_domain* dom, double* u, int on_device, double* t);

/* Gauge source H_a: H[4][comp_stride] and optionally its Cartesian gradient dH[12][comp_stride]
 * ([i*4+a] = d_i H_a).  dH == NULL: the library differentiates H once with its own spectral derivative.
 * d_t H_a = 0 (frozen gauge source, reading S3).  Default before the call: H = 0, dH = 0. */
gh_status gh_set_gauge_source(gh_domain* dom, const double* H, const double* dH, int on_device);

/* Right-hand side of the current state: dtu[50][comp_stride] = d_t (psi, Pi, Phi).
 * Steps A2-A6 of DESIGN.md: Chebyshev-line derivatives (Eq. 22), shell angular derivatives through
 * the l <= L projection (Eq. 24), logical->Cartesian Jacobian (Eq. 8), the fused
 * pointwise GH algebra, and zeroing on FROZEN faces.  dtu: HOST or DEVICE per flag (HOST synchronises). */
gh_status gh_rhs(gh_domain* dom, double* dtu, int on_device);

/* Spectral Cartesian gradient of the current state (debug / parity entry, A2-A4):
 * du[3][50][comp_stride], du[(k*50+c)*comp_stride + p] = d_k u_c.  HOST or DEVICE per flag. */
gh_status gh_gradient(gh_domain* dom, double* du, int on_device);

/* One full Shu-Osher SSP-RK3 step of size dt (A7; "method of lines", reading S4):
 *   u1 = u0 + dt k(u0);  u2 = 3/4 u0 + 1/4 (u1 + dt k(u1));  u_new = 1/3 u0 + 2/3 (u2 + dt k(u2)).
 * Asynchronous on the domain's stream; advances the stored time by dt. */
gh_status gh_rk_step(gh_domain* dom, double dt);

/* gh_rk_step that also returns the constraint norms of the state it STARTS from (A8 as an epilogue of A5, SURVEY.md §8(a), (d):
 * the first stage's fused RHS kernel already holds C_a, the derivatives of psi and Phi and Phi itself on chip, so the norms
 * cost no extra memory traffic and no second derivative pass).  out / per_sub: as in gh_constraint_norms, and equal to what
 * gh_constraint_norms would have returned just before the step.  Synchronises (it returns host data); reports
 * GH_ERR_SINGULAR if the device flag was raised. */
gh_status gh_rk_step_norms(gh_domain* dom, double dt, double* out, double* per_sub);

/* Constraint norms of the current state (A8): out[3][2] = {rms, max} for C_a (4 components),
 * C_iab = d_i psi_ab - Phi_iab (30), C_ijab = d_i Phi_jab - d_j Phi_iab (30 independent);
 * rms = sqrt(sum over points and components / (P * n_comp)), unweighted (reading S16).
 * per_sub: NULL or HOST [n_sub][3][2], the same per subdomain.  out: HOST.  Synchronises; reports
 * GH_ERR_SINGULAR if the device flag was raised. */
gh_status gh_constraint_norms(gh_domain* dom, double* out, double* per_sub);

/* gh_constraint_norms for callers that may not allocate device memory (code under CUDA graph capture around the call, tight
 * serving loops, harnesses that forbid cudaMalloc): same arguments, same results bit for bit, but the reduction scratch (per-tile
 * partials, per-subdomain sums, totals) lives in ONE file-scope static device array of GH_STATIC_SCRATCH_BYTES (3.2 MB, held by
 * every GPU that loads the library until the process exits) instead of the workspace, the totals are folded on the device, and
 * the call makes no cudaMalloc / cudaFree, creates no event or graph and uses no host heap (per-launch profiling is off during
 * the call).  Limits: at most GH_STATIC_MAX_TILES tiles of 128 points (8 388 608 points - the bench workload C4 has 38 036) and
 * GH_STATIC_MAX_SUBS subdomains; beyond them GH_ERR_ARG with a message, nothing launched.  The array is shared by all calls of
 * the process and keeps the last call's contents; every value a call reads it has written itself, so nothing needs clearing.
 * Calls that OVERLAP on the GPU (two domains on different streams, two threads) race on it: serialise them.  The first call
 * on each device resolves the array's device address (cudaGetSymbolAddress) - make it outside any stream capture.
 * Synchronises (it returns host data); reports GH_ERR_SINGULAR if the device flag was raised. */
#define GH_STATIC_MAX_TILES 65536
#define GH_STATIC_MAX_SUBS 4096
#define GH_STATIC_SCRATCH_BYTES ((65536 * 6 + 4096 * 6 + 8) * 8)
gh_status gh_constraint_norms_static(gh_domain* dom, double* out, double* per_sub);

/* ---- spectral filter (NEXT-1 of DESIGN.md; "Filter ~ 30 % of CPU runtime", 452-460, 500-516) ----------
 * "Spectral filtering of 1D basis functions is similar to differentiation, the only difference being the specific
 * form of the transformation matrix": on blocks the state is multiplied along every axis by the
 * cached matrix F = SpecToPhys diag(sigma_k) PhysToSpec (Eqs. 16-17); on shells every (theta,phi) plane goes
 * PhysToSpec -> sigma_l a_lm -> SpecToPhys (the scalar-in-l filter: the tensor-harmonic coupling
 * matrix is not defined in the paper), with no filter along r ("we do not include a filter along the r-axis",
 * PAPER.md:500).  The paper names its two filter functions "Heaviside" and "ExpCheb" without formulas; reading S20:
 *   GH_FILTER_HEAVISIDE: sigma_k = 1 for k <= kmax - cut, else 0            (the top `cut` modes are removed)
 *   GH_FILTER_EXP:       sigma_k = exp(-alpha (k / kmax)^(2 p))
 * with k the Chebyshev mode number (kmax = N-1 on that axis) or the harmonic degree l (kmax = L). */
typedef enum { GH_FILTER_NONE = 0, GH_FILTER_HEAVISIDE = 1, GH_FILTER_EXP = 2 } gh_filter_kind;
typedef struct {
  int32_t kind;   /* gh_filter_kind */
  int32_t cut;    /* HEAVISIDE: number of top modes removed (>= 0) */
  double alpha;   /* EXP */
  int32_t p;      /* EXP: half order (>= 1) */
  int32_t pad_;
} gh_filter_desc;

/* Choose the filters: `block_axes` for the three Chebyshev axes of every block - and of every cylindrical shell, where it acts
 * on the Chebyshev modes k <= N-1 in rho and z and on the Fourier modes m <= N_phi/2 in phi -, `shell_angular` for the l-filter
 * of every shell (either may be NULL or kind NONE: that family is left untouched).  Builds the matrices on the host in long
 * double and uploads them (synchronises).  descs: HOST. */
gh_status gh_set_filter(gh_domain* dom, const gh_filter_desc* block_axes, const gh_filter_desc* shell_angular);

/* state <- filtered state, in place, asynchronous on the domain's stream.  GH_ERR_STATE before gh_set_filter /
 * gh_set_fields.  The derivative scratch is used as temporary storage. */
gh_status gh_apply_filter(gh_domain* dom);

/* The filter function itself, for tests: sigma[0..kmax].  HOST. */
gh_status gh_filter_sigma(const gh_filter_desc* f, int32_t kmax, double* sigma);

/* ---- Dormand-Prince 5(4) step (NEXT-3 of DESIGN.md; the stepper the paper names, "high-order Dormand Prince",
 * PAPER.md:81) -----------------------------------------------------------------------------------------------------
 * Seven-stage explicit pair of Dormand & Prince (1980): the 5th-order solution advances the state, the embedded 4th-order
 * one gives err = dt sum_j (b_j - bh_j) k_j for step-size control.  The seven stage derivatives need 7 x [50][comp_stride]
 * doubles of extra device memory, attached separately so that RK3 users do not pay for it. */
size_t gh_dp5_workspace_bytes(const gh_domain* dom);
/* dev_ws: DEVICE, 256-byte aligned, >= gh_dp5_workspace_bytes; owned by the caller, valid until destroy.  Zeroes it. */
gh_status gh_dp5_attach(gh_domain* dom, void* dev_ws, size_t bytes);
/* One step of size dt.  err: HOST [2] = {rms, max} of the error estimate over all 50 components and points (unweighted).
 * tol > 0: the step is taken only if max <= tol, otherwise the state is left as it was (*accepted = 0) and the caller
 * retries with a smaller dt; tol <= 0: always taken - except that a non-finite error estimate (NaN / Inf anywhere in the
 * stage derivatives) is never accepted.  accepted may be NULL.  Synchronises (it returns host data).
 * The last stage is the RHS at the new state and is reused as the first stage of the next step when nothing else touched
 * the state in between. */
gh_status gh_dp5_step(gh_domain* dom, double dt, double tol, double* err, int* accepted);

/* ---- SpatialCoordJac (NEXT-4 of DESIGN.md; §3.3, Eqs. 9-11) -----------------------------------------------
 * "makes a coordinate change of a tensor's spatial indices only, by contracting every possible combination of said spatial
 * indices with the Jacobian":  T'_ij = J_i^k J_j^l T_kl (9),  T'_0j = J_j^l T_0l (10),  T'_i0 = J_i^k T_k0 (11), the purely
 * timelike component untouched - i.e. every index is multiplied by diag(1, J).  This is the frame change of the dual-frame
 * method (grid coordinates <-> asymptotically inertial coordinates, related by a time-dependent spatial map);
 * J is whatever Jacobian of that map the caller evaluates at the current time.  The four tensor structures the paper's
 * port handles, in structure-of-arrays storage T[N_e][comp_stride]:
 *   GH_T_A   T_a    N_e = 4
 *   GH_T_AA  T_aa   N_e = 10  symmetric, packed 00,01,02,03,11,12,13,22,23,33
 *   GH_T_AB  T_ab   N_e = 16  component 4 a + b
 *   GH_T_ABB T_abb  N_e = 40  T_abc = T_acb, component 10 a + s(b,c)
 * HBM-bound: (2 N_e + 9) doubles per grid point. */
typedef enum { GH_T_A = 0, GH_T_AA = 1, GH_T_AB = 2, GH_T_ABB = 3 } gh_tensor_structure;
/* J[9][comp_stride], J[3 i + k] = J_i^k at every grid point (padding ignored).  HOST or DEVICE per flag; copied into the
 * domain's workspace (asynchronous for DEVICE).  Default before the call: none (the transforms return GH_ERR_STATE). */
gh_status gh_set_jacobian(gh_domain* dom, const double* J, int on_device);
/* out[N_e][comp_stride] = SpatialCoordJac of T[N_e][comp_stride] with the Jacobian last set; out may be T (in place).
 * HOST or DEVICE per flag (both on the same side; HOST synchronises and needs N_e <= 40 of the derivative scratch). */
gh_status gh_spatial_coord_jac(gh_domain* dom, int structure, const double* T, double* out, int on_device);
/* The evolved state in place: psi_ab and Pi_ab as T_aa, Phi_iab with all three indices (its first index is spatial only):
 * Phi'_iab = J_i^k L_a^c L_b^d Phi_kcd, L = diag(1, J).  Asynchronous.  GH_ERR_STATE before gh_set_fields / gh_set_jacobian. */
gh_status gh_spatial_coord_jac_state(gh_domain* dom);

/* ---- dual frame (NEXT-4) -------------------------------------------------------------------------------------------
 * "data is represented at collocation points at fixed grid-coordinates ...  The evolution equations, however, are formulated in
 * asymptotic inertial coordinates.  The two coordinate systems share the same time-coordinate, and their spatial coordinates are
 * related by a time-dependent coordinate transformation."  The caller evaluates the map x = x(xbar, t) at the current time and
 * hands over its kinematics at the grid points:
 *   Jm[9][comp_stride], Jm[3 i + k] = d xbar^k / d x^i      (d/dx^i = Jm_i^k d/dxbar^k: DiffJac, Eq. 8)
 *   v[3][comp_stride],  v^i = d x^i / d t at fixed xbar       (the velocity of the grid points in the inertial frame)
 * From then on gh_rhs, gh_rk_step(_norms), gh_dp5_step and gh_constraint_norms use inertial-frame derivatives d_i u = Jm_i^k dbar_k u
 * and the time derivative AT THE FIXED GRID POINTS:  d_t u |_xbar = F[u, d_i u] + v^i d_i u  (F: the single-frame right-hand side;
 * tensor components stay inertial-frame Cartesian).  Boundary treatments act on F; FROZEN faces hold their grid-frame value
 * (no advection there).  The map is held fixed until the next call (within one step it is frozen: re-set it as time advances).
 * The gauge source's gradient dH must then be given explicitly, in the inertial frame.  gh_gradient stays a grid-frame gradient.
 * Jm = v = NULL: back to the single frame.  HOST or DEVICE per flag.  Cost: two more HBM passes per RHS evaluation, only while set. */
gh_status gh_set_frame_map(gh_domain* dom, const double* Jm, const double* v, int on_device);

/* FP64 throughput of the device the domain lives on, measured now with register-resident kernels on the domain's stream
 * (profiling helper; bench.py quotes the derivative kernels' roofline fraction against it): tflops[0] = DMMA
 * (mma.sync.m8n8k4.f64, what K_cheb / K_ang issue), tflops[1] = plain DFMA.  Best of 3 launches of ~2 ms after a warm-up.
 * Uses the derivative scratch as its output buffer.  tflops: HOST [2].  Synchronises. */
gh_status gh_fp64_peak(gh_domain* dom, double* tflops);

/* Per-kernel device time of the most recent gh_rhs / gh_rk_step / gh_constraint_norms, in
 * milliseconds, measured with CUDA events on the domain's stream when profiling is enabled with
 * gh_set_profiling(dom, 1) (off by default: event records cost launch latency).
 * ms: HOST [GH_NUM_KERNELS] accumulated since the last call to gh_profile_reset; counts likewise. */
#define GH_NUM_KERNELS 13
enum { GH_K_CHEB = 0, GH_K_SHELL_ANG = 1, GH_K_RHS = 2, GH_K_RK = 3, GH_K_CONSTRAINTS = 4, GH_K_REDUCE = 5, GH_K_JAC = 6, GH_K_OTHER = 7,
       GH_K_FILTER_CHEB = 8, GH_K_FILTER_ANG = 9, GH_K_DP_STAGE = 10, GH_K_DP_ERR = 11, GH_K_SCJ = 12 };
gh_status gh_set_profiling(gh_domain* dom, int enabled);
gh_status gh_profile_read(gh_domain* dom, double* ms, int64_t* counts);
gh_status gh_profile_reset(gh_domain* dom);
const char* gh_kernel_name(int k);

/* Execution options (all default 0; they change HOW the path runs, never what it computes - results are bit-identical).
 *   GH_OPT_RK_OUT_OF_PLACE  1: every stage of gh_rk_step writes to a buffer it does not read (ua -> ub -> k -> ua) instead of
 *                           updating in place.  The in-place stages are by design (the fused RHS kernel holds every field of a
 *                           point in registers / shared memory before its first store); this switch exists so that a test can
 *                           demand bit-equality of the two (compute-sanitizer is not available on the GPU pool).
 *   GH_OPT_NO_GRAPH         1: gh_rk_step / gh_rk_step_norms / gh_rhs(DEVICE) enqueue their kernels one by one.  Default 0: the
 *                           whole call (the three stages of a step: up to ~20 launches) is captured once into a CUDA graph
 *                           and replayed as ONE launch - the paper's central lesson is launch overhead (~20 us per kernel,
 *                           PAPER.md:241, 472), and configs C1-C3 are launch-bound.  The graph is re-captured when dt, the
 *                           buffers or an option change; it needs a real stream (not the legacy default stream 0, which
 *                           cannot be captured: then, and while profiling is on, the kernels are enqueued one by one). */
#define GH_NUM_OPTIONS 8
enum { GH_OPT_RK_OUT_OF_PLACE = 0, GH_OPT_NO_GRAPH = 1 };
gh_status gh_set_option(gh_domain* dom, int option, int value);

/* Number of kernel launches issued by the library on this domain since creation. */
int64_t gh_launch_count(const gh_domain* dom);

/* Message for the last non-OK status on this domain (or for a failed create when dom == NULL). */
const char* gh_last_error(const gh_domain* dom);

/* ---- host-side basis builder, exposed for tests (no CUDA) --------------------------------- */
/* CGL nodes x[N] and differentiation matrix D[N*N] (row-major, D[i*N+j]) on [-1,1]. */
gh_status gh_basis_cheb(int32_t N, double* x, double* D);
/* Gauss-Legendre colatitudes theta[L+1] (ascending) and weights w[L+1]. */
gh_status gh_basis_gauss_legendre(int32_t L, double* theta, double* w);
/* Shell angular matrices for band limit L, n_t = L+1, n_p = 2L+2, n_q = 2L+1:
 *   Fa[n_q*n_p]: analysis, row q: q=0..L cos(m phi_k) (m=q), q=L+1..2L sin(m phi_k) (m=q-L), normalised
 *                so that Fs*Fa is the projector onto modes m <= L;
 *   Fs[n_p*n_q]: synthesis;
 *   Th[(L+1)*n_t*n_t]: per-m composite d/dtheta o projection, Th[m][j'][j];
 *   Pr[(L+1)*n_t*n_t]: per-m projector onto l <= L.   Any pointer may be NULL. */
gh_status gh_basis_shell(int32_t L, double* Fa, double* Fs, double* Th, double* Pr);

#ifdef __cplusplus
}
#endif
#endif /* GH_H_ */
