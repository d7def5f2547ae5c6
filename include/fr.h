/* fr.h — C ABI of the B200-native Flux Reconstruction right-hand-side library.
 *
 * One hot path of arxiv/paper_1312_1638 (PyFR): the per-stage RHS of the FR discretisation of the
 * compressible Euler / Navier-Stokes equations on quadrilateral, triangular and hexahedral grids,
 * driven by classical RK4.  Citations are PAPER.md:<line>; A-numbers are the readings in DESIGN.md.
 *
 * Conventions (DESIGN.md "Conventions" has the full statement):
 *  - State matrices are SoA  [point][variable][element], element fastest, leading
 *    dimension ld = fr_leading_dim() >= n_elems (padded so every row starts on a 128-byte boundary).
 *    Variables: rho, rho*v_x, rho*v_y, (rho*v_z,) E   (Eq 20 :474);  N_V = ndims + 2.
 *  - quad/hex reference element [-1,1]^ndims, Gauss-Legendre tensor solution points
 *    rho = i + n*j (+ n^2*k), n = p+1, first coordinate fastest; face f = 2*d + s (d = reference
 *    direction, s = 0 at -1 / 1 at +1); flux point sigma = f*nfp + idx, idx = tensor GL index over the
 *    remaining directions, lowest fastest.  Triangle: reference (-1,-1),(1,-1),(-1,1); solution
 *    points = barycentric lattice (i+1,j+1,k+1)/(p+3) (A6), j outer / i inner; face k = edge
 *    vertex k -> k+1, GL flux points along the edge.
 *  - Geometry nodes: degree-p_g Lagrange on the equispaced lattice of the reference element,
 *    first coordinate fastest (triangle: rows j = 0..p_g, i = 0..p_g-j).
 *  - Every entry point returns 0 on success or a negative FR_E* code; fr_last_error() gives text.
 *    No exception or abort crosses this boundary.  A NULL context is an error, not a crash.
 *  - "host" / "dev" say where a pointer must live.  The library never frees caller memory.
 */
#ifndef FR_B200_H
#define FR_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct fr_ctx fr_ctx;

enum { FR_QUAD = 0, FR_TRI = 1, FR_HEX = 2 };                  /* element types */
enum { FR_EULER = 0, FR_NAVIER_STOKES = 1 };                   /* governing systems */
enum { FR_F32 = 0, FR_F64 = 1 };                               /* storage precision of u / rhs */
enum { FR_BC_SUP_INFLOW = 0, FR_BC_SUB_OUTFLOW = 1, FR_BC_NOSLIP_WALL = 2 }; /* App C :799-825 */
enum { FR_CORR_DG = 0, FR_CORR_SD = 1, FR_CORR_HU = 2 };      /* FR schemes, "DG, SD, and HU as defined in [10]" */
enum { FR_STEPPER_EULER = 0, FR_STEPPER_RK4 = 1, FR_STEPPER_DOPRI5 = 2 }; /* time steppers, Table 1 :263 */

enum {
  FR_OK = 0,
  FR_EINVAL = -1,    /* bad argument / NULL pointer / call order */
  FR_EMESH = -2,     /* J <= 0, unmatched flux points, face referenced twice or never */
  FR_ECUDA = -3,     /* a CUDA runtime call failed (text in fr_last_error) */
  FR_ENOMEM = -4,
  FR_EUNSUPPORTED = -5
};

/* Boundary condition, Appendix C.  SUP_INFLOW uses rho,v,p (Eq 47); SUB_OUTFLOW uses p (Eq 49);
 * NOSLIP_WALL uses cpTw = C_p*T_w and v = v_w (Eq 51-53). */
typedef struct {
  int32_t kind;
  double rho, v[3], p, cpTw;
} fr_bc_desc;

/* Mesh of ONE element type (mixed meshes: DESIGN.md "next").  All pointers: host, read during the
 * call only (the library copies what it needs). */
typedef struct {
  int32_t ndims;           /* 2 | 3 */
  int32_t etype;           /* FR_QUAD | FR_TRI | FR_HEX */
  int32_t p_g;             /* geometry degree >= 1 */
  int32_t n_bcs;           /* entries in bcs; boundary faces index it by bc_id */
  int64_t n_elems;
  int64_t n_ifaces;        /* interior + periodic interfaces, each listed once */
  int64_t n_bfaces;
  const double *nodes;     /* [n_elems][n_nodes(p_g)][ndims] */
  const int32_t *ifaces;   /* [n_ifaces][4] = elemL, faceL, elemR, faceR; L/R order is significant (A12) */
  const double *shifts;    /* [n_ifaces][ndims]: x_L(flux point) = x_R(flux point) + shift (periodic image) */
  const int32_t *bfaces;   /* [n_bfaces][3] = elem, face, bc_id */
  const fr_bc_desc *bcs;   /* [n_bcs] */
} fr_mesh_desc;

/* Mesh of SEVERAL element types sharing faces (PAPER.md:141 "triangles, quadrilaterals"; :603 the mixed unstructured mesh of
 * Table 2): parts of one element type each, and interface records that name the part of each side.  2-D (quadrilaterals and
 * triangles).  All pointers: host, read during the call only. */
typedef struct {
  int32_t etype;           /* FR_QUAD | FR_TRI */
  int32_t p_g;
  int64_t n_elems;
  const double *nodes;     /* [n_elems][n_nodes(p_g)][ndims] */
} fr_mesh_part;

typedef struct {
  int32_t ndims;           /* 2 */
  int32_t n_parts;
  int32_t n_bcs;
  int32_t reserved;
  int64_t n_ifaces, n_bfaces;
  const fr_mesh_part *parts;
  const int32_t *ifaces;   /* [n_ifaces][6] = partL, elemL, faceL, partR, elemR, faceR; L/R order is significant (A12) */
  const double *shifts;    /* [n_ifaces][ndims] */
  const int32_t *bfaces;   /* [n_bfaces][4] = part, elem, face, bc_id */
  const fr_bc_desc *bcs;
} fr_mixed_mesh_desc;

/* Discretisation: order p, system (§4), storage precision, gas constants gamma (Eq 21),
 * mu, Pr (Eq 22-23; mu constant, A9), LDG beta / tau (Eq 25-27 :506-516; tau enters with the dissipative
 * sign, A7).  Point sets are fixed (A6).  correction: FR_CORR_DG (A5; every element type), FR_CORR_SD / FR_CORR_HU
 * (:568; the one-parameter family of the paper's ref [10] with c_SD / c_HU, reading A23; quadrilaterals and hexahedra,
 * FR_CORR_HU needs p >= 1; FR_EINVAL otherwise).
 * rho_ref, v_ref, p_ref: an optional constant reference state (all zero = none).  It is a CONDITIONING hint, not a
 * parameter of the method: the fused kernels then evaluate the inviscid flux and the interface flux in perturbation
 * form about it (constant fluxes have zero discrete divergence, Eq 18 with M1 const = 0), which removes
 * the cancellation of O(p_ref) terms from the rounding error.  The result is the same function of u up to rounding on
 * meshes whose metric terms satisfy the discrete metric identities (affine elements; 2-D elements with p_g <= p; the
 * 3-D cases of reading A10); elsewhere it differs by the freestream residual of the reference state. */
typedef struct {
  int32_t p;
  int32_t system;
  int32_t precision;
  int32_t flags;           /* FR_FLAG_* bits */
  int32_t correction;      /* FR_CORR_* */
  int32_t reserved;        /* 0 */
  double gamma, mu, Pr, ldg_beta, ldg_tau;
  double rho_ref, v_ref[3], p_ref;
} fr_disc_desc;

#define FR_FLAG_FORCE_GENERIC 1
#define FR_FLAG_HOST_ONLY 2      /* build the host tables only (no CUDA call): queries work, fr_rhs fails */
#define FR_FLAG_LEAN 4           /* release the host copies of the mesh and of the setup tables once they are uploaded (meshes of
                                    10^7 elements): fr_get_pairs / fr_get_metrics and a second fr_setup_operators then return
                                    FR_EINVAL; sizes, coordinates, operators, fr_rhs and the steppers are unaffected */

/* Creates a context (owned by the library; release with fr_teardown).  Validates connectivity only;
 * geometric checks happen in fr_setup_operators once the point sets are known. */
int fr_setup_mesh(fr_ctx **out, const fr_mesh_desc *mesh);

/* The same for a mesh of several element types.  State matrices of such a context are ONE buffer holding the parts one after
 * the other: part t is a [N_u(t)][N_V][ld(t)] matrix at byte offset fr_part_info(...).state_offset (256-byte aligned);
 * fr_state_bytes gives the total.  fr_rhs and the steppers take that buffer; the orders 1 <= p <= 4 (fused element kernels of
 * both types) are supported, FR_EUNSUPPORTED otherwise.  Single-type size queries (fr_num_solution_points, fr_num_flux_points,
 * fr_leading_dim, fr_solution_point_coords, fr_get_*) return FR_EINVAL on a mixed context: use the per-part queries. */
int fr_setup_mesh_mixed(fr_ctx **out, const fr_mixed_mesh_desc *mesh);
int64_t fr_num_parts(const fr_ctx *ctx);           /* 1 for a single-type context */
typedef struct {
  int32_t etype, reserved;
  int64_t n_elems, n_solution_points, n_flux_points, leading_dim, state_offset /* bytes */;
} fr_part_info_t;
int fr_part_info(const fr_ctx *ctx, int part, fr_part_info_t *info_host);
int fr_part_solution_point_coords(const fr_ctx *ctx, int part, double *xyz_host); /* [N_u][n_elems][ndims] of the part */

/* Builds M0..M6 (App A :737-768) on the host in extended precision, the metric terms S = J*J^-1, 1/J
 * (Eq 10, 12, 19) at the solution points, the physical normals and J*n (Eq 14, 16) at the flux points,
 * matches flux-point pairs by physical coordinates (:182, :194) and orders them for coalesced access
 * (:693); uploads the constants to the current CUDA device.  May be called again to change p/system.
 * Errors: FR_EMESH on J <= 0 or unmatched / uncovered flux points. */
int fr_setup_operators(fr_ctx *ctx, const fr_disc_desc *disc);

/* Sizes (valid after fr_setup_operators; negative error code otherwise). */
int64_t fr_num_solution_points(const fr_ctx *ctx); /* N_u per element */
int64_t fr_num_flux_points(const fr_ctx *ctx);     /* N_f per element */
int64_t fr_num_vars(const fr_ctx *ctx);            /* N_V */
int64_t fr_num_pairs(const fr_ctx *ctx);           /* interior+periodic flux-point pairs */
int64_t fr_leading_dim(const fr_ctx *ctx);         /* ld of every state matrix */
int64_t fr_state_bytes(const fr_ctx *ctx);         /* N_u*N_V*ld*sizeof(precision) */
int64_t fr_workspace_bytes(const fr_ctx *ctx);     /* scratch for fr_rhs + RK registers for fr_rk4_step */
int64_t fr_stepper_workspace_bytes(const fr_ctx *ctx, int stepper); /* the same for FR_STEPPER_*: Euler 1, RK4 3, DOPRI5 7 registers */
int64_t fr_rhs_kernel_launches(const fr_ctx *ctx); /* kernels one fr_rhs call launches */

/* Physical coordinates of the solution points, host buffer [N_u][n_elems][ndims] doubles. */
int fr_solution_point_coords(const fr_ctx *ctx, double *xyz_host);

/* Operator matrices for operator-level tests: id 0..6 = M0..M6 (row-major doubles, host).
 * fr_operator_dims gives rows, cols. */
int fr_operator_dims(const fr_ctx *ctx, int id, int64_t *rows, int64_t *cols);
int fr_get_operator(const fr_ctx *ctx, int id, double *buf_host);

/* Host copies of the setup tables, for tests.  pairs: int32 [npairs][4] = sigmaL, elemL, sigmaR, elemR in
 * iteration order; normals: [npairs][ndims] unit normal of the L side; jn: [npairs][2] = (J n)_L, (J n)_R
 * (Eq 14, 16-17).  metrics: smat [ndims*ndims][N_u][ld] (S = J*J^-1, Eq 12) and rcpj [N_u][ld] (1/J). */
int fr_get_pairs(const fr_ctx *ctx, int32_t *pairs_host, double *normals_host, double *jn_host);
int fr_get_metrics(const fr_ctx *ctx, double *smat_host, double *rcpj_host);

/* rhs = -div f(u, grad u)  (Eq 19 :243; the seven parts of BASELINE.json north_star).
 * u_dev, rhs_dev: [N_u][N_V][ld] in the context's precision, device; u is not modified; rhs must not
 * alias u.  work_dev: >= fr_workspace_bytes() device bytes, 256-byte aligned, caller-owned.
 * stream: a cudaStream_t (as void*).  Asynchronous; no host synchronisation.  Pad columns
 * (element index >= n_elems) of rhs are left untouched.  Non-finite states are not detected (A19). */
int fr_rhs(fr_ctx *ctx, const void *u_dev, void *rhs_dev, void *work_dev, void *stream);

/* fr_rhs for callers that cannot allocate device memory (code under CUDA graph capture, serving loops, harnesses that forbid
 * cudaMalloc): the scratch of the kernel sequence lives in a static device array of FR_STATIC_WORK_BYTES inside the library
 * instead of a caller-owned work_dev.  Same arguments, layouts and result (bit for bit) as fr_rhs.  Calls no cudaMalloc /
 * cudaFree / allocating library routine; the address of the array is resolved once per device (cudaGetSymbolAddress on the
 * first call with that device current -- make that first call outside graph capture).  Contexts whose right-hand-side scratch
 * (fr_stepper_workspace_bytes(ctx, FR_STEPPER_EULER) minus one state register) exceeds FR_STATIC_WORK_BYTES are rejected with
 * FR_ENOMEM and a message naming both sizes.  Every GPU that loads the library holds the array until the process exits.  ALL
 * calls on a device share it, whatever the context or stream: two calls that overlap on the GPU race; serialise them (one
 * stream, or events).  The array keeps the previous call's contents; the kernels write every scratch value before reading it,
 * so nothing needs clearing between calls. */
#define FR_STATIC_WORK_BYTES (32 * 1024 * 1024)
int fr_rhs_static(fr_ctx *ctx, const void *u_dev, void *rhs_dev, void *stream);

/* fr_rhs with a CUDA event recorded on `stream` before each kernel and after the last; synchronises the
 * stream and returns, for each of the *n_kernels launch groups, its duration ms[i] and a name
 * (names_host: max_kernels x 32 chars).  For measurement only. */
int fr_rhs_profiled(fr_ctx *ctx, const void *u_dev, void *rhs_dev, void *work_dev, void *stream, int max_kernels,
                    int *n_kernels, float *ms_host, char *names_host);

/* One classical RK4 step, u advanced in place; four fr_rhs evaluations.  Pad columns (element index
 * >= n_elems) of u are left untouched by every stepper. */
int fr_rk4_step(fr_ctx *ctx, void *u_dev, double dt, void *work_dev, void *stream);

/* One forward Euler step u <- u + dt R(u) (Table 1 :263).  work_dev: >= fr_stepper_workspace_bytes(FR_STEPPER_EULER). */
int fr_euler_step(fr_ctx *ctx, void *u_dev, double dt, void *work_dev, void *stream);

/* One step of the Dormand-Prince 5(4) pair (Table 1 :263 "DOPRI5"; the published tableau, reading A24): seven fr_rhs
 * evaluations; u advanced in place with the fifth-order weights.  err_dev (device, may be NULL): receives the RMS over
 * all n_elems*N_u*N_V values of the embedded error estimate dt * sum_i (b5_i - b4_i) k_i, reduced in a fixed order
 * (bit-reproducible; FR_EUNSUPPORTED with a non-NULL err_dev on a mixed-mesh context).  Step-size control is the caller's.  work_dev: >= fr_stepper_workspace_bytes(FR_STEPPER_DOPRI5). */
int fr_dopri5_step(fr_ctx *ctx, void *u_dev, double dt, void *work_dev, void *stream, double *err_dev);

/* out = sum_i coef[i] * in[i] over state matrices (device, context precision; n_in <= 8; out may alias an input; pad columns
 * untouched): the register update the steppers above are built from, for callers that write their own stepper -- e.g. one
 * with a halo exchange between the stages (domain decomposition, partition.py). */
int fr_state_lincomb(fr_ctx *ctx, int n_in, const void *const *in_dev, const double *coef_host, void *out_dev, void *stream);

/* End-to-end variant with HOST buffers: copies u_host -> u_dev (H2D), evaluates fr_rhs, copies
 * rhs_dev -> rhs_host (D2H), all asynchronously on `stream` (pinned host memory recommended).
 * u_dev / rhs_dev / work_dev are caller-allocated device staging buffers as in fr_rhs. */
int fr_rhs_host(fr_ctx *ctx, const void *u_host, void *rhs_host, void *u_dev, void *rhs_dev, void *work_dev,
                void *stream);

/* Roofline denominators of the current CUDA device, measured: FP64 and FP32 FMA throughput (TFLOP/s, FMA-chain
 * microbenchmark, 2 flops per FMA) and device-to-device copy bandwidth (GB/s, read + write bytes over 2 GiB).  Needs about
 * 4 GiB of free device memory for a moment; synchronises the device.  Not part of the right-hand-side path. */
int fr_measure_peaks(double *fp64_tflops_host, double *fp32_tflops_host, double *copy_gbs_host);

/* Frees host objects and the library's own constant uploads.  NULL is allowed. */
void fr_teardown(fr_ctx *ctx);

/* Text of the last error on this context (or of the last failed fr_setup_mesh if ctx == NULL).
 * The pointer stays valid until the next failing call on the same context. */
const char *fr_last_error(const fr_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif
