/* neb.h — C ABI of the B200-native neBEM hot path (libneb.so).
 *
 * The calls follow the paper's statement of the problem (arxiv 2606.24154; "P:n" = line n of
 * PAPER.md) and BASELINE.json's north_star:
 *   neb_assemble         = LHMatrix()                         (Eq.(6))
 *   neb_solve            = InvertMatrix() + RHVector() + ValueKnCh() + Solve()  (Alg.1)
 *   neb_eval             = PFAtPoint() = ElePFAtPoint() + KnChPFAtPoint()       (Eq.(3),(4) P:70-78)
 *   neb_add_space_charge = UpdateSpaceCharge()                (Alg.2)
 *   neb_solve again      = UpdateFields(): RHVector() + Solve() on resident factors (Alg.4)
 *
 * Conventions common to every call
 *   - Plain C; no exception crosses the boundary; every call returns a neb_status and
 *     neb_last_error() holds a message for the last non-OK status of that context.
 *   - SI units: metres, volts, coulombs, C/m^2.  eps0 = 8.8541878128e-12 F/m.
 *   - Vectors are SoA: an array "3*n" is x[0..n) then y[0..n) then z[0..n).
 *   - Every array pointer may be a HOST or a DEVICE pointer (detected with
 *     cudaPointerGetAttributes; device pointers must live on the context's device).  Inputs are
 *     borrowed for the duration of the call and copied; outputs are caller-owned.
 *   - Work is ordered on the CUDA stream given to neb_create.  A call synchronises that stream
 *     only when it has to write to host memory.
 *   - Everything runs in the CUDA kernels of this library.  There is no CPU fallback: without a
 *     usable device neb_create fails with NEB_ECUDA.
 *   - State machine: create -> assemble -> (add_space_charge)* -> solve -> eval*; out-of-order
 *     calls return NEB_ESTATE.  neb_set_sigma also unlocks neb_eval.
 */
#ifndef NEB_H
#define NEB_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct neb_ctx neb_ctx; /* opaque; owns every device buffer it allocates */

typedef enum {
  NEB_OK = 0,
  NEB_EINVAL = 1,    /* bad argument (NULL, negative size, unknown kind, degenerate element)  */
  NEB_ENOMEM = 2,    /* device or host allocation failed                                     */
  NEB_ESTATE = 3,    /* call out of order                                                    */
  NEB_ESINGULAR = 4, /* zero or NaN pivot in the LU; OptSVD sweeps that do not converge          */
  NEB_ECUDA = 5      /* CUDA runtime error; message in neb_last_error                        */
} neb_status;

enum { NEB_RECT = 0, NEB_TRI = 1, NEB_WIRE = 2 };       /* element kinds  */
enum { NEB_BC_DIRICHLET = 0, NEB_BC_DIELECTRIC = 1 };   /* row kinds                            */

/* Options for neb_set_option. */
enum {
  NEB_OPT_MATH = 0,     /* 1 (default): hand-written log/atan2/sqrt/rcp sequences; 0: CUDA libm  */
  NEB_OPT_LU_BLOCK = 1, /* LU outer block width (64, 128 or 256) once the trailing matrix is <= 4096 rows;
                           default 64; above: 128 up to 8192 rows, 512 up to 24576, 1024 beyond (panels are 64 wide) */
  NEB_OPT_PROFILE = 2,  /* 1: record per-stage CUDA-event timings (neb_stage_ms); default 0      */
  NEB_OPT_LU_PANEL = 3, /* 0 (default): panel kernel on one thread-block cluster (any height up to 131072 rows);
                           1: the grid-wide cooperative kernel of round 1 (cross-check; n <= 56704) */
  NEB_OPT_EVAL_SPLITS = 5, /* 0 (default): neb_eval splits the elements / charges into as many chunks as fill the GPU for
                           the given number of points (few points -> many chunks); k > 0: always k chunks, so that the
                           fixed-order partial sums, hence the result BITS, do not depend on how many points a call
                           (or a rank of a sharded evaluation) is given                                          */
  NEB_OPT_PAIR_STRIPS = 7, /* 1 (default): two rectangles of the table that are neighbours of one strip (same plane and axes, a
                           shared edge, found by neb_assemble) are evaluated together, sharing the edge's two corner
                           distances and its logarithm; 0: every element on its own.  Read by the next neb_assemble   */
  NEB_OPT_SOLVER = 6,   /* InvertMatrix: 0 (default) = OptLU, the blocked LU; 1 = OptSVD, one-sided Jacobi SVD and the
                           minimum-norm least-squares solution (for meshes with coincident / overlapping panels, whose
                           matrix is rank-deficient: the LU reports NEB_ESINGULAR there).  Read at the next factorisation
                           (the first neb_solve after neb_assemble)                                              */
  NEB_OPT_LU_LOOKAHEAD = 4 /* 1 (default): panel k+1 is factored on an internal stream while the trailing
                           update of panel k runs (cluster panels only); 0: one stream, and
                           NEB_STAGE_LU_GEMM is then timed alone                                 */
};

/* Stages for neb_stage_ms. */
enum {
  NEB_STAGE_GEOMETRY = 0, /* a1 frame tables                                   */
  NEB_STAGE_ASSEMBLE = 1, /* a3 influence matrix kernel                        */
  NEB_STAGE_EQUIL = 2,    /* row equilibration (reading S15)                   */
  NEB_STAGE_LU = 3,       /* a5 factorisation                                  */
  NEB_STAGE_LU_GEMM = 4,  /* a5 trailing update (DMMA) only, subset of LU      */
  NEB_STAGE_RHS = 5,      /* a4                                                */
  NEB_STAGE_TRISOLVE = 6, /* a6                                                */
  NEB_STAGE_EVAL = 7,     /* a7 fused element kernel alone                     */
  NEB_STAGE_CHARGES = 8,  /* a8 point-charge direct sum kernel                 */
  NEB_STAGE_REDUCE = 9,   /* fixed-order sum of the per-chunk partials of a7/a8 */
  NEB_STAGE_FASTVOL = 10, /* FastVolume: node packing and trilinear lookups    */
  NEB_STAGE_COUNT = 11
};
#define NEB_FASTVOL_SLOTS 4

/* Creates a context on `device`.  `cuda_stream` is a cudaStream_t (e.g. torch's current stream),
 * NULL = the legacy default stream.  NEB_ECUDA if the device is absent or not sm_100. */
neb_status neb_create(neb_ctx** out, int device, void* cuda_stream);
void neb_destroy(neb_ctx* ctx);
const char* neb_last_error(const neb_ctx* ctx);
neb_status neb_set_option(neb_ctx* ctx, int32_t option, int64_t value);

/* LHMatrix: builds the frame tables (a1) and the dense n*n fp64 influence matrix (a3)
 * on the device, column-major, and scales its rows (S15).
 *
 * Elements, in GLOBAL coordinates (length n each; vectors 3*n SoA):
 *   kind      NEB_RECT / NEB_TRI / NEB_WIRE
 *   v0        corner (rect), right-angle vertex (tri), start point (wire)
 *   e1, e2    the two PERPENDICULAR edge vectors from v0 (|cos| <= 1e-9, else NEB_EINVAL; rect: sides; tri: legs, hypotenuse from
 *             v0+e1 to v0+e2, P:123-127 with reading S2; wire: e1 = axis vector, e2 ignored).
 *             The unit normal is n = e2 x e1 / |e2 x e1|, so that (e1^, n, e2^) is the paper's
 *             local (X, Y, Z) of P:119.
 *   radius    wire radius r_w (wires only; may be NULL if there are no wires).  A wire's
 *             sigma is a surface density: line density = 2 pi r_w sigma (reading S24).
 *   colloc    3*n collocation points, or NULL = centroids (S4: rectangle centre, triangle
 *             v0+(e1+e2)/3, wire: mid-length on the surface).
 *   bc_kind   NEB_BC_DIRICHLET: row i is  sum_j K_ij sigma_j = bc_value[i] - Phi_sc(p_i)   (Eq.5)
 *             NEB_BC_DIELECTRIC: row i is the normal-displacement condition (reading S8)
 *               sum_j (1/4 pi eps0) n_i.E'_j(p_i) sigma_j + sigma_i/(2 eps0 lambda_i) = -n_i.E_sc(p_i),
 *               lambda_i = (eps_plus - eps_minus)/(eps_plus + eps_minus); eps_plus is the relative
 *               permittivity on the +n side.  bc_value is ignored on these rows.
 *   eps_plus, eps_minus   may be NULL if no row is dielectric.
 *   n_img, img_shift      periodic copies (reading S12): 3*n_img SoA shift vectors, which must
 *             include (0,0,0); every coefficient sums the element's copies.  NULL / 0 = none.
 *             The same copies are applied by neb_eval; never to space charges.  At most 16384 copies
 *             (70 x 70 repetitions); beyond 32 the kernels run once per 32 copies.
 * Errors: NEB_EINVAL (n <= 0, NULL required array, unknown kind, zero-length edge, wire without
 * radius, eps_plus == eps_minus on a dielectric row), NEB_ENOMEM, NEB_ECUDA. */
neb_status neb_assemble(neb_ctx* ctx, int64_t n, const int32_t* kind, const double* v0, const double* e1,
                        const double* e2, const double* radius, const double* colloc, const int32_t* bc_kind,
                        const double* bc_value, const double* eps_plus, const double* eps_minus, int32_t n_img,
                        const double* img_shift);

/* InvertMatrix + RHVector + Solve.  The first call factorises P K = L U in place (blocked,
 * partial pivoting, trailing update on FP64 DMMA; factors stay resident, no explicit inverse:
 * reading S13).  Every call forms the RHS from the boundary values and the current space
 * charges (S10) and does the two triangular solves.  sigma_out (n) may be NULL.
 * Errors: NEB_ESTATE before neb_assemble; NEB_ESINGULAR. */
neb_status neb_solve(neb_ctx* ctx, double* sigma_out);

/* Sets the charge densities used by neb_eval / neb_fastvol_build directly (n values, caller's element
 * order): a test hook, and the way to evaluate a weighting field (sigma from neb_solve_weighting). */
neb_status neb_set_sigma(neb_ctx* ctx, const double* sigma);

/* Adaptive Modelling (Table 2; reading S28): in neb_eval and neb_fastvol_build, a periodic copy of
 * an element whose shift vector is at least far_distance (m) long is represented by the element's total charge
 * sigma_j A_j at the copy's centroid instead of its exact closed form; nearer copies and the element itself stay
 * exact.  An approximation (error of a far copy's contribution ~ (element size / distance)^2), off by default
 * (far_distance = 0); the matrix assembly is never simplified.  Takes effect from the next neb_eval. */
neb_status neb_set_adaptive(neb_ctx* ctx, double far_distance);

/* Weighting field (P:222 CreateWtFldFastVolPF; reading S26): solves K sigma_w = b_w on the RESIDENT LU
 * factors, b_w = bc_value_w on Dirichlet rows (1 on the read-out electrode's panels, 0 on every other
 * conductor), 0 on dielectric rows, no space charge.  bc_value_w and sigma_w_out hold n values in the
 * caller's element order.  Leaves the context's own sigma and right-hand side untouched.
 * Errors: NEB_ESTATE before the first neb_solve (no factors yet). */
neb_status neb_solve_weighting(neb_ctx* ctx, const double* bc_value_w, double* sigma_w_out);
/* The same for n_rhs read-out electrodes at once ("the same inverted matrix ... can be reused"): bc_value_w
 * and sigma_w_out hold n_rhs rows of n values (row k = electrode k).  The triangular solves take up to 8 right-hand
 * sides per pass over the factors, so that 8 electrodes cost one reading of the 8 n^2 bytes of L and U, not eight. */
neb_status neb_solve_weighting_multi(neb_ctx* ctx, int32_t n_rhs, const double* bc_value_w, double* sigma_w_out);

/* FastVolume (P:179, P:222 CreateFastVolPF; reading S25).  neb_fastvol_build precomputes Phi and E, from
 * the context's current sigma (all elements with their periodic copies) and, if with_charges != 0, the
 * space charges, at the nx*ny*nz nodes origin + (i hx, j hy, k hz) of a uniform grid and keeps them on the
 * device in slot `slot` (0 .. NEB_FASTVOL_SLOTS-1; e.g. 0 = field, 1.. = weighting fields); rebuilding a
 * slot frees the old map.  origin and spacing are 3 HOST doubles each.
 * neb_fastvol_eval: trilinear interpolation of each of Phi, Ex, Ey, Ez from the 8 nodes of the cell at m
 * points (3*m SoA, host or device); a point outside the grid's box (beyond a slack of 1e-9 cells) gets NaN.
 * neb_fastvol_get (test hook): the node values as 4 planes Phi, Ex, Ey, Ez of nx*ny*nz doubles, i fastest.
 * Errors: NEB_EINVAL (slot, fewer than 2 nodes on an axis, spacing <= 0, more than 2^28 nodes),
 * NEB_ESTATE (build before sigma exists; eval/get of an empty slot), NEB_ENOMEM. */
neb_status neb_fastvol_build(neb_ctx* ctx, int32_t slot, int32_t nx, int32_t ny, int32_t nz, const double* origin,
                             const double* spacing, int32_t with_charges);
neb_status neb_fastvol_eval(neb_ctx* ctx, int32_t slot, int64_t m, const double* pts, double* phi, double* E);
neb_status neb_fastvol_get(neb_ctx* ctx, int32_t slot, double* values);

/* PFAtPoint: Phi (m) and E (3*m SoA) at m points pts (3*m SoA) from all elements (with
 * their periodic copies) and all space charges; a charge exactly at a point is skipped
 * (reading S11).  Either output may be NULL.  m = 0 is allowed. */
neb_status neb_eval(neb_ctx* ctx, int64_t m, const double* pts, double* phi, double* E);

/* neb_eval without any allocation (for callers under CUDA graph capture, in tight serving loops, or in harnesses that
 * forbid cudaMalloc): the same kernels and the same result as neb_eval to rounding (the elements / charges may be cut
 * into fewer chunks, i.e. a different but equally fixed summation order), with the per-chunk partial sums in a
 * file-scope device array of 32 MiB that every GPU holds from the moment the library is loaded until the process exits,
 * instead of a buffer that grows with m.  Limits: m <= NEB_EVAL_STATIC_MAX_POINTS per call (NEB_EINVAL beyond, with
 * the limit in neb_last_error); pts, phi, E must be DEVICE pointers (NEB_EINVAL otherwise: staging a host buffer would
 * allocate); either output may be NULL.  The call issues kernels on the context's stream and calls no cudaMalloc,
 * cudaFree or other allocating routine.  All contexts of a device share the one array: calls that overlap on the GPU
 * (contexts on different streams) race on it; calls on one stream are ordered and need no clearing in between (every
 * call overwrites the part it reads).  With NEB_OPT_PROFILE = 1 the stage timers synchronise on their events after every
 * stage: leave profiling off (the default) where a synchronisation is not allowed, e.g. under stream capture. */
#define NEB_EVAL_STATIC_MAX_POINTS 65536
neb_status neb_eval_static(neb_ctx* ctx, int64_t m, const double* pts, double* phi, double* E);

/* UpdateSpaceCharge: q point charges, pos 3*q SoA (m), charge in coulomb.
 * replace != 0 discards the charges held so far; q = 0 with replace clears them. */
neb_status neb_add_space_charge(neb_ctx* ctx, int64_t q, const double* pos, const double* charge, int32_t replace);

/* Alg. 3, Point to Line Charge Reduction (Voxelization; reading S27): replaces the point charges
 * the context holds by line charges.  Grid of dims[a] voxels of size voxel[a] (m) from origin[a] (3 HOST values
 * each); voxel index = floor((p - origin)/voxel), clamped to the grid (a point outside counts in the nearest border
 * voxel: the total charge is conserved); every voxel that received at least one point becomes ONE line charge
 * through its centre, parallel to z, spanning its z extent, lambda = (its total charge)/voxel[2]; lines are kept
 * in voxel-index order (x fastest).  From then on neb_eval and the right-hand side of neb_solve sum over the lines
 * (closed form of Eq. 2 integrated along the line; a point exactly on a line's axis is skipped) and over any point
 * charges added LATER with replace = 0; neb_add_space_charge with replace != 0 discards lines and points.
 * A second call voxelises the points added since TOGETHER WITH the lines of the earlier call, each old line entering
 * as its total charge lambda (z_stop - z_start) at its centre, so that the total charge is conserved (the call needs
 * at least one point or line).  n_lines_out (host, may be NULL) receives the number of lines.  Voxel totals are
 * accumulated in fixed point with integer atomics: lambda is bit-reproducible from run to run (exact sum of the
 * charges, each taken with an absolute error below 2^-72 max|q|).  At most 2^26 charges.
 * neb_get_line_charges (test hook): 5*n_lines doubles SoA x, y, z_start, z_stop, lambda.
 * Errors: NEB_EINVAL (non-positive voxel size, dims < 1, more than 2^26 voxels or charges), NEB_ESTATE (no point
 * charges and no lines). */
neb_status neb_voxelize_space_charge(neb_ctx* ctx, const double* origin, const double* voxel, const int32_t* dims,
                                     int64_t* n_lines_out);
neb_status neb_get_line_charges(neb_ctx* ctx, double* lines);

/* Charge push of the synthetic dynamic loop (BASELINE configs[4], reading S23): pos += mu_dt * E,
 * 3*q values, in place.  Stateless; pos and E must both be device or both be host pointers. */
neb_status neb_push(neb_ctx* ctx, int64_t q, double* pos, const double* E, double mu_dt);

/* OptSVD (reading S31 of DESIGN.md).  With NEB_OPT_SOLVER = 1 neb_solve factorises the row-scaled matrix as
 * K V = U diag(s) by one-sided Jacobi rotations (16 npad^2 bytes of device memory: K and V) and returns
 * sigma = sum over s_j > rcond s_max of v_j (u_j . b) / s_j; neb_solve_weighting* and re-solves use the same factors.
 * neb_set_svd_cutoff: rcond in [0, 1), default 1e-10.  neb_get_singular_values (test hook): the npad singular values
 * in column order (the npad - n padding columns contribute exact ones), host or device, and the number of sweeps
 * the factorisation took (host, may be NULL); NEB_ESTATE without SVD factors.  neb_solve returns NEB_ESINGULAR if the
 * rotations have not died out after 60 sweeps (a regular mesh takes 15-20). */
neb_status neb_set_svd_cutoff(neb_ctx* ctx, double rcond);
neb_status neb_get_singular_values(neb_ctx* ctx, double* s_out, int32_t* sweeps);

/* Scale-out of the solve (InvertMatrix with OptLU, Alg. 1, for a matrix spread over
 * several GPUs).  Right-looking block LU with partial pivoting on a matrix whose 256-column blocks are dealt
 * cyclically to `world` contexts, one per GPU, one process each: block g lives on rank g % world; every rank holds
 * all rows of its blocks, the whole geometry and, after the factorisation, all pivots.  The library performs every
 * step of the arithmetic; the exchanges BETWEEN the steps belong to the caller (torch.distributed over NCCL / NVLink:
 * paper_2606_24154_b200/parallel.py, dist_solve): a minimum of the row scales, one broadcast per block, a 256-value
 * sum per block and triangle in the solves, one sum of the solution vector.  Order of calls on EVERY rank:
 *
 *   neb_dist_configure(rank, world)       on a fresh context; world = 1 runs the same code on one context
 *   neb_assemble(...)                     assembles the rank's column blocks only (8 npad ncol_local bytes); the padded
 *                                         dimension npad = neb_dist_npad() is a multiple of 256
 *   neb_dist_row_scales(s, 0)             s (npad, device) <- 1/max_j|K_ij| over THIS rank's columns (+inf: none);
 *   [caller: element-wise MIN over ranks] = the S15 row scales of the whole matrix
 *   neb_dist_row_scales(s, 1)             stores them and scales the local columns
 *   for g = 0 .. npad/256 - 1:
 *     owner g % world: neb_dist_factor_block(g, panel, piv, stream)   factors the block (4 panels of 64 columns on one
 *                                         cluster each, in-block row exchanges, TRSM, rank-64 DMMA updates) and packs
 *                                         rows 256 g .. npad of it into panel ((npad - 256 g) x 256, column-major,
 *                                         device) and its 256 pivot rows into piv (int32, device); stream (a
 *                                         cudaStream_t, NULL = the context's) lets the next block be factored beside
 *                                         the trailing update (look-ahead)
 *     [caller: broadcast panel, piv from the owner]
 *     all ranks: neb_dist_apply_block(g, panel, piv, part)            row exchanges, U12 = L11^-1 A12 and the rank-256
 *                                         DMMA update on the rank's columns right of block g (L read from panel), row
 *                                         exchanges on the columns left of it.  part 0: everything; part 1: only the
 *                                         columns of block g + 1 (no-op unless this rank owns it); part 2: the rest
 *   neb_dist_finish_factor(&singular)     composed row permutation; singular (host) = 1 if one of THIS rank's panels
 *                                         met a zero / NaN pivot [caller: MAX over ranks]
 *   neb_dist_rhs(y)                       y (npad, device) <- the scaled, row-permuted right-hand side (a4, replicated)
 *   forward, g ascending, acc = 0 (npad, device):  [caller: acc[256 g .. +256) <- its sum over the ranks]
 *     neb_dist_tri_block(0, g, y, acc)    owner: y_g <- L_gg^-1 (y_g - acc_g); acc[below] += L[below, g] y_g
 *   backward, g descending, acc = 0:      [same sum]
 *     neb_dist_tri_block(1, g, y, acc)    owner: y_g <- U_gg^-1 (y_g - acc_g); acc[above] += U[above, g] y_g
 *   [caller: x = sum over ranks of (y restricted to the rank's own blocks)]
 *   neb_dist_set_solution(x, sigma_out)   sigma in the caller's element order (n doubles, host or device, may be NULL);
 *                                         neb_eval, neb_fastvol_* and neb_add_space_charge then work as on one GPU
 *                                         (every rank a replica of the element tables); a new right-hand side repeats
 *                                         the steps from neb_dist_rhs on the resident factors.
 * neb_solve, neb_solve_weighting*, neb_get_matrix* return NEB_ESTATE on a distributed context.
 * Errors: NEB_EINVAL (rank/world, block index, a block this rank does not own, host pointers where device ones are
 * required), NEB_ESTATE (order of calls), NEB_ECUDA. */
#define NEB_DIST_BLOCK 256
neb_status neb_dist_configure(neb_ctx* ctx, int32_t rank, int32_t world);
int64_t neb_dist_npad(const neb_ctx* ctx);
neb_status neb_dist_row_scales(neb_ctx* ctx, double* scales, int32_t set);
neb_status neb_dist_factor_block(neb_ctx* ctx, int64_t g, double* panel, int32_t* piv, void* cuda_stream);
neb_status neb_dist_apply_block(neb_ctx* ctx, int64_t g, const double* panel, const int32_t* piv, int32_t part);
neb_status neb_dist_finish_factor(neb_ctx* ctx, int32_t* singular);
neb_status neb_dist_rhs(neb_ctx* ctx, double* y);
neb_status neb_dist_tri_block(neb_ctx* ctx, int32_t upper, int64_t g, double* y, double* acc);
neb_status neb_dist_set_solution(neb_ctx* ctx, const double* x, double* sigma_out);

/* Test hooks.  neb_get_matrix: the UNSCALED matrix in the caller's element order, n*n
 * column-major (K_out[i + j*n] = row i, column j); only between neb_assemble and the first
 * neb_solve (NEB_ESTATE afterwards: the factors overwrite it).  neb_get_rhs: the RHS the last
 * neb_solve used (unscaled, caller's order). */
neb_status neb_get_matrix(neb_ctx* ctx, double* K_out);
/* neb_get_matrix_rows (test hook for sizes whose whole matrix does not fit the host, C3: 20 GB): the UNSCALED rows
 * rows[0..n_rows) (caller's element indices, int32, host or device), as n_rows*n doubles ROW-major in the caller's
 * column order: K_out[r*n + j] = K(rows[r], j).  Same state rule as neb_get_matrix.  NEB_EINVAL for an index
 * outside [0, n). */
neb_status neb_get_matrix_rows(neb_ctx* ctx, int64_t n_rows, const int32_t* rows, double* K_out);
neb_status neb_get_rhs(neb_ctx* ctx, double* b_out);

/* Measurement aids: register-only FP64 microbenchmarks on all SMs.
 * kind 0: DFMA chains; kind 1: mma.sync m8n8k4 f64 (DMMA); kind 2: independent DFMA whose three source operands are
 * three different registers (what the FP64 pipe sustains for instructions shaped like the influence kernels'); kind 3:
 * the same with one multiplicand from the constant bank (a Horner step with a stored coefficient).
 * Result in TFLOP/s (FMA = 2 flop). */
neb_status neb_fp64_peak(neb_ctx* ctx, int32_t kind, double* tflops);

/* Accumulated device time (ms) and number of kernel launches of a stage since the last
 * neb_reset_stats; valid when NEB_OPT_PROFILE is 1.  neb_launch_count counts every kernel this
 * library launched on the context since creation (profiling on or off). */
neb_status neb_stage_ms(neb_ctx* ctx, int32_t stage, double* ms, int64_t* launches);
/* Work counters of the LAST factorisation / assembly, counted by the host code that issues the launches (exact):
 * NEB_COUNTER_GEMM_FLOP   flop of the DMMA trailing updates (2 m n k summed over the gemm_kernel launches);
 * NEB_COUNTER_LU_FLOP     2/3 npad^3, the whole factorisation of the padded matrix;
 * NEB_COUNTER_MATRIX_BYTES bytes of matrix the assembly kernel wrote (8 n npad). */
enum { NEB_COUNTER_GEMM_FLOP = 0, NEB_COUNTER_LU_FLOP = 1, NEB_COUNTER_MATRIX_BYTES = 2, NEB_COUNTER_COUNT = 3 };
neb_status neb_get_counter(neb_ctx* ctx, int32_t which, double* value);
neb_status neb_reset_stats(neb_ctx* ctx);
int64_t neb_launch_count(const neb_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* NEB_H */
