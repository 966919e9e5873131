// neb_internal.h — declarations shared by the translation units of libneb.so (not installed).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string>
#include <vector>

#include "../../include/neb.h"

namespace neb {

constexpr double kEps0 = 8.8541878128e-12;                 // F/m (reading S3)
constexpr double kCoulomb = 1.0 / (4.0 * 3.14159265358979323846 * kEps0);
constexpr int kRec = 20;                                   // doubles per frame-table record
constexpr int kPad = 128;                                  // matrix dimension is padded to a multiple of this
#define NEB_IMG_CHUNK 32                                   // periodic copies per kernel launch (shared-memory table)
constexpr int kDistBlock = 256;                            // columns per block of the distributed factorisation (neb_dist.cu)
constexpr int kMaxImages = 16384;                          // copies per element accepted by neb_assemble

// Frame tables (a1), elements sorted by kind: [rect | tri | wire].  SoA, field-major:
// rec[f * stride + j], f < kRec (fields listed in neb_influence.cuh).
struct GeoTables {
  const double* rec;
  const int32_t* uniform;   // 3 per 64-element window: [0] 1 if all its elements share one set of unit axes (bitwise);
                            // [1], [2] bit k: rectangles 2k, 2k+1 are strip neighbours along local X / Z (tile_uniform_kernel)
  int64_t stride;
  int32_t n_rect, n_tri, n_wire;
};

// One FastVolume map (neb_fastvol.cu): a 32-byte record (Phi, Ex, Ey, Ez) per node, i fastest.
struct FastVol {
  const double4* nodes = nullptr;
  int nx = 0, ny = 0, nz = 0;
  double o[3] = {0, 0, 0}, h[3] = {1, 1, 1};
};

struct StageStat {
  double ms = 0.0;
  int64_t launches = 0;
};

}  // namespace neb

struct neb_ctx {
  int device = 0;
  cudaStream_t stream = nullptr;
  cudaStream_t side_stream = nullptr;   // LU look-ahead: next panel, concurrent with the trailing update
  cudaStream_t left_stream = nullptr;   // LU: row exchanges of the finished columns LEFT of the current block (nothing waits for them
                                        // before the solves), off the streams that carry the factorisation
  cudaEvent_t ev_next = nullptr, ev_panel = nullptr, ev_chain = nullptr, ev_left = nullptr;
  cudaMemPool_t pool = nullptr;   // staging temporaries (stream-ordered, memory kept across syncs)
  int num_sms = 0;
  int cluster_max_ctas = 0;   // largest cluster the device schedules for the LU panel kernel (set by lu_init_device)
  std::string err;

  // options
  int math_fast = 1;
  int lu_nb = 64;
  int profile = 0;
  int lu_lookahead = 1; // 1: factor panel k+1 on the side stream while panel k's trailing update runs
  int panel_mode = 0;   // 0: cluster kernel where it fits, 1: grid-wide cooperative kernel only
  int solver = 0;       // NEB_OPT_SOLVER: 0 = LU (OptLU), 1 = one-sided Jacobi SVD (OptSVD), used by the NEXT factorisation
  double svd_rcond = 1e-10;   // singular values <= svd_rcond x the largest are dropped (neb_set_svd_cutoff)
  int pair_strips = 1;  // NEB_OPT_PAIR_STRIPS: strip-neighbour rectangles evaluated as pairs (read by neb_assemble)
  int eval_splits = 0;  // 0: element/charge chunks chosen from the point count; k: always k chunks (shard-invariant bits)

  // scale-out of the solve (neb_dist.cu): 256-column blocks dealt cyclically to dist_world contexts; 1 = not distributed
  int dist_world = 1, dist_rank = 0;
  int dist_mode = 0;              // set by neb_dist_configure (world = 1 allowed: the same code on one context)
  bool dist_scaled = false;       // the agreed row scales have been applied (neb_dist_row_scales)
  int64_t ncol_loc = 0;           // columns of d_K held here (npad when not distributed)

  // geometry
  int64_t n = 0, npad = 0, stride = 0;
  int32_t n_rect = 0, n_tri = 0, n_wire = 0, n_img = 0;
  double* d_rec = nullptr;        // kRec * stride
  int32_t* d_uniform = nullptr;   // 3 x stride / 64 window flags and pair masks (see GeoTables)
  int32_t* d_perm = nullptr;      // sorted position -> caller index
  double* d_colloc = nullptr;     // 3 * stride, sorted order
  double* d_normal = nullptr;     // 3 * stride, sorted order
  int32_t* d_bc_kind = nullptr;   // sorted
  double* d_bc_value = nullptr;   // sorted
  double* d_diag = nullptr;       // sorted: 1/(2 eps0 lambda) on dielectric rows, else 0
  double* d_img = nullptr;        // copies sorted by length (slot 0 = the zero shift), packed in chunks of NEB_IMG_CHUNK: [chunk][3][32]
  int64_t img_cap = 0;            // chunks allocated
  std::vector<double> h_img_len;  // their lengths (host)
  double adaptive_far = 0.0;      // Adaptive Modelling: copies at least this far are simplified in neb_eval (0 = off)
  int32_t* d_flag = nullptr;      // device error flags (validation, singular pivot)

  // matrix / factors
  double* d_K = nullptr;          // npad x ncol_loc column-major
  double* d_rscale = nullptr;     // npad
  int32_t* d_ipiv = nullptr;      // npad (0-based absolute row)
  int32_t* d_rowperm = nullptr;   // npad: composed row permutation of the factorisation
  double* d_b = nullptr;          // npad, unscaled RHS (sorted order)
  double* d_x = nullptr;          // 16 * npad: running values and solved values of up to 8 right-hand sides (neb_trisolve.cu)
  double* d_dinv = nullptr;       // inverses of the 64x64 diagonal blocks of L and U: 2 * (npad/64) * 4096
  double* d_sigma = nullptr;      // n, caller order
  void* d_panel_ws = nullptr;     // LU panel exchange buffers
  // OptSVD (neb_svd.cu): right singular vectors, squared singular values (+ their maximum in slot npad), weights
  double* d_V = nullptr;
  double* d_s2 = nullptr;
  double* d_svd_w = nullptr;
  int factored_with = 0;          // which factors are resident: 0 LU, 1 SVD
  int svd_sweeps = 0;
  bool assembled = false, factored = false, have_sigma = false;

  // space charges: SoA x,y,z,q (4 * q_cap)
  double* d_charges = nullptr;
  int64_t q = 0, q_cap = 0;
  // line charges from the voxelisation (Alg. 3): SoA x, y, z_start, z_stop, lambda (5 * line_cap)
  double* d_lines = nullptr;
  int64_t n_lines = 0, line_cap = 0;

  neb::FastVol fastvol[NEB_FASTVOL_SLOTS];

  double* d_static_partial = nullptr;   // device address of neb_field.cu's file-scope scratch array (neb_eval_static)

  // scratch for partial sums / staging
  double* d_scratch = nullptr;
  size_t scratch_bytes = 0;

  // stats
  double counter[NEB_COUNTER_COUNT] = {0, 0, 0};
  int64_t launches = 0;
  neb::StageStat stat[NEB_STAGE_COUNT];
  cudaEvent_t ev0[NEB_STAGE_COUNT] = {}, ev1[NEB_STAGE_COUNT] = {};
};

namespace neb {

// error helpers ---------------------------------------------------------------------------------
neb_status fail(neb_ctx* c, neb_status st, const std::string& msg);
#define NEB_CUDA(c, expr)                                                                         \
  do {                                                                                            \
    cudaError_t e_ = (expr);                                                                      \
    if (e_ != cudaSuccess)                                                                        \
      return neb::fail((c), e_ == cudaErrorMemoryAllocation ? NEB_ENOMEM : NEB_ECUDA,             \
                       std::string(#expr) + ": " + cudaGetErrorString(e_));                       \
  } while (0)
#define NEB_TRY(expr)                 \
  do {                                \
    neb_status s_ = (expr);           \
    if (s_ != NEB_OK) return s_;      \
  } while (0)

neb_status ensure_scratch(neb_ctx* c, size_t bytes);
bool is_device_pointer(const void* p);
int64_t dist_local_cols(int64_t npad, int world, int rank);   // neb_dist.cu: columns of the matrix a rank holds

struct StageTimer {   // records device time of a stage when profiling is on
  neb_ctx* c;
  int stage;
  int64_t l0;
  StageTimer(neb_ctx* c_, int stage_);
  ~StageTimer();
};

// neb_field.cu ------------------------------------------------------------------------------------
// Phi/E at m device points (SoA) from the elements (weights in rec field 15) and/or the charges.
neb_status field_at_points(neb_ctx* c, int64_t m, const double* d_pts, bool use_elements, bool use_charges,
                           double* d_phi, double* d_E);
// neb_eval_static: the same evaluation with the partial sums in a fixed file-scope device array (no allocation)
neb_status field_static_init(neb_ctx* c);   // cudaGetSymbolAddress of that array, once per context, from neb_create
neb_status field_at_points_static(neb_ctx* c, int64_t m, const double* d_pts, double* d_phi, double* d_E);
neb_status assemble_matrix(neb_ctx* c);   // a3 + S15 row scales (computed, not yet applied)
neb_status scale_matrix_rows(neb_ctx* c); // applies the row scales in place
neb_status form_rhs(neb_ctx* c);          // a4 -> d_b (unscaled, sorted order)
neb_status finish_sigma(neb_ctx* c, const double* d_x);   // solved values (sorted order) -> d_sigma (caller order) and the table weights

// neb_lu.cu ---------------------------------------------------------------------------------------
neb_status lu_init_device(neb_ctx* c);    // per-device kernel attributes (dynamic shared memory, cluster size); from neb_create
neb_status lu_factor(neb_ctx* c);         // a5, in place on d_K (already row-scaled)
// neb_trisolve.cu: a6, nrhs right-hand sides d_b[k * npad + i] (unscaled, sorted order) -> d_out[k * npad + i]
neb_status lu_solve(neb_ctx* c, const double* d_b, int nrhs, double* d_out);
neb_status trisolve_init_device(neb_ctx* c);
// neb_svd.cu: OptSVD; factors_solve = the solve on whichever factors are resident
neb_status svd_factor(neb_ctx* c);
neb_status svd_solve(neb_ctx* c, const double* d_b, int nrhs, double* d_out);
neb_status factors_solve(neb_ctx* c, const double* d_b, int nrhs, double* d_out);
size_t lu_panel_ws_bytes(int num_sms);
// launch wrappers of the LU update kernels (A: column-major with leading dimension ld; Lp/ldl: the L operand, row index absolute)
void lu_launch_laswp(neb_ctx* c, cudaStream_t st, double* A, int64_t ld, int64_t k, int npiv, int64_t c_lo, int64_t c_hi, int64_t skip_lo, int64_t skip_hi);
void lu_launch_trsm(neb_ctx* c, cudaStream_t st, double* A, int64_t ld, const double* Lp, int64_t ldl, int64_t k, int64_t c_first, int64_t ncols);
void lu_launch_gemm(neb_ctx* c, cudaStream_t st, double* A, int64_t ld, const double* Lp, int64_t ldl, int64_t k, int K, int64_t r0, int64_t m,
                    int64_t c_first, int64_t ncols, bool timed);
neb_status lu_finish_factors(neb_ctx* c);   // rowperm from ipiv

// neb_lu_cluster.cu: panel factorisation on one thread-block cluster (panels of <= 16 x 512 rows)
int panel_cluster_probe();
int64_t panel_cluster_max_rows(neb_ctx* c);
neb_status panel_cluster_launch(neb_ctx* c, double* A, int64_t k, cudaStream_t stream);

// neb_fastvol.cu (device pointers only; the ABI wrappers in neb_api.cu stage host arrays) --------------
neb_status fastvol_build(neb_ctx* c, int slot, int nx, int ny, int nz, const double* origin, const double* spacing, bool with_charges);
neb_status fastvol_eval(neb_ctx* c, int slot, int64_t m, const double* d_pts, double* d_phi, double* d_E);
neb_status fastvol_get(neb_ctx* c, int slot, double* d_values);
neb_status solve_weighting(neb_ctx* c, int nrhs, const double* d_w_caller, double* d_sigma_out);

// neb_voxel.cu -----------------------------------------------------------------------------------
neb_status voxelize_charges(neb_ctx* c, const double* origin, const double* voxel, const int32_t* dims, int64_t* n_lines_out);
void launch_line_kernel(neb_ctx* c, int64_t m, const double* d_pts, int splits, int64_t per_split, double* partial);

// neb_peaks.cu ------------------------------------------------------------------------------------
neb_status fp64_peak(neb_ctx* c, int kind, double* tflops);

}  // namespace neb
