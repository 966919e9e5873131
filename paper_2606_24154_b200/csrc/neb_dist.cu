// neb_dist.cu — SURVEY §8(f).4: scale-out of the solve.  InvertMatrix/OptLU (Alg. 1) for a matrix
// that is spread over several GPUs: right-looking block LU with partial pivoting, 1-D block-cyclic by columns.
//
// Layout.  The padded matrix (npad a multiple of 256) is cut into blocks of kDistBlock = 256 columns; block g lives on
// rank g % world, a rank's blocks side by side in its d_K (column-major, leading dimension npad): the local block
// lb = g / world starts at local column 256 lb.  Rows are not distributed, so the pivot search of a panel and all of a
// block's in-block work (four 64-column panels, their row exchanges, TRSM and rank-64 updates) are local to the
// block's owner and run the single-GPU kernels unchanged (neb_lu_panel.cu, neb_lu.cu) on a base pointer shifted so
// that global column indices land in the local block.
//
// One block step g (neb_dist_factor_block on the owner, neb_dist_apply_block on every rank):
//   owner   factors the block's 256 columns (rows kb = 256 g .. npad) and packs rows kb.. of the block, 256 columns
//           of npad - kb doubles, into `panel`, the 256 pivot rows into `piv`;
//   caller  broadcasts panel and piv from the owner (NCCL over NVLink; (npad - kb) x 2 KB: 100 MB at npad = 5e4);
//   all     apply the block to their own columns right of it: row exchanges, U12 = L11^-1 A12 for the four panels with
//           the rank-64 updates inside the block row, then ONE rank-256 DMMA update of the local trailing columns with
//           L read from the broadcast panel (gemm_kernel's Lp operand); the columns left of the block get the row
//           exchanges only (their L factors follow the rows).
// Look-ahead: `part` splits the update — the rank that owns block g + 1 updates that block's 256 columns first
// (part 1), factors it on a side stream and hands it to the broadcast while its main stream and the other ranks are
// still in the trailing update (part 2): the panel chain and the broadcast hide behind the DMMA work as on one GPU.
//
// Solves (neb_dist_tri_block).  Column-distributed triangular solve: every rank accumulates acc = sum over ITS solved
// blocks j of T[:, j] x_j; at block g the caller sums acc[rows of g] over the ranks (256 doubles), the owner solves the
// 256 x 256 diagonal block and adds its column block's contribution to acc for the rows still open.  The factors are
// read once, spread over the ranks.
//
// The exchanges themselves are the caller's (paper_2606_24154_b200/parallel.py: torch.distributed); every step of the
// arithmetic is here.  With world = 1 the calls run the same code on one context (tested against neb_solve).
#include "neb_internal.h"

namespace neb {

int64_t dist_local_cols(int64_t npad, int world, int rank) {
  if (world <= 1) return npad;
  const int64_t nblk = npad / kDistBlock;
  return (nblk > rank ? (nblk - rank + world - 1) / world : 0) * kDistBlock;
}

namespace {

constexpr int DB = kDistBlock;

// number of local blocks whose global index is < g / <= g
inline int64_t blocks_before(int64_t g, int world, int rank) { return g > rank ? (g - rank + world - 1) / world : 0; }
inline int64_t blocks_upto(int64_t g, int world, int rank) { return g >= rank ? (g - rank) / world + 1 : 0; }

// y[i] = rscale[p] * b[p], p = rowperm[i]: the right-hand side in the factorisation's row order
__global__ void dist_permute_scale_kernel(const double* __restrict__ b, const double* __restrict__ rscale,
                                          const int32_t* __restrict__ rowperm, int64_t npad, double* __restrict__ y) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= npad) return;
  const int p = rowperm[i];
  y[i] = b[p] * rscale[p];
}

__global__ void dist_fix_scales_kernel(double* rscale, int64_t npad) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < npad && !(rscale[i] < 1e300)) rscale[i] = 1.0;
}

// y_g <- T_gg^-1 (y_g - t): the 256 x 256 diagonal block of L (unit lower) or U (upper) by substitution, one CTA of
// 256 threads, thread i owns row i.  T is read column by column straight from L2 (a column = 256 consecutive doubles),
// 8 columns are fetched ahead of the 8 dependent steps that use them.
template <bool UPPER>
__global__ void __launch_bounds__(DB) dist_diag_solve_kernel(const double* __restrict__ T, int64_t ld, const double* __restrict__ t,
                                                             double* __restrict__ y) {
  __shared__ double s_x[2][8];
  const int i = threadIdx.x;
  double v = y[i] - t[i];
  // group gi = columns 8 gi .. 8 gi + 7 (lower) or DB-1-8 gi downwards (upper); the next group's columns are in flight
  // while this group's 8 dependent steps run
  auto column = [&](int gi, int u) { return UPPER ? DB - 1 - (8 * gi + u) : 8 * gi + u; };
  double col[8], nxt[8];
#pragma unroll
  for (int u = 0; u < 8; ++u) col[u] = T[i + (int64_t)column(0, u) * ld];
  for (int gi = 0; gi < DB / 8; ++gi) {
    if (gi + 1 < DB / 8) {
#pragma unroll
      for (int u = 0; u < 8; ++u) nxt[u] = T[i + (int64_t)column(gi + 1, u) * ld];
    }
    double* sx = s_x[gi & 1];
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      const int j = column(gi, u);
      if (i == j) { if (UPPER) v = v / col[u]; sx[u] = v; }      // L has a unit diagonal
      __syncthreads();
      if (UPPER ? (i < j) : (i > j)) v = fma(-col[u], sx[u], v);
    }
#pragma unroll
    for (int u = 0; u < 8; ++u) col[u] = nxt[u];
  }
  y[i] = v;
}

// acc[i] += sum_j T[i][j] x[j], i in [r0, r1), j over the block's 256 columns.  CTA = 64 rows x 4 column groups of
// 64; a warp reads 32 consecutive rows of one column (256 B); the four group sums are added in a fixed order.
__global__ void __launch_bounds__(256) dist_gemv_kernel(const double* __restrict__ T, int64_t ld, const double* __restrict__ x,
                                                        int64_t r0, int64_t r1, double* __restrict__ acc) {
  __shared__ double s_x[DB];
  __shared__ double s_part[4][64];
  s_x[threadIdx.x] = x[threadIdx.x];
  __syncthreads();
  const int r = threadIdx.x & 63, cg = threadIdx.x >> 6;
  const int64_t i = r0 + (int64_t)blockIdx.x * 64 + r;
  double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
  if (i < r1) {
    const double* col = T + i + (int64_t)(cg * 64) * ld;
#pragma unroll 4
    for (int j = 0; j < 64; j += 4) {
      a0 = fma(col[(int64_t)(j + 0) * ld], s_x[cg * 64 + j + 0], a0);
      a1 = fma(col[(int64_t)(j + 1) * ld], s_x[cg * 64 + j + 1], a1);
      a2 = fma(col[(int64_t)(j + 2) * ld], s_x[cg * 64 + j + 2], a2);
      a3 = fma(col[(int64_t)(j + 3) * ld], s_x[cg * 64 + j + 3], a3);
    }
  }
  s_part[cg][r] = (a0 + a1) + (a2 + a3);
  __syncthreads();
  if (cg == 0 && i < r1) acc[i] += (s_part[0][r] + s_part[1][r]) + (s_part[2][r] + s_part[3][r]);
}

neb_status check_dist_block(neb_ctx* c, int64_t g, const char* who) {
  if (!c->assembled) return fail(c, NEB_ESTATE, std::string(who) + " before neb_assemble");
  if (g < 0 || g >= c->npad / DB) return fail(c, NEB_EINVAL, std::string(who) + ": block index outside [0, npad/256)");
  return NEB_OK;
}

}  // namespace
}  // namespace neb

using namespace neb;

extern "C" {

neb_status neb_dist_configure(neb_ctx* c, int32_t rank, int32_t world) {
  if (!c) return NEB_EINVAL;
  if (world < 1 || rank < 0 || rank >= world) return fail(c, NEB_EINVAL, "neb_dist_configure: need 0 <= rank < world");
  if (c->n != 0) return fail(c, NEB_ESTATE, "neb_dist_configure: call it on a fresh context, before the first neb_assemble");
  c->dist_world = world;
  c->dist_rank = rank;
  c->dist_mode = 1;
  return NEB_OK;
}

int64_t neb_dist_npad(const neb_ctx* c) { return c ? c->npad : 0; }

neb_status neb_dist_row_scales(neb_ctx* c, double* scales, int32_t set) {
  if (!c || !scales) return NEB_EINVAL;
  if (!c->dist_mode) return fail(c, NEB_ESTATE, "neb_dist_row_scales without neb_dist_configure");
  if (!c->assembled || c->factored) return fail(c, NEB_ESTATE, "neb_dist_row_scales: only between neb_assemble and the factorisation");
  if (!is_device_pointer(scales)) return fail(c, NEB_EINVAL, "neb_dist_row_scales: scales must be a device pointer");
  NEB_CUDA(c, cudaSetDevice(c->device));
  if (!set) {
    NEB_CUDA(c, cudaMemcpyAsync(scales, c->d_rscale, sizeof(double) * c->npad, cudaMemcpyDeviceToDevice, c->stream));
    return NEB_OK;
  }
  NEB_CUDA(c, cudaMemcpyAsync(c->d_rscale, scales, sizeof(double) * c->npad, cudaMemcpyDeviceToDevice, c->stream));
  dist_fix_scales_kernel<<<(unsigned)((c->npad + 255) / 256), 256, 0, c->stream>>>(c->d_rscale, c->npad);
  c->launches++;
  NEB_CUDA(c, cudaGetLastError());
  NEB_TRY(scale_matrix_rows(c));
  c->dist_scaled = true;
  return NEB_OK;
}

neb_status neb_dist_factor_block(neb_ctx* c, int64_t g, double* panel, int32_t* piv, void* cuda_stream) {
  if (!c || !panel || !piv) return NEB_EINVAL;
  if (!c->dist_mode) return fail(c, NEB_ESTATE, "neb_dist_factor_block without neb_dist_configure");
  NEB_TRY(check_dist_block(c, g, "neb_dist_factor_block"));
  if (!c->dist_scaled) return fail(c, NEB_ESTATE, "neb_dist_factor_block before neb_dist_row_scales(set)");
  if (g % c->dist_world != c->dist_rank) return fail(c, NEB_EINVAL, "neb_dist_factor_block: this rank does not own the block");
  if (!is_device_pointer(panel) || !is_device_pointer(piv)) return fail(c, NEB_EINVAL, "neb_dist_factor_block: panel and piv must be device pointers");
  NEB_CUDA(c, cudaSetDevice(c->device));
  cudaStream_t st = cuda_stream ? (cudaStream_t)cuda_stream : c->stream;
  const int64_t npad = c->npad, ld = npad, kb = g * DB, lc = (g / c->dist_world) * DB;
  if (g == 0) {
    c->counter[NEB_COUNTER_GEMM_FLOP] = 0.0;
    c->counter[NEB_COUNTER_LU_FLOP] = 2.0 / 3.0 * (double)npad * (double)npad * (double)npad;
  }
  // the block's columns under their GLOBAL indices: column kb of `A` is local column lc (only [kb, kb + 256) is touched)
  double* A = c->d_K + (lc - kb) * ld;
  for (int64_t k = kb; k < kb + DB; k += 64) {
    NEB_TRY(panel_cluster_launch(c, A, k, st));
    const int64_t in_cols = kb + DB - (k + 64);
    lu_launch_laswp(c, st, A, ld, k, 64, kb, kb + DB, k, k + 64);
    lu_launch_trsm(c, st, A, ld, A + k * ld, ld, k, k + 64, in_cols);
    lu_launch_gemm(c, st, A, ld, A + k * ld, ld, k, 64, k + 64, npad - (k + 64), k + 64, in_cols, false);
  }
  NEB_CUDA(c, cudaGetLastError());
  const size_t width = sizeof(double) * (size_t)(npad - kb);
  NEB_CUDA(c, cudaMemcpy2DAsync(panel, width, c->d_K + kb + lc * ld, sizeof(double) * (size_t)ld, width, DB, cudaMemcpyDeviceToDevice, st));
  NEB_CUDA(c, cudaMemcpyAsync(piv, c->d_ipiv + kb, sizeof(int32_t) * DB, cudaMemcpyDeviceToDevice, st));
  return NEB_OK;
}

neb_status neb_dist_apply_block(neb_ctx* c, int64_t g, const double* panel, const int32_t* piv, int32_t part) {
  if (!c || !panel || !piv || part < 0 || part > 2) return NEB_EINVAL;
  if (!c->dist_mode) return fail(c, NEB_ESTATE, "neb_dist_apply_block without neb_dist_configure");
  NEB_TRY(check_dist_block(c, g, "neb_dist_apply_block"));
  if (!c->dist_scaled) return fail(c, NEB_ESTATE, "neb_dist_apply_block before neb_dist_row_scales(set)");
  if (!is_device_pointer(panel) || !is_device_pointer(piv)) return fail(c, NEB_EINVAL, "neb_dist_apply_block: panel and piv must be device pointers");
  NEB_CUDA(c, cudaSetDevice(c->device));
  cudaStream_t st = c->stream;
  const int world = c->dist_world, rank = c->dist_rank;
  const int64_t npad = c->npad, ld = npad, kb = g * DB, ldl = npad - kb;
  if (part != 2)   // the pivots of the block (the owner's own are already there; same values)
    NEB_CUDA(c, cudaMemcpyAsync(c->d_ipiv + kb, piv, sizeof(int32_t) * DB, cudaMemcpyDeviceToDevice, st));
  // local columns right of the block: [c_right, ncol_loc); the next block's 256 columns, if they are here, come first
  int64_t c0 = blocks_upto(g, world, rank) * DB, c1 = c->ncol_loc;
  const bool owns_next = (g + 1) < npad / DB && (g + 1) % world == rank;
  if (part == 1) { if (!owns_next) return NEB_OK; c1 = c0 + DB; }
  if (part == 2 && owns_next) c0 += DB;
  const int64_t nc = c1 - c0;
  const double* Pb = panel - kb;                     // Pb[i + j * ldl] = element (absolute row i, block column j)
  if (nc > 0) {
    lu_launch_laswp(c, st, c->d_K, ld, kb, DB, c0, c1, c1, c1);      // the block's 256 exchanges in one launch
    for (int64_t k = kb; k < kb + DB; k += 64) {
      const double* Lk = Pb + (k - kb) * ldl;
      lu_launch_trsm(c, st, c->d_K, ld, Lk, ldl, k, c0, nc);
      lu_launch_gemm(c, st, c->d_K, ld, Lk, ldl, k, 64, k + 64, kb + DB - (k + 64), c0, nc, false);
    }
    lu_launch_gemm(c, st, c->d_K, ld, Pb, ldl, kb, DB, kb + DB, npad - (kb + DB), c0, nc, false);
  }
  if (part != 1) {   // the factors to the left follow the rows
    const int64_t left = blocks_before(g, world, rank) * DB;
    lu_launch_laswp(c, st, c->d_K, ld, kb, DB, 0, left, left, left);
  }
  NEB_CUDA(c, cudaGetLastError());
  return NEB_OK;
}

neb_status neb_dist_finish_factor(neb_ctx* c, int32_t* singular) {
  if (!c) return NEB_EINVAL;
  if (!c->dist_mode || !c->dist_scaled) return fail(c, NEB_ESTATE, "neb_dist_finish_factor: no distributed factorisation in progress");
  NEB_CUDA(c, cudaSetDevice(c->device));
  NEB_TRY(lu_finish_factors(c));
  int32_t h_flag = 0;
  NEB_CUDA(c, cudaMemcpyAsync(&h_flag, c->d_flag, sizeof(int32_t), cudaMemcpyDeviceToHost, c->stream));
  NEB_CUDA(c, cudaStreamSynchronize(c->stream));
  c->factored = true;
  if (singular) *singular = (h_flag & 2) ? 1 : 0;
  return NEB_OK;
}

neb_status neb_dist_rhs(neb_ctx* c, double* y) {
  if (!c || !y) return NEB_EINVAL;
  if (!c->dist_mode || !c->factored) return fail(c, NEB_ESTATE, "neb_dist_rhs before the distributed factorisation");
  if (!is_device_pointer(y)) return fail(c, NEB_EINVAL, "neb_dist_rhs: y must be a device pointer");
  NEB_CUDA(c, cudaSetDevice(c->device));
  NEB_TRY(form_rhs(c));
  dist_permute_scale_kernel<<<(unsigned)((c->npad + 255) / 256), 256, 0, c->stream>>>(c->d_b, c->d_rscale, c->d_rowperm, c->npad, y);
  c->launches++;
  NEB_CUDA(c, cudaGetLastError());
  return NEB_OK;
}

neb_status neb_dist_tri_block(neb_ctx* c, int32_t upper, int64_t g, double* y, double* acc) {
  if (!c || !y || !acc) return NEB_EINVAL;
  if (!c->dist_mode || !c->factored) return fail(c, NEB_ESTATE, "neb_dist_tri_block before the distributed factorisation");
  NEB_TRY(check_dist_block(c, g, "neb_dist_tri_block"));
  if (!is_device_pointer(y) || !is_device_pointer(acc)) return fail(c, NEB_EINVAL, "neb_dist_tri_block: y and acc must be device pointers");
  if (g % c->dist_world != c->dist_rank) return NEB_OK;          // not this rank's block: nothing to do
  NEB_CUDA(c, cudaSetDevice(c->device));
  StageTimer tt(c, NEB_STAGE_TRISOLVE);
  const int64_t npad = c->npad, ld = npad, kb = g * DB, lc = (g / c->dist_world) * DB;
  const double* Tcol = c->d_K + lc * ld;                         // the block's 256 columns, all rows
  if (upper) {
    dist_diag_solve_kernel<true><<<1, DB, 0, c->stream>>>(Tcol + kb, ld, acc + kb, y + kb);
    c->launches++;
    if (kb > 0) {
      dist_gemv_kernel<<<(unsigned)((kb + 63) / 64), 256, 0, c->stream>>>(Tcol, ld, y + kb, 0, kb, acc);
      c->launches++;
    }
  } else {
    dist_diag_solve_kernel<false><<<1, DB, 0, c->stream>>>(Tcol + kb, ld, acc + kb, y + kb);
    c->launches++;
    if (kb + DB < npad) {
      dist_gemv_kernel<<<(unsigned)((npad - kb - DB + 63) / 64), 256, 0, c->stream>>>(Tcol, ld, y + kb, kb + DB, npad, acc);
      c->launches++;
    }
  }
  NEB_CUDA(c, cudaGetLastError());
  return NEB_OK;
}

neb_status neb_dist_set_solution(neb_ctx* c, const double* x, double* sigma_out) {
  if (!c || !x) return NEB_EINVAL;
  if (!c->dist_mode || !c->factored) return fail(c, NEB_ESTATE, "neb_dist_set_solution before the distributed factorisation");
  if (!is_device_pointer(x)) return fail(c, NEB_EINVAL, "neb_dist_set_solution: x must be a device pointer");
  NEB_CUDA(c, cudaSetDevice(c->device));
  NEB_TRY(finish_sigma(c, x));
  if (sigma_out) {
    NEB_CUDA(c, cudaMemcpyAsync(sigma_out, c->d_sigma, sizeof(double) * c->n, cudaMemcpyDefault, c->stream));
    if (!is_device_pointer(sigma_out)) NEB_CUDA(c, cudaStreamSynchronize(c->stream));
  }
  return NEB_OK;
}

}  // extern "C"
