// neb_lu.cu — a5/a6: dense fp64 LU with partial pivoting on the resident, row-scaled influence
// matrix (InvertMatrix with OptLU, Alg. 1; readings S13 "keep the factors, no explicit
// inverse", S15, S16), and the two triangular solves (Solve).
//
// Right-looking blocked factorisation, panel width NB = 64, matrix column-major with leading
// dimension npad (a multiple of 128; the pad block is the identity, so every tile is full):
//   panel_kernel   one cooperative launch per panel: each CTA keeps its slab of panel rows in shared
//                  memory; per column one grid-wide exchange (candidate pivot + candidate row + diagonal
//                  row through global memory, one grid barrier), then the rank-1 update in shared memory
//   laswp_kernel   applies the panel's 64 row exchanges to the columns left and right of the panel
//   trsm_kernel    U12 = L11^-1 A12, one thread per column, the column in registers
//   gemm_kernel    A22 -= L21 U12 on the FP64 tensor cores: mma.sync.m8n8k4.f64 (SASS DMMA), 128x64 CTA
//                  tiles, operands staged by cp.async into padded (conflict-free) shared memory
// tcgen05/UMMA has no f64 kind, so the warp-level DMMA is the FP64 tensor path on sm_100a.
#include <cooperative_groups.h>

#include "neb_internal.h"

namespace neb {

constexpr int NB = 64;           // panel width
constexpr int kMaxBlockPanels = 16;   // widest outer block of lu_factor: 16 panels = 1024 columns
constexpr int PANEL_THREADS = 256;

// ------------------------------------------------------------------------------------------------
// grid barrier for the cooperative panel kernel (all CTAs co-resident: cooperative launch)
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void grid_barrier(unsigned int* counter, unsigned int target) {
  __syncthreads();
  if (threadIdx.x == 0) {
    __threadfence();
    atomicAdd(counter, 1u);
    unsigned int v;
    do {
      asm volatile("ld.acquire.gpu.u32 %0, [%1];" : "=r"(v) : "l"(counter) : "memory");
    } while (v < target);
    __threadfence();
  }
  __syncthreads();
}

struct PanelWs {          // global exchange buffers, double-buffered by step parity
  unsigned int counter;   // monotone barrier counter (reset by the host before each launch)
  int pad_[3];
  double cand_val[2][160];
  int cand_row[2][160];
  double cand_vec[2][160][NB];
  double diag_vec[2][NB];
};

size_t lu_panel_ws_bytes(int) { return sizeof(PanelWs); }

// One panel: columns [k, k+NB), rows [k, npad).  CTA b owns rows [k + b*mc, k + (b+1)*mc) (mc a
// multiple of 32), stored in shared memory column-major: sA[c * mc + r].
__global__ void __launch_bounds__(PANEL_THREADS) panel_kernel(double* __restrict__ A, int64_t ld, int64_t npad, int64_t k,
                                                              int mc, int32_t* __restrict__ ipiv, PanelWs* ws,
                                                              int32_t* __restrict__ flag) {
  extern __shared__ double sA[];
  __shared__ double s_prow[NB], s_drow[NB];
  __shared__ double s_wval[PANEL_THREADS / 32];
  __shared__ int s_wrow[PANEL_THREADS / 32];
  __shared__ int s_win_cta, s_win_row;
  const int tid = threadIdx.x, G = gridDim.x, b = blockIdx.x;
  const int64_t row0 = k + (int64_t)b * mc;
  const int nrows = (int)max((int64_t)0, min((int64_t)mc, npad - row0));   // rows this CTA really owns
  // load slab
  for (int idx = tid; idx < mc * NB; idx += PANEL_THREADS) {
    int r = idx % mc, c = idx / mc;
    sA[idx] = (r < nrows) ? A[(row0 + r) + (k + c) * ld] : 0.0;
  }
  __syncthreads();
  unsigned int epoch = 0;
  for (int j = 0; j < NB; ++j) {
    const int par = j & 1;
    const int64_t dr = k + j;                      // diagonal row of this step
    // (1) local pivot candidate: max |a[r][j]| over owned rows >= dr, ties -> lowest row
    double best = -1.0;
    int brow = 0x7fffffff;
    for (int r = tid; r < nrows; r += PANEL_THREADS) {
      int64_t gr = row0 + r;
      if (gr >= dr) {
        double v = fabs(sA[j * mc + r]);
        if (!(v == v)) v = 0.0;                    // NaN never wins; caught by the zero-pivot test
        if (v > best) { best = v; brow = (int)gr; }
      }
    }
    for (int o = 16; o > 0; o >>= 1) {
      double ov = __shfl_down_sync(0xffffffffu, best, o);
      int orow = __shfl_down_sync(0xffffffffu, brow, o);
      if (ov > best || (ov == best && orow < brow)) { best = ov; brow = orow; }
    }
    if ((tid & 31) == 0) { s_wval[tid >> 5] = best; s_wrow[tid >> 5] = brow; }
    __syncthreads();
    if (tid == 0) {
      for (int w = 1; w < PANEL_THREADS / 32; ++w)
        if (s_wval[w] > best || (s_wval[w] == best && s_wrow[w] < brow)) { best = s_wval[w]; brow = s_wrow[w]; }
      ws->cand_val[par][b] = best;
      ws->cand_row[par][b] = brow;
      s_win_row = brow;                            // local candidate row, for the publication below
    }
    __syncthreads();
    {
      int lrow = s_win_row;
      if (tid < NB && lrow != 0x7fffffff) ws->cand_vec[par][b][tid] = sA[tid * mc + (int)(lrow - row0)];
      if (tid < NB && dr >= row0 && dr < row0 + nrows) ws->diag_vec[par][tid] = sA[tid * mc + (int)(dr - row0)];
    }
    // (2) grid-wide exchange
    epoch += (unsigned)G;
    grid_barrier(&ws->counter, epoch);
    // (3) global winner
    if (tid < 32) {
      double wv = -1.0; int wr = 0x7fffffff, wc = 0;
      for (int c = tid; c < G; c += 32) {
        double v = __ldcg(&ws->cand_val[par][c]);
        int r = __ldcg(&ws->cand_row[par][c]);
        if (v > wv || (v == wv && r < wr)) { wv = v; wr = r; wc = c; }
      }
      for (int o = 16; o > 0; o >>= 1) {
        double ov = __shfl_down_sync(0xffffffffu, wv, o);
        int orow = __shfl_down_sync(0xffffffffu, wr, o);
        int oc = __shfl_down_sync(0xffffffffu, wc, o);
        if (ov > wv || (ov == wv && orow < wr)) { wv = ov; wr = orow; wc = oc; }
      }
      if (tid == 0) {
        s_win_cta = wc; s_win_row = wr;
        if (b == 0) {
          ipiv[dr] = wr;
          if (!(wv > 0.0)) atomicOr(flag, 2);      // zero / NaN pivot: NEB_ESINGULAR
        }
      }
    }
    __syncthreads();
    const int wrow = s_win_row, wcta = s_win_cta;
    if (tid < NB) {
      s_prow[tid] = __ldcg(&ws->cand_vec[par][wcta][tid]);
      s_drow[tid] = __ldcg(&ws->diag_vec[par][tid]);
    }
    __syncthreads();
    // (4) exchange rows dr <-> wrow inside the panel
    if (wrow != (int)dr && tid < NB) {
      if (wrow >= row0 && wrow < row0 + nrows) sA[tid * mc + (int)(wrow - row0)] = s_drow[tid];
      if (dr >= row0 && dr < row0 + nrows) sA[tid * mc + (int)(dr - row0)] = s_prow[tid];
    }
    __syncthreads();
    // (5) multipliers and rank-1 update of the columns to the right, rows below dr
    const double piv = s_prow[j];
    const double invp = (piv != 0.0) ? 1.0 / piv : 0.0;
    const int ncol = NB - 1 - j;
    for (int idx = tid; idx < mc * (ncol + 1); idx += PANEL_THREADS) {
      int r = idx % mc, cc = idx / mc;             // cc = 0: the multiplier column itself
      int64_t gr = row0 + r;
      if (r < nrows && gr > dr) {
        double l = sA[j * mc + r] * invp;
        if (cc == 0) {
          // written after every reader of this column in this pass has its own copy: readers below
          // recompute l from the unscaled value, so defer the store to the second pass
        } else {
          int c = j + cc;
          sA[c * mc + r] = fma(-l, s_prow[c], sA[c * mc + r]);
        }
      }
    }
    __syncthreads();
    for (int r = tid; r < nrows; r += PANEL_THREADS)
      if (row0 + r > dr) sA[j * mc + r] *= invp;
    __syncthreads();
  }
  // write the factored slab back
  for (int idx = tid; idx < mc * NB; idx += PANEL_THREADS) {
    int r = idx % mc, c = idx / mc;
    if (r < nrows) A[(row0 + r) + (k + c) * ld] = sA[idx];
  }
}

// The npiv (<= 256) row exchanges of the panels k, k + 64, ... applied in order to the columns [c_lo, c_hi), minus the
// columns [skip_lo, skip_hi) (the panel's own, and with look-ahead the next panel's, which were exchanged ahead of the
// others).  One thread per column; a whole 256-column block's exchanges take one launch.
__global__ void laswp_kernel(double* __restrict__ A, int64_t ld, int64_t k, int npiv, const int32_t* __restrict__ ipiv, int64_t c_lo,
                             int64_t c_hi, int64_t skip_lo, int64_t skip_hi) {
  __shared__ int s_piv[kMaxBlockPanels * NB];
  for (int t = threadIdx.x; t < npiv; t += blockDim.x) s_piv[t] = ipiv[k + t];
  __syncthreads();
  int64_t c = c_lo + (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= skip_lo) c += skip_hi - skip_lo;
  if (c >= c_hi) return;
  double* col = A + c * ld;
  for (int t = 0; t < npiv; ++t) {
    int p = s_piv[t];
    if (p != k + t) {
      double a = col[k + t], bb = col[p];
      col[k + t] = bb;
      col[p] = a;
    }
  }
}

// U12 = L11^-1 A12: rows [k, k+NB), columns [c_first + 64 b, c_first + 64 (b+1)) for CTA b.  One THREAD per column,
// the whole column (64 rows) in registers: no barrier inside the 63 dependent steps.  The substitution runs as 16
// rolled iterations of 4 steps on a register WINDOW that is rotated by 4 rows per iteration (static register indices,
// a loop body that stays in the instruction cache; the fully unrolled form was fetch-bound).  L11 sits in shared
// memory column-major with 64 rows of zeros below it, so window rows past the block's end are left alone.
constexpr int TRSM_THREADS = NB;
constexpr int TRSM_LD = 2 * NB;
constexpr size_t TRSM_SMEM = (size_t)NB * TRSM_LD * sizeof(double);
// L11 is read from Lp: Lp[i + j * ldl] = element (absolute row i, panel column j); on one GPU Lp = A + k * ld, in the
// distributed factorisation (neb_dist.cu) it is the broadcast panel.
__global__ void __launch_bounds__(TRSM_THREADS) trsm_kernel(double* __restrict__ A, int64_t ld, const double* __restrict__ Lp, int64_t ldl,
                                                            int64_t k, int64_t c_first) {
  extern __shared__ __align__(16) double s_trsm[];             // s_trsm[j * TRSM_LD + i] = L11[i][j], 0 for i >= NB
  const int tid = threadIdx.x;
  double* col = A + k + (c_first + (int64_t)blockIdx.x * NB + tid) * ld;
  double x[NB];
  {
    // thread j stages column j of L11: 32 independent 16-byte loads in flight (a rolled element loop over 64
    // threads would pay one L2 round trip per element)
    const double* lcol = Lp + k + tid * ldl;
#pragma unroll
    for (int i = 0; i < NB; i += 2) {
      const double2 v = *reinterpret_cast<const double2*>(lcol + i);
      x[i] = v.x; x[i + 1] = v.y;
    }
#pragma unroll
    for (int i = 0; i < NB; i += 2) {
      *reinterpret_cast<double2*>(s_trsm + tid * TRSM_LD + i) = make_double2(x[i], x[i + 1]);
      *reinterpret_cast<double2*>(s_trsm + tid * TRSM_LD + NB + i) = make_double2(0.0, 0.0);
    }
  }
#pragma unroll
  for (int i = 0; i < NB; i += 2) {
    const double2 v = *reinterpret_cast<const double2*>(col + i);
    x[i] = v.x; x[i + 1] = v.y;
  }
  __syncthreads();
#pragma unroll 1
  for (int it = 0; it < NB / 4; ++it) {
    const double* Lw = s_trsm + (it * 4) * TRSM_LD + it * 4;    // Lw[b * TRSM_LD + a] = L11[j0 + a][j0 + b], j0 = 4 it
#pragma unroll
    for (int b = 0; b < 4; ++b) {
      const double xj = x[b];
#pragma unroll
      for (int a = b + 1; a < NB; ++a) x[a] = fma(-Lw[b * TRSM_LD + a], xj, x[a]);
    }
    *reinterpret_cast<double2*>(col + it * 4) = make_double2(x[0], x[1]);
    *reinterpret_cast<double2*>(col + it * 4 + 2) = make_double2(x[2], x[3]);
#pragma unroll
    for (int a = 0; a < NB - 4; ++a) x[a] = x[a + 4];
    x[NB - 4] = 0.0; x[NB - 3] = 0.0; x[NB - 2] = 0.0; x[NB - 1] = 0.0;
  }
}

// ------------------------------------------------------------------------------------------------
// Trailing update C -= L * U on the FP64 tensor cores, any depth K (a multiple of 32):
//   C = A[r0 .. r0+m, c_first ..],  L = A[r0 .. r0+m, k .. k+K),  U = A[k .. k+K, c_first ..];
//   L is read through Lp (Lp[i + kk * ldl] = L[i][kk], absolute row i): A + k * ld on one GPU, the broadcast panel in
//   the distributed factorisation (neb_dist.cu).
// CTA tile 128 (rows) x 64 (cols), 8 warps as 4 (rows) x 2 (cols), warp tile 32 x 32 = 4 x 4 DMMA tiles
// (mma.sync.m8n8k4.f64).  The accumulators start from C and stay in registers over the whole K loop; L and U
// arrive in chunks of 32 k through a two-stage cp.async pipeline (the next chunk loads while this one is
// multiplied), so C is read and written ONCE per update whatever its depth: with K = 256 (two-level blocking,
// lu_factor) the update does 32 flop per byte of C instead of 8.
// The mma computes the transposed tile: mma row <-> C column, mma col <-> C row, so that each lane's
// two accumulators are two consecutive rows of one column (16-byte global accesses).
// ------------------------------------------------------------------------------------------------
constexpr int GM = 128, GN = 64, GKC = 32;     // tile and k-chunk
constexpr int LDL = GM + 4;    // shared leading dimensions: stride mod 16 (in doubles) = 4 -> conflict-free
constexpr int LDU = GKC + 4;
constexpr int GEMM_THREADS = 256;
constexpr int GEMM_STAGE = GKC * LDL + GN * LDU;               // doubles per stage
constexpr size_t GEMM_SMEM = (size_t)2 * GEMM_STAGE * sizeof(double);

__device__ __forceinline__ void cp_async16(void* smem, const void* gmem) {
  unsigned s = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(s), "l"(gmem));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N)); }

__device__ __forceinline__ void dmma884(double& d0, double& d1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

#ifndef NEB_GEMM_UNROLL
#define NEB_GEMM_UNROLL 8
#endif
constexpr int kGemmUnroll = NEB_GEMM_UNROLL;   // k4 steps of a chunk unrolled together
#ifndef NEB_GEMM_BAND
#define NEB_GEMM_BAND 32
#endif
constexpr int kBandTiles = NEB_GEMM_BAND;   // row tiles (of 128 rows) per L2 band of the update
__global__ void __launch_bounds__(GEMM_THREADS, 2) gemm_kernel(double* __restrict__ A, int64_t ld, const double* __restrict__ Lp, int64_t ldl,
                                                               int64_t k, int K, int64_t r0, int64_t m, int64_t c_first, int64_t tiles_n) {
  extern __shared__ __align__(16) double smem[];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  // Tile order (1-D grid): bands of kBandTiles row tiles; inside a band column by column, the band's row tiles
  // innermost.  A band's slice of L (kBandTiles x 128 rows x K: 16 MB at K = 512) then stays in L2 while U streams past
  // once per band; with the plain (row tiles fastest, all of them) order L (78 MB at C2, 400 MB at C3 for K = 1024) and U
  // together overflow the 126 MB L2 and every CTA re-reads its operands from HBM (measured: 15.3 GB read by one
  // rank-512 update of C2 whose C is 2.8 GB).
  const unsigned tiles_m = (unsigned)((m + GM - 1) / GM), per_band = kBandTiles * (unsigned)tiles_n;
  const unsigned band = blockIdx.x / per_band, within = blockIdx.x - band * per_band;
  // (the last band may be shorter: its tiles are numbered after all full bands, so the division above is exact for it too)
  const unsigned band_rows = min((unsigned)kBandTiles, tiles_m - band * kBandTiles);
  const unsigned tile_n = within / band_rows, tile_m = band * kBandTiles + (within - tile_n * band_rows);
  const int64_t i0 = r0 + (int64_t)tile_m * GM;           // first row of the tile
  const int64_t j0 = c_first + (int64_t)tile_n * GN;      // first column
  const int rows_here = (int)min((int64_t)GM, r0 + m - i0);   // 64 or 128
  const int nchunks = K / GKC;
  // stage st <- chunk ch: sL[kk * LDL + i] = L[i][ch*32 + kk], sU[j * LDU + kk] = U[ch*32 + kk][j]
  auto issue = [&](int ch, int st) {
    double* sL = smem + st * GEMM_STAGE;
    double* sU = sL + GKC * LDL;
    const int64_t kc = k + (int64_t)ch * GKC;
    for (int idx = tid; idx < GKC * (GM / 2); idx += GEMM_THREADS) {     // 32 k-columns x 64 16-byte chunks
      const int kk = idx / (GM / 2), c2 = idx % (GM / 2);
      if (2 * c2 < rows_here) cp_async16(sL + kk * LDL + 2 * c2, Lp + (i0 + 2 * c2) + ((int64_t)ch * GKC + kk) * ldl);
    }
    for (int idx = tid; idx < GN * (GKC / 2); idx += GEMM_THREADS) {     // 64 columns x 16 chunks
      const int j = idx / (GKC / 2), c2 = idx % (GKC / 2);
      cp_async16(sU + j * LDU + 2 * c2, A + (kc + 2 * c2) + (j0 + j) * ld);
    }
  };
  issue(0, 0);
  cp_async_commit();
  if (nchunks > 1) issue(1, 1);
  cp_async_commit();
  const int wr = warp & 3, wc = warp >> 2;                // warp tile origin: rows wr*32, cols wc*32
  const int g = lane >> 2, t = lane & 3;
  const bool active = wr * 32 < rows_here;
  // accumulators start from C: acc[ni][mi] <-> C[i0 + wr*32 + mi*8 + 2t + {0,1}][j0 + wc*32 + ni*8 + g]
  double acc[4][4][2];
  if (active) {
#pragma unroll
    for (int ni = 0; ni < 4; ++ni)
#pragma unroll
      for (int mi = 0; mi < 4; ++mi) {
        const double2 v = *reinterpret_cast<const double2*>(A + (i0 + wr * 32 + mi * 8 + 2 * t) + (j0 + wc * 32 + ni * 8 + g) * ld);
        acc[ni][mi][0] = v.x; acc[ni][mi][1] = v.y;
      }
  }
#pragma unroll 1
  for (int ch = 0; ch < nchunks; ++ch) {
    cp_async_wait<1>();                                   // chunk ch has landed (one younger group may be in flight)
    __syncthreads();
    const double* sL = smem + (ch & 1) * GEMM_STAGE;
    const double* sU = sL + GKC * LDL;
    if (active) {
#pragma unroll kGemmUnroll
      for (int k4 = 0; k4 < GKC / 4; ++k4) {
        double fa[4], fb[4];
        // mma A operand (row = C column n, col = k): U[k4*4 + t][n = g]
#pragma unroll
        for (int ni = 0; ni < 4; ++ni) fa[ni] = sU[(wc * 32 + ni * 8 + g) * LDU + k4 * 4 + t];
        // mma B operand (row = k, col = C row m): -L[m = g][k4*4 + t]
#pragma unroll
        for (int mi = 0; mi < 4; ++mi) fb[mi] = -sL[(k4 * 4 + t) * LDL + wr * 32 + mi * 8 + g];
#pragma unroll
        for (int ni = 0; ni < 4; ++ni)
#pragma unroll
          for (int mi = 0; mi < 4; ++mi) dmma884(acc[ni][mi][0], acc[ni][mi][1], fa[ni], fb[mi]);
      }
    }
    if (ch + 2 < nchunks) {
      __syncthreads();                                    // everyone is done with this stage: refill it
      issue(ch + 2, ch & 1);
    }
    cp_async_commit();                                    // (possibly empty) keeps the group count in step
  }
  if (active) {
#pragma unroll
    for (int ni = 0; ni < 4; ++ni)
#pragma unroll
      for (int mi = 0; mi < 4; ++mi)
        *reinterpret_cast<double2*>(A + (i0 + wr * 32 + mi * 8 + 2 * t) + (j0 + wc * 32 + ni * 8 + g) * ld) =
            make_double2(acc[ni][mi][0], acc[ni][mi][1]);
  }
}

// ------------------------------------------------------------------------------------------------
// a6: triangular solves on the resident factors
// ------------------------------------------------------------------------------------------------
// Composes the row exchanges into one permutation: rowperm[i] = original row that ends in position i.
// The exchanges are sequential by nature, but few (the matrix is close to diagonally dominant): the
// positions that really exchange are marked in parallel in a bit mask, one thread walks the set bits.
__global__ void __launch_bounds__(1024) compose_perm_kernel(const int32_t* __restrict__ ipiv, int32_t* __restrict__ rowperm, int npad) {
  extern __shared__ int s_perm[];            // npad ints, then (npad+31)/32 mask words
  unsigned* s_mask = reinterpret_cast<unsigned*>(s_perm + npad);
  const int nwords = (npad + 31) / 32;
  for (int i = threadIdx.x; i < npad; i += blockDim.x) s_perm[i] = i;
  for (int w = threadIdx.x >> 5; w < nwords; w += blockDim.x >> 5) {
    int i = w * 32 + (threadIdx.x & 31);
    unsigned m = __ballot_sync(0xffffffffu, i < npad && ipiv[i] != i);
    if ((threadIdx.x & 31) == 0) s_mask[w] = m;
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 0; w < nwords; ++w) {
      unsigned m = s_mask[w];
      while (m) {
        int i = w * 32 + __ffs(m) - 1;
        m &= m - 1;
        int p = ipiv[i];
        int tmp = s_perm[i]; s_perm[i] = s_perm[p]; s_perm[p] = tmp;
      }
    }
  }
  __syncthreads();
  for (int i = threadIdx.x; i < npad; i += blockDim.x) rowperm[i] = s_perm[i];
}

// The same for matrices whose permutation does not fit shared memory (npad > ~5e4): one CTA fills the identity in
// parallel; its first warp then reads 32 pivots at a time (one coalesced load), a ballot finds the positions that really
// exchange, and lane 0 applies those exchanges in order (the exchanges are sequential by nature, but few).
__global__ void __launch_bounds__(1024) compose_perm_global_kernel(const int32_t* __restrict__ ipiv, int32_t* rowperm, int npad) {
  for (int i = threadIdx.x; i < npad; i += blockDim.x) rowperm[i] = i;
  __syncthreads();
  if (threadIdx.x >= 32) return;
  const int lane = threadIdx.x;
  for (int base = 0; base < npad; base += 32) {
    const int i = base + lane;
    const int p = (i < npad) ? ipiv[i] : i;
    unsigned m = __ballot_sync(0xffffffffu, p != i);
    while (m) {                                            // warp-uniform
      const int b = __ffs(m) - 1;
      m &= m - 1;
      const int pp = __shfl_sync(0xffffffffu, p, b);
      if (lane == 0) { const int ii = base + b, tmp = rowperm[ii]; rowperm[ii] = rowperm[pp]; rowperm[pp] = tmp; }
    }
  }
}

// Inverses of the 64x64 diagonal blocks of L (unit lower) and U (upper), once per factorisation, so that a
// solve step is a matrix-vector product instead of a 64-step substitution.  grid = (nblocks, 2), 64 threads;
// thread c computes column c of the inverse by substitution.  dinv[(which * nblk + blk) * 4096 + i + 64 j].
__global__ void __launch_bounds__(NB) diag_inv_kernel(const double* __restrict__ A, int64_t ld, double* __restrict__ dinv, int nblk) {
  extern __shared__ double s_dinv[];
  double(*sT)[NB + 1] = reinterpret_cast<double(*)[NB + 1]>(s_dinv);                     // sT[i][j]
  double(*sXc)[NB + 1] = reinterpret_cast<double(*)[NB + 1]>(s_dinv + NB * (NB + 1));    // sXc[k][c]
  const int c = threadIdx.x, blk = blockIdx.x, upper = blockIdx.y;
  const int64_t kb = (int64_t)blk * NB;
  for (int j = 0; j < NB; ++j) sT[c][j] = A[(kb + c) + (kb + j) * ld];
  __syncthreads();
  if (!upper) {
    for (int i = 0; i < NB; ++i) {
      double acc = (i == c) ? 1.0 : 0.0;
      for (int kk = c; kk < i; ++kk) acc = fma(-sT[i][kk], sXc[kk][c], acc);
      sXc[i][c] = (i < c) ? 0.0 : acc;
    }
  } else {
    for (int i = NB - 1; i >= 0; --i) {
      double acc = (i == c) ? 1.0 : 0.0;
      for (int kk = i + 1; kk <= c; ++kk) acc = fma(-sT[i][kk], sXc[kk][c], acc);
      sXc[i][c] = (i > c) ? 0.0 : acc / sT[i][i];
    }
  }
  __syncthreads();
  double* out = dinv + ((int64_t)upper * nblk + blk) * (NB * NB);
  for (int j = 0; j < NB; ++j) out[c + NB * j] = sXc[c][j];
}

// ------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------
// cudaFuncSetAttribute applies to the CURRENT device only: done once per context, right after cudaSetDevice.
neb_status lu_init_device(neb_ctx* c) {
  NEB_CUDA(c, cudaFuncSetAttribute(panel_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024));
  NEB_CUDA(c, cudaFuncSetAttribute(gemm_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)GEMM_SMEM));
  NEB_CUDA(c, cudaFuncSetAttribute(trsm_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TRSM_SMEM));
  NEB_CUDA(c, cudaFuncSetAttribute(diag_inv_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(2 * NB * (NB + 1) * sizeof(double))));
  NEB_CUDA(c, cudaFuncSetAttribute(compose_perm_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024));
  c->cluster_max_ctas = panel_cluster_probe();
  return trisolve_init_device(c);
}

// Launch wrappers of the update kernels: used by lu_factor below and by the distributed factorisation (neb_dist.cu),
// where A is a rank's local block of columns and the L operand (Lp, ldl) is the broadcast panel.
void lu_launch_laswp(neb_ctx* c, cudaStream_t st, double* A, int64_t ld, int64_t k, int npiv, int64_t c_lo, int64_t c_hi, int64_t skip_lo,
                     int64_t skip_hi) {
  const int64_t ncols = (c_hi - c_lo) - (skip_hi - skip_lo);
  if (ncols <= 0) return;
  laswp_kernel<<<(unsigned)((ncols + 127) / 128), 128, 0, st>>>(A, ld, k, npiv, c->d_ipiv, c_lo, c_hi, skip_lo, skip_hi);
  c->launches++;
}

void lu_launch_trsm(neb_ctx* c, cudaStream_t st, double* A, int64_t ld, const double* Lp, int64_t ldl, int64_t k, int64_t c_first,
                    int64_t ncols) {
  if (ncols <= 0) return;
  trsm_kernel<<<(unsigned)(ncols / NB), TRSM_THREADS, TRSM_SMEM, st>>>(A, ld, Lp, ldl, k, c_first);
  c->launches++;
}

void lu_launch_gemm(neb_ctx* c, cudaStream_t st, double* A, int64_t ld, const double* Lp, int64_t ldl, int64_t k, int K, int64_t r0,
                    int64_t m, int64_t c_first, int64_t ncols, bool timed) {
  if (m <= 0 || ncols <= 0) return;
  c->counter[NEB_COUNTER_GEMM_FLOP] += 2.0 * (double)m * (double)ncols * (double)K;
  const int64_t tiles_n = ncols / GN;
  const unsigned grid = (unsigned)(((m + GM - 1) / GM) * tiles_n);
  if (timed) {
    StageTimer tg(c, NEB_STAGE_LU_GEMM);
    gemm_kernel<<<grid, GEMM_THREADS, GEMM_SMEM, st>>>(A, ld, Lp, ldl, k, K, r0, m, c_first, tiles_n);
  } else {
    gemm_kernel<<<grid, GEMM_THREADS, GEMM_SMEM, st>>>(A, ld, Lp, ldl, k, K, r0, m, c_first, tiles_n);
  }
  c->launches++;
}

// rowperm (the composed row permutation) from ipiv, for the solves
neb_status lu_finish_factors(neb_ctx* c) {
  const int64_t npad = c->npad;
  if ((size_t)npad * sizeof(int) + (size_t)((npad + 31) / 32) * 4 <= 200 * 1024) {
    compose_perm_kernel<<<1, 1024, (size_t)npad * sizeof(int) + (size_t)((npad + 31) / 32) * sizeof(unsigned), c->stream>>>(c->d_ipiv, c->d_rowperm, (int)npad);
  } else {
    compose_perm_global_kernel<<<1, 1024, 0, c->stream>>>(c->d_ipiv, c->d_rowperm, (int)npad);
  }
  c->launches++;
  NEB_CUDA(c, cudaGetLastError());
  return NEB_OK;
}

neb_status lu_factor(neb_ctx* c) {
  const int64_t npad = c->npad, ld = c->npad;
  StageTimer tt(c, NEB_STAGE_LU);
  c->counter[NEB_COUNTER_GEMM_FLOP] = 0.0;
  c->counter[NEB_COUNTER_LU_FLOP] = 2.0 / 3.0 * (double)npad * (double)npad * (double)npad;
  PanelWs* ws = (PanelWs*)c->d_panel_ws;
  // panels run on one cluster (neb_lu_panel.cu) whatever their height; NEB_OPT_LU_PANEL = 1 selects the grid-wide
  // cooperative kernel of round 1 instead (all SMs, no look-ahead, n <= 148 x 384 - 128): kept as a cross-check
  const int64_t cluster_rows = c->panel_mode == 0 ? panel_cluster_max_rows(c) : 0;
#ifndef NEB_LU_CHAIN_ROWS
#define NEB_LU_CHAIN_ROWS 4096
#endif
#ifndef NEB_LU_MID_PANELS
#define NEB_LU_MID_PANELS 2
#endif
  constexpr int64_t kChainRows = NEB_LU_CHAIN_ROWS;     // below this the panel chain, not the update, is the critical path
  cudaStream_t S1 = c->stream, S2 = c->side_stream;

  // panel k on stream st: the cluster kernel where the panel fits, else the grid-wide cooperative kernel
  auto launch_panel = [&](int64_t k, cudaStream_t st) -> neb_status {
    const int64_t mrows = npad - k;
    if (mrows <= cluster_rows) return panel_cluster_launch(c, c->d_K, k, st);
    // rows per CTA: multiple of 32, at most 200 KB of shared memory (390 rows -> 384)
    int G = (int)min((int64_t)c->num_sms, (mrows + 63) / 64);
    int mc = (int)((mrows + G - 1) / G);
    mc = (mc + 31) / 32 * 32;
    size_t smem = (size_t)mc * NB * sizeof(double);
    if (smem > 200 * 1024) return fail(c, NEB_ENOMEM, "LU panel slab exceeds shared memory: n too large for this build");
    G = (int)((mrows + mc - 1) / mc);
    NEB_CUDA(c, cudaMemsetAsync(&ws->counter, 0, sizeof(unsigned int), st));
    double* A = c->d_K;
    int64_t ld_ = ld, npad_ = npad, k_ = k;
    int32_t* ipiv = c->d_ipiv;
    int32_t* flag = c->d_flag;
    void* args[] = {&A, &ld_, &npad_, &k_, &mc, &ipiv, &ws, &flag};
    NEB_CUDA(c, cudaLaunchCooperativeKernel((void*)panel_kernel, dim3(G), dim3(PANEL_THREADS), args, smem, st));
    c->launches++;
    return NEB_OK;
  };
  // row exchanges of panel k on the columns [c_lo, c_hi) \ [skip_lo, skip_hi)
  auto laswp = [&](cudaStream_t st, int64_t k, int npiv, int64_t c_lo, int64_t c_hi, int64_t skip_lo, int64_t skip_hi) {
    lu_launch_laswp(c, st, c->d_K, ld, k, npiv, c_lo, c_hi, skip_lo, skip_hi);
  };
  // C[r0 .. r0+m, c_first .. c_first+ncols) -= A[r0 .., k .. k+K) * A[k .. k+K, c_first ..) on the tensor cores
  const bool timed = !c->lu_lookahead;
  auto gemm = [&](cudaStream_t st, int64_t k, int K, int64_t r0, int64_t m, int64_t c_first, int64_t ncols) {
    lu_launch_gemm(c, st, c->d_K, ld, c->d_K + k * ld, ld, k, K, r0, m, c_first, ncols, timed);
  };
  auto trsm = [&](cudaStream_t st, int64_t k, int64_t c_first, int64_t ncols) {
    lu_launch_trsm(c, st, c->d_K, ld, c->d_K + k * ld, ld, k, c_first, ncols);
  };

  // Two-level right-looking factorisation.  Outer blocks of w columns = w / 64 panels:
  //   chain   for each panel of the block: factor it, then apply its update (row exchanges, U12 = L11^-1 A12,
  //           rank-64 tensor-core update) to the REST OF THE BLOCK only;
  //   wide    the block's row exchanges on all other columns, the block row of U (w / 64 x [TRSM + small update]), and
  //           ONE rank-w tensor-core update of the whole trailing matrix: C is read and written once per w columns
  //           instead of once per 64 (w / 8 flop per byte of C: compute-bound on the DMMA pipe).
  // Look-ahead: the rank-w update is applied to the next block's columns first; that block's chain (latency-bound,
  // one cluster = 16 SMs per panel) then runs on the side stream while the main stream finishes the update on the
  // other SMs.  Only where the panels run on a cluster (the grid-wide panel kernel needs every SM).
  // Block width: the deeper the update, the smaller the share of a tile's life spent reading and writing C (the DMMA
  // pipe idles there unless the SM's other CTA covers it) — 1024 while the trailing matrix exceeds 24576 rows, 512 down to
  // 8192 rows, where the chain of a wider block still hides behind its update; c->lu_nb (64 by default) below: there
  // the chain of panels is the critical path and anything added to it (the in-block updates, a wider look-ahead
  // slice) costs more than the deeper update saves.
  auto block_width = [&](int64_t remaining) -> int64_t {
    if (remaining > 24576) return 16 * NB;     // measured on B200 (C3, whole factorisation): updates at 31.7 TFLOP/s; 512 throughout 30.8, 256 29.3
    if (remaining > 8192) return 8 * NB;
    return remaining > kChainRows ? (int64_t)NEB_LU_MID_PANELS * NB : (int64_t)c->lu_nb;
  };
  bool chain_on_side = false;
  for (int64_t kb = 0; kb < npad;) {
    const int64_t w = min(block_width(npad - kb), npad - kb), nb = kb + w;
    cudaStream_t SC = chain_on_side ? S2 : S1;
    for (int64_t k = kb; k < nb; k += NB) {
      NEB_TRY(launch_panel(k, SC));
      const int64_t in_cols = nb - (k + NB);               // columns of this block right of the panel
      laswp(SC, k, NB, kb, nb, k, k + NB);                 // the block's other columns, left and right of the panel
      trsm(SC, k, k + NB, in_cols);
      gemm(SC, k, NB, k + NB, npad - (k + NB), k + NB, in_cols);
    }
    if (chain_on_side) {
      NEB_CUDA(c, cudaEventRecord(c->ev_panel, S2));
      NEB_CUDA(c, cudaStreamWaitEvent(S1, c->ev_panel, 0));
    }
    // the block's pivots are final: its row exchanges on the finished columns to the LEFT go to a stream of their own
    // (uncoalesced row traffic that nothing needs before the solves; on the main stream it delayed every update)
    cudaStream_t SL = (c->lu_lookahead && c->left_stream) ? c->left_stream : S1;
    if (SL != S1 && kb > 0) {
      NEB_CUDA(c, cudaEventRecord(c->ev_chain, SC));
      NEB_CUDA(c, cudaStreamWaitEvent(SL, c->ev_chain, 0));
    }
    laswp(SL, kb, (int)w, 0, kb, kb, kb);
    const int64_t right = npad - nb;                       // columns (and rows) of the trailing matrix
    // everything the factored block does to the columns [c0, c0 + nc) right of it
    auto wide = [&](int64_t c0, int64_t nc) {
      if (nc <= 0) return;
      laswp(S1, kb, (int)w, c0, c0 + nc, c0 + nc, c0 + nc);   // the block's w exchanges in one launch
      for (int64_t k = kb; k < nb; k += NB) {
        trsm(S1, k, c0, nc);
        gemm(S1, k, NB, k + NB, nb - (k + NB), c0, nc);    // rows of the block row still below this panel
      }
      gemm(S1, kb, (int)w, nb, right, c0, nc);
    };
    const int64_t w_next = right > 0 ? min(block_width(right), right) : 0;
    const bool ahead = c->lu_lookahead && S2 && right > 0 && right <= cluster_rows && right > w_next;
    if (ahead) {
      wide(nb, w_next);                                    // the next block's columns first ...
      NEB_CUDA(c, cudaEventRecord(c->ev_next, S1));
      NEB_CUDA(c, cudaStreamWaitEvent(S2, c->ev_next, 0));
      wide(nb + w_next, right - w_next);                   // ... the rest while its chain runs on the side stream
    } else {
      wide(nb, right);
    }
    chain_on_side = ahead;
    NEB_CUDA(c, cudaGetLastError());
    kb = nb;
  }
  if (c->lu_lookahead && c->left_stream) {
    NEB_CUDA(c, cudaEventRecord(c->ev_left, c->left_stream));
    NEB_CUDA(c, cudaStreamWaitEvent(S1, c->ev_left, 0));
  }
  // composed permutation for the solves
  NEB_TRY(lu_finish_factors(c));
  {
    const int nblk = (int)(npad / NB);
    diag_inv_kernel<<<dim3(nblk, 2), NB, 2 * NB * (NB + 1) * sizeof(double), c->stream>>>(c->d_K, ld, c->d_dinv, nblk);
    c->launches++;
  }
  NEB_CUDA(c, cudaGetLastError());
  return NEB_OK;
}

}  // namespace neb
