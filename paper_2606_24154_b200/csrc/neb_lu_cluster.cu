// neb_lu_cluster.cu — a5: LU panel factorisation for panels of at most 8192 rows, on ONE thread-block
// cluster (up to 16 CTAs x 512 threads, distributed shared memory) instead of the whole grid.
//
// Why: with partial pivoting every column needs a panel-wide argmax and the winner's row before any
// thread can continue.  Through global memory and a grid barrier that exchange costs ~4.8 us per column
// (measured: panel_kernel, 308 us per 64-column panel, 47 % of the C1 step).  A cluster exchanges
// through DSMEM with a hardware cluster barrier: ~0.5 us per column.
//
// Design: a thread owns one matrix ROW BY IDENTITY and keeps the 32 columns of the current half panel in
// registers.  Pivoting is implicit: rows never move, each thread tracks the POSITION its row currently
// occupies (`pos`), which reproduces LAPACK's sequential row exchanges exactly (ipiv[dr] = position of
// the winner at that time; ties -> lowest position).  Per column: warp argmax -> the winning lane publishes
// its row in shared memory -> warp 0 forms the CTA's candidate and PUSHES it (value, position, row) into the
// shared memory of every CTA of the cluster (remote stores) -> one cluster barrier (arrive.release /
// wait.acquire) -> every WARP finds the global winner among the 16 local candidate slots by itself (no second
// CTA barrier, no remote read on the critical path; letting all 16 x 16 warps read the winner's row remotely was
// measured slower: 64 KB through one SM's shared-memory port per column) -> rank-1 update in registers.
// (Starting the next column's search before the rest of the update was also measured slower: the extra live
// registers spill, and spilled locals miss the L1 after every cluster barrier.)  Between the two 32-column halves the
// pivot rows are gathered in CTA 0, which solves the 32x32 triangular system for U12; every row then
// applies the rank-32 update from its own multipliers (stashed in shared memory).  At the end every
// thread writes its row to its final position.
#include <cooperative_groups.h>
#include <cstdio>

#include "neb_internal.h"

namespace cg = cooperative_groups;

namespace neb {

constexpr int PC_THREADS = 512;
constexpr int PC_WARPS = PC_THREADS / 32;
constexpr int PC_H = 32;          // half-panel width
constexpr int PC_MAX_CTAS = 16;

struct PcSmem {
  double L[PC_H][PC_THREADS];         // first-half rows of this CTA's threads: L[c][tid]
  double pub[2][PC_WARPS][PC_H];      // per-warp candidate rows, double-buffered by step parity
  double crow[2][PC_MAX_CTAS][PC_H];  // candidate row of every CTA of the cluster (pushed by its warp 0), by parity
  unsigned long long cval[2][PC_MAX_CTAS];   // |value| bits of every CTA's candidate
  int cpos[2][PC_MAX_CTAS];           // its position (INT_MAX: that CTA has no row left)
  double U[PC_H][PC_H];               // local copy of U12
  double Lp[PC_H][PC_H + 1];          // CTA 0: gathered pivot rows, first half (unit lower L11 / U11)
  double Bp[PC_H][PC_H + 1];          // CTA 0: gathered pivot rows, second half -> U12
  unsigned whi[2][PC_WARPS], wlo[2][PC_WARPS];   // per-warp candidates by parity: |value| bits and position
  int wpos[2][PC_WARPS];
};

// Warp-wide argmax of (|value|, lowest position) with three REDUX.SYNC instead of a 5-round shuffle
// butterfly: non-negative doubles order like their bit patterns, so max(high word), then max(low word)
// among the lanes that hold that high word, then min(position) among the lanes that hold both.
// Lanes that do not take part pass pos = INT_MAX (and hi = lo = 0); result pos = INT_MAX if nobody took part.
__device__ __forceinline__ void warp_argmax(unsigned hi, unsigned lo, int pos, unsigned& mh, unsigned& ml, int& mp) {
  mh = __reduce_max_sync(0xffffffffu, pos != 0x7fffffff ? hi : 0u);
  const bool e1 = (pos != 0x7fffffff) && hi == mh;
  ml = __reduce_max_sync(0xffffffffu, e1 ? lo : 0u);
  const bool e2 = e1 && lo == ml;
  mp = __reduce_min_sync(0xffffffffu, e2 ? pos : 0x7fffffff);
}

// 1/x for a pivot: MUFU.RCP64H seed + two Newton steps + residual correction inside the normal range,
// plain division outside it (one lane only).
__device__ __forceinline__ double pivot_rcp(double x) {
  const double ax = fabs(x);
  if (!(ax > 1e-290 && ax < 1e290)) return (x != 0.0) ? 1.0 / x : 0.0;
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  double e = fma(-x, r, 1.0);
  r = fma(r, e, r);
  e = fma(-x, r, 1.0);
  r = fma(r, e, r);
  e = fma(-x, r, 1.0);
  return fma(r, e, r);
}

// Factorises the 32 columns held in a[] (rows whose position is >= dr0 take part).
// The column loop is rolled in blocks of PC_BS steps (code stays inside the instruction cache).  Register
// indices stay static because the 32-column window is ROTATED by PC_BS after each block: the finished
// columns travel to the tail of the window, where the broadcast pivot row is zero, so the update leaves
// them alone; after 32/PC_BS blocks the window is back in natural order.
constexpr int PC_BS = 4;
#ifdef NEB_PANEL_TRACE
#define PC_MARK(i) do { if (tid == 0) { long long t_ = clock64(); tr[i] += t_ - tl; tl = t_; } } while (0)
#else
#define PC_MARK(i)
#endif
__device__ __forceinline__ void factor_half(double (&a)[PC_H], int& pos, bool valid, int64_t dr0, PcSmem& sm,
                                            cg::cluster_group& cluster, int ncta, int32_t* __restrict__ ipiv,
                                            int32_t* __restrict__ flag) {
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const unsigned rank = cluster.block_rank();
#ifdef NEB_PANEL_TRACE
  long long tr[8] = {0, 0, 0, 0, 0, 0, 0, 0}, tl = clock64();
#endif
#pragma unroll 1
  for (int blk = 0; blk < PC_H / PC_BS; ++blk) {
    const int width = PC_H - blk * PC_BS;          // live columns of the window: indices 0 .. width-1
#pragma unroll
    for (int jj = 0; jj < PC_BS; ++jj) {
      const int j = blk * PC_BS + jj;
      const int par = j & 1;
      const int dr = (int)dr0 + j;
      const bool act = valid && pos >= dr;
      double v = fabs(a[jj]);
      if (!(v == v)) v = 0.0;                      // NaN never wins; caught by the zero-pivot test
      unsigned mh, ml;
      int mp;
      warp_argmax((unsigned)__double2hiint(v), (unsigned)__double2loint(v), act ? pos : 0x7fffffff, mh, ml, mp);
      if (act && pos == mp) {
#pragma unroll
        for (int c = jj; c < PC_H; ++c) sm.pub[par][warp][c] = a[c];
      }
      if (lane == 0) { sm.whi[par][warp] = mh; sm.wlo[par][warp] = ml; sm.wpos[par][warp] = mp; }
      PC_MARK(0);
      __syncthreads();
      PC_MARK(1);
      if (warp == 0) {
        // the CTA's candidate (value, position, row), pushed into every CTA of the cluster (its own included)
        const bool in = lane < PC_WARPS;
        const unsigned h = in ? sm.whi[par][lane] : 0u, l = in ? sm.wlo[par][lane] : 0u;
        const int p = in ? sm.wpos[par][lane] : 0x7fffffff;
        unsigned ch, cl;
        int cp;
        warp_argmax(h, l, p, ch, cl, cp);
        const unsigned who = __ballot_sync(0xffffffffu, in && p == cp && p != 0x7fffffff);
        const int cw = who ? __ffs(who) - 1 : 0;
        // finished columns (rotated to the tail of the window) and unused ones carry 0: the update skips them
        const double x = (lane >= jj && lane < width && cp != 0x7fffffff) ? sm.pub[par][cw][lane] : 0.0;
        for (int r = 0; r < ncta; ++r) cluster.map_shared_rank(&sm, r)->crow[par][rank][lane] = x;
        if (lane < ncta) {
          PcSmem* rs = cluster.map_shared_rank(&sm, lane);
          rs->cval[par][rank] = ((unsigned long long)ch << 32) | cl;
          rs->cpos[par][rank] = cp;
        }
      }
      PC_MARK(2);
      cluster.barrier_arrive();                    // release: the pushes above are visible after the wait
      PC_MARK(3);
      cluster.barrier_wait();
      PC_MARK(4);
      // every warp picks the global winner from its CTA's own copy of the candidates
      unsigned h = 0u, l = 0u;
      int p = 0x7fffffff;
      if (lane < ncta) {
        const unsigned long long cv = sm.cval[par][lane];
        h = (unsigned)(cv >> 32); l = (unsigned)cv; p = sm.cpos[par][lane];
      }
      unsigned gh, gl;
      int gp;
      warp_argmax(h, l, p, gh, gl, gp);
      const bool any = gp != 0x7fffffff;
      const unsigned gwho = __ballot_sync(0xffffffffu, any && p == gp);
      const int gc = gwho ? __ffs(gwho) - 1 : 0;
      const double* prow = sm.crow[par][gc];
      const double piv = prow[jj];
      const double invp = pivot_rcp(piv);
      const int wp = any ? gp : dr;
      if (rank == 0 && tid == 0) {
        ipiv[dr] = wp;
        if (!any || !(fabs(piv) > 0.0)) atomicOr(flag, 2);
      }
      PC_MARK(5);
      pos = (pos == dr) ? wp : ((pos == wp) ? dr : pos);
      if (valid && pos > dr) {
        const double lmul = a[jj] * invp;
        a[jj] = lmul;
#pragma unroll
        for (int c = jj + 1; c < PC_H; ++c) a[c] = fma(-lmul, prow[c], a[c]);
      }
      PC_MARK(6);
    }
    // rotate the window by PC_BS: finished columns go to the tail
    double t[PC_BS];
#pragma unroll
    for (int c = 0; c < PC_BS; ++c) t[c] = a[c];
#pragma unroll
    for (int c = 0; c < PC_H - PC_BS; ++c) a[c] = a[c + PC_BS];
#pragma unroll
    for (int c = 0; c < PC_BS; ++c) a[PC_H - PC_BS + c] = t[c];
    PC_MARK(7);
  }
#ifdef NEB_PANEL_TRACE
  if (tid == 0 && dr0 == 0)
    printf("rank %u: argmax+pub %lld sync %lld cta+push %lld arrive %lld wait %lld global %lld update %lld rotate %lld (cycles, 32 columns)\n",
           rank, tr[0], tr[1], tr[2], tr[3], tr[4], tr[5], tr[6], tr[7]);
#endif
}

__global__ void __launch_bounds__(PC_THREADS, 1) panel_cluster_kernel(double* __restrict__ A, int64_t ld, int64_t npad,
                                                                      int64_t k, int32_t* __restrict__ ipiv,
                                                                      int32_t* __restrict__ flag) {
  extern __shared__ __align__(16) unsigned char pc_raw[];
  PcSmem& sm = *reinterpret_cast<PcSmem*>(pc_raw);
  cg::cluster_group cluster = cg::this_cluster();
  const int ncta = (int)cluster.num_blocks();
  const unsigned rank = cluster.block_rank();
  const int tid = threadIdx.x;
  const int64_t r = k + (int64_t)rank * PC_THREADS + tid;       // the row this thread owns
  const bool valid = r < npad;
  int pos = valid ? (int)r : 0x7ffffff0;
  double a[PC_H];
#pragma unroll
  for (int c = 0; c < PC_H; ++c) a[c] = valid ? A[r + (k + c) * ld] : 0.0;

  factor_half(a, pos, valid, k, sm, cluster, ncta, ipiv, flag);

  // ---- between the halves: stash multipliers, gather the 32 pivot rows in CTA 0, U12 = L11^-1 A12 ----
#pragma unroll
  for (int c = 0; c < PC_H; ++c) sm.L[c][tid] = a[c];
#pragma unroll
  for (int c = 0; c < PC_H; ++c) a[c] = valid ? A[r + (k + PC_H + c) * ld] : 0.0;
  PcSmem* s0 = cluster.map_shared_rank(&sm, 0);
  if (valid && pos < k + PC_H) {
    const int t = pos - (int)k;
#pragma unroll
    for (int c = 0; c < PC_H; ++c) { s0->Lp[t][c] = sm.L[c][tid]; s0->Bp[t][c] = a[c]; }
  }
  cluster.sync();
  if (rank == 0) {
    const int c = tid & 31, w = tid >> 5;
    for (int s = 0; s < PC_H - 1; ++s) {
      for (int t = s + 1 + w; t < PC_H; t += PC_WARPS) sm.Bp[t][c] = fma(-sm.Lp[t][s], sm.Bp[s][c], sm.Bp[t][c]);
      __syncthreads();
    }
  }
  cluster.sync();
  for (int idx = tid; idx < PC_H * PC_H; idx += PC_THREADS) sm.U[idx >> 5][idx & 31] = s0->Bp[idx >> 5][idx & 31];
  __syncthreads();
  if (valid) {
    if (pos < k + PC_H) {
      const int t = pos - (int)k;
#pragma unroll
      for (int c = 0; c < PC_H; ++c) a[c] = sm.U[t][c];
    } else {
#pragma unroll 2
      for (int s = 0; s < PC_H; ++s) {
        const double l = sm.L[s][tid];
#pragma unroll
        for (int c = 0; c < PC_H; ++c) a[c] = fma(-l, sm.U[s][c], a[c]);
      }
    }
  }

  factor_half(a, pos, valid, k + PC_H, sm, cluster, ncta, ipiv, flag);

  if (valid) {
#pragma unroll
    for (int c = 0; c < PC_H; ++c) {
      A[(int64_t)pos + (k + c) * ld] = sm.L[c][tid];
      A[(int64_t)pos + (k + PC_H + c) * ld] = a[c];
    }
  }
  cluster.sync();   // nobody leaves while its shared memory may still be read remotely
}

// Largest cluster size (power of two, <= 16) this device can schedule for the kernel; 0 if none.
int panel_cluster_max_ctas(neb_ctx* c) {
  static int cached = -1;
  if (cached >= 0) return cached;
  cached = 0;
  if (cudaFuncSetAttribute(panel_cluster_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(PcSmem)) != cudaSuccess ||
      cudaFuncSetAttribute(panel_cluster_kernel, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) != cudaSuccess) {
    cudaGetLastError();
    return cached;
  }
  for (int cs = PC_MAX_CTAS; cs >= 1; cs >>= 1) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(cs);
    cfg.blockDim = dim3(PC_THREADS);
    cfg.dynamicSmemBytes = sizeof(PcSmem);
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = cs; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    int nclusters = 0;
    if (cudaOccupancyMaxActiveClusters(&nclusters, panel_cluster_kernel, &cfg) == cudaSuccess && nclusters >= 1) {
      cached = cs;
      break;
    }
    cudaGetLastError();
  }
  (void)c;
  return cached;
}

int64_t panel_cluster_max_rows(neb_ctx* c) { return (int64_t)panel_cluster_max_ctas(c) * PC_THREADS; }

neb_status panel_cluster_launch(neb_ctx* c, int64_t k, cudaStream_t stream) {
  const int64_t mrows = c->npad - k;
  int cs = 1;
  while ((int64_t)cs * PC_THREADS < mrows) cs <<= 1;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(cs);
  cfg.blockDim = dim3(PC_THREADS);
  cfg.dynamicSmemBytes = sizeof(PcSmem);
  cfg.stream = stream;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeClusterDimension;
  at[0].val.clusterDim.x = cs; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
  cfg.attrs = at;
  cfg.numAttrs = 1;
  NEB_CUDA(c, cudaLaunchKernelEx(&cfg, panel_cluster_kernel, c->d_K, c->npad, c->npad, k, c->d_ipiv, c->d_flag));
  c->launches++;
  return NEB_OK;
}

}  // namespace neb
