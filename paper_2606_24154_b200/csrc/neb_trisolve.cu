// neb_trisolve.cu — a6: the two triangular solves on the resident LU factors (Solve; reading S13: factors kept,
// no explicit inverse), for up to 8 right-hand sides per pass ("the same inverted matrix ... can be
// reused" for the weighting potential of every read-out electrode: one pass over the 8 n^2 bytes of L and U serves them
// all).
//
// One persistent, cooperatively launched kernel per triangle (round 1: one launch per 64-column block, 2 n / 64
// launches, every CTA recomputing the same 64 x 64 product from L2: 0.23 of the HBM rate at n = 5e4, launch-bound at
// n = 6e3).  The factors are walked as 64 x 64 tiles.  Row blocks are dealt out cyclically to GROUPS of 64 threads (4
// per CTA, one CTA per SM); a thread owns one row of its group's row blocks.  For every column block t, in order:
//   the group that owns row block t has by then applied all earlier column blocks to it: it multiplies the running
//     values by the precomputed inverse of the diagonal block (diag_inv_kernel) and PUBLISHES the 64 solved values by
//     plain 8-byte stores into a vector that was filled with a sentinel bit pattern;
//   every group polls those 64 values (no flag, no fence: a value is either the sentinel or final), stages them in
//     shared memory and subtracts tile x values from the running values of its row blocks beyond t.
// The chain of n/64 dependent steps is kept short by prefetching, two steps ahead, what the next owner needs that does
// not depend on the solved values — its tile against the preceding column block and its diagonal inverse — into
// shared memory with cp.async; the bulk tiles are loaded into registers BEFORE the poll, so that their HBM latency
// overlaps the wait.  Rows are consecutive across the 64 threads of a group: every tile column is one 512-byte segment.
// Deterministic: each running value is updated by one thread in a fixed order.
#include "neb_internal.h"

namespace neb {

constexpr int TW_THREADS = 256;
constexpr int TW_GROUPS = TW_THREADS / 64;
constexpr int TW_B = 64;                                    // block size
constexpr int TW_MAXK = 8;                                  // right-hand sides per pass
constexpr unsigned long long TW_SENTINEL = 0xffffffffffffffffull;   // a NaN no arithmetic produces; cudaMemset 0xff

struct TwSmem {
  double tile[TW_B * TW_B];                                 // the next owner's tile against the preceding column block
  double dinv[TW_B * TW_B];                                 // ... and the inverse of its diagonal block
  double y[TW_GROUPS][TW_MAXK][TW_B];                       // per group: the solved column block being applied
  double xb[TW_GROUPS][TW_MAXK][TW_B];                      // per group: running values of a diagonal block (for its product)
};

__device__ __forceinline__ void tw_group_sync(int q) { asm volatile("bar.sync %0, 64;" ::"r"(q + 1) : "memory"); }

__device__ __forceinline__ void tw_cp_async16(void* smem, const void* gmem) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((unsigned)__cvta_generic_to_shared(smem)), "l"(gmem));
}

__device__ __forceinline__ double tw_poll(const double* p) {
  unsigned long long v;
  int spin = 0;
  do {
    asm volatile("ld.volatile.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
  } while (v == TW_SENTINEL && ++spin < (1 << 26));
  if (v == TW_SENTINEL) asm volatile("trap;");              // a value that never arrives ends in an error, not a hang
  return __longlong_as_double((long long)v);
}

// acc[k] += sum_j m[j * stride] * v[k][j0 + j], j < N.  The dependent DFMA chain is what the n/64 sequential steps of a
// solve wait for (a DFMA takes ~25 cycles when few warps are resident), so every sum is split into PART partial sums
// (4 independent chains per right-hand side) and the loads are issued ahead of the arithmetic (full unroll).
template <int K>
struct TwPart { static constexpr int value = 4; };   // the same split for every K: a solve gives the same bits alone or in a batch

template <int K, int N>
__device__ __forceinline__ void tw_dot_mem(const double* m, int stride, const double (*v)[TW_B], int j0, double (&acc)[K]) {
  constexpr int PART = TwPart<K>::value;
  double p[K][PART];
#pragma unroll
  for (int k = 0; k < K; ++k)
#pragma unroll
    for (int u = 0; u < PART; ++u) p[k][u] = 0.0;
#pragma unroll
  for (int j = 0; j < N; ++j) {
    const double d = m[j * stride];
#pragma unroll
    for (int k = 0; k < K; ++k) p[k][j % PART] = fma(d, v[k][j0 + j], p[k][j % PART]);
  }
#pragma unroll
  for (int k = 0; k < K; ++k) {
    double t = 0.0;
#pragma unroll
    for (int u = 0; u < PART; ++u) t += p[k][u];
    acc[k] += t;
  }
}

// the same for 32 matrix values held in registers (static register indices)
template <int K>
__device__ __forceinline__ void tw_dot_reg(const double (&a)[32], const double (*v)[TW_B], int j0, double (&acc)[K]) {
  constexpr int PART = TwPart<K>::value;
  double p[K][PART];
#pragma unroll
  for (int k = 0; k < K; ++k)
#pragma unroll
    for (int u = 0; u < PART; ++u) p[k][u] = 0.0;
#pragma unroll
  for (int j = 0; j < 32; ++j)
#pragma unroll
    for (int k = 0; k < K; ++k) p[k][j % PART] = fma(a[j], v[k][j0 + j], p[k][j % PART]);
#pragma unroll
  for (int k = 0; k < K; ++k) {
    double t = 0.0;
#pragma unroll
    for (int u = 0; u < PART; ++u) t += p[k][u];
    acc[k] += t;
  }
}

// xr: running right-hand sides [K][ldx] (consumed); ys: solved values [K][ldx], sentinel-filled on entry.
template <int K, bool UPPER>
__global__ void __launch_bounds__(TW_THREADS, 1) tri_wave_kernel(const double* __restrict__ A, int64_t ld,
                                                                 const double* __restrict__ dinv, double* __restrict__ xr,
                                                                 double* __restrict__ ys, int64_t ldx, int nblk) {
  extern __shared__ __align__(16) unsigned char tw_raw[];
  TwSmem& sm = *reinterpret_cast<TwSmem*>(tw_raw);
  const int tid = threadIdx.x, q = tid >> 6, r = tid & 63;
  const int NG = TW_GROUPS * (int)gridDim.x, gid = q * (int)gridDim.x + (int)blockIdx.x;   // consecutive blocks -> different CTAs
  auto phys = [&](int t) { return UPPER ? nblk - 1 - t : t; };
  int t_own = gid;                                          // my next row block (in processing order)
  bool pre = false;                                         // the shared prefetch buffers hold my next diagonal's data
  // the running values of my next row block stay in registers (its updates and its diagonal product are on the chain
  // of dependent steps: no round trips to L2 there); my later row blocks are updated in global memory
  double xcur[K];
#pragma unroll
  for (int k = 0; k < K; ++k) xcur[k] = (t_own < nblk) ? xr[k * ldx + (int64_t)phys(t_own) * TW_B + r] : 0.0;
  for (int t = 0; t < nblk && t_own < nblk; ++t) {
    const int64_t cb = (int64_t)phys(t) * TW_B;             // first row/column of column block t
    // ---- prefetch for my upcoming diagonal block (needs nothing that is still being computed) ----
    if (t_own >= 1 && (t_own == t + 2 || (t == 0 && t_own == 1))) {
      const int64_t rb = (int64_t)phys(t_own) * TW_B, pb = (int64_t)phys(t_own - 1) * TW_B;
      const double* dsrc = dinv + ((int64_t)(UPPER ? nblk : 0) + phys(t_own)) * (TW_B * TW_B);
      for (int idx = r; idx < TW_B * TW_B / 2; idx += 64) {   // 16-byte pieces: 2 rows of one column
        const int j = idx / (TW_B / 2), i2 = idx % (TW_B / 2);
        tw_cp_async16(&sm.tile[j * TW_B + 2 * i2], A + (rb + 2 * i2) + (pb + j) * ld);
        tw_cp_async16(&sm.dinv[j * TW_B + 2 * i2], dsrc + j * TW_B + 2 * i2);
      }
      asm volatile("cp.async.commit_group;" ::: "memory");
      pre = true;
    }
    // ---- my diagonal block: all earlier column blocks have been applied ----
    if (t_own == t) {
#pragma unroll
      for (int k = 0; k < K; ++k) sm.xb[q][k][r] = xcur[k];
      const double* dsrc = dinv + ((int64_t)(UPPER ? nblk : 0) + phys(t)) * (TW_B * TW_B);
      if (pre) asm volatile("cp.async.wait_group 0;" ::: "memory");
      tw_group_sync(q);
      double acc[K];
#pragma unroll
      for (int k = 0; k < K; ++k) acc[k] = 0.0;
      if (pre) tw_dot_mem<K, TW_B>(sm.dinv + r, TW_B, sm.xb[q], 0, acc);
      else tw_dot_mem<K, TW_B>(dsrc + r, TW_B, sm.xb[q], 0, acc);
#pragma unroll
      for (int k = 0; k < K; ++k) ys[k * ldx + cb + r] = acc[k];       // publish
      pre = false;
      t_own += NG;
      tw_group_sync(q);                                     // xb may be rewritten by my next diagonal
      if (t_own >= nblk) break;
#pragma unroll
      for (int k = 0; k < K; ++k) xcur[k] = xr[k * ldx + (int64_t)phys(t_own) * TW_B + r];
    }
    // ---- apply column block t to my row blocks beyond it; the first of them may be the next diagonal ----
    // matrix data first (independent of the solved values), then the poll
    const int64_t rb0 = (int64_t)phys(t_own) * TW_B;
    const bool next_diag = (t_own == t + 1) && pre;
    double a0[32];
    if (!next_diag) {
#pragma unroll
      for (int j = 0; j < 32; ++j) a0[j] = __ldcs(A + (rb0 + r) + (cb + j) * ld);
    } else {
      asm volatile("cp.async.wait_group 0;" ::: "memory");  // my prefetch (issued two steps ago) has landed
    }
#pragma unroll
    for (int k = 0; k < K; ++k) sm.y[q][k][r] = tw_poll(ys + k * ldx + cb + r);
    tw_group_sync(q);                                       // also makes the group's cp.async data visible to both warps
    for (int tt = t_own; tt < nblk; tt += NG) {
      const int64_t rb = (int64_t)phys(tt) * TW_B;
      double acc[K];
#pragma unroll
      for (int k = 0; k < K; ++k) acc[k] = 0.0;
      if (tt == t_own && next_diag) {
        tw_dot_mem<K, TW_B>(sm.tile + r, TW_B, sm.y[q], 0, acc);
      } else {
        if (tt != t_own) {
#pragma unroll
          for (int j = 0; j < 32; ++j) a0[j] = __ldcs(A + (rb + r) + (cb + j) * ld);
        }
        double a1[32];
#pragma unroll
        for (int j = 0; j < 32; ++j) a1[j] = __ldcs(A + (rb + r) + (cb + 32 + j) * ld);
        tw_dot_reg<K>(a0, sm.y[q], 0, acc);
        tw_dot_reg<K>(a1, sm.y[q], 32, acc);
      }
      if (tt == t_own) {
#pragma unroll
        for (int k = 0; k < K; ++k) xcur[k] -= acc[k];
      } else {
#pragma unroll
        for (int k = 0; k < K; ++k) xr[k * ldx + rb + r] -= acc[k];    // only this thread ever touches this value
      }
    }
    tw_group_sync(q);                                       // y is rewritten at the next step
  }
}

__global__ void permute_scale_multi_kernel(const double* __restrict__ b, const double* __restrict__ rscale,
                                           const int32_t* __restrict__ rowperm, int64_t npad, int nrhs, double* __restrict__ x) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= npad) return;
  const int p = rowperm[i];
  const double s = rscale[p];
  for (int k = 0; k < nrhs; ++k) x[k * npad + i] = b[k * npad + p] * s;
}

template <int K>
static neb_status tw_launch(neb_ctx* c, bool upper, double* xr, double* ys) {
  const int nblk = (int)(c->npad / TW_B);
  const double* A = c->d_K;
  int64_t ld = c->npad, ldx = c->npad;
  const double* dinv = c->d_dinv;
  int nb = nblk;
  void* args[] = {&A, &ld, &dinv, &xr, &ys, &ldx, &nb};
  const void* fn = upper ? (const void*)tri_wave_kernel<K, true> : (const void*)tri_wave_kernel<K, false>;
  NEB_CUDA(c, cudaLaunchCooperativeKernel(fn, dim3(c->num_sms), dim3(TW_THREADS), args, sizeof(TwSmem), c->stream));
  c->launches++;
  return NEB_OK;
}

neb_status trisolve_init_device(neb_ctx* c) {
#define X(K)                                                                                                            \
  NEB_CUDA(c, cudaFuncSetAttribute(tri_wave_kernel<K, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(TwSmem))); \
  NEB_CUDA(c, cudaFuncSetAttribute(tri_wave_kernel<K, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(TwSmem)));
  X(1) X(2) X(4) X(8)
#undef X
  return NEB_OK;
}

// Solves the (row-scaled, factored) system for nrhs right-hand sides d_b[k * npad + i] (unscaled, sorted order);
// solution k in d_out[k * npad + i].  d_out may be c->d_x.  Passes of up to 8 right-hand sides.
neb_status lu_solve(neb_ctx* c, const double* d_b, int nrhs, double* d_out) {
  const int64_t npad = c->npad;
  StageTimer tt(c, NEB_STAGE_TRISOLVE);
  double* R = c->d_x;                                       // running values / final result of a pass
  double* S = c->d_x + (size_t)TW_MAXK * npad;              // forward-solved values
  for (int k0 = 0; k0 < nrhs; k0 += TW_MAXK) {
    const int kn = (nrhs - k0 < TW_MAXK) ? nrhs - k0 : TW_MAXK;
    const int K = kn <= 1 ? 1 : (kn <= 2 ? 2 : (kn <= 4 ? 4 : 8));     // columns beyond kn ride along as zeros
    if (K > kn) NEB_CUDA(c, cudaMemsetAsync(R + (size_t)kn * npad, 0, sizeof(double) * (size_t)(K - kn) * npad, c->stream));
    permute_scale_multi_kernel<<<(unsigned)((npad + 255) / 256), 256, 0, c->stream>>>(d_b + (size_t)k0 * npad, c->d_rscale, c->d_rowperm, npad, kn, R);
    c->launches++;
    NEB_CUDA(c, cudaMemsetAsync(S, 0xff, sizeof(double) * (size_t)K * npad, c->stream));
    // forward: L y = P b (running R, solved S); backward: U x = y (running S, solved R)
    for (int pass = 0; pass < 2; ++pass) {
      double* xr = pass == 0 ? R : S;
      double* ys = pass == 0 ? S : R;
      if (pass == 1) NEB_CUDA(c, cudaMemsetAsync(R, 0xff, sizeof(double) * (size_t)K * npad, c->stream));
      switch (K) {
        case 1: NEB_TRY(tw_launch<1>(c, pass == 1, xr, ys)); break;
        case 2: NEB_TRY(tw_launch<2>(c, pass == 1, xr, ys)); break;
        case 4: NEB_TRY(tw_launch<4>(c, pass == 1, xr, ys)); break;
        default: NEB_TRY(tw_launch<8>(c, pass == 1, xr, ys)); break;
      }
    }
    if (d_out != R || k0 > 0)
      NEB_CUDA(c, cudaMemcpyAsync(d_out + (size_t)k0 * npad, R, sizeof(double) * (size_t)kn * npad, cudaMemcpyDeviceToDevice, c->stream));
  }
  NEB_CUDA(c, cudaGetLastError());
  return NEB_OK;
}

}  // namespace neb
