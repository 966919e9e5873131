// neb_lu_panel.cu — a5: LU panel factorisation (64 columns, partial pivoting) of ANY height on ONE thread-block
// cluster (up to 16 CTAs x 256 threads = 16 SMs), so that it can run beside the trailing update of the previous
// panel on the other SMs (look-ahead) whatever the matrix size.  Replaces round 1's two kernels: the
// register-resident cluster kernel (<= 8192 rows: a thread kept 32 columns of ONE row, ~2.2 us per column, most of it
// a CTA barrier + a cluster barrier whose acquire flushes L1 under spilled registers) and the grid-wide cooperative
// kernel (all 148 SMs, 4.8 us per column through a global-memory barrier, no look-ahead, N <= 56704).
//
// Layout of the work.  A thread owns R rows BY IDENTITY (rows k + i C 256 + cta 256 + tid, i < R: consecutive threads
// hold consecutive rows, so every global access is coalesced) and keeps W columns of them in registers (R W <= 64
// doubles; 256 threads per CTA: a column step is ~500 instructions per warp and issues in order, so few fat threads
// beat many thin ones).  The 64 columns are processed as 64/W sub-panels:
//   left-looking step   the sub-panel's columns are loaded and brought up to date with the columns already factored:
//                       every CTA fetches the (so far jb) pivot rows' raw values and their multipliers, solves
//                       U12 = L11^-1 A12 in shared memory (one warp per column, substitution by shuffles) and each
//                       thread subtracts sum_s l[row][s] U12[s][:] from its rows (its own multipliers come back from
//                       L2, software-pipelined: 8 (m jb) bytes per sub-panel, the only re-read of the algorithm);
//   right-looking steps inside the sub-panel, one per column: pivot search, exchange, rank-1 update in registers; a
//                       multiplier goes to global memory at once and its window slot is cleared, so that finished
//                       columns are zero in every row and the update needs no masks.
// Pivoting is implicit: rows never move while the panel is factored, every thread tracks the POSITION its rows occupy
// (ipiv[j] = position of the winner at that time, as LAPACK's sequential exchanges would give); at the end the rows
// that did change position are moved in chunks (read, cluster barrier, write).  Among candidates of exactly equal
// magnitude the one held by the lowest (row slot, lane, warp, CTA) wins: a fixed, run-to-run reproducible rule.
//
// The per-column exchange has no cluster barrier and no fence:
//   per-warp argmax by two REDUX + one vote; the winning lane writes its candidate record (row entries, |value|,
//   position, row identity, and the reciprocal of the would-be pivot, formed in the shadow of the REDUX)  ->  warps
//   1..7 bar.arrive, warp 0 bar.sync (named barrier: only the consumer waits)  ->  warp 0 picks the CTA's candidate and
//   PUSHES the record into the shared memory of all C CTAs with 16-byte st.async stores, each completing transaction
//   bytes on the DESTINATION's mbarrier  ->  every warp of every CTA waits on its own CTA's mbarrier
//   (mbarrier.try_wait: hardware sleep) and picks the global winner from the C records.
// Two buffers / two mbarriers alternate by column parity: a CTA can only be one column ahead of any other, because
// it needs every CTA's candidate of column j to leave column j.
// The column loop is ROLLED over groups of 4 columns (unrolled, the body of a whole sub-panel would not fit the
// instruction cache; round 1 measured that form fetch-bound): inside a group the window slots are static, after a
// group the W-column window is rotated by 4, so that register indices never depend on the column.
// Measured on B200 (standalone, CUDA events): 82 us for a 64 x 1024 panel (4 CTAs), 115 us at 6144 and 8192 rows (16
// CTAs, 2 rows per thread), 246 us at 19456 rows, 0.9 ms at 50048 rows — 0.9-1.2 us per column where the panel chain
// is the critical path (round 1: 2.2 us), and on 16 SMs only where it hides behind the trailing update.
#include <cooperative_groups.h>

#include "neb_internal.h"

namespace cg = cooperative_groups;

namespace neb {

constexpr int PS_THREADS = 256;
constexpr int PS_WARPS = PS_THREADS / 32;
constexpr int PS_MAXC = 16;       // CTAs per cluster (non-portable size, granted on B200)
constexpr int PS_NB = 64;         // panel width
constexpr int PS_NONE = 0x7fffffff;

template <int W>
struct __align__(16) PsCand {     // one pivot candidate; (W + 4) * 8 bytes, a multiple of 16
  double row[W];                  // its row in window order (slot 0 = the current column)
  unsigned long long val;         // |value| bits
  unsigned long long meta;        // position (low word; PS_NONE: no row left) and identity row (high word)
  double invp;                    // 1 / value
  double pad;
};

template <int W>
struct __align__(16) PsSmem {
  PsCand<W> cand[2][PS_MAXC];                 // every CTA's candidate (remote st.async), by column parity
  PsCand<W> wc[2][PS_WARPS];                  // per-warp candidates
  unsigned long long mbar[2];
  double L11[PS_NB][PS_NB + 1];               // multipliers of the pivot rows (unit lower triangle), by pivot index
  double U[PS_NB][W];                         // U12: the pivot rows in the current sub-panel's columns
  int rowid[PS_NB];                           // identity row of pivot t
};

__device__ __forceinline__ unsigned ps_smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }

__device__ __forceinline__ unsigned ps_mapa(unsigned local_addr, unsigned cta) {
  unsigned r;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(local_addr), "r"(cta));
  return r;
}

// remote (or local) 16-byte store that completes 16 transaction bytes on the destination CTA's mbarrier
__device__ __forceinline__ void ps_st_async16(unsigned remote_addr, unsigned long long v0, unsigned long long v1, unsigned remote_mbar) {
  asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v2.b64 [%0], {%1, %2}, [%3];"
               ::"r"(remote_addr), "l"(v0), "l"(v1), "r"(remote_mbar) : "memory");
}

__device__ __forceinline__ void ps_mbar_wait(unsigned bar, unsigned parity) {
  unsigned done = 0;
  int spin = 0;
  do {
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                 : "=r"(done) : "r"(bar), "r"(parity) : "memory");
  } while (!done && ++spin < (1 << 24));
  if (!done) asm volatile("trap;");       // a lost exchange ends in an error, not in a hang
}

// Warp-wide argmax of |value| bits (non-negative doubles order like their bit patterns) among the lanes with in = true:
// two REDUX and one vote; returns the winning lane (the lowest among exact ties), or -1 if nobody took part.
__device__ __forceinline__ int ps_warp_argmax(bool in, unsigned hi, unsigned lo) {
  const unsigned mh = __reduce_max_sync(0xffffffffu, in ? hi : 0u);
  const bool e1 = in && hi == mh;
  const unsigned ml = __reduce_max_sync(0xffffffffu, e1 ? lo : 0u);
  const unsigned tie = __ballot_sync(0xffffffffu, e1 && lo == ml);
  return tie ? __ffs(tie) - 1 : -1;
}

// 1/x for a would-be pivot, branch-free so that it schedules into the latency shadow of the REDUX chain: MUFU.RCP64H
// seed + one cubic step (relative error ~2^-69 before the final rounding).  Row-scaled matrices keep pivots within
// [1e-290, 1]; a zero or denormal pivot yields inf/NaN here and is reported through the singular flag anyway.
__device__ __forceinline__ double ps_pivot_rcp(double x) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  const double e = fma(-x, r, 1.0);
  const double e2 = fma(e, e, e);
  return fma(r, e2, r);
}

// Everything one column step needs besides the thread's rows.
template <int W>
struct PsCtx {
  PsSmem<W>* sm;
  double* A;
  int64_t ld, k;
  int32_t* ipiv;
  int32_t* flag;
  int C, tid, lane, warp, kk;
  unsigned rank;
  // warp 0: where each of its (at most 5) pushes per column goes — loop-invariant up to the parity offset
  unsigned push_dst[(PS_MAXC * ((W + 4) / 2) + 31) / 32], push_mbar[(PS_MAXC * ((W + 4) / 2) + 31) / 32];
  int push_pc[(PS_MAXC * ((W + 4) / 2) + 31) / 32];
};

// One column of the right-looking sweep; the current column sits in window slot S (static), jcol = its index in the panel.
template <int R, int W, int S>
__device__ __forceinline__ void ps_column(const PsCtx<W>& x, int jcol, double (&a)[R][W], int (&pos)[R], const int (&row)[R],
                                          const bool (&valid)[R], bool& any_swap) {
  PsSmem<W>& sm = *x.sm;
  constexpr int NP = (W + 4) / 2;                           // 16-byte pieces of a candidate record
  constexpr int NPUSH = (PS_MAXC * NP + 31) / 32;
  const int par = jcol & 1, dr = x.kk + jcol, lane = x.lane, warp = x.warp;
  // (1) this thread's best row (lowest row slot among ties), then the warp's; the reciprocal of the thread's value is
  // formed in the shadow of the two REDUX
  unsigned long long best = 0ull;
  int bi = -1;
#pragma unroll
  for (int i = 0; i < R; ++i) {
    double v = fabs(a[i][S]);
    if (!(v == v)) v = 0.0;                                 // NaN never wins; caught by the zero-pivot test
    const unsigned long long bits = (unsigned long long)__double_as_longlong(v);
    if (valid[i] && pos[i] >= dr && (bi < 0 || bits > best)) { best = bits; bi = i; }
  }
  double brow[W];
  int bpos = 0, brid = 0;
#pragma unroll
  for (int c = 0; c < W; ++c) brow[c] = a[0][c];
  bpos = pos[0]; brid = row[0];
#pragma unroll
  for (int i = 1; i < R; ++i) {
    if (i == bi) {
#pragma unroll
      for (int c = 0; c < W; ++c) brow[c] = a[i][c];
      bpos = pos[i]; brid = row[i];
    }
  }
  const int wl = ps_warp_argmax(bi >= 0, (unsigned)(best >> 32), (unsigned)best);
  const double binv = ps_pivot_rcp(brow[S]);
  PsCand<W>& w = sm.wc[par][warp];
  if (lane == (wl < 0 ? 0 : wl)) {
    if (wl >= 0) {
      double2* wr = reinterpret_cast<double2*>(w.row);
#pragma unroll
      for (int c = 0; c < W; c += 2) wr[c / 2] = make_double2(brow[c], brow[c + 1]);
      *reinterpret_cast<ulonglong2*>(&w.val) =
          make_ulonglong2(best, (unsigned long long)(unsigned)bpos | ((unsigned long long)(unsigned)brid << 32));
      w.invp = binv;
    } else {
      w.meta = (unsigned long long)(unsigned)PS_NONE;
    }
  }
  // (2) producer/consumer named barrier: only warp 0 waits for the per-warp candidates
  if (warp != 0) {
    asm volatile("bar.arrive 1, %0;" ::"n"(PS_THREADS) : "memory");
  } else {
    asm volatile("bar.sync 1, %0;" ::"n"(PS_THREADS) : "memory");
    ulonglong2 vm = make_ulonglong2(0ull, (unsigned long long)(unsigned)PS_NONE);
    if (lane < PS_WARPS) vm = *reinterpret_cast<const ulonglong2*>(&sm.wc[par][lane].val);
    const int cw = ps_warp_argmax((int)(unsigned)vm.y != PS_NONE, (unsigned)(vm.x >> 32), (unsigned)vm.x);
    if (lane == 0)
      asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;"
                   ::"r"(ps_smem_u32(&sm.mbar[par])), "r"((unsigned)(NP * 16) * (unsigned)x.C) : "memory");
    // (3) push the CTA's candidate record into every CTA of the cluster (its own included), 16 bytes per store
    const ulonglong2* src = reinterpret_cast<const ulonglong2*>(&sm.wc[par][cw < 0 ? 0 : cw]);
    const unsigned poff = (unsigned)par * (unsigned)(sizeof(PsCand<W>) * PS_MAXC), moff = (unsigned)par * 8u;
    ulonglong2 v[NPUSH];
#pragma unroll
    for (int it = 0; it < NPUSH; ++it)
      if (x.push_pc[it] >= 0) v[it] = src[x.push_pc[it]];
#pragma unroll
    for (int it = 0; it < NPUSH; ++it) {
      if (x.push_pc[it] >= 0) {
        if (cw < 0 && x.push_pc[it] == W / 2) v[it].y = (unsigned long long)(unsigned)PS_NONE;      // an empty candidate
        ps_st_async16(x.push_dst[it] + poff, v[it].x, v[it].y, x.push_mbar[it] + moff);
      }
    }
  }
  // (4) every warp waits for the C records to land in its own CTA and picks the winner
  ps_mbar_wait(ps_smem_u32(&sm.mbar[par]), (unsigned)((jcol >> 1) & 1));
  ulonglong2 gm = make_ulonglong2(0ull, (unsigned long long)(unsigned)PS_NONE);
  if (lane < x.C) gm = *reinterpret_cast<const ulonglong2*>(&sm.cand[par][lane].val);
  const int gc = ps_warp_argmax((int)(unsigned)gm.y != PS_NONE, (unsigned)(gm.x >> 32), (unsigned)gm.x);
  const bool any = gc >= 0;
  const PsCand<W>& win = sm.cand[par][any ? gc : 0];
  const ulonglong2 wm = *reinterpret_cast<const ulonglong2*>(&win.val);
  const int wp = any ? (int)(unsigned)wm.y : dr;
  const double invp = win.invp;
  double prow[W];
#pragma unroll
  for (int c = 0; c < W; c += 2) {
    const double2 t = reinterpret_cast<const double2*>(win.row)[c / 2];
    prow[c] = t.x; prow[c + 1] = t.y;
  }
  if (x.tid == 0) {
    sm.rowid[jcol] = any ? (int)(unsigned)(wm.y >> 32) : dr;
    if (x.rank == 0) {
      x.ipiv[dr] = wp;
      if (!any || wm.x == 0ull) atomicOr(x.flag, 2);        // zero (or NaN -> 0) pivot: NEB_ESINGULAR
    }
  }
  any_swap |= (wp != dr);
  // (5) positions; multipliers go straight to global memory (identity rows) and the window slot is cleared, so that a
  // finished column is zero in every row's window and in every later pivot row: the update needs no masks
#pragma unroll
  for (int i = 0; i < R; ++i) {
    pos[i] = (pos[i] == dr) ? wp : ((pos[i] == wp) ? dr : pos[i]);
    if (valid[i] && pos[i] > dr) {
      const double lmul = a[i][S] * invp;
      x.A[row[i] + (x.k + jcol) * x.ld] = lmul;
      a[i][S] = 0.0;
#pragma unroll
      for (int c = 0; c < W; ++c)
        if (c != S) a[i][c] = fma(-lmul, prow[c], a[i][c]);
    }
  }
}

template <int R, int W>
__global__ void __launch_bounds__(PS_THREADS, 1) panel_stream_kernel(double* __restrict__ A, int64_t ld, int64_t npad, int64_t k,
                                                                     int32_t* __restrict__ ipiv, int32_t* __restrict__ flag) {
  extern __shared__ __align__(16) unsigned char ps_raw[];
  PsSmem<W>& sm = *reinterpret_cast<PsSmem<W>*>(ps_raw);
  cg::cluster_group cluster = cg::this_cluster();
  const int C = (int)cluster.num_blocks();
  const unsigned rank = cluster.block_rank();
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int kk = (int)k;
  constexpr int NP = (W + 4) / 2;
  constexpr int NPUSH = (PS_MAXC * NP + 31) / 32;
  constexpr int UC = W < 4 ? W : 4;                         // columns per iteration of the rolled loop

  if (tid == 0) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(ps_smem_u32(&sm.mbar[0])));
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(ps_smem_u32(&sm.mbar[1])));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  PsCtx<W> x;
  x.sm = &sm; x.A = A; x.ld = ld; x.k = k; x.ipiv = ipiv; x.flag = flag;
  x.C = C; x.tid = tid; x.lane = lane; x.warp = warp; x.kk = kk; x.rank = rank;
#pragma unroll
  for (int it = 0; it < NPUSH; ++it) {
    const int q = lane + 32 * it;
    const int d = q / NP, pc = q - d * NP;
    x.push_pc[it] = (q < C * NP) ? pc : -1;
    x.push_dst[it] = ps_mapa(ps_smem_u32(&sm.cand[0][rank]) + 16u * pc, (unsigned)(d < C ? d : 0));
    x.push_mbar[it] = ps_mapa(ps_smem_u32(&sm.mbar[0]), (unsigned)(d < C ? d : 0));
  }
  // the rows this thread owns, and the position each of them occupies
  int row[R];                                               // npad < 2^31
  int pos[R];
  bool valid[R];
#pragma unroll
  for (int i = 0; i < R; ++i) {
    const int64_t r = k + ((int64_t)i * C + rank) * PS_THREADS + tid;
    valid[i] = r < npad;
    row[i] = valid[i] ? (int)r : 0;
    pos[i] = valid[i] ? (int)r : PS_NONE - 1;               // an absent row never takes part (guarded by valid)
  }
  cluster.sync();                                           // every CTA's mbarriers exist before the first push

  double a[R][W];
  bool any_swap = false;
#pragma unroll 1
  for (int jb = 0; jb < PS_NB; jb += W) {
    // ---- load the sub-panel's columns ----
#pragma unroll
    for (int i = 0; i < R; ++i)
#pragma unroll
      for (int c = 0; c < W; ++c) a[i][c] = valid[i] ? A[row[i] + (k + jb + c) * ld] : 0.0;
    if (jb > 0) {
      // ---- left-looking step: U12 = L11^-1 A12 (every CTA on its own), then rows -= l U12 ----
      // The new pivot rows' multipliers and all pivot rows' raw entries in the new columns; the cluster barrier that
      // ended the last sub-panel made the other threads' stores visible.  All loads first, then the stores.
      {
        constexpr int NL = (W * PS_NB + PS_THREADS - 1) / PS_THREADS, NU = (PS_NB * W + PS_THREADS - 1) / PS_THREADS;
        double vl[NL], vu[NU];
#pragma unroll
        for (int q = 0; q < NL; ++q) {
          const int idx = tid + q * PS_THREADS, t = jb - W + idx / PS_NB, s = idx % PS_NB;
          vl[q] = (idx < W * PS_NB && s < t) ? __ldcg(A + sm.rowid[t] + (k + s) * ld) : 0.0;
        }
#pragma unroll
        for (int q = 0; q < NU; ++q) {
          const int idx = tid + q * PS_THREADS, t = idx / W, c = idx % W;
          vu[q] = (idx < jb * W) ? __ldcg(A + sm.rowid[t] + (k + jb + c) * ld) : 0.0;
        }
#pragma unroll
        for (int q = 0; q < NL; ++q) {
          const int idx = tid + q * PS_THREADS, t = jb - W + idx / PS_NB, s = idx % PS_NB;
          if (idx < W * PS_NB && s < t) sm.L11[t][s] = vl[q];
        }
#pragma unroll
        for (int q = 0; q < NU; ++q) {
          const int idx = tid + q * PS_THREADS;
          if (idx < jb * W) sm.U[idx / W][idx % W] = vu[q];
        }
      }
      __syncthreads();
      // forward substitution, one column per warp (two when W = 16): lanes hold entries lane and lane + 32; the
      // multipliers of the next step are fetched while this step's shuffle and FMA are in flight
      for (int col = warp; col < W; col += PS_WARPS) {
        double x0 = (lane < jb) ? sm.U[lane][col] : 0.0, x1 = (lane + 32 < jb) ? sm.U[lane + 32][col] : 0.0;
        double l0 = sm.L11[lane][0], l1 = sm.L11[lane + 32][0];
        for (int s = 0; s < jb - 1; ++s) {
          const double m0 = l0, m1 = l1;
          l0 = sm.L11[lane][s + 1]; l1 = sm.L11[lane + 32][s + 1];
          const double us = __shfl_sync(0xffffffffu, (s < 32) ? x0 : x1, s & 31);
          if (lane > s && lane < jb) x0 = fma(-m0, us, x0);
          if (lane + 32 > s && lane + 32 < jb) x1 = fma(-m1, us, x1);
        }
        if (lane < jb) sm.U[lane][col] = x0;
        if (lane + 32 < jb) sm.U[lane + 32][col] = x1;
      }
      __syncthreads();
      constexpr int UL = (R >= 16) ? 2 : ((R == 8) ? 4 : 8);    // multiplier loads in flight per row (UL divides W)
#pragma unroll
      for (int i = 0; i < R; ++i) {
        if (!valid[i]) continue;
        if (pos[i] < kk + jb) {
          // a pivot row: its entries are the U12 row just solved
#pragma unroll
          for (int c = 0; c < W; ++c) a[i][c] = sm.U[pos[i] - kk][c];
        } else {
          const double* lrow = A + row[i] + k * ld;            // this row's multipliers, written by this thread
          double l[UL], ln[UL];
#pragma unroll
          for (int u = 0; u < UL; ++u) ln[u] = lrow[(int64_t)u * ld];
#pragma unroll 1
          for (int s0 = 0; s0 < jb; s0 += UL) {
#pragma unroll
            for (int u = 0; u < UL; ++u) l[u] = ln[u];
            if (s0 + UL < jb) {
#pragma unroll
              for (int u = 0; u < UL; ++u) ln[u] = lrow[(int64_t)(s0 + UL + u) * ld];     // next round in flight
            }
#pragma unroll
            for (int u = 0; u < UL; ++u)
#pragma unroll
              for (int c = 0; c < W; ++c) a[i][c] = fma(-l[u], sm.U[s0 + u][c], a[i][c]);
          }
        }
      }
    }
    // ---- right-looking steps inside the sub-panel: rolled over groups of UC columns (static window slots inside a
    // group), the window rotates by UC after each group ----
#pragma unroll 1
    for (int jj = 0; jj < W; jj += UC) {
      ps_column<R, W, 0>(x, jb + jj, a, pos, row, valid, any_swap);
      if (UC > 1) ps_column<R, W, (UC > 1 ? 1 : 0)>(x, jb + jj + 1, a, pos, row, valid, any_swap);
      if (UC > 2) ps_column<R, W, (UC > 2 ? 2 : 0)>(x, jb + jj + 2, a, pos, row, valid, any_swap);
      if (UC > 3) ps_column<R, W, (UC > 3 ? 3 : 0)>(x, jb + jj + 3, a, pos, row, valid, any_swap);
#pragma unroll
      for (int i = 0; i < R; ++i) {
        double t[UC];
#pragma unroll
        for (int c = 0; c < UC; ++c) t[c] = a[i][c];
#pragma unroll
        for (int c = 0; c < W - UC; ++c) a[i][c] = a[i][c + UC];
#pragma unroll
        for (int c = 0; c < UC; ++c) a[i][W - UC + c] = t[c];
      }
    }
    // ---- the sub-panel is done (the window is back in natural order).  Multipliers are in global memory already; the
    // rows that are pivots by now store their U entries (from their own diagonal on; a pivot of an earlier sub-panel:
    // all W columns).  Rows never move: identity rows ----
#pragma unroll
    for (int i = 0; i < R; ++i) {
      if (valid[i] && pos[i] < kk + jb + W) {
        const int t = pos[i] - kk - jb;
#pragma unroll
        for (int c = 0; c < W; ++c)
          if (c >= t) A[row[i] + (k + jb + c) * ld] = a[i][c];
      }
    }
    // the cluster barrier orders these stores before the next left-looking step's loads of other threads' rows
    // (and sm.rowid, written by thread 0, before its readers)
    cluster.sync();
  }

  // ---- rows that changed position move there, PC columns at a time (read, cluster barrier, write) ----
  if (any_swap) {                                            // the same value in every thread of the cluster
    constexpr int PC = (16 / R) < 2 ? 2 : (16 / R);
    double t[R][PC];
#pragma unroll 1
    for (int c0 = 0; c0 < PS_NB; c0 += PC) {
#pragma unroll
      for (int i = 0; i < R; ++i) {
        const bool mv = valid[i] && pos[i] != row[i];
#pragma unroll
        for (int c = 0; c < PC; ++c) t[i][c] = mv ? __ldcg(A + row[i] + (k + c0 + c) * ld) : 0.0;
      }
      cluster.sync();
#pragma unroll
      for (int i = 0; i < R; ++i) {
        if (valid[i] && pos[i] != row[i]) {
#pragma unroll
          for (int c = 0; c < PC; ++c) A[(int64_t)pos[i] + (k + c0 + c) * ld] = t[i][c];
        }
      }
    }
  }
  cluster.sync();   // nobody leaves while its shared memory may still be written remotely
}

// (R, W) pairs instantiated: rows per thread x columns per sub-panel, R W <= 64 doubles in registers
#define NEB_PS_VARIANTS(X) X(1, 16) X(2, 16) X(4, 16) X(8, 8) X(16, 4) X(32, 2)

template <int R, int W>
static bool ps_set_attr() {
  if (cudaFuncSetAttribute(panel_stream_kernel<R, W>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(PsSmem<W>)) != cudaSuccess ||
      cudaFuncSetAttribute(panel_stream_kernel<R, W>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) != cudaSuccess) {
    cudaGetLastError();
    return false;
  }
  return true;
}

// Largest cluster size (power of two, <= 16) the CURRENT device can schedule for the kernel; 0 if none.  Kernel
// attributes are per device: called once per context from neb_create (lu_init_device), result kept in the context.
int panel_cluster_probe() {
#define X(R, W) if (!ps_set_attr<R, W>()) return 0;
  NEB_PS_VARIANTS(X)
#undef X
  for (int cs = PS_MAXC; cs >= 1; cs >>= 1) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(cs);
    cfg.blockDim = dim3(PS_THREADS);
    cfg.dynamicSmemBytes = sizeof(PsSmem<16>);
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = cs; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    int nclusters = 0;
    if (cudaOccupancyMaxActiveClusters(&nclusters, panel_stream_kernel<1, 16>, &cfg) == cudaSuccess && nclusters >= 1) return cs;
    cudaGetLastError();
  }
  return 0;
}

// rows one cluster can factor: 32 rows per thread
int64_t panel_cluster_max_rows(neb_ctx* c) { return (int64_t)c->cluster_max_ctas * PS_THREADS * 32; }

template <int R, int W>
static cudaError_t ps_launch(neb_ctx* c, double* A, int cs, int64_t k, cudaStream_t stream) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(cs);
  cfg.blockDim = dim3(PS_THREADS);
  cfg.dynamicSmemBytes = sizeof(PsSmem<W>);
  cfg.stream = stream;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeClusterDimension;
  at[0].val.clusterDim.x = cs; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
  cfg.attrs = at;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, panel_stream_kernel<R, W>, A, c->npad, c->npad, k, c->d_ipiv, c->d_flag);
}

// A: base such that the panel's columns are A + (k .. k+63) * npad (c->d_K on one GPU; a rank's local block shifted to
// its global column position in the distributed factorisation)
neb_status panel_cluster_launch(neb_ctx* c, double* A, int64_t k, cudaStream_t stream) {
  const int64_t mrows = c->npad - k;
  int cs = 1;
  while (cs < c->cluster_max_ctas && (int64_t)cs * PS_THREADS < mrows) cs <<= 1;
  const int64_t per_thread = (mrows + (int64_t)cs * PS_THREADS - 1) / ((int64_t)cs * PS_THREADS);
  cudaError_t e = cudaErrorInvalidValue;
  bool launched = false;
#define X(R, W) if (!launched && per_thread <= R) { e = ps_launch<R, W>(c, A, cs, k, stream); launched = true; }
  NEB_PS_VARIANTS(X)
#undef X
  if (!launched) return fail(c, NEB_EINVAL, "LU panel: more than 32 rows per thread of the cluster (n too large for this device)");
  if (e != cudaSuccess) return fail(c, NEB_ECUDA, std::string("panel_stream_kernel launch: ") + cudaGetErrorString(e));
  c->launches++;
  return NEB_OK;
}

}  // namespace neb
