// neb_voxel.cu — SURVEY §8(f) item 2: Alg. 3 of the paper, "Point to Line Charge Reduction
// (Voxelization)": dense clusters of point charges are mapped into representative line charges, so that the
// space-charge sums run over N_voxels << N_points sources.  Reading S27: voxel index =
// floor((p - origin)/voxel) clamped to the grid; an occupied voxel (at least one point, Alg. 3's isOccupied)
// becomes one line through its centre, parallel to z, spanning its z extent, lambda = total charge / voxel_z.
//
//   Kernel 1 (scatter)  one thread per point: the charge is added to the voxel's total in 128-bit fixed point by
//                       integer atomics (order-independent: lambda is bit-reproducible), atomicOr of its occupancy flag.
//   Kernel 2 (reduce)   instead of Alg. 3's atomicAdd on a global line counter (arbitrary order), the occupied
//                       voxels are compacted by a scan, so that the line list is in voxel-index order on every run:
//                       count per 1024-voxel block -> exclusive scan of the block counts -> ballot/popc ranks.
//   line_kernel         the direct sum over line charges (same structure as the point-charge kernel a8: a thread owns
//                       a point, line tiles in shared memory), closed form of Eq. (2) integrated along the line,
//                       with the same cancellation-free logarithm as an element edge.
#include "neb_internal.h"
#include "neb_influence.cuh"

namespace neb {

constexpr int kVoxBlock = 1024;
constexpr int kLineTile = 256;
constexpr int kLineThreads = 128;

struct VoxGrid {
  double o[3], d[3];
  int n[3];
};

// Voxel totals are accumulated in 128-bit FIXED POINT with integer atomics, so that they do not depend on the order in
// which the threads arrive (an fp64 atomicAdd would make lambda order-dependent in its last bits): with
// e = 35 - exponent(max |q|) every charge becomes x = q 2^e, |x| < 2^36, split exactly into an integer part and a
// fraction kept to 2^-36; the two parts are summed in two 64-bit integers per voxel (no overflow below 2^26 charges),
// i.e. each charge enters with an absolute error below 2^-72 max|q| and the sum itself is exact.
constexpr int kFixFrac = 36;

// max |charge| as an integer max on the bit pattern (non-negative doubles order like their bits); sources c >= q are
// the line charges of an earlier voxelisation, folded back in as their total charge lambda (z_stop - z_start)
__device__ __forceinline__ double voxel_source_charge(int64_t c, int64_t q, int64_t q_stride, const double* __restrict__ ch,
                                                      int64_t line_cap, const double* __restrict__ lines) {
  if (c < q) return ch[3 * q_stride + c];
  const int64_t l = c - q;
  return lines[4 * line_cap + l] * (lines[3 * line_cap + l] - lines[2 * line_cap + l]);
}

__global__ void voxel_maxabs_kernel(int64_t q, int64_t q_stride, const double* __restrict__ ch, int64_t nl, int64_t line_cap,
                                    const double* __restrict__ lines, unsigned long long* __restrict__ maxbits) {
  int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  unsigned long long b = 0ull;
  if (c < q + nl) {
    double v = fabs(voxel_source_charge(c, q, q_stride, ch, line_cap, lines));
    if (v == v && v < 1.0e300) b = (unsigned long long)__double_as_longlong(v);
  }
  b = __reduce_max_sync(0xffffffffu, (unsigned)(b >> 32)) == (unsigned)(b >> 32) ? b : 0ull;   // cheap pre-filter per warp
  if (b) atomicMax(maxbits, b);
}

__global__ void voxel_scatter_kernel(int64_t q, int64_t q_stride, const double* __restrict__ ch, int64_t nl, int64_t line_cap,
                                     const double* __restrict__ lines, VoxGrid g, const unsigned long long* __restrict__ maxbits,
                                     unsigned long long* __restrict__ tot_hi, unsigned long long* __restrict__ tot_lo,
                                     unsigned* __restrict__ occupied) {
  int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= q + nl) return;
  double p[3];
  if (c < q) { p[0] = ch[c]; p[1] = ch[q_stride + c]; p[2] = ch[2 * q_stride + c]; }
  else {
    const int64_t l = c - q;          // an earlier line: its total charge at its centre
    p[0] = lines[l]; p[1] = lines[line_cap + l]; p[2] = 0.5 * (lines[2 * line_cap + l] + lines[3 * line_cap + l]);
  }
  int64_t idx[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    double t = floor((p[a] - g.o[a]) / g.d[a]);
    t = fmin(fmax(t, 0.0), (double)(g.n[a] - 1));         // points outside count in the nearest border voxel
    idx[a] = (int64_t)t;
  }
  const int64_t v = (idx[2] * g.n[1] + idx[1]) * g.n[0] + idx[0];
  const double mx = __longlong_as_double((long long)*maxbits);
  const int e = (mx > 0.0) ? (kFixFrac - 1) - ilogb(mx) : 0;
  const double x = scalbn(voxel_source_charge(c, q, q_stride, ch, line_cap, lines), e);    // exact; |x| < 2^36
  const double fl = floor(x);
  const long long hi = (long long)fl;
  const long long lo = (long long)scalbn(x - fl, kFixFrac);       // fraction in [0, 1), truncated at 2^-36
  atomicAdd(tot_hi + v, (unsigned long long)hi);
  atomicAdd(tot_lo + v, (unsigned long long)lo);
  atomicOr(occupied + (v >> 5), 1u << (v & 31));
}

// occupied voxels per block of 1024 voxels = 32 flag words
__global__ void voxel_count_kernel(int64_t nwords, const unsigned* __restrict__ occupied, int32_t* __restrict__ block_count) {
  const int64_t w = (int64_t)blockIdx.x * 32 + threadIdx.x;
  int cnt = (w < nwords) ? __popc(occupied[w]) : 0;
  for (int o = 16; o > 0; o >>= 1) cnt += __shfl_down_sync(0xffffffffu, cnt, o);
  if (threadIdx.x == 0) block_count[blockIdx.x] = cnt;
}

// exclusive scan of the block counts by one CTA (at most 65536 blocks); total[0] = number of lines
__global__ void __launch_bounds__(1024) voxel_scan_kernel(int32_t nblocks, const int32_t* __restrict__ block_count,
                                                          int32_t* __restrict__ block_off, int64_t* __restrict__ total) {
  __shared__ int s_warp[32];
  __shared__ int s_carry;
  if (threadIdx.x == 0) s_carry = 0;
  __syncthreads();
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  for (int base = 0; base < nblocks; base += 1024) {
    const int i = base + threadIdx.x;
    const int v = (i < nblocks) ? block_count[i] : 0;
    int inc = v;
    for (int o = 1; o < 32; o <<= 1) {
      const int t = __shfl_up_sync(0xffffffffu, inc, o);
      if (lane >= o) inc += t;
    }
    if (lane == 31) s_warp[warp] = inc;
    __syncthreads();
    if (warp == 0) {
      int w = s_warp[lane];
      for (int o = 1; o < 32; o <<= 1) {
        const int t = __shfl_up_sync(0xffffffffu, w, o);
        if (lane >= o) w += t;
      }
      s_warp[lane] = w;
    }
    __syncthreads();
    const int before = s_carry + (warp ? s_warp[warp - 1] : 0) + inc - v;
    if (i < nblocks) block_off[i] = before;
    __syncthreads();
    if (threadIdx.x == 1023) s_carry = before + v;
    __syncthreads();
  }
  if (threadIdx.x == 0) total[0] = s_carry;
}

// one CTA of 1024 threads per block of 1024 voxels: rank of each occupied voxel, then its line
__global__ void __launch_bounds__(kVoxBlock) voxel_lines_kernel(int64_t nv, VoxGrid g, const unsigned long long* __restrict__ maxbits,
                                                                const unsigned long long* __restrict__ tot_hi,
                                                                const unsigned long long* __restrict__ tot_lo,
                                                                const unsigned* __restrict__ occupied, const int32_t* __restrict__ block_off,
                                                                int64_t cap, double* __restrict__ lines) {
  __shared__ int s_pre[32];
  const int64_t v = (int64_t)blockIdx.x * kVoxBlock + threadIdx.x;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const unsigned word = ((v - lane) < nv) ? occupied[(v - lane) >> 5] : 0u;   // the warp's 32 voxels = one flag word
  const bool occ = (word >> lane) & 1u;
  if (lane == 0) s_pre[warp] = __popc(word);
  __syncthreads();
  if (warp == 0) {
    int w = s_pre[lane], inc = w;
    for (int o = 1; o < 32; o <<= 1) {
      const int t = __shfl_up_sync(0xffffffffu, inc, o);
      if (lane >= o) inc += t;
    }
    s_pre[lane] = inc - w;
  }
  __syncthreads();
  if (!occ) return;
  const int64_t L = (int64_t)block_off[blockIdx.x] + s_pre[warp] + __popc(word & ((1u << lane) - 1u));
  const int64_t i = v % g.n[0], j = (v / g.n[0]) % g.n[1], k = v / ((int64_t)g.n[0] * g.n[1]);
  // one rounded multiply and one rounded add (no FMA contraction): the line positions are reproducible to the bit
  lines[0 * cap + L] = __dadd_rn(g.o[0], __dmul_rn((double)i + 0.5, g.d[0]));
  lines[1 * cap + L] = __dadd_rn(g.o[1], __dmul_rn((double)j + 0.5, g.d[1]));
  lines[2 * cap + L] = __dadd_rn(g.o[2], __dmul_rn((double)k, g.d[2]));
  lines[3 * cap + L] = __dadd_rn(g.o[2], __dmul_rn((double)(k + 1), g.d[2]));
  const double mx = __longlong_as_double((long long)*maxbits);
  const int e = (mx > 0.0) ? (kFixFrac - 1) - ilogb(mx) : 0;
  const double total = scalbn((double)(long long)tot_hi[v] + scalbn((double)(long long)tot_lo[v], -kFixFrac), -e);
  lines[4 * cap + L] = total / g.d[2];
}

// Direct sum over line charges parallel to z.  grid = (ceil(m/128), n_split); partial[(split*4 + c) * m + p],
// without the Coulomb constant (reduce_kernel applies it, as for the point charges).
__global__ void __launch_bounds__(kLineThreads) line_kernel(const double* __restrict__ lines, int64_t nl, int64_t cap,
                                                            const double* __restrict__ pts, int64_t m, int64_t per_split,
                                                            double* __restrict__ partial) {
  __shared__ double sl[5][kLineTile];
  int64_t p = (int64_t)blockIdx.x * kLineThreads + threadIdx.x;
  int64_t pc = min(p, m - 1);
  const double px = pts[pc], py = pts[m + pc], pz = pts[2 * m + pc];
  const int64_t k0 = (int64_t)blockIdx.y * per_split, k1 = min(nl, k0 + per_split);
  double phi = 0, ex = 0, ey = 0, ez = 0;
  for (int64_t base = k0; base < k1; base += kLineTile) {
    const int cnt = (int)min((int64_t)kLineTile, k1 - base);
    __syncthreads();
    for (int idx = threadIdx.x; idx < 5 * kLineTile; idx += kLineThreads) {
      const int f = idx / kLineTile, e = idx % kLineTile;
      if (e < cnt) sl[f][e] = lines[f * cap + base + e];
    }
    __syncthreads();
#pragma unroll 2
    for (int e = 0; e < cnt; ++e) {
      const double dx = px - sl[0][e], dy = py - sl[1][e];
      const double l1 = sl[2][e] - pz, l2 = sl[3][e] - pz, lam = sl[4][e];
      const double rho2 = fma(dx, dx, dy * dy);
      const double R1 = MathFast::sqrt_nn(fma(l1, l1, rho2)), R2 = MathFast::sqrt_nn(fma(l2, l2, rho2));
      // ln[(R2 + l2)/(R1 + l1)] = asinh(l2/rho) - asinh(l1/rho), in the cancellation-free form of an element edge
      const double f = edge_log<MathFast>(l1, l2, R1, R2, rho2, l2 - l1);
      const double i1 = MathFast::rcp_pos(clamp_tiny(R1)), i2 = MathFast::rcp_pos(clamp_tiny(R2));
      const double er = fma(l2, i2, -l1 * i1) * MathFast::rcp_pos(clamp_tiny(rho2));   // E_rho / rho
      const double w = (rho2 > 0.0) ? lam : 0.0;            // a point on the line's axis is skipped (reading S27)
      phi = fma(w, f, phi);
      ex = fma(w * er, dx, ex);
      ey = fma(w * er, dy, ey);
      ez = fma(w, i2 - i1, ez);
    }
  }
  if (p < m) {
    double* o = partial + (int64_t)blockIdx.y * 4 * m;
    o[p] = phi; o[m + p] = ex; o[2 * m + p] = ey; o[3 * m + p] = ez;
  }
}

void launch_line_kernel(neb_ctx* c, int64_t m, const double* d_pts, int splits, int64_t per_split, double* partial) {
  dim3 grid((unsigned)((m + kLineThreads - 1) / kLineThreads), (unsigned)splits);
  line_kernel<<<grid, kLineThreads, 0, c->stream>>>(c->d_lines, c->n_lines, c->line_cap, d_pts, m, per_split, partial);
  c->launches++;
}

neb_status voxelize_charges(neb_ctx* c, const double* origin, const double* voxel, const int32_t* dims, int64_t* n_lines_out) {
  VoxGrid g;
  for (int a = 0; a < 3; ++a) { g.o[a] = origin[a]; g.d[a] = voxel[a]; g.n[a] = dims[a]; }
  const int64_t nv = (int64_t)dims[0] * dims[1] * dims[2];
  const int64_t nwords = (nv + 31) / 32, nblocks = (nv + kVoxBlock - 1) / kVoxBlock;
  // sources: the point charges held now, and the lines of an earlier voxelisation (each as its total charge at its
  // centre), so that charge is conserved over repeated calls
  const int64_t nsrc = c->q + c->n_lines;
  if (nsrc > (1LL << 26)) return fail(c, NEB_EINVAL, "neb_voxelize_space_charge: more than 2^26 charges");
  unsigned long long *tot_hi = nullptr, *tot_lo = nullptr, *maxbits = nullptr;
  unsigned* occ = nullptr;
  int32_t *bcount = nullptr, *boff = nullptr;
  int64_t* d_nl = nullptr;
  double* old_lines = c->d_lines;
  const int64_t old_cap = c->line_cap, old_nl = c->n_lines;
  // the flag words are padded to whole blocks so that voxel_count_kernel's last CTA reads initialised memory
  NEB_CUDA(c, cudaMallocFromPoolAsync((void**)&tot_hi, sizeof(unsigned long long) * (size_t)nv, c->pool, c->stream));
  NEB_CUDA(c, cudaMallocFromPoolAsync((void**)&tot_lo, sizeof(unsigned long long) * (size_t)nv, c->pool, c->stream));
  NEB_CUDA(c, cudaMallocFromPoolAsync((void**)&maxbits, sizeof(unsigned long long), c->pool, c->stream));
  NEB_CUDA(c, cudaMallocFromPoolAsync((void**)&occ, sizeof(unsigned) * (size_t)(nblocks * 32), c->pool, c->stream));
  NEB_CUDA(c, cudaMallocFromPoolAsync((void**)&bcount, sizeof(int32_t) * (size_t)nblocks, c->pool, c->stream));
  NEB_CUDA(c, cudaMallocFromPoolAsync((void**)&boff, sizeof(int32_t) * (size_t)nblocks, c->pool, c->stream));
  NEB_CUDA(c, cudaMallocFromPoolAsync((void**)&d_nl, sizeof(int64_t), c->pool, c->stream));
  NEB_CUDA(c, cudaMemsetAsync(tot_hi, 0, sizeof(unsigned long long) * (size_t)nv, c->stream));
  NEB_CUDA(c, cudaMemsetAsync(tot_lo, 0, sizeof(unsigned long long) * (size_t)nv, c->stream));
  NEB_CUDA(c, cudaMemsetAsync(maxbits, 0, sizeof(unsigned long long), c->stream));
  NEB_CUDA(c, cudaMemsetAsync(occ, 0, sizeof(unsigned) * (size_t)(nblocks * 32), c->stream));
  int64_t nl = 0;
  {
    StageTimer t(c, NEB_STAGE_CHARGES);
    const unsigned sb = (unsigned)((nsrc + 255) / 256);
    voxel_maxabs_kernel<<<sb, 256, 0, c->stream>>>(c->q, c->q_cap, c->d_charges, old_nl, old_cap, old_lines, maxbits);
    voxel_scatter_kernel<<<sb, 256, 0, c->stream>>>(c->q, c->q_cap, c->d_charges, old_nl, old_cap, old_lines, g, maxbits, tot_hi, tot_lo, occ);
    voxel_count_kernel<<<(unsigned)nblocks, 32, 0, c->stream>>>(nwords, occ, bcount);
    voxel_scan_kernel<<<1, 1024, 0, c->stream>>>((int32_t)nblocks, bcount, boff, d_nl);
    c->launches += 4;
  }
  NEB_CUDA(c, cudaMemcpyAsync(&nl, d_nl, sizeof(int64_t), cudaMemcpyDeviceToHost, c->stream));
  NEB_CUDA(c, cudaStreamSynchronize(c->stream));            // the old lines have been read by now
  if (nl > c->line_cap) {
    if (c->d_lines) NEB_CUDA(c, cudaFree(c->d_lines));
    c->d_lines = nullptr;
    c->line_cap = (nl + 255) / 256 * 256;
    NEB_CUDA(c, cudaMalloc((void**)&c->d_lines, sizeof(double) * 5 * (size_t)c->line_cap));
  }
  {
    StageTimer t(c, NEB_STAGE_CHARGES);
    voxel_lines_kernel<<<(unsigned)nblocks, kVoxBlock, 0, c->stream>>>(nv, g, maxbits, tot_hi, tot_lo, occ, boff, c->line_cap, c->d_lines);
    c->launches++;
  }
  NEB_CUDA(c, cudaGetLastError());
  cudaFreeAsync(tot_hi, c->stream);
  cudaFreeAsync(tot_lo, c->stream);
  cudaFreeAsync(maxbits, c->stream);
  cudaFreeAsync(occ, c->stream);
  cudaFreeAsync(bcount, c->stream);
  cudaFreeAsync(boff, c->stream);
  cudaFreeAsync(d_nl, c->stream);
  c->n_lines = nl;
  c->q = 0;                      // the points are now represented by the lines
  if (n_lines_out) *n_lines_out = nl;
  return NEB_OK;
}

}  // namespace neb
