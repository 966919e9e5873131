// neb_field.cu — the element-point kernels of the hot path:
//   a3  assemble_kernel : LHMatrix, K_ij at collocation point i from element j (+ periodic copies)
//   a7  eval_kernel     : PFAtPoint / ElePFAtPoint, Phi and E at M points, fused with the reduction
//                         over the solved charge densities
//   a8  charge_kernel   : KnChPFAtPoint, direct sum over point charges (Alg. 2 P:234-270 re-designed:
//                         many targets per launch, charge tiles in shared memory, no atomics)
//   a4  rhs_kernel      : RHVector + ValueKnCh
// A thread owns one point; element records (frame tables, SoA) are staged tile by tile through shared
// memory and broadcast to the warp.  Tiles are homogeneous in element kind (the tables are sorted by
// kind), every case distinction inside the influence function is a select: warps never diverge.
// Work is split over element (or charge) chunks in grid.y so that small M still fills 148 SMs; the
// per-chunk partial sums are added by reduce_kernel in a fixed order (deterministic, no fp64 atomics).
#include <algorithm>

#include "neb_internal.h"
#include "neb_influence.cuh"

namespace neb {

#ifndef NEB_EVAL_UNROLL
#define NEB_EVAL_UNROLL 2             // elements of a uniform window in flight per thread
#endif
constexpr int kEvalUnroll = NEB_EVAL_UNROLL;
#ifndef NEB_PAIR_UNROLL
#define NEB_PAIR_UNROLL 1
#endif
#ifndef NEB_PAIR_STRIPS
#define NEB_PAIR_STRIPS 1
#endif
constexpr int kPairUnroll = NEB_PAIR_UNROLL;
constexpr bool kPairStrips = NEB_PAIR_STRIPS != 0;   // strip neighbours evaluated as pairs (rect_pair_local)
constexpr int kThreads = 128;   // threads per CTA = points per CTA
constexpr int kTile = 64;       // elements per shared-memory tile
constexpr int kChargeTile = 256;
constexpr int kMaxImg = NEB_IMG_CHUNK;   // periodic copies per launch (kept in shared memory); more copies: more launches

// Element tiles are staged by the TMA unit: one thread arms an mbarrier with the tile's byte count and issues one
// 1-D bulk copy (cp.async.bulk, SASS UBLKCP) per record field (64 elements x 8 bytes, contiguous in the SoA table);
// the copies land in shared memory asynchronously and complete the mbarrier's transaction count.  Two buffers: tile
// i+1 is in flight while the CTA evaluates tile i, so the only CTA-wide barrier per tile is the one that hands a
// fully read buffer back to the producer.
struct __align__(128) TileSmem {
  double rec[2][kRec][kTile];
  double img[3][kMaxImg];
  double limg[3][kMaxImg];    // the image shifts in the axes of the current uniform window
  unsigned long long mbar[2];
};
constexpr unsigned kTileBytes = kRec * kTile * sizeof(double);

__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void tile_pipe_init(TileSmem& sm) {
  if (threadIdx.x == 0) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(smem_u32(&sm.mbar[0])));
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(smem_u32(&sm.mbar[1])));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
}

// Thread 0: start the copy of the 64-element window [tb, tb + 64) (tb a multiple of 64; the table's stride is a
// multiple of 128 and its tail is zero-filled, so every window is in bounds and 16-byte aligned) into buffer seq & 1.
__device__ __forceinline__ void tile_issue(TileSmem& sm, const GeoTables& g, int64_t tb, unsigned seq) {
  const unsigned buf = seq & 1u, bar = smem_u32(&sm.mbar[buf]);
  // the buffer was last READ through the generic proxy (ordered before this point by the CTA barrier): order
  // those reads before the async-proxy writes
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(kTileBytes) : "memory");
#pragma unroll
  for (int f = 0; f < kRec; ++f) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(&sm.rec[buf][f][0])), "l"(g.rec + f * g.stride + tb), "r"((unsigned)(kTile * sizeof(double))), "r"(bar)
                 : "memory");
  }
}

// Every thread: wait until tile seq has landed.  The spin is bounded (each try_wait already blocks for a
// hardware-defined interval), so that a lost copy ends in a trap instead of a hang.
__device__ __forceinline__ void tile_wait(TileSmem& sm, unsigned seq) {
  const unsigned bar = smem_u32(&sm.mbar[seq & 1u]), parity = (seq >> 1) & 1u;
  unsigned done = 0;
  int spin = 0;
  do {
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                 : "=r"(done) : "r"(bar), "r"(parity) : "memory");
  } while (!done && ++spin < (1 << 22));
  if (!done) asm volatile("trap;");
}

__device__ __forceinline__ Frame frame_of(const TileSmem& sm, unsigned buf, int e) {
  Frame f;
  f.v0x = sm.rec[buf][0][e]; f.v0y = sm.rec[buf][1][e]; f.v0z = sm.rec[buf][2][e];
  f.exx = sm.rec[buf][3][e]; f.exy = sm.rec[buf][4][e]; f.exz = sm.rec[buf][5][e];
  f.eyx = sm.rec[buf][6][e]; f.eyy = sm.rec[buf][7][e]; f.eyz = sm.rec[buf][8][e];
  f.ezx = sm.rec[buf][9][e]; f.ezy = sm.rec[buf][10][e]; f.ezz = sm.rec[buf][11][e];
  f.a = sm.rec[buf][12][e]; f.b = sm.rec[buf][13][e]; f.aux = sm.rec[buf][14][e]; f.far2 = sm.rec[buf][16][e];
  return f;
}

// Adaptive Modelling (reading S28): a FAR periodic copy of an element is represented by its total charge at
// the copy's centroid.  d = (point - shift - centroid) in any orthonormal frame; adds area/r and area d/r^3.
__device__ __forceinline__ void far_copy(double area, double dx, double dy, double dz, double& phi, double& fx, double& fy,
                                         double& fz) {
  const double r2 = fma(dx, dx, fma(dy, dy, dz * dz));
  double y = rsqrt_pos(clamp_tiny(r2));             // 1/r: seed + one cubic step, as in the point-charge kernel
  y = is_zero(r2) ? 0.0 : y;
  const double ar = area * y, ar3 = ar * y * y;
  phi += ar;
  fx = fma(ar3, dx, fx); fy = fma(ar3, dy, fy); fz = fma(ar3, dz, fz);
}

// All elements of one kind in [lo, hi): tile loop, image loop, sink(j, weight_j, sum over copies).
// seq = number of tiles this CTA has consumed so far (buffer = seq & 1, mbarrier parity = (seq >> 1) & 1).
// self0 (compile time: a runtime flag cost 4 % on the hot path): slot 0 of this chunk of copies is the element itself
// (the first chunk); later chunks hold shifted copies only.
// NIMG = 1: the element has no periodic copies — known at compile time, so that the copy loops and the Adaptive-Modelling
// branch disappear from the tile loop (one straight block per pair of elements); NIMG = 0: n_img, n_near at run time.
template <class M, int KIND, bool self0, int NIMG, class Sink>
__device__ __forceinline__ void process_kind(const GeoTables& g, int64_t lo, int64_t hi, TileSmem& sm, int n_img, int n_near,
                                             double px, double py, double pz, Sink& sink, unsigned& seq) {
  if (NIMG == 1) { n_img = 1; n_near = 1; }
  const int64_t tb0 = lo & ~(int64_t)(kTile - 1);
  if (threadIdx.x == 0) tile_issue(sm, g, tb0, seq);
  for (int64_t tb = tb0; tb < hi; tb += kTile) {
    if (threadIdx.x == 0 && tb + kTile < hi) tile_issue(sm, g, tb + kTile, seq + 1);
    tile_wait(sm, seq);
    const unsigned buf = seq & 1u;
    const int e0 = (int)max(lo - tb, (int64_t)0), e1 = (int)min(hi - tb, (int64_t)kTile);
    if (KIND != 2 && g.uniform[3 * (tb >> 6)]) {
      // Uniform window: all 64 elements share one set of unit axes (a face of a mesh).  The point's products with
      // the axes are formed once per window, an element's local coordinates are three subtractions, and the field
      // is accumulated in the LOCAL frame and rotated to global once per window instead of once per pair.
      Axes ax;
      ax.exx = sm.rec[buf][3][e0]; ax.exy = sm.rec[buf][4][e0]; ax.exz = sm.rec[buf][5][e0];
      ax.eyx = sm.rec[buf][6][e0]; ax.eyy = sm.rec[buf][7][e0]; ax.eyz = sm.rec[buf][8][e0];
      ax.ezx = sm.rec[buf][9][e0]; ax.ezy = sm.rec[buf][10][e0]; ax.ezz = sm.rec[buf][11][e0];
      if (n_img > 1) {
        if (threadIdx.x < n_img) {
          const double sx = sm.img[0][threadIdx.x], sy = sm.img[1][threadIdx.x], sz = sm.img[2][threadIdx.x];
          sm.limg[0][threadIdx.x] = fma(sx, ax.exx, fma(sy, ax.exy, sz * ax.exz));
          sm.limg[1][threadIdx.x] = fma(sx, ax.eyx, fma(sy, ax.eyy, sz * ax.eyz));
          sm.limg[2][threadIdx.x] = fma(sx, ax.ezx, fma(sy, ax.ezy, sz * ax.ezz));
        }
        __syncthreads();
      }
      const double PX = fma(px, ax.exx, fma(py, ax.exy, pz * ax.exz));
      const double PY = fma(px, ax.eyx, fma(py, ax.eyy, pz * ax.eyz));
      const double PZ = fma(px, ax.ezx, fma(py, ax.ezy, pz * ax.ezz));
      sink.tile_begin(ax);
      // strip neighbours (rectangles 2k, 2k + 1 of the window sharing an edge: masks from tile_uniform_kernel) are
      // evaluated as a pair, 6 corner distances and 7 edge logarithms for the two instead of 8 and 8; the masks are
      // the same for every thread of the grid, so the choice costs no divergence
      const unsigned mask_x = (KIND == 0 && kPairStrips) ? (unsigned)g.uniform[3 * (tb >> 6) + 1] : 0u;
      const unsigned mask_z = (KIND == 0 && kPairStrips) ? (unsigned)g.uniform[3 * (tb >> 6) + 2] : 0u;
      auto single = [&](int e) {
        const double a = sm.rec[buf][12][e], b = sm.rec[buf][13][e], aux = sm.rec[buf][14][e], far2 = sm.rec[buf][16][e];
        const double X0 = PX - sm.rec[buf][17][e], Y0 = PY - sm.rec[buf][18][e], Z0 = PZ - sm.rec[buf][19][e];
        double phi = 0.0, lx = 0.0, ly = 0.0, lz = 0.0;
        if (self0) {
          local_pair<M, KIND>(a, b, aux, far2, X0, Y0, Z0, phi, lx, ly, lz);
          if (sink.self_pv(tb + e)) { lx = 0.0; ly = 0.0; lz = 0.0; }   // principal value (S5, S8)
        }
#pragma unroll 1
        for (int s = self0 ? 1 : 0; s < n_near; ++s) {
          double p1, x1, y1, z1;
          local_pair<M, KIND>(a, b, aux, far2, X0 - sm.limg[0][s], Y0 - sm.limg[1][s], Z0 - sm.limg[2][s], p1, x1, y1, z1);
          phi += p1; lx += x1; ly += y1; lz += z1;
        }
        if (n_near < n_img) {
          // far copies (Adaptive Modelling): total charge at the copy's centroid, in the window's axes
          const double area = (KIND == 0) ? aux : 0.5 * a * b;
          const double cxl = X0 - ((KIND == 0) ? 0.5 : (1.0 / 3.0)) * a, czl = Z0 - ((KIND == 0) ? 0.5 : (1.0 / 3.0)) * b;
#pragma unroll 1
          for (int s = n_near; s < n_img; ++s) far_copy(area, cxl - sm.limg[0][s], Y0 - sm.limg[1][s], czl - sm.limg[2][s], phi, lx, ly, lz);
        }
        sink.local(tb + e, sm.rec[buf][15][e], phi, lx, ly, lz);
      };
      int e = e0;
      if (e & 1) { single(e); ++e; }                        // pairs sit at even positions of the window
#pragma unroll kPairUnroll
      for (; e + 1 < e1; e += 2) {
        const bool along_x = (mask_x >> (e >> 1)) & 1u, along_z = (mask_z >> (e >> 1)) & 1u;
        if (KIND == 0 && n_near == n_img && (along_x || along_z)) {
          // the pair in the first element's frame; a strip along local Z is the same figure with X and Z exchanged
          const double a1 = sm.rec[buf][12][e], b1 = sm.rec[buf][13][e], a2 = sm.rec[buf][12][e + 1], b2 = sm.rec[buf][13][e + 1];
          const double la1 = along_x ? a1 : b1, la2 = along_x ? a2 : b2, lb = along_x ? b1 : a1;
          const double ab1 = sm.rec[buf][14][e], ab2 = sm.rec[buf][14][e + 1], fa = sm.rec[buf][16][e], fb = sm.rec[buf][16][e + 1];
          const double X0 = PX - sm.rec[buf][17][e], Y0 = PY - sm.rec[buf][18][e], Z0 = PZ - sm.rec[buf][19][e];
          const double S0 = along_x ? X0 : Z0, T0 = along_x ? Z0 : X0;      // along / across the strip
          double p1 = 0.0, s1 = 0.0, y1 = 0.0, t1 = 0.0, p2 = 0.0, s2 = 0.0, y2 = 0.0, t2 = 0.0;
          if (self0) {
            rect_pair_local<M>(la1, la2, lb, ab1, ab2, fa, fb, S0, Y0, T0, p1, s1, y1, t1, p2, s2, y2, t2);
            if (sink.self_pv(tb + e)) { s1 = 0.0; y1 = 0.0; t1 = 0.0; }
            if (sink.self_pv(tb + e + 1)) { s2 = 0.0; y2 = 0.0; t2 = 0.0; }
          }
#pragma unroll 1
          for (int s = self0 ? 1 : 0; s < n_near; ++s) {
            const double sx = sm.limg[0][s], sz = sm.limg[2][s];
            double q1, u1, v1, w1, q2, u2, v2, w2;
            rect_pair_local<M>(la1, la2, lb, ab1, ab2, fa, fb, S0 - (along_x ? sx : sz), Y0 - sm.limg[1][s], T0 - (along_x ? sz : sx),
                               q1, u1, v1, w1, q2, u2, v2, w2);
            p1 += q1; s1 += u1; y1 += v1; t1 += w1; p2 += q2; s2 += u2; y2 += v2; t2 += w2;
          }
          sink.local(tb + e, sm.rec[buf][15][e], p1, along_x ? s1 : t1, y1, along_x ? t1 : s1);
          sink.local(tb + e + 1, sm.rec[buf][15][e + 1], p2, along_x ? s2 : t2, y2, along_x ? t2 : s2);
        } else {
          single(e);
          single(e + 1);
        }
      }
      if (e < e1) single(e);
      sink.tile_end(ax);
    } else {
      sink.gtile_begin();
#pragma unroll 2
      for (int e = e0; e < e1; ++e) {
        Frame fr = frame_of(sm, buf, e);
        // slot 0 is the unshifted copy (the host puts it there).  For the pair (collocation point of element j,
        // element j) its field is dropped: principal value of a flat element's normal field on itself (S5, S8)
        Infl acc = {0.0, 0.0, 0.0, 0.0};
        if (self0) {
          acc = influence<M, KIND>(fr, px, py, pz);      // slot 0 of the first chunk holds the zero shift
          if (sink.self_pv(tb + e)) { acc.ex = 0.0; acc.ey = 0.0; acc.ez = 0.0; }
        }
#pragma unroll 1
        for (int s = self0 ? 1 : 0; s < n_near; ++s) {
          Infl o = influence<M, KIND>(fr, px - sm.img[0][s], py - sm.img[1][s], pz - sm.img[2][s]);
          acc.phi += o.phi; acc.ex += o.ex; acc.ey += o.ey; acc.ez += o.ez;
        }
        if (n_near < n_img) {
          // far copies (Adaptive Modelling): total charge at the copy's centroid, in global coordinates
          const double wc = (KIND == 0) ? 0.5 : ((KIND == 1) ? (1.0 / 3.0) : 0.5), wz = (KIND == 2) ? 0.0 : wc;
          const double area = (KIND == 0) ? fr.aux : ((KIND == 1) ? 0.5 * fr.a * fr.b : fr.aux * fr.a);
          const double gx = px - fma(wc * fr.a, fr.exx, fma(wz * fr.b, fr.ezx, fr.v0x));
          const double gy = py - fma(wc * fr.a, fr.exy, fma(wz * fr.b, fr.ezy, fr.v0y));
          const double gz = pz - fma(wc * fr.a, fr.exz, fma(wz * fr.b, fr.ezz, fr.v0z));
#pragma unroll 1
          for (int s = n_near; s < n_img; ++s) far_copy(area, gx - sm.img[0][s], gy - sm.img[1][s], gz - sm.img[2][s], acc.phi, acc.ex, acc.ey, acc.ez);
        }
        sink(tb + e, sm.rec[buf][15][e], acc);
      }
      sink.gtile_end();
    }
    __syncthreads();                               // the buffer is free for the tile after next
    ++seq;
  }
}

template <class M, bool self0, int NIMG, class Sink>
__device__ __forceinline__ void process_range(const GeoTables& g, int64_t j0, int64_t j1, TileSmem& sm, int n_img, int n_near,
                                              double px, double py, double pz, Sink& sink) {
  int64_t r1 = g.n_rect, t1 = r1 + g.n_tri, w1 = t1 + g.n_wire;
  int64_t lo, hi;
  unsigned seq = 0;
  lo = max(j0, (int64_t)0); hi = min(j1, r1);
  if (lo < hi) process_kind<M, 0, self0, NIMG>(g, lo, hi, sm, n_img, n_near, px, py, pz, sink, seq);
  lo = max(j0, r1); hi = min(j1, t1);
  if (lo < hi) process_kind<M, 1, self0, NIMG>(g, lo, hi, sm, n_img, n_near, px, py, pz, sink, seq);
  lo = max(j0, t1); hi = min(j1, w1);
  if (lo < hi) process_kind<M, 2, self0, NIMG>(g, lo, hi, sm, n_img, n_near, px, py, pz, sink, seq);
}

// img: one chunk of the copy table, [3][kMaxImg] (the host packs the sorted shifts in chunks of kMaxImg)
__device__ __forceinline__ void load_images(TileSmem& sm, const double* img, int n_img) {
  for (int idx = threadIdx.x; idx < 3 * kMaxImg; idx += blockDim.x) {
    const int k = idx / kMaxImg, sidx = idx % kMaxImg;
    sm.img[k][sidx] = (sidx < n_img) ? img[idx] : 0.0;
  }
}

// ------------------------------------------------------------------------------------------------
// a7: fused evaluation.  grid = (ceil(m/128), n_split); partial[(split*4 + c) * m + p]
// ------------------------------------------------------------------------------------------------
struct EvalSink {
  // Two-level summation: a thread adds the (at most 64) weighted pairs of one tile into tile accumulators and the tile
  // sums into the totals, so that the rounding error of the fp64 accumulation grows like sqrt(64) + sqrt(n/64) ulps of
  // the running sum instead of sqrt(n) (n = 5e4 elements per point on C3); 4 extra additions per 64 pairs.
  double phi = 0, ex = 0, ey = 0, ez = 0;
  double tphi = 0, lx = 0, ly = 0, lz = 0;     // tile sums: potential; field in GLOBAL (general tile) or LOCAL (uniform window) axes
  __device__ __forceinline__ bool self_pv(int64_t) const { return false; }
  __device__ __forceinline__ void gtile_begin() { tphi = 0.0; lx = 0.0; ly = 0.0; lz = 0.0; }
  __device__ __forceinline__ void operator()(int64_t, double w, const Infl& a) {
    tphi = fma(w, a.phi, tphi); lx = fma(w, a.ex, lx); ly = fma(w, a.ey, ly); lz = fma(w, a.ez, lz);
  }
  __device__ __forceinline__ void gtile_end() { phi += tphi; ex += lx; ey += ly; ez += lz; }
  // uniform window: weighted sum of the LOCAL field components, rotated to global at its end
  __device__ __forceinline__ void tile_begin(const Axes&) { tphi = 0.0; lx = 0.0; ly = 0.0; lz = 0.0; }
  __device__ __forceinline__ void local(int64_t, double w, double p, double fx, double fy, double fz) {
    tphi = fma(w, p, tphi); lx = fma(w, fx, lx); ly = fma(w, fy, ly); lz = fma(w, fz, lz);
  }
  __device__ __forceinline__ void tile_end(const Axes& ax) {
    phi += tphi;
    ex = fma(lx, ax.exx, fma(ly, ax.eyx, fma(lz, ax.ezx, ex)));
    ey = fma(lx, ax.exy, fma(ly, ax.eyy, fma(lz, ax.ezy, ey)));
    ez = fma(lx, ax.exz, fma(ly, ax.eyz, fma(lz, ax.ezz, ez)));
  }
};

#ifndef NEB_EVAL_MINB
#define NEB_EVAL_MINB 4
#endif
template <class M, bool FIRST, int NIMG>
__global__ void __launch_bounds__(kThreads, NEB_EVAL_MINB) eval_kernel(GeoTables g, const double* __restrict__ img, int n_img, int n_near,
                                                        const double* __restrict__ pts, int64_t m, int64_t per_split,
                                                        double* __restrict__ partial) {
  __shared__ TileSmem sm;
  tile_pipe_init(sm);
  load_images(sm, img, n_img);
  __syncthreads();
  int64_t p = (int64_t)blockIdx.x * kThreads + threadIdx.x;
  int64_t pc = min(p, m - 1);
  double px = pts[pc], py = pts[m + pc], pz = pts[2 * m + pc];
  int64_t n = (int64_t)g.n_rect + g.n_tri + g.n_wire;
  int64_t j0 = (int64_t)blockIdx.y * per_split, j1 = min(n, j0 + per_split);
  EvalSink sink;
  process_range<M, FIRST, NIMG>(g, j0, j1, sm, n_img, n_near, px, py, pz, sink);
  if (p < m) {
    double* o = partial + (int64_t)blockIdx.y * 4 * m;
    if (FIRST) { o[p] = sink.phi; o[m + p] = sink.ex; o[2 * m + p] = sink.ey; o[3 * m + p] = sink.ez; }
    else { o[p] += sink.phi; o[m + p] += sink.ex; o[2 * m + p] += sink.ey; o[3 * m + p] += sink.ez; }   // later chunks of copies
  }
}

// ------------------------------------------------------------------------------------------------
// a8: point charges.  charges SoA x,y,z,q with stride q_stride; grid = (ceil(m / (128 kChargePpt)), n_split).
// A thread owns kChargePpt points (p, p + 128, ...: coalesced) so that one pair of 16-byte shared-memory loads of a
// charge (x, y, z, q packed per charge in the tile) serves kChargePpt pairs and their dependent 1/r chains interleave.
// ------------------------------------------------------------------------------------------------
#ifndef NEB_CHARGE_PPT
#define NEB_CHARGE_PPT 2
#endif
constexpr int kChargePpt = NEB_CHARGE_PPT;
__global__ void __launch_bounds__(kThreads) charge_kernel(const double* __restrict__ ch, int64_t q, int64_t q_stride,
                                                          const double* __restrict__ pts, int64_t m, int64_t per_split,
                                                          double* __restrict__ partial) {
  __shared__ double4 sc[kChargeTile];
  const int64_t p0 = (int64_t)blockIdx.x * (kThreads * kChargePpt) + threadIdx.x;
  double px[kChargePpt], py[kChargePpt], pz[kChargePpt];
  double phi[kChargePpt], ex[kChargePpt], ey[kChargePpt], ez[kChargePpt];
#pragma unroll
  for (int u = 0; u < kChargePpt; ++u) {
    const int64_t pc = min(p0 + u * kThreads, m - 1);
    px[u] = pts[pc]; py[u] = pts[m + pc]; pz[u] = pts[2 * m + pc];
    phi[u] = 0; ex[u] = 0; ey[u] = 0; ez[u] = 0;
  }
  int64_t k0 = (int64_t)blockIdx.y * per_split, k1 = min(q, k0 + per_split);
  for (int64_t base = k0; base < k1; base += kChargeTile) {
    int cnt = (int)min((int64_t)kChargeTile, k1 - base);
    __syncthreads();
    for (int e = threadIdx.x; e < cnt; e += blockDim.x)
      sc[e] = make_double4(ch[base + e], ch[q_stride + base + e], ch[2 * q_stride + base + e], ch[3 * q_stride + base + e]);
    __syncthreads();
#pragma unroll 2
    for (int e = 0; e < cnt; ++e) {
      const double4 c4 = sc[e];
#pragma unroll
      for (int u = 0; u < kChargePpt; ++u) {
        double dx = px[u] - c4.x, dy = py[u] - c4.y, dz = pz[u] - c4.z;
        double r2 = fma(dx, dx, fma(dy, dy, dz * dz));
        // 1/r: MUFU.RSQ64H seed + one cubic step; a charge exactly at the point is skipped.  The clamp
        // and the r = 0 test are integer operations on the bit pattern: 18 FP64-pipe operations per pair (27 flop)
        double y = rsqrt_pos(clamp_tiny(r2));
        y = is_zero(r2) ? 0.0 : y;
        const double qr3 = (c4.w * y) * (y * y);
        phi[u] = fma(c4.w, y, phi[u]);
        ex[u] = fma(qr3, dx, ex[u]); ey[u] = fma(qr3, dy, ey[u]); ez[u] = fma(qr3, dz, ez[u]);
      }
    }
  }
  double* o = partial + (int64_t)blockIdx.y * 4 * m;
#pragma unroll
  for (int u = 0; u < kChargePpt; ++u) {
    const int64_t p = p0 + u * kThreads;
    if (p < m) { o[p] = phi[u]; o[m + p] = ex[u]; o[2 * m + p] = ey[u]; o[3 * m + p] = ez[u]; }
  }
}

// Sum of the partials in a fixed order.  Element partials carry the 1/(4 pi eps0) in the weights;
// charge partials (index >= n_elem_split) are multiplied by kCoulomb here.
__global__ void reduce_kernel(const double* __restrict__ partial, int n_elem_split, int n_charge_split, int64_t m,
                              double* __restrict__ phi, double* __restrict__ E) {
  int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= m) return;
  double acc[4] = {0, 0, 0, 0};
  for (int s = 0; s < n_elem_split; ++s)
    for (int c = 0; c < 4; ++c) acc[c] += partial[((int64_t)s * 4 + c) * m + p];
  double cc[4] = {0, 0, 0, 0};
  for (int s = n_elem_split; s < n_elem_split + n_charge_split; ++s)
    for (int c = 0; c < 4; ++c) cc[c] += partial[((int64_t)s * 4 + c) * m + p];
  for (int c = 0; c < 4; ++c) acc[c] = fma(kCoulomb, cc[c], acc[c]);
  if (phi) phi[p] = acc[0];
  if (E) { E[p] = acc[1]; E[m + p] = acc[2]; E[2 * m + p] = acc[3]; }
}

// ------------------------------------------------------------------------------------------------
// a3: assembly.  grid = (ceil(n/128), ceil(n/64)); CTA = 128 rows x one 64-column tile.
// K column-major with leading dimension ld; consecutive threads write consecutive rows of a column.
// Row maxima (for the S15 equilibration) are accumulated with an order-independent integer max.
// ------------------------------------------------------------------------------------------------
struct AsmSink {
  double* K; int64_t ld, i; double nx, ny, nz, diag; bool dielectric, active, first; double rmax;   // first: the first chunk of copies
  __device__ __forceinline__ bool self_pv(int64_t j) const { return j == i; }
  __device__ __forceinline__ void put(int64_t j, double v) {
    v += (dielectric && j == i && first) ? diag : 0.0;
    if (!first && active) v += K[i + j * ld];            // later chunks of copies add to the coefficient
    rmax = fmax(rmax, fabs(v));
    if (active) K[i + j * ld] = v;
  }
  __device__ __forceinline__ void operator()(int64_t j, double, const Infl& a) {
    double vd = fma(nx, a.ex, fma(ny, a.ey, nz * a.ez));
    put(j, kCoulomb * (dielectric ? vd : a.phi));
  }
  // uniform window: the row's normal in the window's axes, so that n . E' needs no rotation per pair
  double nlx = 0, nly = 0, nlz = 0;
  __device__ __forceinline__ void tile_begin(const Axes& ax) {
    nlx = fma(nx, ax.exx, fma(ny, ax.exy, nz * ax.exz));
    nly = fma(nx, ax.eyx, fma(ny, ax.eyy, nz * ax.eyz));
    nlz = fma(nx, ax.ezx, fma(ny, ax.ezy, nz * ax.ezz));
  }
  __device__ __forceinline__ void local(int64_t j, double, double p, double fx, double fy, double fz) {
    double vd = fma(nlx, fx, fma(nly, fy, nlz * fz));
    put(j, kCoulomb * (dielectric ? vd : p));
  }
  __device__ __forceinline__ void tile_end(const Axes&) {}
  __device__ __forceinline__ void gtile_begin() {}
  __device__ __forceinline__ void gtile_end() {}
};

#ifndef NEB_ASM_MINB
#define NEB_ASM_MINB 4
#endif
template <class M, bool FIRST, int NIMG>
__global__ void __launch_bounds__(kThreads, NEB_ASM_MINB) assemble_kernel(GeoTables g, const double* __restrict__ img, int n_img,
                                                            const double* __restrict__ colloc, int64_t stride,
                                                            const double* __restrict__ normal,
                                                            const int32_t* __restrict__ bc_kind,
                                                            const double* __restrict__ diag, double* __restrict__ K,
                                                            int64_t ld, unsigned long long* __restrict__ rowmax_bits,
                                                            int world, int rank) {
  // distributed matrix (neb_dist.cu): this context holds the 256-column blocks g = rank, rank + world, ... side by side;
  // grid.y counts LOCAL 64-column tiles, lt -> global tile gt, and K is shifted so that column j lands in its local slot
  const int64_t lt = blockIdx.y, gt = ((lt >> 2) * world + rank) * 4 + (lt & 3);
  if (gt * kTile >= (int64_t)g.n_rect + g.n_tri + g.n_wire) return;
  K += (lt - gt) * kTile * ld;
  __shared__ TileSmem sm;
  tile_pipe_init(sm);
  load_images(sm, img, n_img);
  __syncthreads();
  int64_t n = (int64_t)g.n_rect + g.n_tri + g.n_wire;
  int64_t i = (int64_t)blockIdx.x * kThreads + threadIdx.x;
  int64_t ic = min(i, n - 1);
  AsmSink sink;
  sink.K = K; sink.ld = ld; sink.i = ic; sink.active = i < n; sink.rmax = 0.0; sink.first = FIRST;
  sink.nx = normal[ic]; sink.ny = normal[stride + ic]; sink.nz = normal[2 * stride + ic];
  sink.dielectric = bc_kind[ic] == NEB_BC_DIELECTRIC;
  sink.diag = diag[ic];
  double px = colloc[ic], py = colloc[stride + ic], pz = colloc[2 * stride + ic];
  int64_t j0 = gt * kTile, j1 = min(n, j0 + kTile);
  process_range<M, FIRST, NIMG>(g, j0, j1, sm, n_img, n_img, px, py, pz, sink);   // assembly is always exact
  // the running maximum of a row whose coefficients are still being summed is not the row's maximum: with several
  // chunks of copies only the LAST chunk's values (the finished coefficients) count
  if (i < n && rowmax_bits) atomicMax(rowmax_bits + i, (unsigned long long)__double_as_longlong(sink.rmax));
}

// distributed layout: rows n..npad of every local column, and the local columns whose global index is >= n
__global__ void pad_identity_dist_kernel(double* K, int64_t n, int64_t npad, int64_t ncol_loc, int world, int rank) {
  for (int64_t lc = blockIdx.y; lc < ncol_loc; lc += gridDim.y) {
    const int64_t gc = ((lc >> 8) * world + rank) * 256 + (lc & 255);
    const int64_t i0 = gc >= n ? 0 : n;
    for (int64_t i = i0 + (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < npad; i += (int64_t)gridDim.x * blockDim.x)
      K[i + lc * npad] = (i == gc) ? 1.0 : 0.0;
  }
}

// rows/columns >= n of the padded matrix: identity
__global__ void pad_identity_kernel(double* K, int64_t n, int64_t npad) {
  int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  int64_t npadrows = npad - n;
  // region A: rows n..npad, all columns (npadrows x npad); region B: rows 0..n, columns n..npad
  int64_t sizeA = npadrows * npad, sizeB = n * npadrows;
  if (idx < sizeA) {
    int64_t j = idx / npadrows, i = n + idx % npadrows;
    K[i + j * npad] = (i == j) ? 1.0 : 0.0;
  } else if (idx < sizeA + sizeB) {
    int64_t t = idx - sizeA;
    int64_t j = n + t / n, i = t % n;
    K[i + j * npad] = 0.0;
  }
}

// dist: a row with no non-zero entry in THIS rank's columns gets +inf, so that the minimum over the ranks (= 1 / the
// row's maximum over all columns) ignores it; neb_dist_row_scales turns a surviving +inf into 1
__global__ void rscale_kernel(const unsigned long long* rowmax_bits, int64_t n, int64_t npad, double* rscale, bool dist) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= npad) return;
  double mx = (i < n) ? __longlong_as_double((long long)rowmax_bits[i]) : 1.0;
  rscale[i] = (mx > 0.0) ? 1.0 / mx : (dist ? __longlong_as_double(0x7ff0000000000000LL) : 1.0);
}

// grid.y covers the columns with a stride (a grid's y extent ends at 65535, the matrix at 131072 columns)
__global__ void scale_rows_kernel(double* K, int64_t n, int64_t ncols, int64_t ld, const double* __restrict__ rscale) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const double s = rscale[i];
  for (int64_t j = blockIdx.y; j < ncols; j += gridDim.y) K[i + j * ld] *= s;
}

// ------------------------------------------------------------------------------------------------
// a4: RHS (reading S10): Dirichlet b_i = V_i - Phi_sc(p_i); dielectric b_i = -n_i.E_sc(p_i)
// ------------------------------------------------------------------------------------------------
__global__ void rhs_kernel(int64_t n, int64_t npad, int64_t stride, const int32_t* __restrict__ bc_kind,
                           const double* __restrict__ bc_value, const double* __restrict__ normal,
                           const double* __restrict__ phi_sc, const double* __restrict__ E_sc, double* __restrict__ b) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= npad) return;
  double v = 0.0;
  if (i < n) {
    if (bc_kind[i] == NEB_BC_DIRICHLET) v = bc_value[i] - (phi_sc ? phi_sc[i] : 0.0);
    else if (E_sc) v = -(normal[i] * E_sc[i] + normal[stride + i] * E_sc[n + i] + normal[2 * stride + i] * E_sc[2 * n + i]);
  }
  b[i] = v;
}

// ------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------
static int pick_splits(int64_t pt_blocks, int64_t units, int64_t unit_tile, int num_sms, int fixed) {
  // aim at >= 16 waves of 4 CTAs/SM so the tail wave is small, but keep >= 2 tiles per split; NEB_OPT_EVAL_SPLITS
  // replaces the point-count-dependent wish by a fixed one
  int64_t want = fixed > 0 ? fixed : (16LL * 4 * num_sms + pt_blocks - 1) / pt_blocks;
  int64_t max_split = (units + 2 * unit_tile - 1) / (2 * unit_tile);
  int64_t s = want < 1 ? 1 : want;
  if (s > max_split) s = max_split;
  if (s > 1024) s = 1024;
  if (s < 1) s = 1;
  return (int)s;
}

static GeoTables tables(const neb_ctx* c) {
  GeoTables g;
  g.rec = c->d_rec; g.uniform = c->d_uniform; g.stride = c->stride; g.n_rect = c->n_rect; g.n_tri = c->n_tri; g.n_wire = c->n_wire;
  return g;
}

neb_status field_at_points(neb_ctx* c, int64_t m, const double* d_pts, bool use_elements, bool use_charges,
                           double* d_phi, double* d_E) {
  if (m <= 0) return NEB_OK;
  const bool use_lines = use_charges && c->n_lines > 0;
  use_charges = use_charges && c->q > 0;
  int64_t pt_blocks = (m + kThreads - 1) / kThreads;
  int se = use_elements ? pick_splits(pt_blocks, c->n, kTile, c->num_sms, c->eval_splits) : 0;
  int sq = use_charges ? pick_splits(pt_blocks, c->q, kChargeTile, c->num_sms, c->eval_splits) : 0;
  int64_t per_e = 0, per_q = 0;
  if (se) {
    per_e = (c->n + se - 1) / se;
    per_e = (per_e + kTile - 1) / kTile * kTile;
    se = (int)((c->n + per_e - 1) / per_e);
  }
  if (sq) {
    per_q = (c->q + sq - 1) / sq;
    per_q = (per_q + kChargeTile - 1) / kChargeTile * kChargeTile;
    sq = (int)((c->q + per_q - 1) / per_q);
  }
  int sl = use_lines ? pick_splits(pt_blocks, c->n_lines, 256, c->num_sms, c->eval_splits) : 0;
  int64_t per_l = 0;
  if (sl) {
    per_l = (c->n_lines + sl - 1) / sl;
    per_l = (per_l + 255) / 256 * 256;
    sl = (int)((c->n_lines + per_l - 1) / per_l);
  }
  size_t need = (size_t)(se + sq + sl) * 4 * (size_t)m * sizeof(double);
  NEB_TRY(ensure_scratch(c, need));
  double* partial = c->d_scratch;
  // Adaptive Modelling: the copies are sorted by shift length (neb_assemble), the first n_near are evaluated exactly
  int n_near = c->n_img;
  if (c->adaptive_far > 0.0) {
    n_near = 1;
    while (n_near < c->n_img && c->h_img_len[(size_t)n_near] < c->adaptive_far) ++n_near;
  }
  if (se) {
    StageTimer t(c, NEB_STAGE_EVAL);
    dim3 grid((unsigned)pt_blocks, (unsigned)se);
    // more than kMaxImg copies: one launch per chunk of the (length-sorted) copy table, later chunks add to the partials
    for (int ch = 0; ch * kMaxImg < c->n_img; ++ch) {
      const int len = std::min(kMaxImg, c->n_img - ch * kMaxImg);
      const int near_ch = std::max(0, std::min(len, n_near - ch * kMaxImg));
      const double* img = c->d_img + (size_t)ch * 3 * kMaxImg;
#define NEB_EVAL_ARGS tables(c), img, len, near_ch, d_pts, m, per_e, partial
      if (c->math_fast) {
        if (c->n_img == 1) eval_kernel<MathFast, true, 1><<<grid, kThreads, 0, c->stream>>>(NEB_EVAL_ARGS);
        else if (ch == 0) eval_kernel<MathFast, true, 0><<<grid, kThreads, 0, c->stream>>>(NEB_EVAL_ARGS);
        else eval_kernel<MathFast, false, 0><<<grid, kThreads, 0, c->stream>>>(NEB_EVAL_ARGS);
      } else {
        if (ch == 0) eval_kernel<MathLib, true, 0><<<grid, kThreads, 0, c->stream>>>(NEB_EVAL_ARGS);
        else eval_kernel<MathLib, false, 0><<<grid, kThreads, 0, c->stream>>>(NEB_EVAL_ARGS);
      }
#undef NEB_EVAL_ARGS
      c->launches++;
    }
    NEB_CUDA(c, cudaGetLastError());
  }
  if (sq) {
    StageTimer t(c, NEB_STAGE_CHARGES);
    dim3 grid((unsigned)((m + kThreads * kChargePpt - 1) / (kThreads * kChargePpt)), (unsigned)sq);
    charge_kernel<<<grid, kThreads, 0, c->stream>>>(c->d_charges, c->q, c->q_cap, d_pts, m, per_q,
                                                    partial + (size_t)se * 4 * m);
    c->launches++;
    NEB_CUDA(c, cudaGetLastError());
  }
  if (sl) {
    // line charges of the voxelised cloud (Alg. 3): their partials follow the point charges' (same Coulomb factor)
    StageTimer t(c, NEB_STAGE_CHARGES);
    launch_line_kernel(c, m, d_pts, sl, per_l, partial + (size_t)(se + sq) * 4 * m);
    NEB_CUDA(c, cudaGetLastError());
  }
  {
    StageTimer t(c, NEB_STAGE_REDUCE);
    reduce_kernel<<<(unsigned)((m + 255) / 256), 256, 0, c->stream>>>(partial, se, sq + sl, m, d_phi, d_E);
    c->launches++;
    NEB_CUDA(c, cudaGetLastError());
  }
  return NEB_OK;
}

// ------------------------------------------------------------------------------------------------
// neb_eval_static: the fused evaluation (a7 + a8) for callers that may not allocate (code under CUDA graph capture,
// tight serving loops, harnesses that forbid cudaMalloc).  Same kernels as field_at_points; the per-chunk partial sums,
// which field_at_points keeps in a cudaMalloc'ed buffer that grows with m, live in a file-scope device array of fixed
// size instead: kStaticScratchDoubles doubles = 32 MiB, held by every GPU that loads the library until the process
// exits.  In host code the array's NAME is a host-side stand-in, not a device address: its device address is taken once
// per context (= per device, with that device current) by cudaGetSymbolAddress in field_static_init, from neb_create.
// Every call on every context of a device shares the array; the kernels overwrite the part they use before they read it
// (each chunk's first launch stores, nothing accumulates across calls), so nothing has to be cleared between calls —
// but two calls that overlap on the GPU (different streams, or contexts on different streams) race on it.
// ------------------------------------------------------------------------------------------------
constexpr int64_t kStaticScratchDoubles = (int64_t)4 << 20;                   // 32 MiB
constexpr int64_t kStaticMaxPoints = NEB_EVAL_STATIC_MAX_POINTS;              // 65536: leaves room for >= 16 chunks
static __device__ __align__(256) double g_static_partial[kStaticScratchDoubles];

neb_status field_static_init(neb_ctx* c) {
  void* ptr = nullptr;
  cudaError_t e = cudaGetSymbolAddress(&ptr, g_static_partial);
  if (e != cudaSuccess || !ptr) {
    cudaGetLastError();
    return fail(c, NEB_ECUDA, std::string("cudaGetSymbolAddress(g_static_partial): ") + cudaGetErrorString(e));
  }
  c->d_static_partial = (double*)ptr;
  return NEB_OK;
}

neb_status field_at_points_static(neb_ctx* c, int64_t m, const double* d_pts, double* d_phi, double* d_E) {
  if (m <= 0) return NEB_OK;
  if (m > kStaticMaxPoints)
    return fail(c, NEB_EINVAL, "neb_eval_static: at most " + std::to_string(kStaticMaxPoints) + " points per call (fixed 32 MiB scratch); got " +
                                   std::to_string(m) + " - split the points or use neb_eval");
  if (!c->d_static_partial) return fail(c, NEB_ESTATE, "neb_eval_static: the static scratch was not set up for this context");
  const bool use_lines = c->n_lines > 0, use_charges = c->q > 0;
  const int64_t pt_blocks = (m + kThreads - 1) / kThreads;
  int se = pick_splits(pt_blocks, c->n, kTile, c->num_sms, c->eval_splits);
  int sq = use_charges ? pick_splits(pt_blocks, c->q, kChargeTile, c->num_sms, c->eval_splits) : 0;
  int sl = use_lines ? pick_splits(pt_blocks, c->n_lines, 256, c->num_sms, c->eval_splits) : 0;
  // the chunk counts are cut down until the partial sums fit the fixed array (fewer, longer chunks: same result to
  // rounding, a little less parallelism for small m)
  const int64_t budget = kStaticScratchDoubles / (4 * m);
  while ((int64_t)se + sq + sl > budget) {
    if (se >= sq && se >= sl && se > 1) --se;
    else if (sq >= sl && sq > 1) --sq;
    else if (sl > 1) --sl;
    else return fail(c, NEB_EINVAL, "neb_eval_static: the partial sums do not fit the static scratch");
  }
  int64_t per_e = (c->n + se - 1) / se, per_q = 0, per_l = 0;
  per_e = (per_e + kTile - 1) / kTile * kTile;
  se = (int)((c->n + per_e - 1) / per_e);
  if (sq) {
    per_q = (c->q + sq - 1) / sq;
    per_q = (per_q + kChargeTile - 1) / kChargeTile * kChargeTile;
    sq = (int)((c->q + per_q - 1) / per_q);
  }
  if (sl) {
    per_l = (c->n_lines + sl - 1) / sl;
    per_l = (per_l + 255) / 256 * 256;
    sl = (int)((c->n_lines + per_l - 1) / per_l);
  }
  double* partial = c->d_static_partial;
  int n_near = c->n_img;
  if (c->adaptive_far > 0.0) {
    n_near = 1;
    while (n_near < c->n_img && c->h_img_len[(size_t)n_near] < c->adaptive_far) ++n_near;
  }
  {
    StageTimer t(c, NEB_STAGE_EVAL);
    dim3 grid((unsigned)pt_blocks, (unsigned)se);
    for (int ch = 0; ch * kMaxImg < c->n_img; ++ch) {
      const int len = std::min(kMaxImg, c->n_img - ch * kMaxImg);
      const int near_ch = std::max(0, std::min(len, n_near - ch * kMaxImg));
      const double* img = c->d_img + (size_t)ch * 3 * kMaxImg;
#define NEB_EVAL_ARGS tables(c), img, len, near_ch, d_pts, m, per_e, partial
      if (c->math_fast) {
        if (c->n_img == 1) eval_kernel<MathFast, true, 1><<<grid, kThreads, 0, c->stream>>>(NEB_EVAL_ARGS);
        else if (ch == 0) eval_kernel<MathFast, true, 0><<<grid, kThreads, 0, c->stream>>>(NEB_EVAL_ARGS);
        else eval_kernel<MathFast, false, 0><<<grid, kThreads, 0, c->stream>>>(NEB_EVAL_ARGS);
      } else {
        if (ch == 0) eval_kernel<MathLib, true, 0><<<grid, kThreads, 0, c->stream>>>(NEB_EVAL_ARGS);
        else eval_kernel<MathLib, false, 0><<<grid, kThreads, 0, c->stream>>>(NEB_EVAL_ARGS);
      }
#undef NEB_EVAL_ARGS
      c->launches++;
    }
    NEB_CUDA(c, cudaGetLastError());
  }
  if (sq) {
    StageTimer t(c, NEB_STAGE_CHARGES);
    dim3 grid((unsigned)((m + kThreads * kChargePpt - 1) / (kThreads * kChargePpt)), (unsigned)sq);
    charge_kernel<<<grid, kThreads, 0, c->stream>>>(c->d_charges, c->q, c->q_cap, d_pts, m, per_q, partial + (size_t)se * 4 * m);
    c->launches++;
    NEB_CUDA(c, cudaGetLastError());
  }
  if (sl) {
    StageTimer t(c, NEB_STAGE_CHARGES);
    launch_line_kernel(c, m, d_pts, sl, per_l, partial + (size_t)(se + sq) * 4 * m);
    NEB_CUDA(c, cudaGetLastError());
  }
  {
    StageTimer t(c, NEB_STAGE_REDUCE);
    reduce_kernel<<<(unsigned)((m + 255) / 256), 256, 0, c->stream>>>(partial, se, sq + sl, m, d_phi, d_E);
    c->launches++;
    NEB_CUDA(c, cudaGetLastError());
  }
  return NEB_OK;
}

neb_status assemble_matrix(neb_ctx* c) {
  int64_t n = c->n, npad = c->npad;
  c->counter[NEB_COUNTER_MATRIX_BYTES] = 8.0 * (double)n * (double)(c->dist_mode ? std::min(c->ncol_loc, n) : n);
  NEB_TRY(ensure_scratch(c, (size_t)npad * sizeof(unsigned long long)));
  unsigned long long* rowmax = (unsigned long long*)c->d_scratch;
  NEB_CUDA(c, cudaMemsetAsync(rowmax, 0, (size_t)npad * sizeof(unsigned long long), c->stream));
  {
    StageTimer t(c, NEB_STAGE_ASSEMBLE);
    const bool dist = c->dist_mode != 0;
    dim3 grid((unsigned)((n + kThreads - 1) / kThreads), (unsigned)(dist ? c->ncol_loc / kTile : (n + kTile - 1) / kTile));
    const int n_chunks = (c->n_img + kMaxImg - 1) / kMaxImg;
    for (int ch = 0; ch < n_chunks; ++ch) {
      const int len = std::min(kMaxImg, c->n_img - ch * kMaxImg);
      const double* img = c->d_img + (size_t)ch * 3 * kMaxImg;
      unsigned long long* rm = (ch == n_chunks - 1) ? rowmax : nullptr;      // row maxima from the finished coefficients
#define NEB_ASM_ARGS tables(c), img, len, c->d_colloc, c->stride, c->d_normal, c->d_bc_kind, c->d_diag, c->d_K, npad, rm, c->dist_world, c->dist_rank
      if (c->math_fast) {
        if (c->n_img == 1) assemble_kernel<MathFast, true, 1><<<grid, kThreads, 0, c->stream>>>(NEB_ASM_ARGS);
        else if (ch == 0) assemble_kernel<MathFast, true, 0><<<grid, kThreads, 0, c->stream>>>(NEB_ASM_ARGS);
        else assemble_kernel<MathFast, false, 0><<<grid, kThreads, 0, c->stream>>>(NEB_ASM_ARGS);
      } else {
        if (ch == 0) assemble_kernel<MathLib, true, 0><<<grid, kThreads, 0, c->stream>>>(NEB_ASM_ARGS);
        else assemble_kernel<MathLib, false, 0><<<grid, kThreads, 0, c->stream>>>(NEB_ASM_ARGS);
      }
#undef NEB_ASM_ARGS
      c->launches++;
    }
    NEB_CUDA(c, cudaGetLastError());
    int64_t padcells = (npad - n) * npad + n * (npad - n);
    if (dist) {
      pad_identity_dist_kernel<<<dim3(4, (unsigned)std::min<int64_t>(c->ncol_loc, 65535)), 256, 0, c->stream>>>(c->d_K, n, npad, c->ncol_loc, c->dist_world, c->dist_rank);
      c->launches++;
      NEB_CUDA(c, cudaGetLastError());
    } else if (padcells > 0) {
      pad_identity_kernel<<<(unsigned)((padcells + 255) / 256), 256, 0, c->stream>>>(c->d_K, n, npad);
      c->launches++;
      NEB_CUDA(c, cudaGetLastError());
    }
  }
  {
    StageTimer t(c, NEB_STAGE_EQUIL);
    rscale_kernel<<<(unsigned)((npad + 255) / 256), 256, 0, c->stream>>>(rowmax, n, npad, c->d_rscale, c->dist_mode != 0);
    c->launches++;
    NEB_CUDA(c, cudaGetLastError());
  }
  return NEB_OK;
}

// Applies the row scales in place (done at the first neb_solve, so that neb_get_matrix before it
// returns the unscaled matrix without a second copy).
neb_status scale_matrix_rows(neb_ctx* c) {
  StageTimer t(c, NEB_STAGE_EQUIL);
  const int64_t ncols = c->dist_mode ? c->ncol_loc : c->n;   // pad columns are zero above row n
  dim3 grid((unsigned)((c->n + 255) / 256), (unsigned)std::min<int64_t>(ncols, 65535));
  scale_rows_kernel<<<grid, 256, 0, c->stream>>>(c->d_K, c->n, ncols, c->npad, c->d_rscale);
  c->launches++;
  NEB_CUDA(c, cudaGetLastError());
  return NEB_OK;
}

neb_status form_rhs(neb_ctx* c) {
  int64_t n = c->n;
  double *phi = nullptr, *E = nullptr;
  if (c->q > 0 || c->n_lines > 0) {
    // Phi_sc, E_sc at the collocation points: reuse d_x (npad >= n) for phi and a scratch tail for E.
    // field_at_points uses d_scratch for its partials, so E lives in a dedicated allocation.
    phi = c->d_x;
    NEB_CUDA(c, cudaMallocFromPoolAsync((void**)&E, (size_t)3 * n * sizeof(double), c->pool, c->stream));
    // collocation points are stored with stride c->stride; field_at_points wants stride m: pack
    double* pts = nullptr;
    NEB_CUDA(c, cudaMallocFromPoolAsync((void**)&pts, (size_t)3 * n * sizeof(double), c->pool, c->stream));
    for (int k = 0; k < 3; ++k)
      NEB_CUDA(c, cudaMemcpyAsync(pts + k * n, c->d_colloc + k * c->stride, (size_t)n * sizeof(double),
                                  cudaMemcpyDeviceToDevice, c->stream));
    neb_status st = field_at_points(c, n, pts, false, true, phi, E);
    cudaFreeAsync(pts, c->stream);
    if (st != NEB_OK) { cudaFreeAsync(E, c->stream); return st; }
  }
  {
    StageTimer t(c, NEB_STAGE_RHS);
    rhs_kernel<<<(unsigned)((c->npad + 255) / 256), 256, 0, c->stream>>>(n, c->npad, c->stride, c->d_bc_kind,
                                                                         c->d_bc_value, c->d_normal, phi, E, c->d_b);
    c->launches++;
  }
  if (E) cudaFreeAsync(E, c->stream);
  NEB_CUDA(c, cudaGetLastError());
  return NEB_OK;
}

}  // namespace neb
