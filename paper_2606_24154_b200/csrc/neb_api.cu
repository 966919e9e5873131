// neb_api.cu — the C ABI of include/neb.h: context, pointer staging, a1 frame tables, call ordering.
#include <math.h>
#include <string.h>

#include <algorithm>
#include <vector>

#include "neb_internal.h"

namespace neb {

neb_status fail(neb_ctx* c, neb_status st, const std::string& msg) {
  if (c) c->err = msg;
  return st;
}

neb_status ensure_scratch(neb_ctx* c, size_t bytes) {
  if (bytes <= c->scratch_bytes) return NEB_OK;
  if (c->d_scratch) {
    NEB_CUDA(c, cudaStreamSynchronize(c->stream));
    NEB_CUDA(c, cudaFree(c->d_scratch));
    c->d_scratch = nullptr;
    c->scratch_bytes = 0;
  }
  size_t want = bytes + bytes / 8;
  NEB_CUDA(c, cudaMalloc((void**)&c->d_scratch, want));
  c->scratch_bytes = want;
  return NEB_OK;
}

StageTimer::StageTimer(neb_ctx* c_, int stage_) : c(c_), stage(stage_), l0(c_->launches) {
  if (c->profile) cudaEventRecord(c->ev0[stage], c->stream);
}
StageTimer::~StageTimer() {
  if (c->profile) {
    cudaEventRecord(c->ev1[stage], c->stream);
    cudaEventSynchronize(c->ev1[stage]);
    float ms = 0.f;
    cudaEventElapsedTime(&ms, c->ev0[stage], c->ev1[stage]);
    c->stat[stage].ms += ms;
  }
  c->stat[stage].launches += c->launches - l0;
}

// ---- pointer staging -------------------------------------------------------------------------------
static bool is_device_ptr(const void* p) {
  cudaPointerAttributes a;
  if (cudaPointerGetAttributes(&a, p) != cudaSuccess) {
    cudaGetLastError();
    return false;
  }
  return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

bool is_device_pointer(const void* p) { return is_device_ptr(p); }

struct Staging {   // temporaries of one ABI call
  neb_ctx* c;
  std::vector<void*> temps;
  bool host_in = false;   // an input was copied from host memory and the stream has not been synchronised since
  explicit Staging(neb_ctx* c_) : c(c_) {}
  ~Staging() {
    // inputs are borrowed for the duration of the call (neb.h): a copy from PINNED host memory is truly
    // asynchronous, so the call may not return before it has been read
    if (host_in) cudaStreamSynchronize(c->stream);
    for (void* p : temps) cudaFreeAsync(p, c->stream);
  }
  // device view of an input array (copied if it lives on the host)
  neb_status in(const void* p, size_t bytes, const void** out) {
    *out = nullptr;
    if (!p || bytes == 0) return NEB_OK;
    if (is_device_ptr(p)) { *out = p; return NEB_OK; }
    void* d = nullptr;
    NEB_CUDA(c, cudaMallocFromPoolAsync(&d, bytes, c->pool, c->stream));
    temps.push_back(d);
    NEB_CUDA(c, cudaMemcpyAsync(d, p, bytes, cudaMemcpyHostToDevice, c->stream));
    host_in = true;
    *out = d;
    return NEB_OK;
  }
  // device buffer standing for an output array; host_dst != nullptr means copy back at finish()
  struct Out { void* dev; void* host; size_t bytes; };
  std::vector<Out> outs;
  neb_status out(void* p, size_t bytes, void** dev) {
    *dev = nullptr;
    if (!p || bytes == 0) return NEB_OK;
    if (is_device_ptr(p)) { *dev = p; return NEB_OK; }
    void* d = nullptr;
    NEB_CUDA(c, cudaMallocFromPoolAsync(&d, bytes, c->pool, c->stream));
    temps.push_back(d);
    outs.push_back({d, p, bytes});
    *dev = d;
    return NEB_OK;
  }
  neb_status finish() {
    if (outs.empty()) return NEB_OK;
    for (auto& o : outs) NEB_CUDA(c, cudaMemcpyAsync(o.host, o.dev, o.bytes, cudaMemcpyDeviceToHost, c->stream));
    NEB_CUDA(c, cudaStreamSynchronize(c->stream));
    host_in = false;
    outs.clear();
    return NEB_OK;
  }
};

// ---- a1: frame tables -------------------------------------------------------------------------------
// Stable partition of the element indices by kind (single CTA): perm[sorted position] = caller index.
__global__ void __launch_bounds__(1024) kind_partition_kernel(const int32_t* __restrict__ kind, int n, int32_t* __restrict__ perm,
                                                              int32_t* __restrict__ counts, int32_t* __restrict__ flag) {
  __shared__ int s_cnt[3], s_run[3], s_warp[32][3];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  if (tid < 3) s_cnt[tid] = 0;
  __syncthreads();
  int local[3] = {0, 0, 0};
  for (int i = tid; i < n; i += 1024) {
    int k = kind[i];
    if (k < 0 || k > 2) atomicOr(flag, 1);
    else local[k]++;
  }
  for (int kk = 0; kk < 3; ++kk) atomicAdd(&s_cnt[kk], local[kk]);
  __syncthreads();
  if (tid == 0) {
    s_run[0] = 0; s_run[1] = s_cnt[0]; s_run[2] = s_cnt[0] + s_cnt[1];
    counts[0] = s_cnt[0]; counts[1] = s_cnt[1]; counts[2] = s_cnt[2];
  }
  __syncthreads();
  for (int chunk = 0; chunk < n; chunk += 1024) {
    int i = chunk + tid;
    int k = (i < n) ? kind[i] : -1;
    if (k < 0 || k > 2) k = -1;
    int rank = 0;
    for (int kk = 0; kk < 3; ++kk) {
      unsigned bal = __ballot_sync(0xffffffffu, k == kk);
      if (k == kk) rank = __popc(bal & ((1u << lane) - 1u));
      if (lane == 0) s_warp[warp][kk] = __popc(bal);
    }
    __syncthreads();
    if (k >= 0) {
      int pre = 0;
      for (int w = 0; w < warp; ++w) pre += s_warp[w][k];
      perm[s_run[k] + pre + rank] = i;
    }
    __syncthreads();
    if (tid < 3) {
      int tot = 0;
      for (int w = 0; w < 32; ++w) tot += s_warp[w][tid];
      s_run[tid] += tot;
    }
    __syncthreads();
  }
}

// One thread per sorted position: unit frame, edge lengths, collocation point, normal, row data.
__global__ void frames_kernel(int64_t n, int64_t stride, const int32_t* __restrict__ perm, const int32_t* __restrict__ kind,
                              const double* __restrict__ v0, const double* __restrict__ e1, const double* __restrict__ e2,
                              const double* __restrict__ radius, const double* __restrict__ colloc_in,
                              const int32_t* __restrict__ bc_kind_in, const double* __restrict__ bc_value_in,
                              const double* __restrict__ eps_plus, const double* __restrict__ eps_minus,
                              double* __restrict__ rec, double* __restrict__ colloc, double* __restrict__ normal,
                              int32_t* __restrict__ bc_kind, double* __restrict__ bc_value, double* __restrict__ diag,
                              int32_t* __restrict__ flag) {
  int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= n) return;
  int64_t j = perm[s];
  int k = kind[j];
  double p0[3] = {v0[j], v0[n + j], v0[2 * n + j]};
  double a1[3] = {e1[j], e1[n + j], e1[2 * n + j]};
  double a2[3] = {e2[j], e2[n + j], e2[2 * n + j]};
  double la = sqrt(a1[0] * a1[0] + a1[1] * a1[1] + a1[2] * a1[2]);
  if (!(la > 0.0)) { atomicOr(flag, 4); la = 1.0; }
  double ex[3] = {a1[0] / la, a1[1] / la, a1[2] / la};
  double ey[3] = {0, 0, 0}, ez[3] = {0, 0, 0};
  double lb = 0.0, aux = 0.0;
  double cp[3];
  if (k == NEB_WIRE) {
    double rw = radius ? radius[j] : 0.0;
    if (!(rw > 0.0)) { atomicOr(flag, 8); rw = 1.0; }
    lb = rw;
    aux = 2.0 * 3.14159265358979323846 * rw;
    // default collocation: mid-length, on the surface, along axis x (least-aligned coordinate axis)
    int m = 0;
    if (fabs(ex[1]) < fabs(ex[m])) m = 1;
    if (fabs(ex[2]) < fabs(ex[m])) m = 2;
    double ax[3] = {m == 0 ? 1.0 : 0.0, m == 1 ? 1.0 : 0.0, m == 2 ? 1.0 : 0.0};
    double pr[3] = {ex[1] * ax[2] - ex[2] * ax[1], ex[2] * ax[0] - ex[0] * ax[2], ex[0] * ax[1] - ex[1] * ax[0]};
    double lp = sqrt(pr[0] * pr[0] + pr[1] * pr[1] + pr[2] * pr[2]);
    for (int c = 0; c < 3; ++c) cp[c] = p0[c] + 0.5 * a1[c] + rw * pr[c] / lp;
  } else {
    double l2 = sqrt(a2[0] * a2[0] + a2[1] * a2[1] + a2[2] * a2[2]);
    if (!(l2 > 0.0)) { atomicOr(flag, 4); l2 = 1.0; }
    double z0[3] = {a2[0] / l2, a2[1] / l2, a2[2] / l2};
    // n = e2 x e1 / |e2 x e1| (local Y); then local Z = X x Y so the frame is orthonormal
    double c0 = z0[1] * ex[2] - z0[2] * ex[1], c1 = z0[2] * ex[0] - z0[0] * ex[2], c2 = z0[0] * ex[1] - z0[1] * ex[0];
    double lc = sqrt(c0 * c0 + c1 * c1 + c2 * c2);
    // the edges must be perpendicular (the closed forms are those of a rectangle / RIGHT triangle): |cos| <= 1e-9
    const double cs = z0[0] * ex[0] + z0[1] * ex[1] + z0[2] * ex[2];
    if (!(fabs(cs) <= 1e-9) || !(lc > 0.5)) { atomicOr(flag, 4); lc = 1.0; }
    ey[0] = c0 / lc; ey[1] = c1 / lc; ey[2] = c2 / lc;
    ez[0] = ex[1] * ey[2] - ex[2] * ey[1];
    ez[1] = ex[2] * ey[0] - ex[0] * ey[2];
    ez[2] = ex[0] * ey[1] - ex[1] * ey[0];
    lb = a2[0] * ez[0] + a2[1] * ez[1] + a2[2] * ez[2];
    double w = (k == NEB_RECT) ? 0.5 : (1.0 / 3.0);
    for (int c = 0; c < 3; ++c) cp[c] = p0[c] + w * (a1[c] + a2[c]);
    if (k == NEB_TRI) aux = 1.0 / sqrt(la * la + lb * lb);
    else aux = la * lb;
  }
  if (colloc_in) { cp[0] = colloc_in[j]; cp[1] = colloc_in[n + j]; cp[2] = colloc_in[2 * n + j]; }
  double* r = rec + s;
  r[0 * stride] = p0[0]; r[1 * stride] = p0[1]; r[2 * stride] = p0[2];
  r[3 * stride] = ex[0]; r[4 * stride] = ex[1]; r[5 * stride] = ex[2];
  r[6 * stride] = ey[0]; r[7 * stride] = ey[1]; r[8 * stride] = ey[2];
  r[9 * stride] = ez[0]; r[10 * stride] = ez[1]; r[11 * stride] = ez[2];
  r[12 * stride] = la; r[13 * stride] = lb; r[14 * stride] = aux; r[15 * stride] = 0.0;
  {
    // far-field radius of the warp-uniform shortcut (neb_influence.cuh): 2.5 longest edges beyond the reach from v0
    double diag = sqrt(la * la + lb * lb);
    double lmax = (k == NEB_TRI) ? diag : fmax(la, fabs(lb));
    double rf = 2.5 * lmax + diag;
    r[16 * stride] = rf * rf;
  }
  r[17 * stride] = fma(p0[0], ex[0], fma(p0[1], ex[1], p0[2] * ex[2]));
  r[18 * stride] = fma(p0[0], ey[0], fma(p0[1], ey[1], p0[2] * ey[2]));
  r[19 * stride] = fma(p0[0], ez[0], fma(p0[1], ez[1], p0[2] * ez[2]));
  for (int c = 0; c < 3; ++c) { colloc[c * stride + s] = cp[c]; normal[c * stride + s] = ey[c]; }
  int bk = bc_kind_in[j];
  if (bk != NEB_BC_DIRICHLET && bk != NEB_BC_DIELECTRIC) { atomicOr(flag, 16); bk = NEB_BC_DIRICHLET; }
  double dg = 0.0;
  if (bk == NEB_BC_DIELECTRIC) {
    double ep = eps_plus ? eps_plus[j] : 1.0, em = eps_minus ? eps_minus[j] : 1.0;
    if (!(ep > 0.0) || !(em > 0.0) || ep == em || k == NEB_WIRE) { atomicOr(flag, 32); }
    else dg = (ep + em) / (2.0 * kEps0 * (ep - em));     // 1 / (2 eps0 lambda), reading S8
  }
  bc_kind[s] = bk;
  bc_value[s] = bc_value_in ? bc_value_in[j] : 0.0;
  diag[s] = dg;
}

// One 64-thread CTA per 64-element window of the sorted table.  uniform[3 w] = 1 if all its elements have bit-identical
// unit axes (a face of a mesh); uniform[3 w + 1], [3 w + 2] = bit k set when the rectangles 2k and 2k + 1 of the window
// are neighbours of one strip — same plane, same axes, the second one starts where the first one ends along local X
// (mask 1) or local Z (mask 2), equal extent across — so that the pair shares an edge and two corners and is evaluated
// by rect_pair_local (neb_influence.cuh).  Agreement is asked to 1e-13 of the smaller side: the table's coordinates
// carry rounding errors of ~1e-16 x |v0|, and treating the shared edge as one line moves it by no more than that.
__global__ void __launch_bounds__(64) tile_uniform_kernel(int64_t n, int64_t stride, const double* __restrict__ rec,
                                                          const int32_t* __restrict__ counts, int pairs_enabled,
                                                          int32_t* __restrict__ uniform) {
  __shared__ unsigned s_bx[2], s_bz[2];
  const int64_t j0 = (int64_t)blockIdx.x * 64, j = j0 + threadIdx.x;
  int same = 1;
  if (j < n) {
#pragma unroll
    for (int f = 3; f < 12; ++f)
      same &= __double_as_longlong(rec[f * stride + j]) == __double_as_longlong(rec[f * stride + j0]);
  }
  bool chain_x = false, chain_z = false;
  if (pairs_enabled && (threadIdx.x & 1) == 0 && j + 1 < (int64_t)counts[0]) {
    bool axes = true;
#pragma unroll
    for (int f = 3; f < 12; ++f) axes = axes && __double_as_longlong(rec[f * stride + j]) == __double_as_longlong(rec[f * stride + j + 1]);
    const double a0 = rec[12 * stride + j], a1 = rec[12 * stride + j + 1], b0 = rec[13 * stride + j], b1 = rec[13 * stride + j + 1];
    const double dx = rec[17 * stride + j + 1] - rec[17 * stride + j], dy = rec[18 * stride + j + 1] - rec[18 * stride + j],
                 dz = rec[19 * stride + j + 1] - rec[19 * stride + j];
    const double t = 1e-13 * fmin(a0, b0);
    chain_x = axes && fabs(b1 - b0) <= t && fabs(dy) <= t && fabs(dz) <= t && fabs(dx - a0) <= t;
    chain_z = axes && fabs(a1 - a0) <= t && fabs(dy) <= t && fabs(dx) <= t && fabs(dz - b0) <= t;
  }
  const unsigned bx = __ballot_sync(0xffffffffu, chain_x), bz = __ballot_sync(0xffffffffu, chain_z);
  if ((threadIdx.x & 31) == 0) { s_bx[threadIdx.x >> 5] = bx; s_bz[threadIdx.x >> 5] = bz; }
  same = __syncthreads_and(same);
  if (threadIdx.x == 0) {
    unsigned mx = 0, mz = 0;
    for (int k = 0; k < 32; ++k) {                        // pair k = lanes 2k, 2k + 1 of the window
      mx |= ((s_bx[k >> 4] >> (2 * (k & 15))) & 1u) << k;
      mz |= ((s_bz[k >> 4] >> (2 * (k & 15))) & 1u) << k;
    }
    uniform[3 * blockIdx.x] = (j0 < n) ? same : 0;
    uniform[3 * blockIdx.x + 1] = same ? (int32_t)mx : 0;
    uniform[3 * blockIdx.x + 2] = same ? (int32_t)mz : 0;
  }
}

__global__ void set_weights_kernel(int64_t n, int64_t stride, const int32_t* __restrict__ perm, const double* __restrict__ sigma_caller,
                                   double* __restrict__ rec) {
  int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (s < n) rec[15 * stride + s] = sigma_caller[perm[s]] * kCoulomb;
}

__global__ void finish_sigma_kernel(int64_t n, int64_t stride, const int32_t* __restrict__ perm, const double* __restrict__ x,
                                    double* __restrict__ rec, double* __restrict__ sigma_caller) {
  int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (s < n) {
    double v = x[s];
    rec[15 * stride + s] = v * kCoulomb;
    sigma_caller[perm[s]] = v;
  }
}

__global__ void unpermute_matrix_kernel(int64_t n, int64_t ld, const int32_t* __restrict__ perm, const double* __restrict__ K,
                                        double* __restrict__ out) {
  int64_t si = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (si >= n) return;
  for (int64_t sj = blockIdx.y; sj < n; sj += gridDim.y) out[(int64_t)perm[si] + (int64_t)perm[sj] * n] = K[si + sj * ld];
}

__global__ void inverse_perm_kernel(int64_t n, const int32_t* __restrict__ perm, int32_t* __restrict__ inv) {
  int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (s < n) inv[perm[s]] = (int32_t)s;
}

// out[r * n + perm[sj]] = K[inv[rows[r]] + sj * ld]; grid = (ceil(n/256), n_rows)
__global__ void gather_rows_kernel(int64_t n, int64_t ld, const int32_t* __restrict__ perm, const int32_t* __restrict__ inv,
                                   const int32_t* __restrict__ rows, const double* __restrict__ K, double* __restrict__ out,
                                   int32_t* __restrict__ flag) {
  int64_t sj = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t r = blockIdx.y;
  const int32_t i = rows[r];
  if (i < 0 || i >= n) { if (sj == 0) atomicOr(flag, 64); return; }
  if (sj < n) out[r * n + perm[sj]] = K[(int64_t)inv[i] + sj * ld];
}

__global__ void unpermute_vector_kernel(int64_t n, const int32_t* __restrict__ perm, const double* __restrict__ v, double* __restrict__ out) {
  int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (s < n) out[perm[s]] = v[s];
}

__global__ void push_kernel(int64_t n3, double* __restrict__ pos, const double* __restrict__ E, double mu_dt) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n3) pos[i] = fma(mu_dt, E[i], pos[i]);
}

static void free_problem(neb_ctx* c) {
  void* ptrs[] = {c->d_rec, c->d_uniform, c->d_perm, c->d_colloc, c->d_normal, c->d_bc_kind, c->d_bc_value, c->d_diag, c->d_img,
                  c->d_K, c->d_rscale, c->d_ipiv, c->d_rowperm, c->d_b, c->d_x, c->d_sigma, c->d_dinv, c->d_V, c->d_s2, c->d_svd_w};
  for (void* p : ptrs)
    if (p) cudaFree(p);
  c->d_rec = nullptr; c->d_uniform = nullptr; c->d_perm = nullptr; c->d_colloc = nullptr; c->d_normal = nullptr; c->d_bc_kind = nullptr;
  c->d_bc_value = nullptr; c->d_diag = nullptr; c->d_img = nullptr; c->d_K = nullptr; c->d_rscale = nullptr;
  c->d_ipiv = nullptr; c->d_rowperm = nullptr; c->d_b = nullptr; c->d_x = nullptr; c->d_sigma = nullptr; c->d_dinv = nullptr;
  c->d_V = nullptr; c->d_s2 = nullptr; c->d_svd_w = nullptr;
  c->assembled = c->factored = c->have_sigma = false;
  c->n = c->npad = c->stride = 0;
  c->img_cap = 0;
}

neb_status finish_sigma(neb_ctx* c, const double* d_x) {
  finish_sigma_kernel<<<(unsigned)((c->n + 255) / 256), 256, 0, c->stream>>>(c->n, c->stride, c->d_perm, d_x, c->d_rec, c->d_sigma);
  c->launches++;
  NEB_CUDA(c, cudaGetLastError());
  c->have_sigma = true;
  return NEB_OK;
}

}  // namespace neb

using namespace neb;

extern "C" {

neb_status neb_create(neb_ctx** out, int device, void* cuda_stream) {
  if (!out) return NEB_EINVAL;
  *out = nullptr;
  int count = 0;
  if (cudaGetDeviceCount(&count) != cudaSuccess || device < 0 || device >= count) {
    cudaGetLastError();
    return NEB_ECUDA;
  }
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return NEB_ECUDA;
  if (prop.major != 10) return NEB_ECUDA;   // built for sm_100a only; no other code path exists
  if (cudaSetDevice(device) != cudaSuccess) return NEB_ECUDA;
  neb_ctx* c = new neb_ctx();
  c->device = device;
  c->stream = (cudaStream_t)cuda_stream;
  c->num_sms = prop.multiProcessorCount;
  bool ok = cudaMalloc((void**)&c->d_flag, sizeof(int32_t)) == cudaSuccess &&
            cudaMemset(c->d_flag, 0, sizeof(int32_t)) == cudaSuccess &&
            cudaMalloc(&c->d_panel_ws, lu_panel_ws_bytes(c->num_sms)) == cudaSuccess;
  if (ok) {
    // staging temporaries come from a pool of the context's own that keeps its memory across synchronisations
    // (the default pool hands everything back to the driver at each sync: milliseconds per re-allocation)
    cudaMemPoolProps pp = {};
    pp.allocType = cudaMemAllocationTypePinned;
    pp.handleTypes = cudaMemHandleTypeNone;
    pp.location.type = cudaMemLocationTypeDevice;
    pp.location.id = device;
    unsigned long long keep = ~0ULL;
    ok = cudaMemPoolCreate(&c->pool, &pp) == cudaSuccess &&
         cudaMemPoolSetAttribute(c->pool, cudaMemPoolAttrReleaseThreshold, &keep) == cudaSuccess;
  }
  if (ok) {
    int lo = 0, hi = 0;
    cudaDeviceGetStreamPriorityRange(&lo, &hi);   // hi = numerically lowest = greatest priority
    ok = cudaStreamCreateWithPriority(&c->side_stream, cudaStreamNonBlocking, hi) == cudaSuccess &&
         cudaStreamCreateWithPriority(&c->left_stream, cudaStreamNonBlocking, lo) == cudaSuccess &&
         cudaEventCreateWithFlags(&c->ev_chain, cudaEventDisableTiming) == cudaSuccess &&
         cudaEventCreateWithFlags(&c->ev_left, cudaEventDisableTiming) == cudaSuccess &&
         cudaEventCreateWithFlags(&c->ev_next, cudaEventDisableTiming) == cudaSuccess &&
         cudaEventCreateWithFlags(&c->ev_panel, cudaEventDisableTiming) == cudaSuccess;
  }
  for (int s = 0; ok && s < NEB_STAGE_COUNT; ++s)
    ok = cudaEventCreate(&c->ev0[s]) == cudaSuccess && cudaEventCreate(&c->ev1[s]) == cudaSuccess;
  ok = ok && lu_init_device(c) == NEB_OK;
  ok = ok && field_static_init(c) == NEB_OK;   // device address of the fixed scratch of neb_eval_static
  if (!ok) {
    neb_destroy(c);
    return NEB_ECUDA;
  }
  *out = c;
  return NEB_OK;
}

void neb_destroy(neb_ctx* c) {
  if (!c) return;
  cudaSetDevice(c->device);
  cudaStreamSynchronize(c->stream);
  free_problem(c);
  if (c->d_flag) cudaFree(c->d_flag);
  if (c->d_panel_ws) cudaFree(c->d_panel_ws);
  if (c->d_charges) cudaFree(c->d_charges);
  if (c->d_lines) cudaFree(c->d_lines);
  if (c->d_scratch) cudaFree(c->d_scratch);
  for (int s = 0; s < NEB_FASTVOL_SLOTS; ++s)
    if (c->fastvol[s].nodes) cudaFree((void*)c->fastvol[s].nodes);
  if (c->pool) cudaMemPoolDestroy(c->pool);
  if (c->side_stream) { cudaStreamSynchronize(c->side_stream); cudaStreamDestroy(c->side_stream); }
  if (c->left_stream) { cudaStreamSynchronize(c->left_stream); cudaStreamDestroy(c->left_stream); }
  if (c->ev_chain) cudaEventDestroy(c->ev_chain);
  if (c->ev_left) cudaEventDestroy(c->ev_left);
  if (c->ev_next) cudaEventDestroy(c->ev_next);
  if (c->ev_panel) cudaEventDestroy(c->ev_panel);
  for (int s = 0; s < NEB_STAGE_COUNT; ++s) {
    if (c->ev0[s]) cudaEventDestroy(c->ev0[s]);
    if (c->ev1[s]) cudaEventDestroy(c->ev1[s]);
  }
  delete c;
}

const char* neb_last_error(const neb_ctx* c) { return c ? c->err.c_str() : "null context"; }

neb_status neb_set_option(neb_ctx* c, int32_t option, int64_t value) {
  if (!c) return NEB_EINVAL;
  switch (option) {
    case NEB_OPT_MATH: c->math_fast = value ? 1 : 0; return NEB_OK;
    case NEB_OPT_LU_BLOCK:
      if (value != 64 && value != 128 && value != 256) return fail(c, NEB_EINVAL, "LU outer block width must be 64, 128 or 256");
      c->lu_nb = (int)value;
      return NEB_OK;
    case NEB_OPT_PROFILE: c->profile = value ? 1 : 0; return NEB_OK;
    case NEB_OPT_LU_PANEL: c->panel_mode = value ? 1 : 0; return NEB_OK;
    case NEB_OPT_LU_LOOKAHEAD: c->lu_lookahead = value ? 1 : 0; return NEB_OK;
    case NEB_OPT_EVAL_SPLITS:
      if (value < 0 || value > 1024) return fail(c, NEB_EINVAL, "eval splits must be 0 (automatic) .. 1024");
      c->eval_splits = (int)value;
      return NEB_OK;
    case NEB_OPT_PAIR_STRIPS: c->pair_strips = value ? 1 : 0; return NEB_OK;
    case NEB_OPT_SOLVER:
      if (value != 0 && value != 1) return fail(c, NEB_EINVAL, "solver must be 0 (LU) or 1 (SVD)");
      c->solver = (int)value;
      return NEB_OK;
    default: return fail(c, NEB_EINVAL, "unknown option");
  }
}

neb_status neb_assemble(neb_ctx* c, int64_t n, const int32_t* kind, const double* v0, const double* e1, const double* e2,
                        const double* radius, const double* colloc, const int32_t* bc_kind, const double* bc_value,
                        const double* eps_plus, const double* eps_minus, int32_t n_img, const double* img_shift) {
  if (!c) return NEB_EINVAL;
  // the LU panel runs on one cluster of cluster_max_ctas x 256 threads with at most 32 rows per thread: 131072 rows on
  // a B200 (the matrix itself, 8 n^2 bytes, reaches the 180 GB of HBM at n ~ 1.4e5)
  const int64_t n_max = std::max<int64_t>(panel_cluster_max_rows(c), (int64_t)c->num_sms * 384) - kPad;
  if (n <= 0 || n > n_max || !kind || !v0 || !e1 || !e2 || !bc_kind)
    return fail(c, NEB_EINVAL, "neb_assemble: n must be in 1.." + std::to_string(n_max) + " and kind, v0, e1, e2, bc_kind non-NULL");
  if (n_img < 0 || n_img > kMaxImages || (n_img > 0 && !img_shift))
    return fail(c, NEB_EINVAL, "neb_assemble: 0 <= n_img <= " + std::to_string(kMaxImages));
  NEB_CUDA(c, cudaSetDevice(c->device));
  const bool reuse = (c->n == n && c->d_K != nullptr);   // same size as the last problem: keep the buffers
  if (!reuse) {
    NEB_CUDA(c, cudaStreamSynchronize(c->stream));
    free_problem(c);
    c->n = n;
    const int64_t pad = c->dist_mode ? kDistBlock : kPad;     // distributed: whole 256-column blocks
    c->npad = (n + pad - 1) / pad * pad;
    c->stride = c->npad;
    c->ncol_loc = dist_local_cols(c->npad, c->dist_world, c->dist_rank);
  }
  c->assembled = c->factored = c->have_sigma = false;
  c->dist_scaled = false;
  const int64_t st = c->stride, npad = c->npad;
  if (!reuse) {
    NEB_CUDA(c, cudaMalloc((void**)&c->d_rec, sizeof(double) * kRec * st));
    NEB_CUDA(c, cudaMalloc((void**)&c->d_uniform, sizeof(int32_t) * 3 * (st / 64)));
    NEB_CUDA(c, cudaMalloc((void**)&c->d_perm, sizeof(int32_t) * st));
    NEB_CUDA(c, cudaMalloc((void**)&c->d_colloc, sizeof(double) * 3 * st));
    NEB_CUDA(c, cudaMalloc((void**)&c->d_normal, sizeof(double) * 3 * st));
    NEB_CUDA(c, cudaMalloc((void**)&c->d_bc_kind, sizeof(int32_t) * st));
    NEB_CUDA(c, cudaMalloc((void**)&c->d_bc_value, sizeof(double) * st));
    NEB_CUDA(c, cudaMalloc((void**)&c->d_diag, sizeof(double) * st));
    NEB_CUDA(c, cudaMalloc((void**)&c->d_rscale, sizeof(double) * npad));
    NEB_CUDA(c, cudaMalloc((void**)&c->d_ipiv, sizeof(int32_t) * npad));
    NEB_CUDA(c, cudaMalloc((void**)&c->d_rowperm, sizeof(int32_t) * npad));
    NEB_CUDA(c, cudaMalloc((void**)&c->d_b, sizeof(double) * npad));
    NEB_CUDA(c, cudaMalloc((void**)&c->d_x, sizeof(double) * 16 * npad));
    NEB_CUDA(c, cudaMalloc((void**)&c->d_dinv, sizeof(double) * 2 * (npad / 64) * 4096));
    NEB_CUDA(c, cudaMalloc((void**)&c->d_sigma, sizeof(double) * n));
    NEB_CUDA(c, cudaMalloc((void**)&c->d_K, sizeof(double) * (size_t)npad * (size_t)c->ncol_loc));
  }
  c->n_img = n_img > 0 ? n_img : 1;
  const int64_t n_chunks = (c->n_img + NEB_IMG_CHUNK - 1) / NEB_IMG_CHUNK;
  if (n_chunks > c->img_cap || !c->d_img) {
    if (c->d_img) { NEB_CUDA(c, cudaStreamSynchronize(c->stream)); NEB_CUDA(c, cudaFree(c->d_img)); c->d_img = nullptr; }
    NEB_CUDA(c, cudaMalloc((void**)&c->d_img, sizeof(double) * 3 * NEB_IMG_CHUNK * n_chunks));
    c->img_cap = n_chunks;
  }
  c->h_img_len.assign((size_t)c->n_img, 0.0);
  NEB_CUDA(c, cudaMemsetAsync(c->d_img, 0, sizeof(double) * 3 * NEB_IMG_CHUNK * n_chunks, c->stream));
  NEB_CUDA(c, cudaMemsetAsync(c->d_rec, 0, sizeof(double) * kRec * st, c->stream));
  NEB_CUDA(c, cudaMemsetAsync(c->d_flag, 0, sizeof(int32_t), c->stream));

  Staging sg(c);
  const void *dk, *dv0, *de1, *de2, *drad, *dcol, *dbk, *dbv, *dep, *dem;
  NEB_TRY(sg.in(kind, sizeof(int32_t) * n, &dk));
  NEB_TRY(sg.in(v0, sizeof(double) * 3 * n, &dv0));
  NEB_TRY(sg.in(e1, sizeof(double) * 3 * n, &de1));
  NEB_TRY(sg.in(e2, sizeof(double) * 3 * n, &de2));
  NEB_TRY(sg.in(radius, sizeof(double) * n, &drad));
  NEB_TRY(sg.in(colloc, sizeof(double) * 3 * n, &dcol));
  NEB_TRY(sg.in(bc_kind, sizeof(int32_t) * n, &dbk));
  NEB_TRY(sg.in(bc_value, sizeof(double) * n, &dbv));
  NEB_TRY(sg.in(eps_plus, sizeof(double) * n, &dep));
  NEB_TRY(sg.in(eps_minus, sizeof(double) * n, &dem));
  if (n_img > 0) {
    // the unshifted copy goes to slot 0 (the kernels treat slot 0 of the first chunk as the element itself); it must be present
    std::vector<double> h_img((size_t)3 * n_img);
    NEB_CUDA(c, cudaMemcpy(h_img.data(), img_shift, sizeof(double) * 3 * n_img, cudaMemcpyDefault));
    std::vector<double> len((size_t)n_img);
    std::vector<int> order((size_t)n_img);
    int zero = -1;
    for (int s = 0; s < n_img; ++s) {
      const double x = h_img[s], y = h_img[(size_t)n_img + s], z = h_img[(size_t)2 * n_img + s];
      if (zero < 0 && x == 0.0 && y == 0.0 && z == 0.0) zero = s;
      len[s] = sqrt(x * x + y * y + z * z);
      order[s] = s;
    }
    if (zero < 0) { free_problem(c); return fail(c, NEB_EINVAL, "neb_assemble: img_shift must include (0,0,0)"); }
    // copies sorted by the length of their shift (stable): the zero shift lands in slot 0, and the far copies of
    // Adaptive Modelling (neb_set_adaptive) form the tail; packed in chunks of NEB_IMG_CHUNK, [chunk][3][32]
    std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return len[a] < len[b]; });
    std::vector<double> packed((size_t)3 * NEB_IMG_CHUNK * n_chunks, 0.0);
    for (int s = 0; s < n_img; ++s) {
      const size_t base = (size_t)(s / NEB_IMG_CHUNK) * 3 * NEB_IMG_CHUNK + (size_t)(s % NEB_IMG_CHUNK);
      for (int k = 0; k < 3; ++k) packed[base + (size_t)k * NEB_IMG_CHUNK] = h_img[(size_t)k * n_img + order[s]];
      c->h_img_len[s] = len[order[s]];
    }
    NEB_CUDA(c, cudaMemcpyAsync(c->d_img, packed.data(), sizeof(double) * packed.size(), cudaMemcpyHostToDevice, c->stream));
    NEB_CUDA(c, cudaStreamSynchronize(c->stream));   // packed is a local buffer
  }
  int32_t* d_counts = nullptr;
  NEB_CUDA(c, cudaMallocFromPoolAsync((void**)&d_counts, 3 * sizeof(int32_t), c->pool, c->stream));
  sg.temps.push_back(d_counts);
  {
    StageTimer t(c, NEB_STAGE_GEOMETRY);
    kind_partition_kernel<<<1, 1024, 0, c->stream>>>((const int32_t*)dk, (int)n, c->d_perm, d_counts, c->d_flag);
    c->launches++;
    frames_kernel<<<(unsigned)((n + 127) / 128), 128, 0, c->stream>>>(
        n, st, c->d_perm, (const int32_t*)dk, (const double*)dv0, (const double*)de1, (const double*)de2,
        (const double*)drad, (const double*)dcol, (const int32_t*)dbk, (const double*)dbv, (const double*)dep,
        (const double*)dem, c->d_rec, c->d_colloc, c->d_normal, c->d_bc_kind, c->d_bc_value, c->d_diag, c->d_flag);
    c->launches++;
    tile_uniform_kernel<<<(unsigned)(st / 64), 64, 0, c->stream>>>(n, st, c->d_rec, d_counts, c->pair_strips, c->d_uniform);
    c->launches++;
    NEB_CUDA(c, cudaGetLastError());
  }
  int32_t h_counts[3], h_flag = 0;
  NEB_CUDA(c, cudaMemcpyAsync(h_counts, d_counts, sizeof(h_counts), cudaMemcpyDeviceToHost, c->stream));
  NEB_CUDA(c, cudaMemcpyAsync(&h_flag, c->d_flag, sizeof(int32_t), cudaMemcpyDeviceToHost, c->stream));
  NEB_CUDA(c, cudaStreamSynchronize(c->stream));
  if (h_flag != 0) {
    std::string why = "neb_assemble: invalid input:";
    if (h_flag & 1) why += " unknown element kind;";
    if (h_flag & 4) why += " zero-length or non-perpendicular edge;";
    if (h_flag & 8) why += " wire without a positive radius;";
    if (h_flag & 16) why += " unknown bc_kind;";
    if (h_flag & 32) why += " dielectric row with eps_plus == eps_minus, a non-positive permittivity, or on a wire;";
    free_problem(c);
    return fail(c, NEB_EINVAL, why);
  }
  c->n_rect = h_counts[0]; c->n_tri = h_counts[1]; c->n_wire = h_counts[2];
  // the image set must contain the zero shift in slot 0 for the kernels' first evaluation: any order is
  // fine mathematically, the kernels simply sum all n_img copies
  NEB_TRY(assemble_matrix(c));
  c->assembled = true;
  return NEB_OK;
}

neb_status neb_solve(neb_ctx* c, double* sigma_out) {
  if (!c) return NEB_EINVAL;
  if (!c->assembled) return fail(c, NEB_ESTATE, "neb_solve before neb_assemble");
  if (c->dist_mode) return fail(c, NEB_ESTATE, "neb_solve on a distributed context: the factorisation runs through the neb_dist_* calls");
  NEB_CUDA(c, cudaSetDevice(c->device));
  if (!c->factored) {
    NEB_TRY(scale_matrix_rows(c));
    c->factored_with = c->solver;
    if (c->solver == 1) NEB_TRY(svd_factor(c));
    else NEB_TRY(lu_factor(c));
    int32_t h_flag = 0;
    NEB_CUDA(c, cudaMemcpyAsync(&h_flag, c->d_flag, sizeof(int32_t), cudaMemcpyDeviceToHost, c->stream));
    NEB_CUDA(c, cudaStreamSynchronize(c->stream));
    c->factored = true;   // the matrix is overwritten either way
    if (h_flag & 2) {
      c->assembled = false;
      return fail(c, NEB_ESINGULAR, "neb_solve: zero or NaN pivot");
    }
  }
  NEB_TRY(form_rhs(c));
  NEB_TRY(factors_solve(c, c->d_b, 1, c->d_x));
  NEB_TRY(finish_sigma(c, c->d_x));
  if (sigma_out) {
    if (is_device_ptr(sigma_out)) {
      NEB_CUDA(c, cudaMemcpyAsync(sigma_out, c->d_sigma, sizeof(double) * c->n, cudaMemcpyDeviceToDevice, c->stream));
    } else {
      NEB_CUDA(c, cudaMemcpyAsync(sigma_out, c->d_sigma, sizeof(double) * c->n, cudaMemcpyDeviceToHost, c->stream));
      NEB_CUDA(c, cudaStreamSynchronize(c->stream));
    }
  }
  return NEB_OK;
}

neb_status neb_set_sigma(neb_ctx* c, const double* sigma) {
  if (!c || !sigma) return NEB_EINVAL;
  if (!c->assembled && c->n == 0) return fail(c, NEB_ESTATE, "neb_set_sigma before neb_assemble");
  NEB_CUDA(c, cudaSetDevice(c->device));
  Staging sg(c);
  const void* ds;
  NEB_TRY(sg.in(sigma, sizeof(double) * c->n, &ds));
  NEB_CUDA(c, cudaMemcpyAsync(c->d_sigma, ds, sizeof(double) * c->n, cudaMemcpyDeviceToDevice, c->stream));
  set_weights_kernel<<<(unsigned)((c->n + 255) / 256), 256, 0, c->stream>>>(c->n, c->stride, c->d_perm, c->d_sigma, c->d_rec);
  c->launches++;
  NEB_CUDA(c, cudaGetLastError());
  c->have_sigma = true;
  return NEB_OK;
}

neb_status neb_eval(neb_ctx* c, int64_t m, const double* pts, double* phi, double* E) {
  if (!c || m < 0 || (m > 0 && !pts)) return NEB_EINVAL;
  if (!c->have_sigma) return fail(c, NEB_ESTATE, "neb_eval before neb_solve / neb_set_sigma");
  if (m == 0) return NEB_OK;
  NEB_CUDA(c, cudaSetDevice(c->device));
  Staging sg(c);
  const void* dp;
  void *dphi, *dE;
  NEB_TRY(sg.in(pts, sizeof(double) * 3 * m, &dp));
  NEB_TRY(sg.out(phi, sizeof(double) * m, &dphi));
  NEB_TRY(sg.out(E, sizeof(double) * 3 * m, &dE));
  NEB_TRY(field_at_points(c, m, (const double*)dp, true, true, (double*)dphi, (double*)dE));
  return sg.finish();
}

neb_status neb_set_svd_cutoff(neb_ctx* c, double rcond) {
  if (!c || !(rcond >= 0.0) || !(rcond < 1.0)) return NEB_EINVAL;
  c->svd_rcond = rcond;
  return NEB_OK;
}

neb_status neb_get_singular_values(neb_ctx* c, double* s_out, int32_t* sweeps) {
  if (!c || !s_out) return NEB_EINVAL;
  if (!c->factored || c->factored_with != 1) return fail(c, NEB_ESTATE, "neb_get_singular_values: no SVD factors (NEB_OPT_SOLVER = 1, then neb_solve)");
  NEB_CUDA(c, cudaSetDevice(c->device));
  std::vector<double> h((size_t)c->npad);
  NEB_CUDA(c, cudaMemcpyAsync(h.data(), c->d_s2, sizeof(double) * c->npad, cudaMemcpyDeviceToHost, c->stream));
  NEB_CUDA(c, cudaStreamSynchronize(c->stream));
  for (double& v : h) v = sqrt(v);
  NEB_CUDA(c, cudaMemcpy(s_out, h.data(), sizeof(double) * c->npad, cudaMemcpyDefault));
  if (sweeps) *sweeps = c->svd_sweeps;
  return NEB_OK;
}

neb_status neb_eval_static(neb_ctx* c, int64_t m, const double* pts, double* phi, double* E) {
  if (!c || m < 0 || (m > 0 && !pts)) return NEB_EINVAL;
  if (!c->have_sigma) return fail(c, NEB_ESTATE, "neb_eval_static before neb_solve / neb_set_sigma");
  if (m == 0) return NEB_OK;
  NEB_CUDA(c, cudaSetDevice(c->device));
  // device pointers only: staging a host buffer would need a temporary, and this entry point allocates nothing
  if (!is_device_ptr(pts) || (phi && !is_device_ptr(phi)) || (E && !is_device_ptr(E)))
    return fail(c, NEB_EINVAL, "neb_eval_static: pts, phi and E must be device pointers");
  return field_at_points_static(c, m, pts, phi, E);
}

neb_status neb_set_adaptive(neb_ctx* c, double far_distance) {
  if (!c || !(far_distance >= 0.0)) return NEB_EINVAL;
  c->adaptive_far = far_distance;
  return NEB_OK;
}

neb_status neb_solve_weighting_multi(neb_ctx* c, int32_t n_rhs, const double* bc_value_w, double* sigma_w_out) {
  if (!c || n_rhs < 1 || !bc_value_w || !sigma_w_out) return NEB_EINVAL;
  if (!c->factored || !c->assembled) return fail(c, NEB_ESTATE, "neb_solve_weighting before the first neb_solve (no LU factors)");
  if (c->dist_mode) return fail(c, NEB_ESTATE, "neb_solve_weighting: not available on a distributed context");
  NEB_CUDA(c, cudaSetDevice(c->device));
  Staging sg(c);
  const void* dw;
  void* dout;
  NEB_TRY(sg.in(bc_value_w, sizeof(double) * (size_t)n_rhs * c->n, &dw));
  NEB_TRY(sg.out(sigma_w_out, sizeof(double) * (size_t)n_rhs * c->n, &dout));
  NEB_TRY(solve_weighting(c, n_rhs, (const double*)dw, (double*)dout));
  return sg.finish();
}

neb_status neb_solve_weighting(neb_ctx* c, const double* bc_value_w, double* sigma_w_out) {
  return neb_solve_weighting_multi(c, 1, bc_value_w, sigma_w_out);
}

neb_status neb_fastvol_build(neb_ctx* c, int32_t slot, int32_t nx, int32_t ny, int32_t nz, const double* origin,
                             const double* spacing, int32_t with_charges) {
  if (!c || !origin || !spacing) return NEB_EINVAL;
  if (slot < 0 || slot >= NEB_FASTVOL_SLOTS || nx < 2 || ny < 2 || nz < 2 || (int64_t)nx * ny * nz > (1LL << 28))
    return fail(c, NEB_EINVAL, "neb_fastvol_build: slot out of range, fewer than 2 nodes on an axis, or more than 2^28 nodes");
  for (int a = 0; a < 3; ++a)
    if (!(spacing[a] > 0.0) || !isfinite(origin[a]) || !isfinite(spacing[a]))
      return fail(c, NEB_EINVAL, "neb_fastvol_build: spacing must be positive and finite");
  if (!c->have_sigma) return fail(c, NEB_ESTATE, "neb_fastvol_build before neb_solve / neb_set_sigma");
  NEB_CUDA(c, cudaSetDevice(c->device));
  return fastvol_build(c, slot, nx, ny, nz, origin, spacing, with_charges != 0);
}

neb_status neb_fastvol_eval(neb_ctx* c, int32_t slot, int64_t m, const double* pts, double* phi, double* E) {
  if (!c || m < 0 || (m > 0 && !pts) || slot < 0 || slot >= NEB_FASTVOL_SLOTS) return NEB_EINVAL;
  if (!c->fastvol[slot].nodes) return fail(c, NEB_ESTATE, "neb_fastvol_eval: empty slot (call neb_fastvol_build)");
  if (m == 0) return NEB_OK;
  NEB_CUDA(c, cudaSetDevice(c->device));
  Staging sg(c);
  const void* dp;
  void *dphi, *dE;
  NEB_TRY(sg.in(pts, sizeof(double) * 3 * m, &dp));
  NEB_TRY(sg.out(phi, sizeof(double) * m, &dphi));
  NEB_TRY(sg.out(E, sizeof(double) * 3 * m, &dE));
  NEB_TRY(fastvol_eval(c, slot, m, (const double*)dp, (double*)dphi, (double*)dE));
  return sg.finish();
}

neb_status neb_fastvol_get(neb_ctx* c, int32_t slot, double* values) {
  if (!c || !values || slot < 0 || slot >= NEB_FASTVOL_SLOTS) return NEB_EINVAL;
  const FastVol& fv = c->fastvol[slot];
  if (!fv.nodes) return fail(c, NEB_ESTATE, "neb_fastvol_get: empty slot");
  NEB_CUDA(c, cudaSetDevice(c->device));
  Staging sg(c);
  void* dout;
  NEB_TRY(sg.out(values, sizeof(double) * 4 * (size_t)fv.nx * fv.ny * fv.nz, &dout));
  NEB_TRY(fastvol_get(c, slot, (double*)dout));
  return sg.finish();
}

neb_status neb_add_space_charge(neb_ctx* c, int64_t q, const double* pos, const double* charge, int32_t replace) {
  if (!c || q < 0 || (q > 0 && (!pos || !charge))) return NEB_EINVAL;
  NEB_CUDA(c, cudaSetDevice(c->device));
  if (replace) { c->q = 0; c->n_lines = 0; }
  if (q == 0) return NEB_OK;
  int64_t need = c->q + q;
  if (need > c->q_cap) {
    int64_t cap = need > 2 * c->q_cap ? need : 2 * c->q_cap;
    cap = (cap + 255) / 256 * 256;
    double* nd = nullptr;
    NEB_CUDA(c, cudaMalloc((void**)&nd, sizeof(double) * 4 * cap));
    for (int f = 0; f < 4 && c->q > 0; ++f)
      NEB_CUDA(c, cudaMemcpyAsync(nd + f * cap, c->d_charges + f * c->q_cap, sizeof(double) * c->q, cudaMemcpyDeviceToDevice, c->stream));
    if (c->d_charges) {
      NEB_CUDA(c, cudaStreamSynchronize(c->stream));
      NEB_CUDA(c, cudaFree(c->d_charges));
    }
    c->d_charges = nd;
    c->q_cap = cap;
  }
  cudaMemcpyKind kp = is_device_ptr(pos) ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
  cudaMemcpyKind kq = is_device_ptr(charge) ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
  for (int f = 0; f < 3; ++f)
    NEB_CUDA(c, cudaMemcpyAsync(c->d_charges + f * c->q_cap + c->q, pos + f * q, sizeof(double) * q, kp, c->stream));
  NEB_CUDA(c, cudaMemcpyAsync(c->d_charges + 3 * c->q_cap + c->q, charge, sizeof(double) * q, kq, c->stream));
  // borrowed host buffers (pinned memory copies asynchronously) must have been read before the call returns
  if (kp == cudaMemcpyHostToDevice || kq == cudaMemcpyHostToDevice) NEB_CUDA(c, cudaStreamSynchronize(c->stream));
  c->q = need;
  return NEB_OK;
}

neb_status neb_voxelize_space_charge(neb_ctx* c, const double* origin, const double* voxel, const int32_t* dims, int64_t* n_lines_out) {
  if (!c || !origin || !voxel || !dims) return NEB_EINVAL;
  for (int a = 0; a < 3; ++a)
    if (!(voxel[a] > 0.0) || !isfinite(voxel[a]) || !isfinite(origin[a]) || dims[a] < 1)
      return fail(c, NEB_EINVAL, "neb_voxelize_space_charge: voxel sizes must be positive and finite, dims >= 1");
  if ((int64_t)dims[0] * dims[1] * dims[2] > (1LL << 26)) return fail(c, NEB_EINVAL, "neb_voxelize_space_charge: more than 2^26 voxels");
  if (c->q == 0 && c->n_lines == 0) return fail(c, NEB_ESTATE, "neb_voxelize_space_charge: no point charges (neb_add_space_charge first)");
  NEB_CUDA(c, cudaSetDevice(c->device));
  return voxelize_charges(c, origin, voxel, dims, n_lines_out);
}

neb_status neb_get_line_charges(neb_ctx* c, double* lines) {
  if (!c || !lines) return NEB_EINVAL;
  if (c->n_lines == 0) return NEB_OK;
  NEB_CUDA(c, cudaSetDevice(c->device));
  cudaMemcpyKind kind = is_device_ptr(lines) ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost;
  for (int f = 0; f < 5; ++f)
    NEB_CUDA(c, cudaMemcpyAsync(lines + f * c->n_lines, c->d_lines + f * c->line_cap, sizeof(double) * c->n_lines, kind, c->stream));
  NEB_CUDA(c, cudaStreamSynchronize(c->stream));
  return NEB_OK;
}

neb_status neb_push(neb_ctx* c, int64_t q, double* pos, const double* E, double mu_dt) {
  if (!c || q < 0 || (q > 0 && (!pos || !E))) return NEB_EINVAL;
  if (q == 0) return NEB_OK;
  NEB_CUDA(c, cudaSetDevice(c->device));
  bool dp = is_device_ptr(pos), dE = is_device_ptr(E);
  if (dp != dE) return fail(c, NEB_EINVAL, "neb_push: pos and E must both be host or both be device pointers");
  Staging sg(c);
  const void* din;
  const void* dEv;
  void* dpos;
  NEB_TRY(sg.in(E, sizeof(double) * 3 * q, &dEv));
  if (dp) dpos = pos;
  else {
    NEB_TRY(sg.in(pos, sizeof(double) * 3 * q, &din));
    dpos = const_cast<void*>(din);
    sg.outs.push_back({dpos, pos, sizeof(double) * 3 * (size_t)q});
  }
  push_kernel<<<(unsigned)((3 * q + 255) / 256), 256, 0, c->stream>>>(3 * q, (double*)dpos, (const double*)dEv, mu_dt);
  c->launches++;
  NEB_CUDA(c, cudaGetLastError());
  return sg.finish();
}

neb_status neb_get_matrix(neb_ctx* c, double* K_out) {
  if (!c || !K_out) return NEB_EINVAL;
  if (!c->assembled || c->factored) return fail(c, NEB_ESTATE, "neb_get_matrix: only between neb_assemble and the first neb_solve");
  if (c->dist_mode) return fail(c, NEB_ESTATE, "neb_get_matrix: not available on a distributed context (each rank holds only its column blocks)");
  NEB_CUDA(c, cudaSetDevice(c->device));
  Staging sg(c);
  void* dout;
  NEB_TRY(sg.out(K_out, sizeof(double) * (size_t)c->n * (size_t)c->n, &dout));
  dim3 grid((unsigned)((c->n + 255) / 256), (unsigned)std::min<int64_t>(c->n, 65535));
  unpermute_matrix_kernel<<<grid, 256, 0, c->stream>>>(c->n, c->npad, c->d_perm, c->d_K, (double*)dout);
  c->launches++;
  NEB_CUDA(c, cudaGetLastError());
  return sg.finish();
}

neb_status neb_get_matrix_rows(neb_ctx* c, int64_t n_rows, const int32_t* rows, double* K_out) {
  if (!c || n_rows < 0 || (n_rows > 0 && (!rows || !K_out))) return NEB_EINVAL;
  if (!c->assembled || c->factored) return fail(c, NEB_ESTATE, "neb_get_matrix_rows: only between neb_assemble and the first neb_solve");
  if (c->dist_mode) return fail(c, NEB_ESTATE, "neb_get_matrix_rows: not available on a distributed context (each rank holds only its column blocks)");
  if (n_rows == 0) return NEB_OK;
  if (n_rows > 65535) return fail(c, NEB_EINVAL, "neb_get_matrix_rows: at most 65535 rows per call");
  NEB_CUDA(c, cudaSetDevice(c->device));
  Staging sg(c);
  const void* drows;
  void* dout;
  int32_t* inv = nullptr;
  NEB_TRY(sg.in(rows, sizeof(int32_t) * n_rows, &drows));
  NEB_TRY(sg.out(K_out, sizeof(double) * (size_t)n_rows * (size_t)c->n, &dout));
  NEB_CUDA(c, cudaMallocFromPoolAsync((void**)&inv, sizeof(int32_t) * c->n, c->pool, c->stream));
  sg.temps.push_back(inv);
  NEB_CUDA(c, cudaMemsetAsync(c->d_flag, 0, sizeof(int32_t), c->stream));
  inverse_perm_kernel<<<(unsigned)((c->n + 255) / 256), 256, 0, c->stream>>>(c->n, c->d_perm, inv);
  dim3 grid((unsigned)((c->n + 255) / 256), (unsigned)n_rows);
  gather_rows_kernel<<<grid, 256, 0, c->stream>>>(c->n, c->npad, c->d_perm, inv, (const int32_t*)drows, c->d_K, (double*)dout, c->d_flag);
  c->launches += 2;
  NEB_CUDA(c, cudaGetLastError());
  int32_t h_flag = 0;
  NEB_CUDA(c, cudaMemcpyAsync(&h_flag, c->d_flag, sizeof(int32_t), cudaMemcpyDeviceToHost, c->stream));
  NEB_CUDA(c, cudaStreamSynchronize(c->stream));
  if (h_flag & 64) return fail(c, NEB_EINVAL, "neb_get_matrix_rows: row index outside [0, n)");
  return sg.finish();
}

neb_status neb_get_rhs(neb_ctx* c, double* b_out) {
  if (!c || !b_out) return NEB_EINVAL;
  if (!c->have_sigma || !c->factored) return fail(c, NEB_ESTATE, "neb_get_rhs before neb_solve");
  NEB_CUDA(c, cudaSetDevice(c->device));
  Staging sg(c);
  void* dout;
  NEB_TRY(sg.out(b_out, sizeof(double) * c->n, &dout));
  unpermute_vector_kernel<<<(unsigned)((c->n + 255) / 256), 256, 0, c->stream>>>(c->n, c->d_perm, c->d_b, (double*)dout);
  c->launches++;
  NEB_CUDA(c, cudaGetLastError());
  return sg.finish();
}

neb_status neb_fp64_peak(neb_ctx* c, int32_t kind, double* tflops) {
  if (!c || !tflops) return NEB_EINVAL;
  NEB_CUDA(c, cudaSetDevice(c->device));
  return fp64_peak(c, kind, tflops);
}

neb_status neb_stage_ms(neb_ctx* c, int32_t stage, double* ms, int64_t* launches) {
  if (!c || stage < 0 || stage >= NEB_STAGE_COUNT) return NEB_EINVAL;
  if (ms) *ms = c->stat[stage].ms;
  if (launches) *launches = c->stat[stage].launches;
  return NEB_OK;
}

neb_status neb_get_counter(neb_ctx* c, int32_t which, double* value) {
  if (!c || !value || which < 0 || which >= NEB_COUNTER_COUNT) return NEB_EINVAL;
  *value = c->counter[which];
  return NEB_OK;
}

neb_status neb_reset_stats(neb_ctx* c) {
  if (!c) return NEB_EINVAL;
  for (int s = 0; s < NEB_STAGE_COUNT; ++s) c->stat[s] = StageStat();
  return NEB_OK;
}

int64_t neb_launch_count(const neb_ctx* c) { return c ? c->launches : 0; }

}  // extern "C"
