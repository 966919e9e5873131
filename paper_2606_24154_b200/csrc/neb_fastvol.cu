// neb_fastvol.cu — SURVEY §8(f) item 1: FastVolume ("Fast Volume", P:222 CreateFastVolPF /
// CreateWtFldFastVolPF) and the weighting-field solve.
//
//   neb_fastvol_build   Phi and E at the nodes of a uniform 3-D grid, by the fused evaluation kernel (a7/a8) —
//                       the "computationally expensive step performed only once" — stored as one 32-byte record
//                       (Phi, Ex, Ey, Ez) per node, so that a lookup touches one sector per corner;
//   neb_fastvol_eval    "a simple trilinear interpolation from the values stored at the nearest nodes": a gather of
//                       8 records per point, bound by L2/HBM, not by arithmetic;
//   neb_solve_weighting the charge densities for a weighting potential (read-out electrode at 1, every other
//                       conductor at 0, no space charge), on the RESIDENT LU factors; with neb_set_sigma +
//                       neb_fastvol_build into another slot this gives the weighting-field map.
// Readings S25 (uniform grid, NaN outside, 1e-9-cell slack at the faces) and S26 (weighting RHS) in DESIGN.md §3.
#include <math.h>

#include "neb_internal.h"

namespace neb {

__global__ void fastvol_nodes_kernel(int64_t nn, int nx, int ny, double ox, double oy, double oz, double hx, double hy,
                                     double hz, double* __restrict__ pts) {
  int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= nn) return;
  const int i = (int)(t % nx), j = (int)((t / nx) % ny), k = (int)(t / ((int64_t)nx * ny));
  pts[t] = ox + i * hx;              // same expression as the oracle's node generator (one multiply, one add)
  pts[nn + t] = oy + j * hy;
  pts[2 * nn + t] = oz + k * hz;
}

__global__ void fastvol_pack_kernel(int64_t nn, const double* __restrict__ phi, const double* __restrict__ E,
                                    double4* __restrict__ nodes) {
  int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t < nn) nodes[t] = make_double4(phi[t], E[t], E[nn + t], E[2 * nn + t]);
}

__global__ void fastvol_unpack_kernel(int64_t nn, const double4* __restrict__ nodes, double* __restrict__ values) {
  int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= nn) return;
  const double4 v = nodes[t];
  values[t] = v.x; values[nn + t] = v.y; values[2 * nn + t] = v.z; values[3 * nn + t] = v.w;
}

// cell coordinate of x on one axis: false if outside (with the 1e-9-cell slack of reading S25)
__device__ __forceinline__ bool cell_of(double x, double o, double h, int n, int& i, double& f) {
  double t = (x - o) / h;
  if (!(t >= -1e-9 && t <= (double)(n - 1) + 1e-9)) return false;
  t = fmin(fmax(t, 0.0), (double)(n - 1));
  i = min((int)floor(t), n - 2);
  f = t - (double)i;
  return true;
}

// one node record through the read-only path: ONE 32-byte load of its sector (sm_100: ld.global.nc.v4.f64, SASS LDG.E.256)
// instead of two 16-byte loads — the lookup is bound by the L1/TEX request rate (every lane gathers its own sectors):
// 1e7 lookups in C2's map 0.450 -> 0.427 ms
__device__ __forceinline__ double4 load_node(const double4* p) {
  double4 v;
  asm("ld.global.nc.v4.f64 {%0, %1, %2, %3}, [%4];" : "=d"(v.x), "=d"(v.y), "=d"(v.z), "=d"(v.w) : "l"(p));
  return v;
}

__device__ __forceinline__ double4 lerp4(const double4& a, const double4& b, double f) {
  return make_double4(fma(f, b.x - a.x, a.x), fma(f, b.y - a.y, a.y), fma(f, b.z - a.z, a.z), fma(f, b.w - a.w, a.w));
}

__global__ void __launch_bounds__(256) fastvol_eval_kernel(FastVol fv, int64_t m, const double* __restrict__ pts,
                                                           double* __restrict__ phi, double* __restrict__ E) {
  int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= m) return;
  int i, j, k;
  double fx, fy, fz;
  const bool in = cell_of(pts[p], fv.o[0], fv.h[0], fv.nx, i, fx) && cell_of(pts[m + p], fv.o[1], fv.h[1], fv.ny, j, fy) &&
                  cell_of(pts[2 * m + p], fv.o[2], fv.h[2], fv.nz, k, fz);
  double4 r = make_double4(NAN, NAN, NAN, NAN);
  if (in) {
    const double4* n0 = fv.nodes + ((int64_t)k * fv.ny + j) * fv.nx + i;
    const int64_t sy = fv.nx, sz = (int64_t)fv.nx * fv.ny;
    const double4 v000 = load_node(n0), v100 = load_node(n0 + 1), v010 = load_node(n0 + sy), v110 = load_node(n0 + sy + 1);
    const double4 v001 = load_node(n0 + sz), v101 = load_node(n0 + sz + 1), v011 = load_node(n0 + sz + sy), v111 = load_node(n0 + sz + sy + 1);
    const double4 c00 = lerp4(v000, v100, fx), c10 = lerp4(v010, v110, fx), c01 = lerp4(v001, v101, fx), c11 = lerp4(v011, v111, fx);
    r = lerp4(lerp4(c00, c10, fy), lerp4(c01, c11, fy), fz);
  }
  if (phi) phi[p] = r.x;
  if (E) { E[p] = r.y; E[m + p] = r.z; E[2 * m + p] = r.w; }
}

// weighting right-hand sides in the sorted order (reading S26): b[k * npad + s], k < nrhs
__global__ void weighting_rhs_kernel(int64_t n, int64_t npad, int nrhs, const int32_t* __restrict__ perm, const int32_t* __restrict__ bc_kind,
                                     const double* __restrict__ w_caller, double* __restrict__ b) {
  int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= npad) return;
  const bool use = s < n && bc_kind[s] == NEB_BC_DIRICHLET;
  const int64_t j = use ? perm[s] : 0;
  for (int k = 0; k < nrhs; ++k) b[k * npad + s] = use ? w_caller[k * n + j] : 0.0;
}

__global__ void unpermute_multi_kernel(int64_t n, int64_t npad, int nrhs, const int32_t* __restrict__ perm, const double* __restrict__ x,
                                       double* __restrict__ out) {
  int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= n) return;
  const int64_t j = perm[s];
  for (int k = 0; k < nrhs; ++k) out[k * n + j] = x[k * npad + s];
}

neb_status fastvol_build(neb_ctx* c, int slot, int nx, int ny, int nz, const double* o, const double* h, bool with_charges) {
  const int64_t nn = (int64_t)nx * ny * nz;
  FastVol& fv = c->fastvol[slot];
  if (fv.nodes) {
    NEB_CUDA(c, cudaStreamSynchronize(c->stream));
    NEB_CUDA(c, cudaFree((void*)fv.nodes));
    fv = FastVol();
  }
  double4* nodes = nullptr;
  NEB_CUDA(c, cudaMalloc((void**)&nodes, sizeof(double4) * (size_t)nn));
  double *pts = nullptr, *phi = nullptr, *E = nullptr;
  NEB_CUDA(c, cudaMallocFromPoolAsync((void**)&pts, sizeof(double) * 3 * (size_t)nn, c->pool, c->stream));
  NEB_CUDA(c, cudaMallocFromPoolAsync((void**)&phi, sizeof(double) * (size_t)nn, c->pool, c->stream));
  NEB_CUDA(c, cudaMallocFromPoolAsync((void**)&E, sizeof(double) * 3 * (size_t)nn, c->pool, c->stream));
  const unsigned blocks = (unsigned)((nn + 255) / 256);
  fastvol_nodes_kernel<<<blocks, 256, 0, c->stream>>>(nn, nx, ny, o[0], o[1], o[2], h[0], h[1], h[2], pts);
  c->launches++;
  neb_status st = field_at_points(c, nn, pts, true, with_charges, phi, E);
  if (st == NEB_OK) {
    StageTimer t(c, NEB_STAGE_FASTVOL);
    fastvol_pack_kernel<<<blocks, 256, 0, c->stream>>>(nn, phi, E, nodes);
    c->launches++;
  }
  cudaFreeAsync(pts, c->stream);
  cudaFreeAsync(phi, c->stream);
  cudaFreeAsync(E, c->stream);
  if (st != NEB_OK || cudaGetLastError() != cudaSuccess) {
    cudaFree(nodes);
    return st != NEB_OK ? st : fail(c, NEB_ECUDA, "neb_fastvol_build: kernel launch failed");
  }
  fv.nodes = nodes; fv.nx = nx; fv.ny = ny; fv.nz = nz;
  for (int a = 0; a < 3; ++a) { fv.o[a] = o[a]; fv.h[a] = h[a]; }
  return NEB_OK;
}

neb_status fastvol_eval(neb_ctx* c, int slot, int64_t m, const double* d_pts, double* d_phi, double* d_E) {
  StageTimer t(c, NEB_STAGE_FASTVOL);
  fastvol_eval_kernel<<<(unsigned)((m + 255) / 256), 256, 0, c->stream>>>(c->fastvol[slot], m, d_pts, d_phi, d_E);
  c->launches++;
  NEB_CUDA(c, cudaGetLastError());
  return NEB_OK;
}

neb_status fastvol_get(neb_ctx* c, int slot, double* d_values) {
  const FastVol& fv = c->fastvol[slot];
  const int64_t nn = (int64_t)fv.nx * fv.ny * fv.nz;
  fastvol_unpack_kernel<<<(unsigned)((nn + 255) / 256), 256, 0, c->stream>>>(nn, fv.nodes, d_values);
  c->launches++;
  NEB_CUDA(c, cudaGetLastError());
  return NEB_OK;
}

neb_status solve_weighting(neb_ctx* c, int nrhs, const double* d_w_caller, double* d_sigma_out) {
  const int64_t n = c->n, npad = c->npad;
  // the physical right-hand side (neb_get_rhs) and sigma stay as they are: the solve runs on temporaries
  double *tb = nullptr, *tx = nullptr;
  NEB_CUDA(c, cudaMallocFromPoolAsync((void**)&tb, sizeof(double) * (size_t)nrhs * npad, c->pool, c->stream));
  NEB_CUDA(c, cudaMallocFromPoolAsync((void**)&tx, sizeof(double) * (size_t)nrhs * npad, c->pool, c->stream));
  weighting_rhs_kernel<<<(unsigned)((npad + 255) / 256), 256, 0, c->stream>>>(n, npad, nrhs, c->d_perm, c->d_bc_kind, d_w_caller, tb);
  c->launches++;
  neb_status st = factors_solve(c, tb, nrhs, tx);
  if (st == NEB_OK) {
    unpermute_multi_kernel<<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>(n, npad, nrhs, c->d_perm, tx, d_sigma_out);
    c->launches++;
  }
  cudaFreeAsync(tb, c->stream);
  cudaFreeAsync(tx, c->stream);
  if (st == NEB_OK) NEB_CUDA(c, cudaGetLastError());
  return st;
}

}  // namespace neb
