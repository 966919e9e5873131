// neb_svd.cu — SURVEY §8(f).4, second half: InvertMatrix with OptSVD ("in the case of complex MPGD geometries,
// due to the repetition of basic primitives, there exist overlapping surfaces ... Singular Value Decomposition can be
// used to obtain the solution").  Reading S31: the solution is the minimum-norm least-squares solution of the
// row-equilibrated system, sigma = sum over s_j > rcond s_max of v_j (u_j . b) / s_j.
//
// One-sided Jacobi (Hestenes) on the resident matrix: plane rotations from the right make the columns of A = K V
// mutually orthogonal; then A = U diag(s), s_j = |a_j|, and  sigma = V w,  w_j = (a_j . b) / s_j^2  for the kept j.
// No bidiagonalisation, no explicit U: the method works on columns, which is how the matrix is stored, every
// rotation is two dot products and two column updates (pure streaming, HBM/L2-bound), and its singular values are
// accurate to RELATIVE precision — what matters for the cut between "tiny" and "zero".
//   svd_round_kernel   one round of the round-robin ordering: npad/2 disjoint column pairs, one CTA each (Gram entries
//                      by a fixed-order block reduction, rotation of the two columns of A and of V)
//   a sweep = npad - 1 rounds; sweeps repeat until one of them rotates nothing (|a_p . a_q| <= tol |a_p| |a_q| for all pairs)
//   svd_norms_kernel, svd_weights_kernel, svd_apply_kernel   the solve: s_j^2, w, sigma = V w
// Cost per sweep: npad^2/2 pairs x (3 dot products + 2 rotated column pairs) = 9 npad^3 flop and 40 npad^3 bytes
// through L2/HBM, 6-12 sweeps: one to two orders of magnitude above the LU, as the paper says ("LU ... is usually much
// faster"); meant for the meshes that need it (n up to ~1e4), memory 16 npad^2 bytes (A and V).
#include "neb_internal.h"

namespace neb {
namespace {

constexpr int SV_THREADS = 256;

__device__ __forceinline__ double block_sum(double v, double* s_red) {
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  __syncthreads();
  if (lane == 0) s_red[warp] = v;
  __syncthreads();
  double t = 0.0;
  for (int w = 0; w < SV_THREADS / 32; ++w) t += s_red[w];      // every thread adds the warp sums in the same order
  return t;
}

__global__ void svd_identity_kernel(double* V, int64_t n) {
  int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx < n * n) V[idx] = (idx / n == idx % n) ? 1.0 : 0.0;
}

// Round r of the round-robin tournament on n columns (n even): column n-1 stays, the others rotate; pair k of the
// round is (n-1, r) for k = 0 and ((r + k) mod (n-1), (r - k) mod (n-1)) otherwise — every pair meets once per sweep.
__global__ void __launch_bounds__(SV_THREADS) svd_round_kernel(double* __restrict__ A, double* __restrict__ V, int64_t ld, int n, int round,
                                                               double tol, const double* __restrict__ max_norm2,
                                                               unsigned int* __restrict__ rotations) {
  __shared__ double s_red[SV_THREADS / 32];
  const int m = n - 1, k = blockIdx.x;
  int i = (k == 0) ? m : (round + k) % m;
  int j = (k == 0) ? round : (round - k + m) % m;
  const int p = min(i, j), q = max(i, j);
  double* ap = A + (int64_t)p * ld;
  double* aq = A + (int64_t)q * ld;
  double alpha = 0.0, beta = 0.0, gamma = 0.0;
  for (int r = threadIdx.x; r < n; r += SV_THREADS) {
    const double x = ap[r], y = aq[r];
    alpha = fma(x, x, alpha); beta = fma(y, y, beta); gamma = fma(x, y, gamma);
  }
  alpha = block_sum(alpha, s_red);
  beta = block_sum(beta, s_red);
  gamma = block_sum(gamma, s_red);
  if (!(fabs(gamma) > tol * sqrt(alpha * beta))) return;            // orthogonal already (also: a zero column, NaN)
  // a column that has shrunk below 1e-15 of the largest initial column IS a null direction (its remaining entries are
  // rounding noise with no direction of their own: relative orthogonality against noise would never be reached)
  const double floor2 = 1e-30 * max_norm2[0];
  if (alpha < floor2 || beta < floor2) return;
  const double zeta = (beta - alpha) / (2.0 * gamma);
  const double t = copysign(1.0, zeta) / (fabs(zeta) + sqrt(fma(zeta, zeta, 1.0)));
  const double cs = rsqrt(fma(t, t, 1.0)), sn = cs * t;
  for (int r = threadIdx.x; r < n; r += SV_THREADS) {
    const double x = ap[r], y = aq[r];
    ap[r] = fma(cs, x, -sn * y);
    aq[r] = fma(sn, x, cs * y);
  }
  double* vp = V + (int64_t)p * ld;
  double* vq = V + (int64_t)q * ld;
  for (int r = threadIdx.x; r < n; r += SV_THREADS) {
    const double x = vp[r], y = vq[r];
    vp[r] = fma(cs, x, -sn * y);
    vq[r] = fma(sn, x, cs * y);
  }
  if (threadIdx.x == 0) atomicAdd(rotations, 1u);
}

// s2[j] = |a_j|^2; one CTA per column
__global__ void __launch_bounds__(SV_THREADS) svd_norms_kernel(const double* __restrict__ A, int64_t ld, int n, double* __restrict__ s2) {
  __shared__ double s_red[SV_THREADS / 32];
  const double* a = A + (int64_t)blockIdx.x * ld;
  double v = 0.0;
  for (int r = threadIdx.x; r < n; r += SV_THREADS) v = fma(a[r], a[r], v);
  v = block_sum(v, s_red);
  if (threadIdx.x == 0) s2[blockIdx.x] = v;
}

// s2[n] = max_j s2[j] (one CTA; max is order-independent)
__global__ void __launch_bounds__(1024) svd_max_kernel(double* s2, int n) {
  __shared__ double s_m[32];
  double v = 0.0;
  for (int j = threadIdx.x; j < n; j += 1024) v = fmax(v, s2[j]);
  for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
  if ((threadIdx.x & 31) == 0) s_m[threadIdx.x >> 5] = v;
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < 32; ++w) v = fmax(v, s_m[w]);
    s2[n] = v;
  }
}

// w[j] = (a_j . (rscale * b)) / s_j^2 where s_j > rcond s_max, else 0; one CTA per column
__global__ void __launch_bounds__(SV_THREADS) svd_weights_kernel(const double* __restrict__ A, int64_t ld, int n, const double* __restrict__ s2,
                                                                 double rcond2, const double* __restrict__ b, const double* __restrict__ rscale,
                                                                 double* __restrict__ w) {
  __shared__ double s_red[SV_THREADS / 32];
  const int j = blockIdx.x;
  const double* a = A + (int64_t)j * ld;
  double v = 0.0;
  for (int r = threadIdx.x; r < n; r += SV_THREADS) v = fma(a[r], b[r] * rscale[r], v);
  v = block_sum(v, s_red);
  if (threadIdx.x == 0) w[j] = (s2[j] > rcond2 * s2[n]) ? v / s2[j] : 0.0;
}

// x[i] = sum_j V[i][j] w[j]: CTA = 64 rows x 4 column groups, groups added in a fixed order
__global__ void __launch_bounds__(256) svd_apply_kernel(const double* __restrict__ V, int64_t ld, int n, const double* __restrict__ w,
                                                        double* __restrict__ x) {
  __shared__ double s_part[4][64];
  const int r = threadIdx.x & 63, cg = threadIdx.x >> 6;
  const int i = blockIdx.x * 64 + r;
  double a0 = 0.0, a1 = 0.0;
  if (i < n) {
    const int per = (n + 3) / 4, j0 = cg * per, j1 = min(n, j0 + per);
    int j = j0;
    for (; j + 1 < j1; j += 2) {
      a0 = fma(V[i + (int64_t)j * ld], w[j], a0);
      a1 = fma(V[i + (int64_t)(j + 1) * ld], w[j + 1], a1);
    }
    if (j < j1) a0 = fma(V[i + (int64_t)j * ld], w[j], a0);
  }
  s_part[cg][r] = a0 + a1;
  __syncthreads();
  if (cg == 0 && i < n) x[i] = (s_part[0][r] + s_part[1][r]) + (s_part[2][r] + s_part[3][r]);
}

}  // namespace

// One-sided Jacobi SVD of the row-scaled matrix in d_K (overwritten by U diag(s)); V and s^2 kept for the solves.
neb_status svd_factor(neb_ctx* c) {
  const int64_t npad = c->npad;
  if (npad > (1 << 30)) return fail(c, NEB_EINVAL, "OptSVD: n too large");
  StageTimer tt(c, NEB_STAGE_LU);
  if (!c->d_V) {
    NEB_CUDA(c, cudaMalloc((void**)&c->d_V, sizeof(double) * (size_t)npad * (size_t)npad));
    NEB_CUDA(c, cudaMalloc((void**)&c->d_s2, sizeof(double) * (size_t)(npad + 1)));
    NEB_CUDA(c, cudaMalloc((void**)&c->d_svd_w, sizeof(double) * (size_t)npad));
  }
  const int n = (int)npad;
  svd_identity_kernel<<<(unsigned)((npad * npad + 255) / 256), 256, 0, c->stream>>>(c->d_V, npad);
  c->launches++;
  unsigned int* d_rot = nullptr;
  NEB_CUDA(c, cudaMallocFromPoolAsync((void**)&d_rot, sizeof(unsigned int), c->pool, c->stream));
  svd_norms_kernel<<<n, SV_THREADS, 0, c->stream>>>(c->d_K, npad, n, c->d_s2);
  svd_max_kernel<<<1, 1024, 0, c->stream>>>(c->d_s2, n);      // d_s2[n] = largest squared column norm of the scaled matrix
  c->launches += 2;
  const double tol = 1e-15;
  constexpr int kMaxSweeps = 60;
  c->svd_sweeps = 0;
  bool converged = false;
  for (int sweep = 0; sweep < kMaxSweeps; ++sweep) {
    NEB_CUDA(c, cudaMemsetAsync(d_rot, 0, sizeof(unsigned int), c->stream));
    for (int r = 0; r < n - 1; ++r) {
      svd_round_kernel<<<n / 2, SV_THREADS, 0, c->stream>>>(c->d_K, c->d_V, npad, n, r, tol, c->d_s2 + n, d_rot);
      c->launches++;
    }
    unsigned int h_rot = 0;
    NEB_CUDA(c, cudaMemcpyAsync(&h_rot, d_rot, sizeof(unsigned int), cudaMemcpyDeviceToHost, c->stream));
    NEB_CUDA(c, cudaStreamSynchronize(c->stream));
    c->svd_sweeps = sweep + 1;
    if (h_rot == 0) { converged = true; break; }
  }
  cudaFreeAsync(d_rot, c->stream);
  if (!converged) return fail(c, NEB_ESINGULAR, "OptSVD: the Jacobi sweeps did not converge (NaN/inf in the matrix?)");
  svd_norms_kernel<<<n, SV_THREADS, 0, c->stream>>>(c->d_K, npad, n, c->d_s2);
  svd_max_kernel<<<1, 1024, 0, c->stream>>>(c->d_s2, n);
  c->launches += 2;
  NEB_CUDA(c, cudaGetLastError());
  return NEB_OK;
}

// d_out[k * npad + i] = the minimum-norm least-squares solution for right-hand side k (d_b unscaled, sorted order)
neb_status svd_solve(neb_ctx* c, const double* d_b, int nrhs, double* d_out) {
  const int64_t npad = c->npad;
  const int n = (int)npad;
  StageTimer tt(c, NEB_STAGE_TRISOLVE);
  const double rcond2 = c->svd_rcond * c->svd_rcond;
  for (int k = 0; k < nrhs; ++k) {
    svd_weights_kernel<<<n, SV_THREADS, 0, c->stream>>>(c->d_K, npad, n, c->d_s2, rcond2, d_b + (size_t)k * npad, c->d_rscale, c->d_svd_w);
    svd_apply_kernel<<<(n + 63) / 64, 256, 0, c->stream>>>(c->d_V, npad, n, c->d_svd_w, d_out + (size_t)k * npad);
    c->launches += 2;
  }
  NEB_CUDA(c, cudaGetLastError());
  return NEB_OK;
}

// The solve on whatever factors are resident: LU (two triangular solves) or SVD
neb_status factors_solve(neb_ctx* c, const double* d_b, int nrhs, double* d_out) {
  return c->factored_with == 1 ? svd_solve(c, d_b, nrhs, d_out) : lu_solve(c, d_b, nrhs, d_out);
}

}  // namespace neb
