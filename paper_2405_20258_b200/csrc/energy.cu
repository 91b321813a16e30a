// (a5) E_c = (1/2 pi) sum_k W_k Tr[ln(1 - chi_s(i w_k)) + chi_s(i w_k)]   (PAPER.md:35 eq. 1, :160, :174).
// Tr ln A = ln det A; 1 - chi_s is Hermitian positive definite (reading R10), so the determinant
// comes from a Cholesky factor: ln det = 2 sum_i ln L_ii.  All N_w matrices are factored as one batch.  The factor
// is taken of the deviation from the identity (see negate_kernel) so the integrand keeps full relative accuracy.
#include "rpa_internal.h"

namespace {

// W[k] = -chi_s[k]  (= (1 - chi_s[k]) - 1: the Cholesky below works on the deviation from the identity, so that
// t_k, which is O(|chi|^2) while ln det and Tr chi are each O(|chi|), is formed without cancellation)
__global__ void negate_kernel(const cplx* __restrict__ chi, long long total, cplx* __restrict__ W) {
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < total; i += (long long)gridDim.x * blockDim.x) {
    cplx x = chi[i];
    W[i] = make_double2(-x.x, -x.y);
  }
}

// With d_i = L_ii^2 - 1 (pivot deviations) and chi_ii = -d_i - sum_{j<i} |L_ij|^2:
//   t[k] = ln det(1 - chi) + Tr chi = sum_i [log1p(d_i) - d_i] - sum_{i>j} |L_ij|^2
__global__ void logdet_kernel(const cplx* __restrict__ L, int n, const double* __restrict__ dvec, double* __restrict__ t) {
  __shared__ double sh[32];
  const int k = blockIdx.x;
  const cplx* a = L + (long long)k * n * n;
  const double* d = dvec + (long long)k * n;
  double s = 0.0;
  for (int i = threadIdx.x; i < n; i += blockDim.x) s += log1p(d[i]) - d[i];
  for (long long idx = threadIdx.x; idx < (long long)n * n; idx += blockDim.x) {
    int i = (int)(idx / n), j = (int)(idx - (long long)i * n);
    if (j < i) { cplx x = a[idx]; s -= x.x * x.x + x.y * x.y; }
  }
  for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
  if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = s;
  __syncthreads();
  if (threadIdx.x < 32) {
    s = threadIdx.x < (blockDim.x >> 5) ? sh[threadIdx.x] : 0.0;
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (threadIdx.x == 0) t[k] = s;
  }
}

__global__ void quadrature_kernel(const double* __restrict__ t, const double* __restrict__ weight, int n_w, double* e) {
  if (threadIdx.x == 0 && blockIdx.x == 0) {
    double s = 0.0;
    for (int k = 0; k < n_w; k++) s += weight[k] * t[k];
    e[0] = s / (2.0 * 3.14159265358979323846);
  }
}

// X[k] = identity (n x n) for every matrix of the batch
__global__ void identity_kernel(cplx* __restrict__ X, int n, long long total) {
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < total; i += (long long)gridDim.x * blockDim.x) {
    const long long r = i % ((long long)n * n);
    X[i] = make_double2((r / n) == (r % n) ? 1.0 : 0.0, 0.0);
  }
}
__global__ void conj_kernel(cplx* __restrict__ X, long long total) {
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < total; i += (long long)gridDim.x * blockDim.x)
    X[i].y = -X[i].y;
}

}  // namespace

size_t energy_workspace_bytes(const rpa_ctx* ctx, int n_eig, int n_w) {
  (void)ctx;
  return ws_round((size_t)n_w * n_eig * n_eig * sizeof(cplx)) + 2 * ws_round((size_t)(n_w + 1) * sizeof(double)) + ws_round((size_t)n_w * n_eig * sizeof(double)) + 256;
}

int energy_run(rpa_ctx* ctx, WsAlloc& ws, const cplx* chi_s, int n_eig, const double* weight, int n_w, double* e_c,
               double* per_freq) {
  ProfScope prof_scope(ctx, RPA_PROF_ENERGY);
  cplx* W = ws.get<cplx>((size_t)n_w * n_eig * n_eig);
  double* dvec = ws.get<double>((size_t)n_w * n_eig);
  double* t = ws.get<double>(n_w + 1);
  int* info = ws.get<int>(n_w + 1);
  if (!ws.ok) return rpa_fail(ctx, RPA_ERR_WORKSPACE, "rpa_correlation_energy: workspace too small (need %zu bytes)", ws.off);
  negate_kernel<<<ctx->sm_count * 8, 256, 0, ctx->stream>>>(chi_s, (long long)n_w * n_eig * n_eig, W);
  RPA_LAUNCH_CHECK(ctx);
  int rc = zpotrf_batched(ctx, W, n_eig, n_eig, n_w, (long long)n_eig * n_eig, info, 1, dvec);
  if (rc) return rc;
  logdet_kernel<<<n_w, 1024, 0, ctx->stream>>>(W, n_eig, dvec, t);
  RPA_LAUNCH_CHECK(ctx);
  quadrature_kernel<<<1, 32, 0, ctx->stream>>>(t, weight, n_w, t + n_w);
  RPA_LAUNCH_CHECK(ctx);
  std::vector<double> th(n_w + 1);
  std::vector<int> ih(n_w);
  RPA_CUDA(ctx, cudaMemcpyAsync(th.data(), t, (n_w + 1) * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
  RPA_CUDA(ctx, cudaMemcpyAsync(ih.data(), info, n_w * sizeof(int), cudaMemcpyDeviceToHost, ctx->stream));
  RPA_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
  for (int k = 0; k < n_w; k++)
    if (ih[k] != 0)
      return rpa_fail(ctx, RPA_ERR_NOT_POSDEF, "1 - chi_s(i w_%d) is not positive definite (pivot %d): chi_s not negative-semidefinite",
                      k, ih[k]);
  *e_c = th[n_w];
  if (per_freq)
    for (int k = 0; k < n_w; k++) per_freq[k] = th[k];
  return RPA_OK;
}

// (next-3) eps_s^-1(i w_k) = (1 - chi_s(i w_k))^-1 from the same Cholesky factor as E_c (the factorisation
// "also gives eps^-1", kept for GW):  1 - chi_s = L L^H  =>  eps^-1 = L^-H L^-1 = X^H X with X = L^-1.
size_t epsinv_workspace_bytes(const rpa_ctx* ctx, int n_eig, int n_w) {
  (void)ctx;
  return 2 * ws_round((size_t)n_w * n_eig * n_eig * sizeof(cplx)) + ws_round((size_t)n_w * n_eig * sizeof(double)) + ws_round((size_t)(n_w + 1) * sizeof(int)) + 256;
}

int epsinv_run(rpa_ctx* ctx, WsAlloc& ws, const cplx* chi_s, int n, int n_w, cplx* eps_inv) {
  const long long nn = (long long)n * n;
  cplx* W = ws.get<cplx>((size_t)n_w * nn);
  cplx* X = ws.get<cplx>((size_t)n_w * nn);
  double* dvec = ws.get<double>((size_t)n_w * n);
  int* info = ws.get<int>(n_w + 1);
  if (!ws.ok) return rpa_fail(ctx, RPA_ERR_WORKSPACE, "rpa_epsilon_inverse: workspace too small (need %zu bytes)", ws.off);
  negate_kernel<<<ctx->sm_count * 8, 256, 0, ctx->stream>>>(chi_s, n_w * nn, W);
  RPA_LAUNCH_CHECK(ctx);
  int rc = zpotrf_batched(ctx, W, n, n, n_w, nn, info, 1, dvec);
  if (rc) return rc;
  identity_kernel<<<ctx->sm_count * 8, 256, 0, ctx->stream>>>(X, n, n_w * nn);
  RPA_LAUNCH_CHECK(ctx);
  for (int k = 0; k < n_w; k++)
    if ((rc = ztrsm_left_lower(ctx, W + k * nn, n, n, X + k * nn, n, n))) return rc;
  ZgemmParams g;   // R[m][n'] = sum_k X[k][m] conj(X[k][n']) = conj((X^H X)[m][n'])
  g.A = X; g.lda = n; g.a_km = true; g.B = X; g.ldb = n; g.b_kn = true; g.C = eps_inv; g.ldc = n;
  g.M = n; g.N = n; g.K = n; g.conj_b = true; g.herm = true;
  g.batch = n_w; g.strideA = nn; g.strideB = nn; g.strideC = nn;
  if ((rc = zgemm_dmma(ctx, g))) return rc;
  conj_kernel<<<ctx->sm_count * 8, 256, 0, ctx->stream>>>(eps_inv, n_w * nn);
  RPA_LAUNCH_CHECK(ctx);
  std::vector<int> ih(n_w);
  RPA_CUDA(ctx, cudaMemcpyAsync(ih.data(), info, n_w * sizeof(int), cudaMemcpyDeviceToHost, ctx->stream));
  RPA_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
  for (int k = 0; k < n_w; k++)
    if (ih[k] != 0)
      return rpa_fail(ctx, RPA_ERR_NOT_POSDEF, "1 - chi_s(i w_%d) is not positive definite (pivot %d)", k, ih[k]);
  return RPA_OK;
}
