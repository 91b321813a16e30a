// (a5) E_c = (1/2 pi) sum_k W_k Tr[ln(1 - chi_s(i w_k)) + chi_s(i w_k)]   (PAPER.md:35 eq. 1, :160, :174).
// Tr ln A = ln det A; 1 - chi_s is Hermitian positive definite (reading R10), so the determinant
// comes from a Cholesky factor: ln det = 2 sum_i ln L_ii.  All N_w matrices are factored as one batch.
#include "rpa_internal.h"

namespace {

// W[k] = 1 - chi_s[k];  tr[k] = Re Tr chi_s[k]
__global__ void one_minus_kernel(const cplx* __restrict__ chi, int n, cplx* __restrict__ W, double* __restrict__ tr) {
  const int k = blockIdx.y, i = blockIdx.x;
  const cplx* src = chi + ((long long)k * n + i) * n;
  cplx* dst = W + ((long long)k * n + i) * n;
  for (int j = threadIdx.x; j < n; j += blockDim.x) {
    cplx x = src[j];
    dst[j] = make_double2((i == j ? 1.0 : 0.0) - x.x, -x.y);
    if (i == j) atomicAdd(&tr[k], x.x);
  }
}

// t[k] = 2 sum_i ln L_ii + tr[k]; the last block to finish forms E_c = (1/2 pi) sum_k weight_k t_k
__global__ void logdet_kernel(const cplx* __restrict__ L, int n, const double* __restrict__ tr, double* __restrict__ t) {
  __shared__ double sh[32];
  const int k = blockIdx.x;
  const cplx* a = L + (long long)k * n * n;
  double s = 0.0;
  for (int i = threadIdx.x; i < n; i += blockDim.x) s += log(a[(long long)i * n + i].x);
  for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
  if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = s;
  __syncthreads();
  if (threadIdx.x < 32) {
    s = threadIdx.x < (blockDim.x >> 5) ? sh[threadIdx.x] : 0.0;
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (threadIdx.x == 0) t[k] = 2.0 * s + tr[k];
  }
}

__global__ void quadrature_kernel(const double* __restrict__ t, const double* __restrict__ weight, int n_w, double* e) {
  if (threadIdx.x == 0 && blockIdx.x == 0) {
    double s = 0.0;
    for (int k = 0; k < n_w; k++) s += weight[k] * t[k];
    e[0] = s / (2.0 * 3.14159265358979323846);
  }
}

}  // namespace

size_t energy_workspace_bytes(const rpa_ctx* ctx, int n_eig, int n_w) {
  (void)ctx;
  return ws_round((size_t)n_w * n_eig * n_eig * sizeof(cplx)) + 3 * ws_round((size_t)(n_w + 1) * sizeof(double)) + 256;
}

int energy_run(rpa_ctx* ctx, WsAlloc& ws, const cplx* chi_s, int n_eig, const double* weight, int n_w, double* e_c,
               double* per_freq) {
  cplx* W = ws.get<cplx>((size_t)n_w * n_eig * n_eig);
  double* tr = ws.get<double>(n_w + 1);
  double* t = ws.get<double>(n_w + 1);
  int* info = ws.get<int>(n_w + 1);
  if (!ws.ok) return rpa_fail(ctx, RPA_ERR_WORKSPACE, "rpa_correlation_energy: workspace too small (need %zu bytes)", ws.off);
  RPA_CUDA(ctx, cudaMemsetAsync(tr, 0, (n_w + 1) * sizeof(double), ctx->stream));
  dim3 grid(n_eig, n_w);
  one_minus_kernel<<<grid, 128, 0, ctx->stream>>>(chi_s, n_eig, W, tr);
  RPA_LAUNCH_CHECK(ctx);
  int rc = zpotrf_batched(ctx, W, n_eig, n_eig, n_w, (long long)n_eig * n_eig, info);
  if (rc) return rc;
  logdet_kernel<<<n_w, 256, 0, ctx->stream>>>(W, n_eig, tr, t);
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
