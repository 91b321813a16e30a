// Blocked complex-FP64 Cholesky (lower, in place, batched) and a blocked left triangular solve.
// Used by (a5) E_c: L L^H = 1 - chi_s(i omega_k) (PAPER.md:160 with reading R10: Hermitian positive definite, so
// Cholesky replaces the paper's LU; the determinant is the same) and by the CholeskyQR step of (a3).
// Right-looking: potf2 on a 64 x 64 diagonal block in one CTA, a warp-per-row panel solve, and the trailing
// Hermitian update on the DMMA GEMM (zgemm_dmma, herm + accumulate, alpha = -1).
#include "rpa_internal.h"

namespace {
constexpr int NB = 64;
constexpr int LDB = NB + 1;

__device__ __forceinline__ cplx cmulc(cplx a, cplx b) {  // a * conj(b)
  return make_double2(a.x * b.x + a.y * b.y, a.y * b.x - a.x * b.y);
}
__device__ __forceinline__ cplx cmul_(cplx a, cplx b) {
  return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}

// factor the nb x nb diagonal block at (k0,k0) of each matrix of the batch
// shift != 0: the stored diagonal is A_ii - 1 (deviation from the identity), pivots are 1 + stored, and the pivot
// deviations d_i = L_ii^2 - 1 go to dvec (so ln det = sum log1p(d_i) keeps full relative accuracy for A close to 1).
__global__ void __launch_bounds__(256) potf2_kernel(cplx* A, long long lda, long long stride, int k0, int nb, int* info,
                                                    int shift, double* dvec, long long dstride) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx* s = reinterpret_cast<cplx*>(smem_raw);  // [nb][LDB]
  cplx* a = A + blockIdx.x * stride + (long long)k0 * lda + k0;
  const int tid = threadIdx.x;
  for (int idx = tid; idx < nb * nb; idx += blockDim.x) {
    int i = idx / nb, j = idx - i * nb;
    s[i * LDB + j] = a[(long long)i * lda + j];
  }
  __syncthreads();
  for (int j = 0; j < nb; j++) {
    const double dev = s[j * LDB + j].x;
    double d = shift ? 1.0 + dev : dev;
    if (shift && dvec && tid == 0) dvec[blockIdx.x * dstride + k0 + j] = dev;
    if (!(d > 0.0)) {
      if (tid == 0 && info[blockIdx.x] == 0) info[blockIdx.x] = k0 + j + 1;
      d = 1.0;  // keep going with finite numbers; the caller reads info
    }
    const double r = sqrt(d), rinv = 1.0 / r;
    __syncthreads();
    if (tid == 0) s[j * LDB + j] = make_double2(r, 0.0);
    for (int i = j + 1 + tid; i < nb; i += blockDim.x) {
      cplx x = s[i * LDB + j];
      s[i * LDB + j] = make_double2(x.x * rinv, x.y * rinv);
    }
    __syncthreads();
    const int rem = nb - j - 1;
    for (int idx = tid; idx < rem * rem; idx += blockDim.x) {
      int i = j + 1 + idx / rem, k = j + 1 + idx % rem;
      if (k <= i) {
        cplx u = cmulc(s[i * LDB + j], s[k * LDB + j]);
        s[i * LDB + k].x -= u.x; s[i * LDB + k].y -= u.y;
      }
    }
    __syncthreads();
  }
  for (int idx = tid; idx < nb * nb; idx += blockDim.x) {
    int i = idx / nb, j = idx - i * nb;
    a[(long long)i * lda + j] = (j <= i) ? s[i * LDB + j] : make_double2(0.0, 0.0);
  }
}

// panel: rows i >= k0+nb of columns k0..k0+nb:  A21 <- A21 L11^{-H}.  One warp per row, L11 in shared memory.
__global__ void __launch_bounds__(256) panel_trsm_kernel(cplx* A, long long lda, long long stride, int n, int k0, int nb) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx* s = reinterpret_cast<cplx*>(smem_raw);  // L11 [nb][LDB]
  cplx* base = A + blockIdx.y * stride;
  const cplx* l11 = base + (long long)k0 * lda + k0;
  for (int idx = threadIdx.x; idx < nb * nb; idx += blockDim.x) {
    int i = idx / nb, j = idx - i * nb;
    s[i * LDB + j] = l11[(long long)i * lda + j];
  }
  __syncthreads();
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int row = k0 + nb + blockIdx.x * 8 + warp;
  if (row >= n) return;
  cplx* x = base + (long long)row * lda + k0;
  cplx x0 = lane < nb ? x[lane] : make_double2(0, 0);
  cplx x1 = lane + 32 < nb ? x[lane + 32] : make_double2(0, 0);
  for (int j = 0; j < nb; j++) {
    // finalise x[j], broadcast, update the columns t > j
    cplx xj = (j < 32) ? x0 : x1;
    const double dinv = 1.0 / s[j * LDB + j].x;
    xj.x *= dinv; xj.y *= dinv;
    xj.x = __shfl_sync(0xffffffffu, xj.x, j & 31);
    xj.y = __shfl_sync(0xffffffffu, xj.y, j & 31);
    if (lane == (j & 31)) { if (j < 32) x0 = xj; else x1 = xj; }
    if (lane > j && lane < nb) { cplx u = cmulc(xj, s[lane * LDB + j]); x0.x -= u.x; x0.y -= u.y; }
    if (lane + 32 > j && lane + 32 < nb) { cplx u = cmulc(xj, s[(lane + 32) * LDB + j]); x1.x -= u.x; x1.y -= u.y; }
  }
  if (lane < nb) x[lane] = x0;
  if (lane + 32 < nb) x[lane + 32] = x1;
}

// X_b <- L_bb^{-1} X_b for the nb rows starting at r0 of X [p][ncols]; one thread per column, TC columns per CTA.
constexpr int TC = 32;
__global__ void __launch_bounds__(TC) diag_solve_kernel(const cplx* L, long long ldl, cplx* X, long long ldx, int ncols, int r0,
                                                       int nb) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx* sl = reinterpret_cast<cplx*>(smem_raw);  // [nb][LDB]
  cplx* sx = sl + NB * LDB;                      // [nb][TC+1]
  const cplx* l = L + (long long)r0 * ldl + r0;
  for (int idx = threadIdx.x; idx < nb * nb; idx += blockDim.x) {
    int i = idx / nb, j = idx - i * nb;
    sl[i * LDB + j] = l[(long long)i * ldl + j];
  }
  const int c = blockIdx.x * TC + threadIdx.x;
  const bool ok = c < ncols;
  for (int i = 0; i < nb; i++) sx[i * (TC + 1) + threadIdx.x] = ok ? X[(long long)(r0 + i) * ldx + c] : make_double2(0, 0);
  __syncthreads();
  // row-oriented forward substitution: x_i = (b_i - sum_{k<i} L_ik x_k) / L_ii.  The sum only READS shared memory (the
  // column-oriented form updated every later row through shared memory, one dependent read-modify-write per term), with
  // two independent accumulator pairs.
  for (int i = 0; i < nb; i++) {
    double ar0 = 0.0, ai0 = 0.0, ar1 = 0.0, ai1 = 0.0;
    int k = 0;
    for (; k + 1 < i; k += 2) {
      const cplx l0 = sl[i * LDB + k], x0 = sx[k * (TC + 1) + threadIdx.x];
      const cplx l1 = sl[i * LDB + k + 1], x1 = sx[(k + 1) * (TC + 1) + threadIdx.x];
      ar0 += l0.x * x0.x - l0.y * x0.y; ai0 += l0.x * x0.y + l0.y * x0.x;
      ar1 += l1.x * x1.x - l1.y * x1.y; ai1 += l1.x * x1.y + l1.y * x1.x;
    }
    if (k < i) {
      const cplx l0 = sl[i * LDB + k], x0 = sx[k * (TC + 1) + threadIdx.x];
      ar0 += l0.x * x0.x - l0.y * x0.y; ai0 += l0.x * x0.y + l0.y * x0.x;
    }
    cplx xi = sx[i * (TC + 1) + threadIdx.x];
    const double dinv = 1.0 / sl[i * LDB + i].x;
    xi.x = (xi.x - (ar0 + ar1)) * dinv; xi.y = (xi.y - (ai0 + ai1)) * dinv;
    sx[i * (TC + 1) + threadIdx.x] = xi;
  }
  if (ok)
    for (int i = 0; i < nb; i++) X[(long long)(r0 + i) * ldx + c] = sx[i * (TC + 1) + threadIdx.x];
}
}  // namespace

// Lower Cholesky of `batch` Hermitian n x n matrices (row-major, lower triangle read), in place.  d_info[b] = 0 or
// 1 + the first column with a non-positive pivot.  shift/dvec: see potf2_kernel (dvec is [batch][n]).
int zpotrf_batched(rpa_ctx* ctx, cplx* A, int n, long long lda, int batch, long long stride, int* d_info, int shift,
                   double* dvec) {
  RPA_CUDA(ctx, cudaMemsetAsync(d_info, 0, batch * sizeof(int), ctx->stream));
  const size_t smem = (size_t)NB * LDB * sizeof(cplx);
  if (ctx->attr_once(RPA_ATTR_POTRF)) {
    RPA_CUDA(ctx, cudaFuncSetAttribute(potf2_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    RPA_CUDA(ctx, cudaFuncSetAttribute(panel_trsm_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  }
  for (int k0 = 0; k0 < n; k0 += NB) {
    const int nb = n - k0 < NB ? n - k0 : NB;
    potf2_kernel<<<batch, 256, smem, ctx->stream>>>(A, lda, stride, k0, nb, d_info, shift, dvec, (long long)n);
    RPA_LAUNCH_CHECK(ctx);
    const int rem = n - k0 - nb;
    if (rem <= 0) break;
    dim3 grid((rem + 7) / 8, batch);
    panel_trsm_kernel<<<grid, 256, smem, ctx->stream>>>(A, lda, stride, n, k0, nb);
    RPA_LAUNCH_CHECK(ctx);
    ZgemmParams g;
    g.A = A + (long long)(k0 + nb) * lda + k0; g.lda = lda; g.a_km = false;
    g.B = g.A; g.ldb = lda; g.b_kn = false;
    g.C = A + (long long)(k0 + nb) * lda + (k0 + nb); g.ldc = lda;
    g.M = rem; g.N = rem; g.K = nb; g.conj_b = true; g.herm = true; g.accumulate = true; g.alpha = -1.0;
    g.batch = batch; g.strideA = stride; g.strideB = stride; g.strideC = stride; g.split_k = 1;
    int rc = zgemm_dmma(ctx, g);
    if (rc) return rc;
  }
  return RPA_OK;
}

// X <- L^{-1} X, L lower triangular p x p (row-major), X [p][ncols] row-major.
int ztrsm_left_lower(rpa_ctx* ctx, const cplx* L, long long ldl, int p, cplx* X, long long ldx, int ncols) {
  const size_t smem = ((size_t)NB * LDB + (size_t)NB * (TC + 1)) * sizeof(cplx);
  if (ctx->attr_once(RPA_ATTR_TRSM))
    RPA_CUDA(ctx, cudaFuncSetAttribute(diag_solve_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  for (int r0 = 0; r0 < p; r0 += NB) {
    const int nb = p - r0 < NB ? p - r0 : NB;
    if (r0 > 0) {
      ZgemmParams g;
      g.A = L + (long long)r0 * ldl; g.lda = ldl; g.a_km = false;
      g.B = X; g.ldb = ldx; g.b_kn = true;
      g.C = X + (long long)r0 * ldx; g.ldc = ldx;
      g.M = nb; g.N = ncols; g.K = r0; g.conj_b = false; g.accumulate = true; g.alpha = -1.0; g.split_k = 1;
      int rc = zgemm_dmma(ctx, g);
      if (rc) return rc;
    }
    diag_solve_kernel<<<(ncols + TC - 1) / TC, TC, smem, ctx->stream>>>(L, ldl, X, ldx, ncols, r0, nb);
    RPA_LAUNCH_CHECK(ctx);
  }
  return RPA_OK;
}
