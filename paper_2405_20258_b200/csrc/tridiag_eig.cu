// Lowest eigenpairs of a Hermitian matrix by the classical dense route, all on the device:
//   (1) Householder tridiagonalisation  H = Q T Q^H  (unblocked, LAPACK zhetd2 'L' arithmetic) in ONE cooperative launch
//       with one pass over the trailing matrix and one grid-wide barrier per column,
//   (2) the n_eig smallest eigenvalues of the real symmetric tridiagonal T by bisection on the Sturm count,
//   (3) their eigenvectors by inverse iteration (tridiagonal LU with partial pivoting),
//   (4) back-transformation  c_i = Q z_i  (reflectors applied in reverse order; compact-WY blocks + DMMA GEMMs for n >= 1024),
// followed, in basis.cu, by a CholeskyQR clean-up.  Used by the basis stage (a3) whenever a part of the
// spectrum is wanted (4 N_eig <= 3 n, n <= 12800): a Jacobi sweep costs ~n dependent grid-wide rounds and 12 n^3 flop.
#include <algorithm>
#include <cooperative_groups.h>

#include "rpa_internal.h"

namespace cg = cooperative_groups;

namespace {

__device__ __forceinline__ double wsum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
// block-wide sums of NV doubles (256 threads), result in every thread
template <int NV>
__device__ __forceinline__ void bsum(double (&v)[NV], double* sh /* [NV][8] */) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
  for (int k = 0; k < NV; k++) { v[k] = wsum(v[k]); if (lane == 0) sh[k * 8 + warp] = v[k]; }
  __syncthreads();
#pragma unroll
  for (int k = 0; k < NV; k++) { double s = 0.0; for (int w = 0; w < 8; w++) s += sh[k * 8 + w]; v[k] = s; }
  __syncthreads();
}
__device__ __forceinline__ cplx cmulf(cplx a, cplx b) { return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }

// (1) A: n x n Hermitian, row-major, both triangles (destroyed).  Vh[k][:] = reflector v_k (v_k[j] = 0 for j <= k,
// v_k[k+1] = 1), tau[k]; T = tridiag(e, d, e).  256 threads per CTA, one warp per matrix row in the O(m^2) phase.
// Householder vector of x (x_0 = alpha, |x_1..|^2 = xn2), LAPACK zlarfg: H x = beta e_0, v = x / (alpha - beta) below the 1.
struct Reflector { cplx tau, sc; double beta; };
__device__ __forceinline__ Reflector make_reflector(double alr, double ali, double xn2) {
  Reflector r;
  r.tau = make_double2(0.0, 0.0); r.sc = make_double2(0.0, 0.0); r.beta = alr;
  if (xn2 > 0.0 || ali != 0.0) {
    const double nrm = sqrt(alr * alr + ali * ali + xn2);
    r.beta = alr >= 0.0 ? -nrm : nrm;
    r.tau = make_double2((r.beta - alr) / r.beta, -ali / r.beta);
    const double dr = alr - r.beta, di = ali, den = dr * dr + di * di;     // 1 / (alpha - beta)
    r.sc = make_double2(dr / den, -di / den);
  }
  return r;
}

// block-wide sums for any block size (<= 1024 threads), result in every thread
template <int NV>
__device__ __forceinline__ void bsumx(double (&v)[NV], double* sh /* [NV][32] */) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwc = blockDim.x >> 5;
#pragma unroll
  for (int k = 0; k < NV; k++) { v[k] = wsum(v[k]); if (lane == 0) sh[k * 32 + warp] = v[k]; }
  __syncthreads();
#pragma unroll
  for (int k = 0; k < NV; k++) { double s = 0.0; for (int w = 0; w < nwc; w++) s += sh[k * 32 + w]; v[k] = s; }
  __syncthreads();
}
// column chunks a row of the trailing matrix (m rows) is split into, so that all nw warps of the grid have work when
// m < nw; each chunk leaves a partial sum of p_next (summed in a fixed order by the readers: deterministic)
constexpr int HT_CMAX = 8;
template <int MODE>
__device__ __host__ __forceinline__ int ht_chunks(int m, int nw, int cmax) {
  if (MODE != 0 || m < 1) return 1;                           // modes 1, 2 read p in the inner loop: one chunk
  int c = nw / m;                                             // (balancing the rounds of the slowest warp instead was slower)
  c = c < m / 64 ? c : m / 64;                                // at least 64 columns per chunk
  return c < 1 ? 1 : c > cmax ? cmax : c;
}

// (1') the same reduction with ONE pass over the trailing matrix and ONE grid-wide barrier per column: while a warp applies
// the rank-2 update of column k to its row, it also accumulates that row's product with the NEXT reflector v_{k+1}, which
// every CTA has formed beforehand from the updated row k+1 (one row: cheap, redundant).  MODE 0: v, v_next, w in shared
// memory; 1: v, v_next (w_j = p_j + al2 v_j on the fly); 2: v_next only (v read back from Vh).
// MODE 3 (n <= 32 HT_RMAX, one warp per matrix row, 256 threads): as mode 0, but every warp keeps ITS row of the trailing
// matrix in registers for the whole reduction (lane l holds columns l, l + 32, ...), so the rank-2 update and the product
// with the next reflector touch no memory but the shared-memory vectors; only the row the next column needs is written
// back (to A, where every CTA reads it after the barrier).
constexpr int HT_RMAX = 24;
template <int MODE>
__global__ void __launch_bounds__(MODE == 3 ? 256 : 1024) hetrd_fused_kernel(cplx* __restrict__ A, int n, cplx* __restrict__ Vh, cplx* __restrict__ tau,
                                                          double* __restrict__ d, double* __restrict__ e, cplx* __restrict__ P /* [2][HT_CMAX][n] */, int cmax) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx* buf0 = reinterpret_cast<cplx*>(smem_raw);            // v_next / v alternate between buf0 and buf1 (MODE 2: buf0 only)
  cplx* buf1 = buf0 + n;
  cplx* w = buf0 + 2 * n;                                    // MODE 0, 3
  __shared__ double sh[2 * 32];
  cg::grid_group grid = cg::this_grid();
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int nthr = blockDim.x, nwc = nthr >> 5;
  const int gw = blockIdx.x * nwc + warp, nw = gridDim.x * nwc;
  if (n < 2) { if (blockIdx.x == 0 && tid == 0) { d[0] = A[0].x; e[0] = 0.0; } return; }
  // ---- prologue: v_0 from row 0, p_0 = tau_0 A22 v_0
  cplx* v = MODE == 2 ? nullptr : buf0;
  cplx* vn = MODE == 2 ? buf0 : buf1;
  cplx t;
  {
    double s[1] = {0.0};
    for (int i = 2 + tid; i < n; i += nthr) { const cplx x = __ldcg(A + i); s[0] += x.x * x.x + x.y * x.y; }
    bsumx<1>(s, sh);
    const cplx a0 = __ldcg(A + 1);
    const Reflector r = make_reflector(a0.x, -a0.y, s[0]);
    t = r.tau;
    cplx* v0 = buf0;
    for (int i = tid; i < n; i += nthr) {
      cplx vi = make_double2(0.0, 0.0);
      if (i == 1) vi = make_double2(1.0, 0.0);
      else if (i > 1) { const cplx x = __ldcg(A + i); vi = cmulf(make_double2(x.x, -x.y), r.sc); }
      v0[i] = vi;
    }
    __syncthreads();
    if (blockIdx.x == 0) {
      for (int i = tid; i < n; i += nthr) Vh[i] = v0[i];
      if (tid == 0) { tau[0] = t; e[0] = r.beta; d[0] = __ldcg(A).x; }
    }
    for (int i = 1 + gw; i < n; i += nw) {
      const cplx* ri = A + (long long)i * n;
      double pr = 0.0, pi = 0.0;
      for (int j = 1 + lane; j < n; j += 32) { const cplx a = __ldcg(ri + j), b = v0[j]; pr += a.x * b.x - a.y * b.y; pi += a.x * b.y + a.y * b.x; }
      pr = wsum(pr); pi = wsum(pi);
      if (lane == 0) P[i] = cmulf(t, make_double2(pr, pi));    // chunk 0 of buffer 0
    }
    grid.sync();
  }
  cplx areg[MODE == 3 ? HT_RMAX : 1];
  if (MODE == 3 && gw < n) {
#pragma unroll
    for (int r = 0; r < HT_RMAX; r++) {
      const int j = lane + 32 * r;
      areg[r] = j < n ? __ldcg(A + (long long)gw * n + j) : make_double2(0.0, 0.0);
    }
  }
  for (int k = 0; k + 1 < n; k++) {
    // p_k = sum of the partial sums the row chunks of the last pass left; p_{k+1} goes to the other half (CTAs are not in step)
    const cplx* pk = P + (size_t)(k & 1) * HT_CMAX * n;
    cplx* pnext = P + (size_t)((k + 1) & 1) * HT_CMAX * n;
    const int cprev = k == 0 ? 1 : ht_chunks<MODE>(n - k - 1, nw, cmax), ccur = ht_chunks<MODE>(n - k - 2, nw, cmax);
    auto pval = [&](int i) -> cplx {
      cplx x = __ldcg(pk + i);
      for (int c = 1; c < cprev; c++) { const cplx y = __ldcg(pk + (size_t)c * n + i); x.x += y.x; x.y += y.y; }
      return x;
    };
    // MODE 3: this thread's elements of row k+1 (needed after the reductions below) are requested now, so their L2 round
    // trip overlaps the one of p_k
    cplx r1pre[MODE == 3 ? (32 * HT_RMAX + 255) / 256 : 1];
    if (MODE == 3) {
#pragma unroll
      for (int m = 0; m < (32 * HT_RMAX + 255) / 256; m++) {
        const int j = k + 1 + tid + m * 256;
        r1pre[m] = j < n ? __ldcg(A + (long long)(k + 1) * n + j) : make_double2(0.0, 0.0);
      }
    }
    const cplx* vrow = Vh + (long long)k * n;                 // MODE 2: v_k as written by CTA 0 one barrier ago
    auto vval = [&](int i) -> cplx { return MODE == 2 ? vrow[i] : v[i]; };
    // ---- w = p - (tau/2) (p^H v) v
    double q[2] = {0.0, 0.0};
    for (int i = k + 1 + tid; i < n; i += nthr) {
      const cplx x = pval(i), b = vval(i);
      if (MODE == 0 || MODE == 3) w[i] = x;                    // p stays in shared memory for the second loop (same thread)
      q[0] += x.x * b.x + x.y * b.y; q[1] += x.x * b.y - x.y * b.x;
    }
    bsumx<2>(q, sh);
    const cplx al2 = cmulf(make_double2(-0.5 * t.x, -0.5 * t.y), make_double2(q[0], q[1]));
    if (MODE == 0 || MODE == 3) {
      for (int i = k + 1 + tid; i < n; i += nthr) { const cplx x = w[i], av = cmulf(al2, v[i]); w[i] = make_double2(x.x + av.x, x.y + av.y); }
      __syncthreads();
    }
    auto wval = [&](int i) -> cplx {
      if (MODE == 0 || MODE == 3) return w[i];
      const cplx x = pval(i), av = cmulf(al2, vval(i));
      return make_double2(x.x + av.x, x.y + av.y);
    };
    const bool upd = t.x != 0.0 || t.y != 0.0;
    auto updated = [&](cplx a, cplx vi, cplx wi, cplx vj, cplx wj) -> cplx {   // a - v_i conj(w_j) - w_i conj(v_j)
      if (upd) {
        a.x -= vi.x * wj.x + vi.y * wj.y + wi.x * vj.x + wi.y * vj.y;
        a.y -= vi.y * wj.x - vi.x * wj.y + wi.y * vj.x - wi.x * vj.y;
      }
      return a;
    };
    // ---- the updated row k+1 -> next reflector (every CTA, redundantly)
    const int k1 = k + 1;
    cplx tn = make_double2(0.0, 0.0);
    {
      const cplx* r1 = A + (long long)k1 * n;
      const cplx vi = vval(k1), wi = wval(k1);
      double s[1] = {0.0};
      if (MODE == 3) {
#pragma unroll
        for (int m = 0; m < (32 * HT_RMAX + 255) / 256; m++) {
          const int j = k1 + tid + m * 256;
          if (j < n) {
            const cplx a = updated(r1pre[m], vi, wi, vval(j), wval(j));
            vn[j] = a;
            if (j >= k1 + 2) s[0] += a.x * a.x + a.y * a.y;
          }
        }
      }
      for (int j = k1 + tid; MODE != 3 && j < n; j += nthr) {
        const cplx a = updated(__ldcg(r1 + j), vi, wi, vval(j), wval(j));
        vn[j] = a;
        if (j >= k1 + 2) s[0] += a.x * a.x + a.y * a.y;
      }
      bsumx<1>(s, sh);                                          // (its barriers also order the vn writes)
      const double dk1 = vn[k1].x;
      Reflector r; r.tau = make_double2(0.0, 0.0); r.sc = r.tau; r.beta = 0.0;
      if (k1 + 1 < n) { const cplx a0 = vn[k1 + 1]; r = make_reflector(a0.x, -a0.y, s[0]); }
      tn = r.tau;
      __syncthreads();
      for (int i = tid; i < n; i += nthr) {
        cplx vi2 = make_double2(0.0, 0.0);
        if (i == k1 + 1) vi2 = make_double2(1.0, 0.0);
        else if (i > k1 + 1) { const cplx x = vn[i]; vi2 = cmulf(make_double2(x.x, -x.y), r.sc); }
        vn[i] = vi2;
      }
      __syncthreads();
      if (blockIdx.x == 0) {
        if (k1 + 1 < n) for (int i = tid; i < n; i += nthr) Vh[(long long)k1 * n + i] = vn[i];
        if (tid == 0) { d[k1] = dk1; e[k1] = k1 + 1 < n ? r.beta : 0.0; if (k1 + 1 < n) tau[k1] = tn; }
      }
    }
    if (k1 + 1 >= n) break;
    // ---- A22 -= v w^H + w v^H and p_next = tau_next A22' v_next in the same pass (warp per row; row k+1 is dead)
    if (MODE == 3) {
      const int i = gw;                                        // this warp's row, resident in areg
      if (i > k1 && i < n) {
        const cplx vi = v[i], wi = w[i];
        double pr = 0.0, pi = 0.0;
#pragma unroll
        for (int r = 0; r < HT_RMAX; r++) {
          const int j = lane + 32 * r;
          if (j > k1 && j < n) {
            const cplx a = updated(areg[r], vi, wi, v[j], w[j]);
            areg[r] = a;
            if (i == k1 + 1) __stcg(A + (long long)i * n + j, a);   // the row the next column's reflector is formed from
            const cplx b = vn[j];
            pr += a.x * b.x - a.y * b.y; pi += a.x * b.y + a.y * b.x;
          }
        }
        pr = wsum(pr); pi = wsum(pi);
        if (lane == 0) pnext[i] = cmulf(tn, make_double2(pr, pi));
      }
    }
    const int m = n - k1 - 1, clen = ((m + ccur - 1) / ccur + 31) & ~31;     // rows (= columns) k1+1 .. n-1 in ccur column chunks
    for (long long task = gw; MODE != 3 && task < (long long)m * ccur; task += nw) {
      const int i = k1 + 1 + (int)(task / ccur), c = (int)(task % ccur);
      const int j0 = k1 + 1 + c * clen, j1 = min(n, j0 + clen);
      cplx* ri = A + (long long)i * n;
      const cplx vi = vval(i), wi = wval(i);
      double pr = 0.0, pi = 0.0;
#pragma unroll 4
      for (int j = j0 + lane; j < j1; j += 32) {
        const cplx a = updated(__ldcg(ri + j), vi, wi, vval(j), wval(j));
        __stcg(ri + j, a);
        const cplx b = vn[j];
        pr += a.x * b.x - a.y * b.y; pi += a.x * b.y + a.y * b.x;
      }
      pr = wsum(pr); pi = wsum(pi);
      if (lane == 0) pnext[(size_t)c * n + i] = cmulf(tn, make_double2(pr, pi));
    }
    grid.sync();
    t = tn;
    if (MODE == 2) { /* v_next stays in buf0; v is read from Vh */ }
    else { cplx* tmp = v; v = vn; vn = tmp; }
  }
}

}  // namespace

namespace {

// (2) lam[i] = i-th smallest eigenvalue of T, i < n_eig: bisection on the Sturm count (one thread per eigenvalue)
__global__ void __launch_bounds__(256) bisect_kernel(const double* __restrict__ d, const double* __restrict__ e, int n, int n_eig,
                                                     double* __restrict__ lam, double* __restrict__ tnorm) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  double* sd = reinterpret_cast<double*>(smem_raw);   // [n]
  double* se2 = sd + n;                               // [n] e_j^2
  __shared__ double s_gl, s_gu, s_piv;
  for (int j = threadIdx.x; j < n; j += blockDim.x) { sd[j] = d[j]; const double x = j + 1 < n ? e[j] : 0.0; se2[j] = x * x; }
  __syncthreads();
  if (threadIdx.x == 0) {
    double gl = sd[0], gu = sd[0], emax = 0.0;
    for (int j = 0; j < n; j++) {
      const double r = (j > 0 ? sqrt(se2[j - 1]) : 0.0) + (j + 1 < n ? sqrt(se2[j]) : 0.0);
      gl = fmin(gl, sd[j] - r); gu = fmax(gu, sd[j] + r); emax = fmax(emax, se2[j]);
    }
    const double tn = fmax(fabs(gl), fabs(gu));
    s_gl = gl - 2.2e-16 * tn * n - 1e-300; s_gu = gu + 2.2e-16 * tn * n + 1e-300;
    s_piv = 2.3e-308 * fmax(1.0, emax);
    if (blockIdx.x == 0) tnorm[0] = tn;
  }
  __syncthreads();
  // one warp per eigenvalue: 32 trial points per step (the interval shrinks 33-fold per Sturm sweep)
  const int lane = threadIdx.x & 31;
  const int idx = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  if (idx >= n_eig) return;
  double lo = s_gl, hi = s_gu;
  const double piv = s_piv;
  for (int it = 0; it < 40; it++) {
    const double h = (hi - lo) / 33.0;
    if (hi - lo <= 2.0 * 2.2e-16 * fmax(fabs(lo), fabs(hi)) + 2.0 * piv || !(h > 0.0)) break;
    const double x = lo + h * (lane + 1);
    double q = sd[0] - x;
    int c = q < 0.0;
    for (int j = 1; j < n; j++) {
      if (fabs(q) < piv) q = -piv;
      q = sd[j] - x - se2[j - 1] / q;
      c += q < 0.0;
    }
    const unsigned m = __ballot_sync(0xffffffffu, c >= idx + 1);   // counts are monotone in x: a suffix of lanes
    const int first = m ? __ffs(m) - 1 : 32;
    const double nlo = first == 0 ? lo : lo + h * first, nhi = first == 32 ? hi : lo + h * (first + 1);
    lo = nlo; hi = nhi;
  }
  if (lane == 0) lam[idx] = 0.5 * (lo + hi);
}

// (3) z_i = eigenvector of T for lam[i] by inverse iteration.  The solves are sequential in j, so what matters is the
// latency of a step: IV_NT eigenvectors per CTA (one lane each), their LU factors in shared memory, layout [6][n][IV_NT].
constexpr int IV_NT = 4;
// element stride of the factor arrays: int in shared memory (a 64-bit stride there gave wrong vectors at n = 146, 147 with nvcc 12.9)
template <bool SMEM> struct IvStride { using type = long long; };
template <> struct IvStride<true> { using type = int; };
template <bool SMEM>   // SMEM: launched with 32 threads, IV_NT of them active; otherwise 128 threads, gws = [6][n][n_eig]
__global__ void __launch_bounds__(SMEM ? 32 : 128) invit_kernel(const double* __restrict__ d, const double* __restrict__ e, int n, int n_eig,
                             const double* __restrict__ lam, const double* __restrict__ tnorm, double* __restrict__ gws,
                             cplx* __restrict__ Z) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int idx = SMEM ? blockIdx.x * IV_NT + threadIdx.x : blockIdx.x * blockDim.x + threadIdx.x;
  if ((SMEM && threadIdx.x >= IV_NT) || idx >= n_eig) return;
  const typename IvStride<SMEM>::type S = SMEM ? IV_NT : n_eig;
  double* dl = SMEM ? reinterpret_cast<double*>(smem_raw) + threadIdx.x : gws + idx;   // multipliers  dl[j] at dl[j * S]
  double* dd = dl + (long long)n * S;      // U diagonal
  double* du = dd + (long long)n * S;      // U first superdiagonal
  double* du2 = du + (long long)n * S;     // U second superdiagonal
  double* pv = du2 + (long long)n * S;     // 1.0 if rows j, j+1 were swapped
  double* x = pv + (long long)n * S;       // the iterate
  const double tn = fmax(tnorm[0], 1e-300), eps = 2.2e-16;
  // a tiny index-dependent shift keeps (numerically) equal eigenvalues from giving identical vectors
  const double sigma = lam[idx] + eps * tn * (double)((idx % 7) - 3);
  for (int j = 0; j < n; j++) { dd[j * S] = d[j] - sigma; du[j * S] = j + 1 < n ? e[j] : 0.0; dl[j * S] = j + 1 < n ? e[j] : 0.0; du2[j * S] = 0.0; }
  // LU with partial pivoting (dgttrf)
  for (int j = 0; j + 1 < n; j++) {
    const double dj = dd[j * S], lj = dl[j * S];
    if (fabs(dj) >= fabs(lj)) {
      double piv = dj;
      if (piv == 0.0) { piv = eps * tn; dd[j * S] = piv; }
      const double f = lj / piv;
      dl[j * S] = f; pv[j * S] = 0.0;
      dd[(j + 1) * S] -= f * du[j * S];
    } else {
      const double f = dj / lj;
      dd[j * S] = lj; dl[j * S] = f; pv[j * S] = 1.0;
      const double t = du[j * S];
      du[j * S] = dd[(j + 1) * S];
      dd[(j + 1) * S] = t - f * dd[(j + 1) * S];
      if (j + 2 < n) { du2[j * S] = du[(j + 1) * S]; du[(j + 1) * S] = -f * du[(j + 1) * S]; }
    }
  }
  if (dd[(n - 1) * S] == 0.0) dd[(n - 1) * S] = eps * tn;
  // start vector: deterministic pseudo-random signs
  for (int j = 0; j < n; j++) {
    unsigned h = (unsigned)(j * 2654435761u) ^ (unsigned)(idx * 40503u + 12345u);
    h ^= h >> 15; h *= 2246822519u; h ^= h >> 13;
    x[j * S] = 0.5 + (double)(h & 0xffff) * (1.0 / 65536.0);
  }
  for (int iter = 0; iter < 3; iter++) {
    // forward (L with the row interchanges)
    for (int j = 0; j + 1 < n; j++) {
      if (pv[j * S] == 0.0) x[(j + 1) * S] -= dl[j * S] * x[j * S];
      else { const double t = x[j * S]; x[j * S] = x[(j + 1) * S]; x[(j + 1) * S] = t - dl[j * S] * x[j * S]; }
    }
    // back substitution (U)
    x[(n - 1) * S] /= dd[(n - 1) * S];
    if (n > 1) x[(n - 2) * S] = (x[(n - 2) * S] - du[(n - 2) * S] * x[(n - 1) * S]) / dd[(n - 2) * S];
    for (int j = n - 3; j >= 0; j--) x[j * S] = (x[j * S] - du[j * S] * x[(j + 1) * S] - du2[j * S] * x[(j + 2) * S]) / dd[j * S];
    // normalise (max norm first: the solve amplifies by ~1/eps)
    double mx = 0.0;
    for (int j = 0; j < n; j++) mx = fmax(mx, fabs(x[j * S]));
    const double r = mx > 0.0 ? 1.0 / mx : 1.0;
    double s2 = 0.0;
    for (int j = 0; j < n; j++) { const double t = x[j * S] * r; x[j * S] = t; s2 += t * t; }
    const double r2 = s2 > 0.0 ? 1.0 / sqrt(s2) : 1.0;
    for (int j = 0; j < n; j++) x[j * S] *= r2;
  }
  for (int j = 0; j < n; j++) Z[(long long)idx * n + j] = make_double2(x[j * S], 0.0);
}

// (4) rows of Z <- Q z:  y <- H_0 H_1 ... H_{n-2} y,  H_k = I - tau_k v_k v_k^H.  NV vectors per CTA, kept in shared memory.
constexpr int BT_NV = 1;      // vectors per CTA (300 vectors -> 300 CTAs, two per SM)
constexpr int BT_NE = 4;      // elements of a reflector per thread: n <= 1024 (larger matrices take the blocked route)
__global__ void __launch_bounds__(256) backtransform_kernel(const cplx* __restrict__ Vh, const cplx* __restrict__ tau, int n, int n_eig,
                                                            cplx* __restrict__ Z) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx* y = reinterpret_cast<cplx*>(smem_raw);   // [BT_NV][n]
  __shared__ double sh[2 * BT_NV * 8];
  const int tid = threadIdx.x, v0 = blockIdx.x * BT_NV, nv = min(BT_NV, n_eig - v0);
  for (int idx = tid; idx < BT_NV * n; idx += 256) {
    const int u = idx / n, j = idx - u * n;
    y[idx] = u < nv ? Z[(long long)(v0 + u) * n + j] : make_double2(0.0, 0.0);
  }
  __syncthreads();
  // The elements of v_k this thread needs (at most BT_NE: the kernel serves n < 1024) live in registers for both phases, and
  // v_{k-1}, tau_{k-1} are requested before the reduction of reflector k, so their L2 round trip hides behind it.
  cplx vcur[BT_NE], tcur;
  auto loadv = [&](int k, cplx (&v)[BT_NE], cplx& t) {
    t = k >= 0 ? tau[k] : make_double2(0.0, 0.0);
#pragma unroll
    for (int m = 0; m < BT_NE; m++) {
      const int j = k + 1 + tid + 256 * m;
      v[m] = (k >= 0 && j < n) ? Vh[(long long)k * n + j] : make_double2(0.0, 0.0);
    }
  };
  loadv(n - 2, vcur, tcur);
  for (int k = n - 2; k >= 0; k--) {
    cplx vnx[BT_NE], tnx;
    loadv(k - 1, vnx, tnx);
    const cplx t = tcur;
    if (t.x != 0.0 || t.y != 0.0) {
      double s[2 * BT_NV];
#pragma unroll
      for (int u = 0; u < 2 * BT_NV; u++) s[u] = 0.0;
#pragma unroll
      for (int m = 0; m < BT_NE; m++) {
        const int j = k + 1 + tid + 256 * m;
        if (j < n) {
          const cplx v = vcur[m];
#pragma unroll
          for (int u = 0; u < BT_NV; u++) { const cplx yy = y[u * n + j]; s[2 * u] += v.x * yy.x + v.y * yy.y; s[2 * u + 1] += v.x * yy.y - v.y * yy.x; }
        }
      }
      bsum<2 * BT_NV>(s, sh);
#pragma unroll
      for (int m = 0; m < BT_NE; m++) {
        const int j = k + 1 + tid + 256 * m;
        if (j < n) {
          const cplx v = vcur[m];
#pragma unroll
          for (int u = 0; u < BT_NV; u++) {
            const cplx f = cmulf(t, make_double2(s[2 * u], s[2 * u + 1]));     // tau (v^H y)
            const cplx g = cmulf(f, v);
            y[u * n + j].x -= g.x; y[u * n + j].y -= g.y;
          }
        }
      }
      __syncthreads();
    }
#pragma unroll
    for (int m = 0; m < BT_NE; m++) vcur[m] = vnx[m];
    tcur = tnx;
  }
  for (int idx = tid; idx < nv * n; idx += 256) {
    const int u = idx / n, j = idx - u * n;
    Z[(long long)(v0 + u) * n + j] = y[idx];
  }
}

}  // namespace

namespace {
// Compact-WY factor of a block of nb reflectors (LAPACK zlarft, forward / columnwise):  H_k0 ... H_k0+nb-1 = I - V T V^H.
// G[r][s] = sum_j v_r[j] conj(v_s[j]) (Gram of the block).  Writes Tc = conj(T), row-major [nb][ldt], zero below the diagonal.
__global__ void __launch_bounds__(256) larft_kernel(const cplx* __restrict__ G, int ldg, const cplx* __restrict__ tau, int nb,
                                                    cplx* __restrict__ Tc, int ldt) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx (*T)[65] = reinterpret_cast<cplx (*)[65]>(smem_raw);   // [64][65]
  cplx* x = reinterpret_cast<cplx*>(smem_raw) + 64 * 65;      // [64]
  const int tid = threadIdx.x;
  for (int idx = tid; idx < nb * nb; idx += 256) T[idx / nb][idx % nb] = make_double2(0.0, 0.0);
  __syncthreads();
  for (int i = 0; i < nb; i++) {
    const cplx ti = tau[i];
    if (tid < i) x[tid] = G[(long long)i * ldg + tid];          // (V^H v_i)[s] = G[i][s]
    __syncthreads();
    if (tid < i) {                                              // T[0:i, i] = -tau_i T[0:i, 0:i] x
      cplx acc = make_double2(0.0, 0.0);
      for (int s = tid; s < i; s++) { const cplx a = T[tid][s], b = x[s]; acc.x += a.x * b.x - a.y * b.y; acc.y += a.x * b.y + a.y * b.x; }
      T[tid][i] = make_double2(-(ti.x * acc.x - ti.y * acc.y), -(ti.x * acc.y + ti.y * acc.x));
    }
    if (tid == 0) T[i][i] = ti;
    __syncthreads();
  }
  for (int idx = tid; idx < nb * nb; idx += 256) { const cplx a = T[idx / nb][idx % nb]; Tc[(long long)(idx / nb) * ldt + idx % nb] = make_double2(a.x, -a.y); }
}
}  // namespace

// rows of Y [n_eig][n] <- Q y with Q = H_0 ... H_{n-2}, blocked: three DMMA GEMMs per block of 64 reflectors.
// Wk: scratch of n_eig * 64 * 2 + 64 * 64 * 2 complex numbers.
static int backtransform_wy(rpa_ctx* ctx, const cplx* Vh, const cplx* tau, int n, int n_eig, cplx* Y, cplx* Wk) {
  const int NBK = 64;
  cplx* W = Wk;
  cplx* U = W + (size_t)n_eig * NBK;
  cplx* G = U + (size_t)n_eig * NBK;
  cplx* Tc = G + NBK * NBK;
  const int nref = n - 1;
  RPA_CUDA(ctx, cudaFuncSetAttribute(larft_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 96 * 1024));
  for (int k0 = ((nref - 1) / NBK) * NBK; k0 >= 0; k0 -= NBK) {
    const int nb = std::min(NBK, nref - k0);
    const cplx* Vb = Vh + (long long)k0 * n;
    int rc;
    ZgemmParams g;   // G = Vb Vb^H
    g.A = Vb; g.lda = n; g.a_km = false; g.B = Vb; g.ldb = n; g.b_kn = false; g.C = G; g.ldc = NBK;
    g.M = nb; g.N = nb; g.K = n; g.conj_b = true; g.herm = true;
    if ((rc = zgemm_dmma(ctx, g))) return rc;
    larft_kernel<<<1, 256, (64 * 65 + 64) * sizeof(cplx), ctx->stream>>>(G, NBK, tau + k0, nb, Tc, NBK);
    RPA_LAUNCH_CHECK(ctx);
    ZgemmParams w;   // W[i][r] = sum_j Y[i][j] conj(Vb[r][j])  = (V^H y_i)[r]
    w.A = Y; w.lda = n; w.a_km = false; w.B = Vb; w.ldb = n; w.b_kn = false; w.C = W; w.ldc = NBK;
    w.M = n_eig; w.N = nb; w.K = n; w.conj_b = true;
    if ((rc = zgemm_dmma(ctx, w))) return rc;
    ZgemmParams u;   // U[i][r] = sum_s W[i][s] T[r][s]  (B = conj(T), conjugated again by the kernel)
    u.A = W; u.lda = NBK; u.a_km = false; u.B = Tc; u.ldb = NBK; u.b_kn = false; u.C = U; u.ldc = NBK;
    u.M = n_eig; u.N = nb; u.K = nb; u.conj_b = true; u.split_k = 1;
    if ((rc = zgemm_dmma(ctx, u))) return rc;
    ZgemmParams y;   // Y[i][j] -= sum_r U[i][r] Vb[r][j]
    y.A = U; y.lda = NBK; y.a_km = false; y.B = Vb; y.ldb = n; y.b_kn = true; y.C = Y; y.ldc = n;
    y.M = n_eig; y.N = n; y.K = nb; y.conj_b = false; y.accumulate = true; y.alpha = -1.0; y.split_k = 1;
    if ((rc = zgemm_dmma(ctx, y))) return rc;
  }
  return RPA_OK;
}

size_t tridiag_workspace_bytes(int n, int n_eig) {
  size_t b = ws_round((size_t)n * sizeof(cplx)) + ws_round((size_t)2 * HT_CMAX * n * sizeof(cplx)) + ws_round((size_t)n * sizeof(double)) * 2 + 1024;
  if ((size_t)6 * n * IV_NT * sizeof(double) > 200 * 1024) b += ws_round((size_t)6 * n * n_eig * sizeof(double));   // II factors in global memory
  if (n >= 1024) b += ws_round(((size_t)2 * n_eig * 64 + 2 * 64 * 64) * sizeof(cplx));                      // blocked back-transformation
  return b;
}

// H (n x n Hermitian, row-major, leading dimension ld, not modified) -> C [n_eig][n] (rows = eigenvectors of the n_eig
// smallest eigenvalues, unit norm up to rounding, NOT yet re-orthogonalised), lambda dev [n_eig] ascending.
// Abuf, Vbuf: n x n scratch each.  Returns RPA_OK, or a negative code (the caller may fall back to Jacobi).
int tridiag_eigh_lowest(rpa_ctx* ctx, WsAlloc& ws, const cplx* H, long long ld, int n, int n_eig, cplx* Abuf, cplx* Vbuf, cplx* C,
                        double* lambda) {
  const bool iv_smem = (size_t)6 * n * sizeof(double) <= 190 * 1024;
  const bool wy = n >= 1024;
  cplx* tau = ws.get<cplx>(n);
  cplx* p = ws.get<cplx>((size_t)2 * HT_CMAX * n);
  double* d = ws.get<double>(n);
  double* e = ws.get<double>(n);
  double* tnorm = ws.get<double>(8);
  double* iws = iv_smem ? nullptr : ws.get<double>((size_t)6 * n * n_eig);
  cplx* Wk = wy ? ws.get<cplx>((size_t)2 * n_eig * 64 + 2 * 64 * 64) : nullptr;
  if (!ws.ok) return rpa_fail(ctx, RPA_ERR_WORKSPACE, "rpa_subspace_basis: workspace too small (need %zu bytes)", ws.off);
  RPA_CUDA(ctx, cudaMemcpy2DAsync(Abuf, (size_t)n * sizeof(cplx), H, (size_t)ld * sizeof(cplx), (size_t)n * sizeof(cplx), n,
                                  cudaMemcpyDeviceToDevice, ctx->stream));
  int coop = 0, per_sm = 0;
  cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, ctx->device);
  const size_t row = (size_t)n * sizeof(cplx), cap = 200 * 1024;
  int mode = 3 * row <= cap ? 0 : 2 * row <= cap ? 1 : 2;   // what of v, v_next, w fits in shared memory
  if (ctx->opt.hetrd_mode >= 0) mode = std::max(mode, std::min(2, ctx->opt.hetrd_mode));   // tests: the large-n variants on small matrices
  const size_t smem1 = (size_t)(3 - mode) * row;
  if (!coop || smem1 > cap) return RPA_ERR_INVALID;
  const void* fn = mode == 0 ? (const void*)hetrd_fused_kernel<0> : mode == 1 ? (const void*)hetrd_fused_kernel<1> : (const void*)hetrd_fused_kernel<2>;
  // rows resident in registers (mode 3) when a warp per row fits on the device and a row fits in a warp's registers
  bool rowreg = mode == 0 && n <= 32 * HT_RMAX && ctx->opt.hetrd_mode < 0 && ctx->opt.hetrd_threads == 0;
  if (rowreg) {
    int ps = 0;
    const void* f3 = (const void*)hetrd_fused_kernel<3>;
    RPA_CUDA(ctx, cudaFuncSetAttribute(f3, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024));
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&ps, f3, 256, smem1) != cudaSuccess || (long long)ps * ctx->sm_count < (n + 7) / 8) rowreg = false;
    else fn = f3;
  }
  RPA_CUDA(ctx, cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024));
  // large matrices stream from HBM: one CTA of 32 warps per SM (the shared-memory rows allow no second CTA); small ones are
  // bound by the barrier latency: few small CTAs
  int nthr = n > 3072 ? 1024 : n > 1536 ? 512 : 256;
  if (ctx->opt.hetrd_threads > 0) nthr = std::max(64, std::min(1024, ctx->opt.hetrd_threads & ~31));
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, nthr, smem1) != cudaSuccess || per_sm < 1) return RPA_ERR_INVALID;
  // small matrices: no more warps than rows (a cheaper barrier); large ones: every SM (rows are split into chunks when warps > rows)
  const int grid = rowreg ? (n + 7) / 8 : nthr > 256 ? ctx->sm_count * per_sm : std::min(ctx->sm_count * std::min(per_sm, 2), (n + 7) / 8);
  cplx* A_ = Abuf; int n_ = n; cplx* V_ = Vbuf; cplx* tau_ = tau; double* d_ = d; double* e_ = e; cplx* p_ = p;
  int cmax = HT_CMAX;
  void* args[] = {&A_, &n_, &V_, &tau_, &d_, &e_, &p_, &cmax};
  RPA_CUDA(ctx, cudaLaunchCooperativeKernel(fn, dim3(grid), dim3(nthr), args, smem1, ctx->stream));
  ctx->launches++;
  RPA_CUDA(ctx, cudaFuncSetAttribute(bisect_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024));
  bisect_kernel<<<(n_eig + 7) / 8, 256, (size_t)2 * n * sizeof(double), ctx->stream>>>(d, e, n, n_eig, lambda, tnorm);
  RPA_LAUNCH_CHECK(ctx);
  if (iv_smem) {
    const int nt = IV_NT;
    const size_t smem3 = (size_t)6 * n * nt * sizeof(double);
    if (smem3 <= 200 * 1024) {
      RPA_CUDA(ctx, cudaFuncSetAttribute(invit_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024));
      invit_kernel<true><<<(n_eig + nt - 1) / nt, 32, smem3, ctx->stream>>>(d, e, n, n_eig, lambda, tnorm, nullptr, C);
    } else {   // IV_NT vectors do not fit: one per CTA would waste the SMs, use global memory instead
      iws = ws.get<double>((size_t)6 * n * n_eig);
      if (!ws.ok) return rpa_fail(ctx, RPA_ERR_WORKSPACE, "rpa_subspace_basis: workspace too small (need %zu bytes)", ws.off);
      invit_kernel<false><<<(n_eig + 127) / 128, 128, 0, ctx->stream>>>(d, e, n, n_eig, lambda, tnorm, iws, C);
    }
  } else {
    invit_kernel<false><<<(n_eig + 127) / 128, 128, 0, ctx->stream>>>(d, e, n, n_eig, lambda, tnorm, iws, C);
  }
  RPA_LAUNCH_CHECK(ctx);
  if (wy) return backtransform_wy(ctx, Vbuf, tau, n, n_eig, C, Wk);
  const size_t smem4 = (size_t)BT_NV * n * sizeof(cplx);
  RPA_CUDA(ctx, cudaFuncSetAttribute(backtransform_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 96 * 1024));
  backtransform_kernel<<<(n_eig + BT_NV - 1) / BT_NV, 256, smem4, ctx->stream>>>(Vbuf, tau, n, n_eig, C);
  RPA_LAUNCH_CHECK(ctx);
  return RPA_OK;
}
