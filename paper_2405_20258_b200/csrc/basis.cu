// (a3) Static subspace basis: the n_eig eigenpairs of the Hermitian negative-semidefinite chi~0(0) with the greatest
// |lambda| (reading R9).  Block subspace iteration with CholeskyQR orthonormalisation and an on-device
// one-sided (Hestenes) Jacobi Rayleigh-Ritz, as north_star prescribes; when the block (n_eig + guard vectors) would
// cover more than half of the matrix the iteration degenerates to its p = n case: Jacobi on chi~0(0) itself.
//
// Row convention throughout: a "vector" is a contiguous row.  Acol[i][:] is the i-th column of G V (G = -H >= 0),
// Vcol[i][:] the i-th column of V.  Because G is Hermitian, Acol starts as conj(G).
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <numeric>

#include <cooperative_groups.h>

#include "rpa_internal.h"

namespace cg = cooperative_groups;

namespace {

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// block-wide sum of NV doubles per thread; result valid in all threads
template <int NV>
__device__ __forceinline__ void block_sum(double (&v)[NV], double* sh /* [NV][32] */) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
#pragma unroll
  for (int k = 0; k < NV; k++) {
    v[k] = warp_sum(v[k]);
    if (lane == 0) sh[k * 32 + warp] = v[k];
  }
  __syncthreads();
#pragma unroll
  for (int k = 0; k < NV; k++) {
    double x = lane < nw ? sh[k * 32 + lane] : 0.0;
    v[k] = warp_sum(x);
  }
  __syncthreads();
}

// Acol = -conj(src) (src row-major n x n with leading dimension ld), Vcol = identity
__global__ void jacobi_init_kernel(const cplx* __restrict__ src, long long ld, int n, cplx* __restrict__ A,
                                   cplx* __restrict__ V, int negate_conj, int with_v) {
  const int i = blockIdx.x;
  for (int k = threadIdx.x; k < n; k += blockDim.x) {
    cplx x = src[(long long)i * ld + k];
    A[(long long)i * n + k] = negate_conj ? make_double2(-x.x, x.y) : make_double2(-x.x, -x.y);
    if (with_v) V[(long long)i * n + k] = make_double2(i == k ? 1.0 : 0.0, 0.0);
  }
}

__global__ void row_norm2_max_kernel(const cplx* __restrict__ A, int n, double* out) {
  __shared__ double sh[32];
  double v[1] = {0.0};
  const cplx* a = A + (long long)blockIdx.x * n;
  for (int k = threadIdx.x; k < n; k += blockDim.x) v[0] += a[k].x * a[k].x + a[k].y * a[k].y;
  block_sum<1>(v, sh);
  if (threadIdx.x == 0) atomicMax((unsigned long long*)out, (unsigned long long)__double_as_longlong(v[0]));
}

// one round of the round-robin ordering: CTA k rotates the pair (i,j) of columns.
// WITH_V: also rotate the accumulated V (needed only when eigenvectors of numerically null eigenvalues are wanted;
// otherwise the eigenvectors are the normalised columns of the converged A = G V, and V is never touched, which halves
// the traffic).  STASH: the two columns are kept in shared memory between the dot products and the update.
template <bool WITH_V, bool STASH>
__device__ __forceinline__ void rotate_pair(cplx* __restrict__ A, cplx* __restrict__ V, int n, int m_even, int round, int k,
                                            double rot_tol, const double* __restrict__ gmax, double* __restrict__ off_max,
                                            cplx* st, double* sh) {
  int i, j;
  if (k == 0) { i = m_even - 1; j = round; }
  else { i = (round + k) % (m_even - 1); j = (round - k + (m_even - 1)) % (m_even - 1); }
  if (i >= n || j >= n) return;
  if (i > j) { int t = i; i = j; j = t; }
  cplx* ai = A + (long long)i * n;
  cplx* aj = A + (long long)j * n;
  double v[4] = {0, 0, 0, 0};
  for (int t = threadIdx.x; t < n; t += blockDim.x) {
    cplx x = ai[t], y = aj[t];
    if (STASH) { st[t] = x; st[n + t] = y; }
    v[0] += x.x * x.x + x.y * x.y;
    v[1] += y.x * y.x + y.y * y.y;
    v[2] += x.x * y.x + x.y * y.y;   // Re conj(x) y
    v[3] += x.x * y.y - x.y * y.x;   // Im conj(x) y
  }
  block_sum<4>(v, sh);
  const double alpha = v[0], beta = v[1];
  const double gabs = sqrt(v[2] * v[2] + v[3] * v[3]);
  const double null2 = 1e-24 * gmax[0];
  if (alpha <= null2 && beta <= null2) return;   // two numerically null columns: nothing to resolve
  const double denom = sqrt(alpha * beta);
  if (!(denom > 0.0) || gabs == 0.0) return;
  const double off = gabs / denom;
  if (threadIdx.x == 0) atomicMax((unsigned long long*)off_max, (unsigned long long)__double_as_longlong(off));
  if (off <= rot_tol) return;
  const double zeta = (beta - alpha) / (2.0 * gabs);
  const double t = (zeta >= 0.0 ? 1.0 : -1.0) / (fabs(zeta) + sqrt(1.0 + zeta * zeta));
  const double c = 1.0 / sqrt(1.0 + t * t), s = c * t;
  const double pr = v[2] / gabs, pi = v[3] / gabs;   // e^{i phi}
  // a_i' = c a_i - s e^{-i phi} a_j ;  a_j' = s e^{i phi} a_i + c a_j
  cplx* vi = V + (long long)i * n;
  cplx* vj = V + (long long)j * n;
  const int total = WITH_V ? 2 * n : n;
  for (int tt = threadIdx.x; tt < total; tt += blockDim.x) {
    cplx* pi_ = tt < n ? ai + tt : vi + (tt - n);
    cplx* pj_ = tt < n ? aj + tt : vj + (tt - n);
    cplx x, y;
    if (STASH && tt < n) { x = st[tt]; y = st[n + tt]; } else { x = *pi_; y = *pj_; }
    cplx ey = make_double2(pr * y.x + pi * y.y, pr * y.y - pi * y.x);   // e^{-i phi} y
    cplx ex = make_double2(pr * x.x - pi * x.y, pr * x.y + pi * x.x);   // e^{+i phi} x
    *pi_ = make_double2(c * x.x - s * ey.x, c * x.y - s * ey.y);
    *pj_ = make_double2(s * ex.x + c * y.x, s * ex.y + c * y.y);
  }
}

template <bool WITH_V, bool STASH>
__global__ void __launch_bounds__(256) jacobi_round_kernel(cplx* __restrict__ A, cplx* __restrict__ V, int n, int m_even,
                                                          int round, double rot_tol, const double* __restrict__ gmax,
                                                          double* __restrict__ off_max) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  __shared__ double sh[4 * 32];
  rotate_pair<WITH_V, STASH>(A, V, n, m_even, round, blockIdx.x, rot_tol, gmax, off_max, reinterpret_cast<cplx*>(smem_raw), sh);
}

// All sweeps in ONE cooperative launch: every round is followed by a grid-wide barrier instead of a kernel boundary,
// and convergence is decided on the device (off[sweep] = largest |a_i^H a_j| / (|a_i||a_j|) seen in that sweep).
// info[0] = sweeps done, info[1] = converged.
template <bool WITH_V, bool STASH>
__global__ void __launch_bounds__(256) jacobi_persistent_kernel(cplx* __restrict__ A, cplx* __restrict__ V, int n, int m_even,
                                                               double rot_tol, double stop, int max_sweeps,
                                                               const double* __restrict__ gmax, double* __restrict__ off,
                                                               int* __restrict__ info) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  __shared__ double sh[4 * 32];
  cg::grid_group grid = cg::this_grid();
  const int npairs = m_even / 2;
  int sweep = 0;
  bool conv = false;
  for (; sweep < max_sweeps && !conv; sweep++) {
    for (int r = 0; r < m_even - 1; r++) {
      for (int k = blockIdx.x; k < npairs; k += gridDim.x) {
        rotate_pair<WITH_V, STASH>(A, V, n, m_even, r, k, rot_tol, gmax, off + sweep, reinterpret_cast<cplx*>(smem_raw), sh);
        __syncthreads();
      }
      grid.sync();
    }
    conv = ((volatile double*)off)[sweep] <= stop;
  }
  if (blockIdx.x == 0 && threadIdx.x == 0) { info[0] = sweep; info[1] = conv ? 1 : 0; }
}

// WITH_V: theta_i = Re v_i^H a_i (eigenvalue of G, keeps the sign of tiny ones); otherwise theta_i = ||a_i|| (G >= 0).
// lam = -theta;  scale[i] = 1/||a_i|| (0 for a null column)
__global__ void rayleigh_kernel(const cplx* __restrict__ A, const cplx* __restrict__ V, int n, int with_v, double* lam,
                                double* scale) {
  __shared__ double sh[3 * 32];
  double v[3] = {0.0, 0.0, 0.0};
  const cplx* a = A + (long long)blockIdx.x * n;
  const cplx* w = V + (long long)blockIdx.x * n;
  for (int k = threadIdx.x; k < n; k += blockDim.x) {
    v[0] += a[k].x * a[k].x + a[k].y * a[k].y;
    if (with_v) { v[1] += w[k].x * a[k].x + w[k].y * a[k].y; v[2] += w[k].x * w[k].x + w[k].y * w[k].y; }
  }
  block_sum<3>(v, sh);
  if (threadIdx.x == 0) {
    const double nrm = sqrt(v[0]);
    // a zero row of V is a padding vector of the block iteration, not an eigenvector: it sorts after everything
    lam[blockIdx.x] = with_v ? (v[2] < 0.5 ? 1.0 : -v[1]) : -nrm;
    scale[blockIdx.x] = nrm > 0.0 ? 1.0 / nrm : 0.0;
  }
}

// dst[r][:] = scale[order[r]] * src[order[r]][:]   (scale == nullptr: plain gather)
__global__ void gather_scaled_rows_kernel(const cplx* __restrict__ src, long long lds, const int* __restrict__ order,
                                          const double* __restrict__ scale, int ncols, cplx* __restrict__ dst, long long ldd) {
  const int o = order[blockIdx.x];
  const cplx* s = src + (long long)o * lds;
  const double f = scale ? scale[o] : 1.0;
  cplx* d = dst + (long long)blockIdx.x * ldd;
  for (int k = threadIdx.x; k < ncols; k += blockDim.x) d[k] = make_double2(s[k].x * f, s[k].y * f);
}

__global__ void gather_rows_kernel(const cplx* __restrict__ src, long long lds, const int* __restrict__ order, int ncols,
                                   cplx* __restrict__ dst, long long ldd) {
  const cplx* s = src + (long long)order[blockIdx.x] * lds;
  cplx* d = dst + (long long)blockIdx.x * ldd;
  for (int k = threadIdx.x; k < ncols; k += blockDim.x) d[k] = s[k];
}

__global__ void random_rows_kernel(cplx* X, long long total, unsigned long long seed) {
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < total; i += (long long)gridDim.x * blockDim.x) {
    unsigned long long z = seed + 0x9E3779B97F4A7C15ull * (unsigned long long)(2 * i + 1);
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull; z = (z ^ (z >> 27)) * 0x94D049BB133111EBull; z ^= z >> 31;
    unsigned long long y = z * 0xD6E8FEB86659FD93ull; y ^= y >> 32;
    X[i] = make_double2((double)(z >> 11) * (1.0 / 9007199254740992.0) - 0.5,
                        (double)(y >> 11) * (1.0 / 9007199254740992.0) - 0.5);
  }
}

// res[i] = || Y[i] - theta_i X[i] ||_2  (theta = lam[i])
__global__ void residual_kernel(const cplx* __restrict__ X, const cplx* __restrict__ Y, const double* __restrict__ lam, int n,
                                double* res) {
  __shared__ double sh[32];
  double v[1] = {0.0};
  const cplx* x = X + (long long)blockIdx.x * n;
  const cplx* y = Y + (long long)blockIdx.x * n;
  const double th = lam[blockIdx.x];
  for (int k = threadIdx.x; k < n; k += blockDim.x) {
    double a = y[k].x - th * x[k].x, b = y[k].y - th * x[k].y;
    v[0] += a * a + b * b;
  }
  block_sum<1>(v, sh);
  if (threadIdx.x == 0) res[blockIdx.x] = sqrt(v[0]);
}

// q[0] = max_i res[i], q[1] = max_ij |S[i][j] - delta_ij|  (both >= 0: the bit patterns of non-negative doubles order like
// unsigned integers, so the maximum is an integer atomicMax).  One row of S per CTA; q must be zeroed first.
__global__ void quality_kernel(const double* __restrict__ res, const cplx* __restrict__ S, int p, double* __restrict__ q) {
  __shared__ double sh[32];
  const int i = blockIdx.x;
  double m = 0.0;
  for (int j = threadIdx.x; j < p; j += blockDim.x) {
    const cplx x = S[(long long)i * p + j];
    m = fmax(m, fmax(fabs(x.x - (i == j ? 1.0 : 0.0)), fabs(x.y)));
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
  if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = m;
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < (int)(blockDim.x >> 5); w++) m = fmax(m, sh[w]);
    atomicMax(reinterpret_cast<unsigned long long*>(q + 1), (unsigned long long)__double_as_longlong(m));
    atomicMax(reinterpret_cast<unsigned long long*>(q), (unsigned long long)__double_as_longlong(res[i]));
  }
}

struct JacobiWs {
  cplx* A; cplx* V; double* lam; double* scale; int* order; double* scal;  // scal[0] = gmax, scal[1] = off_max
  double* off; int* info;   // [64] per-sweep off-norm, [2] sweeps / converged (persistent kernel)
  cplx* Wb = nullptr; cplx* Ub = nullptr;   // [n_pad/64][64][64] Gram matrices / rotations of the block iteration
  bool with_v = false;
};

template <bool WITH_V, bool STASH>
void launch_round(rpa_ctx* ctx, JacobiWs& jw, int n, int m_even, int r, size_t smem) {
  jacobi_round_kernel<WITH_V, STASH><<<m_even / 2, 256, smem, ctx->stream>>>(jw.A, jw.V, n, m_even, r, 1e-15, jw.scal,
                                                                              jw.scal + 1);
  ctx->launches++;
}

// ---------------------------------------------------------------------------------------------------------------
// Block one-sided Jacobi (GEMM-rich form of the Hestenes iteration above): the vectors are taken in blocks of JB = 32;
// a step pairs adjacent blocks, forms the 64 x 64 Gram matrix W of each pair with the DMMA GEMM, runs one cyclic sweep
// of two-sided Jacobi rotations on W in shared memory accumulating the unitary U (pair_rotations_kernel), and applies
// A_pair <- U A_pair with the DMMA GEMM.  Odd-even transposition ordering: even steps pair blocks (0,1),(2,3),...,
// odd steps (1,2),(3,4),..., and the two blocks of a pair always swap places, so after nblk steps every pair of
// blocks has met exactly once and pairs are always contiguous in memory.
constexpr int JB = 32, JP = 2 * JB, JLD = JP + 1;

__global__ void __launch_bounds__(256) pair_rotations_kernel(const cplx* __restrict__ Wg, cplx* __restrict__ Ug, double rot_tol,
                                                             const double* __restrict__ gmax, double* __restrict__ off_max) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx* W = reinterpret_cast<cplx*>(smem_raw);   // [JP][JLD]
  cplx* U = W + JP * JLD;                        // [JP][JLD]
  __shared__ double rc_[JB], rs_[JB], rx_[JB], ry_[JB];
  __shared__ int rp_[JB], rq_[JB];
  __shared__ double sh[32];
  const int tid = threadIdx.x;
  const cplx* wg = Wg + (long long)blockIdx.x * JP * JP;
  for (int idx = tid; idx < JP * JP; idx += 256) {
    const int i = idx / JP, k = idx - i * JP;
    W[i * JLD + k] = wg[idx];
    U[i * JLD + k] = make_double2(i == k ? 1.0 : 0.0, 0.0);
  }
  __syncthreads();
  const double null2 = 1e-24 * gmax[0];
  {  // largest normalised off-diagonal element of this pair's Gram matrix (convergence measure of the sweep)
    double off = 0.0;
    for (int idx = tid; idx < JP * JP; idx += 256) {
      const int i = idx / JP, k = idx - i * JP;
      if (k < i) {
        const double a = W[i * JLD + i].x, b = W[k * JLD + k].x;
        if (a > null2 && b > null2) {   // a numerically null vector has no direction to converge
          const double den = sqrt(a * b);
          const cplx w = W[i * JLD + k];
          if (den > 0.0) off = fmax(off, sqrt(w.x * w.x + w.y * w.y) / den);
        }
      }
    }
    for (int o = 16; o > 0; o >>= 1) off = fmax(off, __shfl_xor_sync(0xffffffffu, off, o));
    if ((tid & 31) == 0) sh[tid >> 5] = off;
    __syncthreads();
    if (tid == 0) {
      for (int w = 1; w < 8; w++) off = fmax(off, sh[w]);
      atomicMax((unsigned long long*)off_max, (unsigned long long)__double_as_longlong(off));
    }
  }
  const int lane = tid & 31, wrp = tid >> 5;
  for (int r = 0; r < JP - 1; r++) {
    if (tid < JB) {
      int i, j;
      if (tid == 0) { i = JP - 1; j = r; }
      else { i = (r + tid) % (JP - 1); j = (r - tid + (JP - 1)) % (JP - 1); }
      if (i > j) { int t = i; i = j; j = t; }
      const double alpha = W[i * JLD + i].x, beta = W[j * JLD + j].x;
      const cplx w = W[i * JLD + j];
      const double g2 = w.x * w.x + w.y * w.y, ab = alpha * beta;
      double c = 1.0, s = 0.0, ex = 1.0, ey = 0.0;
      // rotation parameters with reciprocal square roots only (this chain is the critical path of a round)
      if (!(alpha <= null2 && beta <= null2) && ab > 0.0 && g2 > rot_tol * rot_tol * ab) {
        const double rg = rsqrt(g2);                               // 1 / |W_ij|
        const double zeta = (beta - alpha) * 0.5 * rg;
        const double z1 = 1.0 + zeta * zeta;
        const double t = (zeta >= 0.0 ? 1.0 : -1.0) * __drcp_rn(fabs(zeta) + z1 * rsqrt(z1));
        c = rsqrt(1.0 + t * t); s = c * t;
        ex = w.x * rg; ey = w.y * rg;                              // e^{i theta} = W_ij / |W_ij|
      }
      rp_[tid] = i; rq_[tid] = j; rc_[tid] = c; rs_[tid] = s; rx_[tid] = ex; ry_[tid] = ey;
    }
    __syncthreads();
    // W <- R W R^H on 2 x 2 blocks: block (k, l) = rows {i_k, j_k} x columns {i_l, j_l} is read and written by one thread
    // only, so the row and the column rotation are applied together and in place.
    //   rows:    x_i' = c x_i - s e^{i theta} x_j ;  x_j' = s x_i + c e^{i theta} x_j          (rotation of pair k)
    //   columns: y_i' = c y_i - s e^{-i theta} y_j ; y_j' = s y_i + c e^{-i theta} y_j         (rotation of pair l)
    {
      const int pl = rp_[lane], ql = rq_[lane];
      const double cl = rc_[lane], sl = rs_[lane], xl = rx_[lane], yl = ry_[lane];
#pragma unroll
      for (int m = 0; m < JB / 8; m++) {
        const int k = wrp + 8 * m;
        const double ck = rc_[k], sk = rs_[k];
        if (sk == 0.0 && sl == 0.0) continue;
        const int pk = rp_[k], qk = rq_[k];
        const double xk = rx_[k], yk = ry_[k];
        cplx w00 = W[pk * JLD + pl], w01 = W[pk * JLD + ql], w10 = W[qk * JLD + pl], w11 = W[qk * JLD + ql];
        // rows
        cplx e0 = make_double2(xk * w10.x - yk * w10.y, xk * w10.y + yk * w10.x);   // e^{i theta_k} w10
        cplx e1 = make_double2(xk * w11.x - yk * w11.y, xk * w11.y + yk * w11.x);
        cplx r00 = make_double2(ck * w00.x - sk * e0.x, ck * w00.y - sk * e0.y);
        cplx r10 = make_double2(sk * w00.x + ck * e0.x, sk * w00.y + ck * e0.y);
        cplx r01 = make_double2(ck * w01.x - sk * e1.x, ck * w01.y - sk * e1.y);
        cplx r11 = make_double2(sk * w01.x + ck * e1.x, sk * w01.y + ck * e1.y);
        // columns
        cplx f0 = make_double2(xl * r01.x + yl * r01.y, xl * r01.y - yl * r01.x);   // e^{-i theta_l} r01
        cplx f1 = make_double2(xl * r11.x + yl * r11.y, xl * r11.y - yl * r11.x);
        W[pk * JLD + pl] = make_double2(cl * r00.x - sl * f0.x, cl * r00.y - sl * f0.y);
        W[pk * JLD + ql] = make_double2(sl * r00.x + cl * f0.x, sl * r00.y + cl * f0.y);
        W[qk * JLD + pl] = make_double2(cl * r10.x - sl * f1.x, cl * r10.y - sl * f1.y);
        W[qk * JLD + ql] = make_double2(sl * r10.x + cl * f1.x, sl * r10.y + cl * f1.y);
      }
      // U <- R U (rows only)
      const int col = tid & (JP - 1), k0 = tid >> 6;
#pragma unroll
      for (int m = 0; m < JB / 4; m++) {
        const int k = k0 + 4 * m;
        const double ck = rc_[k], sk = rs_[k];
        if (sk == 0.0) continue;
        const int pk = rp_[k], qk = rq_[k];
        const double xk = rx_[k], yk = ry_[k];
        const cplx ui = U[pk * JLD + col], uj = U[qk * JLD + col];
        const cplx ej = make_double2(xk * uj.x - yk * uj.y, xk * uj.y + yk * uj.x);
        U[pk * JLD + col] = make_double2(ck * ui.x - sk * ej.x, ck * ui.y - sk * ej.y);
        U[qk * JLD + col] = make_double2(sk * ui.x + ck * ej.x, sk * ui.y + ck * ej.y);
      }
    }
    __syncthreads();
  }
  // U with its two row blocks swapped: the blocks of the pair exchange places (odd-even transposition ordering)
  cplx* ug = Ug + (long long)blockIdx.x * JP * JP;
  for (int idx = tid; idx < JP * JP; idx += 256) {
    const int i = idx / JP, k = idx - i * JP;
    ug[idx] = U[((i + JB) % JP) * JLD + k];
  }
}

// matrices smaller than this use the vector iteration (1024; RPA_JACOBI_BLOCK_MIN, read by rpa_create, overrides)
int jacobi_block_min(const rpa_ctx* ctx) { return ctx->opt.jacobi_block_min; }

// One sweep (nblk steps) of the block iteration on the n_pad = nblk * JB vectors of length n in A (and V if with_v).
int block_jacobi_sweep(rpa_ctx* ctx, cplx* A, cplx* V, bool with_v, int n, int nblk, cplx* Wb, cplx* Ub, const double* gmax,
                       double* off_slot) {
  const size_t smem = (size_t)2 * JP * JLD * sizeof(cplx);
  for (int step = 0; step < nblk; step++) {
    const int b0 = step & 1;
    const int npairs = (nblk - b0) / 2;
    if (npairs <= 0) continue;
    cplx* a0 = A + (long long)b0 * JB * n;
    ZgemmParams g;   // W[pair] = A_pair A_pair^H
    g.A = a0; g.lda = n; g.a_km = false; g.B = a0; g.ldb = n; g.b_kn = false; g.C = Wb; g.ldc = JP;
    g.M = JP; g.N = JP; g.K = n; g.conj_b = true; g.herm = true;
    g.batch = npairs; g.strideA = (long long)JP * n; g.strideB = g.strideA; g.strideC = JP * JP;
    int rc = zgemm_dmma(ctx, g);
    if (rc) return rc;
    pair_rotations_kernel<<<npairs, 256, smem, ctx->stream>>>(Wb, Ub, 1e-15, gmax, off_slot);
    RPA_LAUNCH_CHECK(ctx);
    for (int which = 0; which < (with_v ? 2 : 1); which++) {   // X_pair <- U X_pair, in place (a CTA reads its whole
      cplx* x0 = (which ? V : A) + (long long)b0 * JB * n;     // 64-row column strip before it writes it)
      ZgemmParams u;
      u.A = Ub; u.lda = JP; u.a_km = false; u.B = x0; u.ldb = n; u.b_kn = true; u.C = x0; u.ldc = n;
      u.M = JP; u.N = n; u.K = JP; u.conj_b = false; u.split_k = 1;
      u.batch = npairs; u.strideA = JP * JP; u.strideB = (long long)JP * n; u.strideC = u.strideB;
      if ((rc = zgemm_dmma(ctx, u))) return rc;
    }
  }
  return RPA_OK;
}

// Eigen-decomposition of G = -H (H given as src, Hermitian negative semidefinite n x n) by one-sided Jacobi on the
// columns of G.  On return lam_h / order_h (host) and jw.order (device) sort the eigenvalues of H ascending (most
// negative first).  The leading n_need eigenvectors are then fetched with jacobi_vectors().  V is accumulated only if
// some wanted eigenvalue is numerically null (its column of G V cannot be normalised); that case reruns with V.
int jacobi_eigh(rpa_ctx* ctx, const cplx* src, long long ld, int n, bool src_is_hc, int n_need, bool try_without_v,
                JacobiWs& jw, std::vector<int>& order_h, std::vector<double>& lam_h) {
  if (ctx->attr_once(RPA_ATTR_JACOBI)) {
    RPA_CUDA(ctx, cudaFuncSetAttribute(jacobi_round_kernel<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 100 * 1024));
    RPA_CUDA(ctx, cudaFuncSetAttribute(jacobi_round_kernel<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 100 * 1024));
    RPA_CUDA(ctx, cudaFuncSetAttribute(pair_rotations_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                       (int)((size_t)2 * JP * JLD * sizeof(cplx))));
  }
  const bool verbose = ctx->opt.verbose;
  for (int attempt = try_without_v ? 0 : 1; attempt < 2; attempt++) {
    const bool with_v = attempt == 1;
    jw.with_v = with_v;
    // src_is_hc: src already holds Hc = H^T (RR matrix), so Acol = -src; otherwise src = H and Acol = -conj(H)
    jacobi_init_kernel<<<n, 256, 0, ctx->stream>>>(src, ld, n, jw.A, jw.V, src_is_hc ? 0 : 1, with_v ? 1 : 0);
    RPA_LAUNCH_CHECK(ctx);
    RPA_CUDA(ctx, cudaMemsetAsync(jw.scal, 0, 2 * sizeof(double), ctx->stream));
    row_norm2_max_kernel<<<n, 256, 0, ctx->stream>>>(jw.A, n, jw.scal);
    RPA_LAUNCH_CHECK(ctx);
    const int m_even = (n + 1) & ~1;
    const double stop = std::max(1e-14, 4.0 * std::sqrt((double)n) * 1.1e-16);
    const bool block = jw.Wb != nullptr && n >= jacobi_block_min(ctx);
    const int n_rows = block ? (n + JB - 1) / JB * JB : n;   // vectors held in jw.A (the block iteration pads with zeros)
    const size_t stash_bytes = (size_t)2 * n * sizeof(cplx);
    const bool stash = stash_bytes <= 96 * 1024;
    bool converged = n < 2;
    int sweep = 0;
    bool persistent = false;
    if (block && !converged) {
      // GEMM-rich block iteration; padding vectors (rows n .. n_rows) are zero and stay zero
      if (n_rows > n) {
        RPA_CUDA(ctx, cudaMemsetAsync(jw.A + (size_t)n * n, 0, (size_t)(n_rows - n) * n * sizeof(cplx), ctx->stream));
        if (with_v) RPA_CUDA(ctx, cudaMemsetAsync(jw.V + (size_t)n * n, 0, (size_t)(n_rows - n) * n * sizeof(cplx), ctx->stream));
      }
      RPA_CUDA(ctx, cudaMemsetAsync(jw.off, 0, 64 * sizeof(double), ctx->stream));
      double prev = 1e300;
      for (; sweep < 60 && !converged; sweep++) {
        int rc = block_jacobi_sweep(ctx, jw.A, jw.V, with_v, n, n_rows / JB, jw.Wb, jw.Ub, jw.scal, jw.off + sweep);
        if (rc) return rc;
        double off = 0.0;
        RPA_CUDA(ctx, cudaMemcpyAsync(&off, jw.off + sweep, sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
        RPA_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
        if (verbose) fprintf(stderr, "[rpa] block jacobi n=%d sweep %d off %.3e\n", n, sweep, off);
        // off is measured on the Gram matrices BEFORE the sweep's rotations; rounding of the Gram sums floors it near
        // sqrt(n) eps, so a sweep that no longer improves a tiny off also ends the iteration
        converged = off <= stop || (off <= 1e-12 && off > 0.5 * prev);
        prev = off;
      }
      persistent = true;   // skip the per-round launch loop below
    }
    if (!block && !converged) {
      // one cooperative launch for all sweeps, if the device can co-schedule a useful number of CTAs
      const void* fn = with_v ? (stash ? (const void*)jacobi_persistent_kernel<true, true> : (const void*)jacobi_persistent_kernel<true, false>)
                              : (stash ? (const void*)jacobi_persistent_kernel<false, true> : (const void*)jacobi_persistent_kernel<false, false>);
      const size_t smem = stash ? stash_bytes : 0;
      int per_sm = 0, coop = 0;
      cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, ctx->device);
      if (stash) cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, 100 * 1024);
      if (coop && cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, 256, smem) == cudaSuccess && per_sm > 0) {
        int grid = std::min(m_even / 2, per_sm * ctx->sm_count);
        RPA_CUDA(ctx, cudaMemsetAsync(jw.off, 0, 64 * sizeof(double), ctx->stream));
        cplx* A_ = jw.A; cplx* V_ = jw.V; int n_ = n, me = m_even, maxs = 60;
        double rt = 1e-15, st_ = stop;
        const double* gm = jw.scal; double* off_ = jw.off; int* info_ = jw.info;
        void* args[] = {&A_, &V_, &n_, &me, &rt, &st_, &maxs, &gm, &off_, &info_};
        cudaError_t e = cudaLaunchCooperativeKernel(fn, dim3(grid), dim3(256), args, smem, ctx->stream);
        if (e == cudaSuccess) {
          ctx->launches++;
          int info_h[2] = {0, 0};
          RPA_CUDA(ctx, cudaMemcpyAsync(info_h, jw.info, 2 * sizeof(int), cudaMemcpyDeviceToHost, ctx->stream));
          RPA_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
          sweep = info_h[0]; converged = info_h[1] != 0; persistent = true;
        } else {
          (void)cudaGetLastError();   // fall back to one launch per round
        }
      }
    }
    for (; !persistent && sweep < 60 && !converged; sweep++) {
      RPA_CUDA(ctx, cudaMemsetAsync(jw.scal + 1, 0, sizeof(double), ctx->stream));
      for (int r = 0; r < m_even - 1; r++) {
        if (with_v) { if (stash) launch_round<true, true>(ctx, jw, n, m_even, r, stash_bytes); else launch_round<true, false>(ctx, jw, n, m_even, r, 0); }
        else { if (stash) launch_round<false, true>(ctx, jw, n, m_even, r, stash_bytes); else launch_round<false, false>(ctx, jw, n, m_even, r, 0); }
      }
      RPA_CUDA(ctx, cudaGetLastError());
      double off = 0.0;
      RPA_CUDA(ctx, cudaMemcpyAsync(&off, jw.scal + 1, sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
      RPA_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
      converged = off <= stop;
    }
    if (verbose) fprintf(stderr, "[rpa] jacobi n=%d with_v=%d stash=%d persistent=%d sweeps=%d\n", n, (int)with_v, (int)stash, (int)persistent, sweep);
    if (verbose && persistent && !block) {
      double offh[64];
      cudaMemcpy(offh, jw.off, sizeof(offh), cudaMemcpyDeviceToHost);
      for (int k = 0; k < sweep && k < 64; k++) fprintf(stderr, "[rpa]   sweep %d off %.3e\n", k, offh[k]);
    }
    ctx->jac_n = n; ctx->jac_sweeps = sweep; ctx->jac_kind = block ? 1 : 0;
    if (!converged) return rpa_fail(ctx, RPA_ERR_NO_CONVERGENCE, "one-sided Jacobi did not converge in 60 sweeps (n = %d)", n);
    rayleigh_kernel<<<n_rows, 256, 0, ctx->stream>>>(jw.A, jw.V, n, with_v ? 1 : 0, jw.lam, jw.scale);
    RPA_LAUNCH_CHECK(ctx);
    lam_h.resize(n_rows);
    RPA_CUDA(ctx, cudaMemcpyAsync(lam_h.data(), jw.lam, n_rows * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    RPA_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    order_h.resize(n_rows);
    std::iota(order_h.begin(), order_h.end(), 0);
    std::stable_sort(order_h.begin(), order_h.end(), [&](int a, int b) { return lam_h[a] < lam_h[b]; });
    RPA_CUDA(ctx, cudaMemcpyAsync(jw.order, order_h.data(), n_rows * sizeof(int), cudaMemcpyHostToDevice, ctx->stream));
    if (with_v) break;
    // without V the wanted eigenvectors are a_i / ||a_i||: fine unless a wanted eigenvalue is numerically null
    const double smallest = std::fabs(lam_h[order_h[std::min(n_need, n) - 1]]);
    if (smallest > 1e-9 * std::fabs(lam_h[order_h[0]])) break;
  }
  return RPA_OK;
}

// dst[r][:] (r < count) = eigenvector of the r-th smallest eigenvalue of H
int jacobi_vectors(rpa_ctx* ctx, const JacobiWs& jw, int n, int count, cplx* dst, long long ldd) {
  gather_scaled_rows_kernel<<<count, 256, 0, ctx->stream>>>(jw.with_v ? jw.V : jw.A, n, jw.order,
                                                           jw.with_v ? nullptr : jw.scale, n, dst, ldd);
  RPA_LAUNCH_CHECK(ctx);
  return RPA_OK;
}

int block_size(int n, int n_eig) {
  int p = std::max(2 * n_eig, n_eig + 16);
  return std::min(p, n);
}
bool use_direct(int n, int n_eig) { return 2 * block_size(n, n_eig) > n; }
// tridiagonalisation + bisection + inverse iteration (tridiag_eig.cu): part of the spectrum, v and the Sturm data in shared memory
bool use_tridiag(const rpa_ctx* ctx, int n, int n_eig) { return n >= 32 && n <= 12800 && 4 * n_eig <= 3 * n && !ctx->opt.no_tridiag; }

}  // namespace

size_t basis_workspace_bytes(const rpa_ctx* ctx, int n, int n_eig) {
  const size_t small = ws_round((size_t)(n + JB) * sizeof(double)) * 4 + ws_round((size_t)(n + JB) * sizeof(int)) + 8 * 256;
  auto jac = [](size_t m) {   // A, V (padded to whole blocks) and the Gram / rotation matrices of the block iteration
    return 2 * ws_round((m + JB) * m * sizeof(cplx)) + 2 * ws_round(((m + JB) / JP + 1) * JP * JP * sizeof(cplx));
  };
  const size_t direct = jac(n) + small + tridiag_workspace_bytes(n, n_eig) + ws_round((size_t)n_eig * n_eig * sizeof(cplx));
  if (use_direct(n, n_eig)) return direct;
  const size_t p = block_size(n, n_eig);
  const size_t iter = 3 * ws_round(p * n * sizeof(cplx)) + 2 * ws_round(p * p * sizeof(cplx)) + jac(p) + small;
  return use_tridiag(ctx, n, n_eig) ? std::max(direct, iter) : iter;
}

int basis_run(rpa_ctx* ctx, WsAlloc& ws, const cplx* chi0, int n, int n_eig, double tol, cplx* C, double* lambda,
              int* iters_out) {
  ProfScope prof_scope(ctx, RPA_PROF_BASIS);
  if (tol <= 0.0) tol = 1e-11;
  std::vector<int> order_h;
  std::vector<double> lam_h;
  JacobiWs jw;
  jw.lam = ws.get<double>(n + JB);
  jw.scale = ws.get<double>(n + JB);
  double* d_lam_sorted = ws.get<double>(n);
  double* d_res = ws.get<double>(n);
  jw.order = ws.get<int>(n + JB);
  jw.scal = ws.get<double>(4);
  jw.off = ws.get<double>(64);
  jw.info = ws.get<int>(4);
  int* d_info = ws.get<int>(4);
  double* d_quality = ws.get<double>(2);
  int rc;
  // What the header promises for every route (P13): residuals ||chi0 c_i - lambda_i c_i|| <= tol |lambda_1| and
  // C C^H = 1.  X [p][n] are the vectors, lam_dev their eigenvalues, Y [p][n] and S [p][p] scratch.  Returns 1 when the
  // p vectors meet the targets, 0 when not, < 0 on error; the two measures are kept for rpa_basis_quality.
  const double ortho_tol = std::max(10.0 * tol, 1e-11);
  auto verify = [&](const cplx* X, const double* lam_dev, int p, cplx* Y, cplx* S) -> int {
    ZgemmParams g;   // Y[i][G] = sum_G' chi0[G][G'] X[i][G']  (chi0 Hermitian)
    g.A = X; g.lda = n; g.a_km = false; g.B = chi0; g.ldb = n; g.b_kn = true; g.C = Y; g.ldc = n;
    g.M = p; g.N = n; g.K = n; g.conj_b = true;
    int r = zgemm_dmma(ctx, g);
    if (r) return r;
    residual_kernel<<<p, 256, 0, ctx->stream>>>(X, Y, lam_dev, n, d_res);
    RPA_LAUNCH_CHECK(ctx);
    ZgemmParams h;   // S = X X^H
    h.A = X; h.lda = n; h.a_km = false; h.B = X; h.ldb = n; h.b_kn = false; h.C = S; h.ldc = p;
    h.M = p; h.N = p; h.K = n; h.conj_b = true; h.herm = true;
    if ((r = zgemm_dmma(ctx, h))) return r;
    RPA_CUDA(ctx, cudaMemsetAsync(d_quality, 0, 2 * sizeof(double), ctx->stream));
    quality_kernel<<<p, 256, 0, ctx->stream>>>(d_res, S, p, d_quality);
    RPA_LAUNCH_CHECK(ctx);
    double q[3] = {0.0, 0.0, 0.0};
    RPA_CUDA(ctx, cudaMemcpyAsync(q, d_quality, 2 * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    RPA_CUDA(ctx, cudaMemcpyAsync(q + 2, lam_dev, sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    RPA_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    const double scale = std::fabs(q[2]) > 0.0 ? std::fabs(q[2]) : 1.0;
    ctx->basis_residual = q[0] / scale; ctx->basis_ortho = q[1];
    if (ctx->opt.verbose)
      fprintf(stderr, "[rpa] basis check: n=%d p=%d residual %.3e |lambda_1| (target %.1e), max|C C^H - 1| %.3e (target %.1e)\n", n, p,
              ctx->basis_residual, tol, ctx->basis_ortho, ortho_tol);
    return (std::isfinite(q[0]) && std::isfinite(q[1]) && ctx->basis_residual <= tol && ctx->basis_ortho <= ortho_tol) ? 1 : 0;
  };
  const WsAlloc ws_iter = ws;   // the block iteration below restarts from here when the tridiagonal route fails
  const bool direct = use_direct(n, n_eig);
  if (direct || use_tridiag(ctx, n, n_eig)) {
    jw.A = ws.get<cplx>((size_t)(n + JB) * n);
    jw.V = ws.get<cplx>((size_t)(n + JB) * n);
    jw.Wb = ws.get<cplx>((size_t)((n + JB) / JP + 1) * JP * JP);
    jw.Ub = ws.get<cplx>((size_t)((n + JB) / JP + 1) * JP * JP);
    if (!ws.ok) return rpa_fail(ctx, RPA_ERR_WORKSPACE, "rpa_subspace_basis: workspace too small (need %zu bytes)", ws.off);
    if (use_tridiag(ctx, n, n_eig)) {
      // part of the spectrum: tridiagonalisation + bisection + inverse iteration (tridiag_eig.cu), then a
      // CholeskyQR2 clean-up of the n_eig vectors; any failure (e.g. a numerically singular Gram matrix because wanted
      // eigenvalues coincide) falls through to the Jacobi iteration below
      WsAlloc wt = ws;
      cplx* S = wt.get<cplx>((size_t)n_eig * n_eig);
      rc = tridiag_eigh_lowest(ctx, wt, chi0, n, n, n_eig, jw.A, jw.V, C, lambda);
      if (rc == RPA_ERR_WORKSPACE) return rc;
      bool ok = rc == RPA_OK && wt.ok;
      for (int pass = 0; pass < 1 && ok; pass++) {   // the vectors arrive orthogonal to ~eps / gap: one CholeskyQR pass restores eps
        ZgemmParams g;
        g.A = C; g.lda = n; g.a_km = false; g.B = C; g.ldb = n; g.b_kn = false; g.C = S; g.ldc = n_eig;
        g.M = n_eig; g.N = n_eig; g.K = n; g.conj_b = true; g.herm = true;
        if ((rc = zgemm_dmma(ctx, g))) return rc;
        if ((rc = zpotrf_batched(ctx, S, n_eig, n_eig, 1, 0, d_info))) return rc;
        int info_h = 0;
        RPA_CUDA(ctx, cudaMemcpyAsync(&info_h, d_info, sizeof(int), cudaMemcpyDeviceToHost, ctx->stream));
        RPA_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
        if (info_h != 0) { ok = false; break; }
        if ((rc = ztrsm_left_lower(ctx, S, n_eig, n_eig, C, n, n))) return rc;
      }
      if (ok) {   // the route has no convergence test of its own (and no reorthogonalisation inside clusters): check it
        const int v = verify(C, lambda, n_eig, jw.A, jw.V);
        if (v < 0) return v;
        ok = v == 1;
      }
      if (ctx->opt.verbose) fprintf(stderr, "[rpa] tridiagonal eigensolver n=%d n_eig=%d %s\n", n, n_eig, ok ? "ok" : "failed -> Jacobi / block iteration");
      if (ok) {
        ctx->jac_n = n; ctx->jac_sweeps = 0; ctx->jac_kind = 2;
        RPA_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
        if (iters_out) *iters_out = 0;
        return RPA_OK;
      }
      (void)cudaGetLastError();
    }
  }
  if (direct) {
    if ((rc = jacobi_eigh(ctx, chi0, n, n, false, n_eig, n_eig < n, jw, order_h, lam_h))) return rc;
    if ((rc = jacobi_vectors(ctx, jw, n, n_eig, C, n))) return rc;
    std::vector<double> ls(n_eig);
    for (int i = 0; i < n_eig; i++) ls[i] = lam_h[order_h[i]];
    RPA_CUDA(ctx, cudaMemcpyAsync(lambda, ls.data(), n_eig * sizeof(double), cudaMemcpyHostToDevice, ctx->stream));
    RPA_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    if (iters_out) *iters_out = 0;
    const int v = verify(C, lambda, n_eig, jw.A, jw.V);   // the eigenvectors have left jw.A / jw.V
    if (v < 0) return v;
    if (v == 0)
      return rpa_fail(ctx, RPA_ERR_NO_CONVERGENCE, "rpa_subspace_basis: Jacobi eigenvectors miss the targets: residual %.3e |lambda_1| (tol %.1e), "
                      "max|C C^H - 1| %.3e (tol %.1e)", ctx->basis_residual, tol, ctx->basis_ortho, ortho_tol);
    return RPA_OK;
  }

  // ---- block subspace iteration ----
  ws = ws_iter;
  const int p = block_size(n, n_eig);
  cplx* X = ws.get<cplx>((size_t)p * n);
  cplx* Y = ws.get<cplx>((size_t)p * n);
  cplx* Z = ws.get<cplx>((size_t)p * n);
  cplx* S = ws.get<cplx>((size_t)p * p);
  cplx* Vs = ws.get<cplx>((size_t)p * p);
  jw.A = ws.get<cplx>((size_t)(p + JB) * p);
  jw.V = ws.get<cplx>((size_t)(p + JB) * p);
  jw.Wb = ws.get<cplx>((size_t)((p + JB) / JP + 1) * JP * JP);
  jw.Ub = ws.get<cplx>((size_t)((p + JB) / JP + 1) * JP * JP);
  if (!ws.ok) return rpa_fail(ctx, RPA_ERR_WORKSPACE, "rpa_subspace_basis: workspace too small (need %zu bytes)", ws.off);

  auto gemm_apply = [&](const cplx* Xin, cplx* Yout) {  // Yout[j][G] = sum_G' chi0[G][G'] Xin[j][G']
    ZgemmParams g;
    g.A = Xin; g.lda = n; g.a_km = false; g.B = chi0; g.ldb = n; g.b_kn = true; g.C = Yout; g.ldc = n;
    g.M = p; g.N = n; g.K = n; g.conj_b = true;
    return zgemm_dmma(ctx, g);
  };
  auto gram = [&](const cplx* Ain, const cplx* Bin, cplx* out) {  // out[i][j] = sum_G Ain[i][G] conj(Bin[j][G])
    ZgemmParams g;
    g.A = Ain; g.lda = n; g.a_km = false; g.B = Bin; g.ldb = n; g.b_kn = false; g.C = out; g.ldc = p;
    g.M = p; g.N = p; g.K = n; g.conj_b = true; g.herm = (Ain == Bin);
    return zgemm_dmma(ctx, g);
  };
  auto rotate = [&](const cplx* Q, const cplx* Xin, cplx* Xout) {  // Xout[i][G] = sum_j Q[i][j] Xin[j][G]
    ZgemmParams g;
    g.A = Q; g.lda = p; g.a_km = false; g.B = Xin; g.ldb = n; g.b_kn = true; g.C = Xout; g.ldc = n;
    g.M = p; g.N = n; g.K = p; g.conj_b = false;
    return zgemm_dmma(ctx, g);
  };
  auto orthonormalise = [&](cplx* W) -> int {  // CholeskyQR: W W^H = L L^H, W <- L^{-1} W
    int r;
    if ((r = gram(W, W, S))) return r;
    if ((r = zpotrf_batched(ctx, S, p, p, 1, 0, d_info))) return r;
    if ((r = ztrsm_left_lower(ctx, S, p, p, W, n, n))) return r;
    return RPA_OK;
  };

  random_rows_kernel<<<ctx->sm_count * 4, 256, 0, ctx->stream>>>(X, (long long)p * n, 0x2405ull);
  RPA_LAUNCH_CHECK(ctx);
  if ((rc = orthonormalise(X))) return rc;
  if ((rc = orthonormalise(X))) return rc;
  const int max_it = 400, rr_every = 6;
  int it = 0;
  bool done = false;
  double worst = 0.0;
  while (it < max_it && !done) {
    for (int s = 0; s < rr_every; s++, it++) {   // power steps: X <- orth(chi0 X)
      if ((rc = gemm_apply(X, Y))) return rc;
      std::swap(X, Y);
      if ((rc = orthonormalise(X))) return rc;
    }
    if ((rc = orthonormalise(X))) return rc;     // second pass (CholeskyQR2) before Rayleigh-Ritz
    if ((rc = gemm_apply(X, Y))) return rc;      // Y = chi0 X
    if ((rc = gram(Y, X, S))) return rc;         // Hc[i][j] = x_j^H chi0 x_i
    if ((rc = jacobi_eigh(ctx, S, p, p, true, p, true, jw, order_h, lam_h))) return rc;
    if ((rc = jacobi_vectors(ctx, jw, p, p, Vs, p))) return rc;
    if ((rc = rotate(Vs, X, Z))) return rc;      // Ritz vectors
    std::swap(X, Z);
    if ((rc = rotate(Vs, Y, Z))) return rc;      // chi0 applied to the Ritz vectors
    std::swap(Y, Z);
    std::vector<double> ls(p);
    for (int i = 0; i < p; i++) ls[i] = lam_h[order_h[i]];
    RPA_CUDA(ctx, cudaMemcpyAsync(d_lam_sorted, ls.data(), p * sizeof(double), cudaMemcpyHostToDevice, ctx->stream));
    residual_kernel<<<n_eig, 256, 0, ctx->stream>>>(X, Y, d_lam_sorted, n, d_res);
    RPA_LAUNCH_CHECK(ctx);
    std::vector<double> res(n_eig);
    RPA_CUDA(ctx, cudaMemcpyAsync(res.data(), d_res, n_eig * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    RPA_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    worst = *std::max_element(res.begin(), res.end());
    done = worst <= tol * std::fabs(ls[0]);
  }
  if (iters_out) *iters_out = it;
  if (!done)
    return rpa_fail(ctx, RPA_ERR_NO_CONVERGENCE, "subspace iteration: residual %.3e after %d iterations (target %.3e)", worst,
                    it, tol);
  RPA_CUDA(ctx, cudaMemcpy2DAsync(C, (size_t)n * sizeof(cplx), X, (size_t)n * sizeof(cplx), (size_t)n * sizeof(cplx), n_eig,
                                  cudaMemcpyDeviceToDevice, ctx->stream));
  RPA_CUDA(ctx, cudaMemcpyAsync(lambda, d_lam_sorted, n_eig * sizeof(double), cudaMemcpyDeviceToDevice, ctx->stream));
  {
    const int v = verify(C, lambda, n_eig, Y, S);   // residuals were the stopping test; this adds orthonormality
    if (v < 0) return v;
    if (v == 0)
      return rpa_fail(ctx, RPA_ERR_NO_CONVERGENCE, "rpa_subspace_basis: Ritz vectors miss the targets: residual %.3e |lambda_1| (tol %.1e), "
                      "max|C C^H - 1| %.3e (tol %.1e)", ctx->basis_residual, tol, ctx->basis_ortho, ortho_tol);
  }
  return RPA_OK;
}
