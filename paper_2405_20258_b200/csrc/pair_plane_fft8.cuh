// pair_plane_fft8_kernel<N>: the hot kernel of MTXEL for square xy planes with N = 8 * R2 (N = 24, 40, 48, 64: every
// config of BASELINE.json).  Same role as the generic pair_plane_kernel (see mtxel.cu), but the two 1-D transforms of a
// plane are a compile-time two-pass decimation-in-frequency FFT held in registers:
//
//   pass A (radix 8):   thread (line, j), j < R2, takes x[j + q R2], q < 8, from the line, does an 8-point butterfly and
//                       multiplies by w_N^{j s}; y_s goes back in place to position s R2 + j.
//   pass B (pruned):    only the kept frequencies k are formed:  X[k] = sum_q z[s R2 + q] w_R2^{q s2},  s = k mod 8,
//                       s2 = k / 8 -- the last radix-R2 pass restricted to the epsilon-sphere outputs (eq. 3
//                       evaluated on the epsilon sphere only).
//
// Per valence band: [product fused into the loads of pass A on the rows | pass A | pass B -> kept y-frequencies,
// transposed] __syncthreads [pass A on the kept columns] __syncthreads [pass B -> the nk1 x nk2 kept plane
// frequencies, written to T].  Rows are private to a warp, so passes A and B of the row transforms are separated by
// __syncwarp() only; the twiddles w_N^{j s} live in registers for the whole valence loop and the next band's u_v
// elements are prefetched into registers while the current band is transformed.
#pragma once
#include "fft_smem.cuh"

namespace fft8 {

using fftsm::cplx;

template <int N>
struct Geo {
  static constexpr int R2 = N / 8;            // lanes per line in pass A
  static constexpr int RW = 32 / R2;          // lines per warp
  static constexpr int NWARP = (N + RW - 1) / RW;
  // line pitch (16-byte elements): odd so that lanes on consecutive lines never share a bank group in pass B, and
  // = R2 (mod 8) where possible so that pass A is conflict free too
  static constexpr int P = (R2 == 8) ? N + 1 : ((R2 & 1) ? N + R2 : N + 1);
};

template <int N>
__global__ void __launch_bounds__(Geo<N>::NWARP * 32)
pair_plane_fft8_kernel(const cplx* __restrict__ u_v, const cplx* __restrict__ u_c, int nvb, int ncc, int N3,
                       const cplx* __restrict__ tw /* [N] exp(-2 pi i k/N) */, const int* __restrict__ kfreq1,
                       const int* __restrict__ kfreq2, int nk1, int nk2, cplx* __restrict__ T) {
  constexpr int R2 = Geo<N>::R2, RW = Geo<N>::RW, P = Geo<N>::P, NTHR = Geo<N>::NWARP * 32;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx* sc = reinterpret_cast<cplx*>(smem_raw);   // [N][P]  u_c plane
  cplx* wk = sc + N * P;                          // [N][P]  rows being transformed
  cplx* cb0 = wk + N * P;                         // 2 x [nk2][P] kept y-frequencies, x contiguous
  cplx* root = cb0 + 2 * nk2 * P;                 // [R2]  w_R2^t
  int* s_k1 = reinterpret_cast<int*>(root + R2);  // [nk1] (s | s2 << 8) of the kept x-frequencies
  int* s_k2 = s_k1 + nk1;                         // [nk2]
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int z = blockIdx.x / ncc, c = blockIdx.x - z * ncc;
  constexpr int plane = N * N;
  const long long n_r = (long long)plane * N3;
  const cplx* ucp = u_c + (long long)c * n_r + (long long)z * plane;
  for (int idx = tid; idx < plane; idx += NTHR) {
    int x = idx / N, y = idx - x * N;
    sc[x * P + y] = ucp[idx];
  }
  for (int i = tid; i < R2; i += NTHR) root[i] = tw[i * 8];
  for (int i = tid; i < nk1; i += NTHR) { int k = kfreq1[i]; s_k1[i] = (k & 7) | ((k >> 3) << 8); }
  for (int i = tid; i < nk2; i += NTHR) { int k = kfreq2[i]; s_k2[i] = (k & 7) | ((k >> 3) << 8); }

  // role of this lane in pass A: line slot ls (row r0 + ls, or kept column c0 + ls), position j
  const int ls = lane / R2, j = lane - ls * R2;
  const bool lane_on = lane < RW * R2;
  const int r0 = warp * RW;                       // first row of this warp
  const int row = r0 + ls;
  const bool row_on = lane_on && row < N;
  const int nrow = min(RW, N - r0);               // > 0 for every warp by construction
  const int col = warp * RW + ls;                 // kept column handled in the x transforms
  const bool col_on = lane_on && col < nk2;
  cplx twj[8];
#pragma unroll
  for (int s = 1; s < 8; s++) twj[s] = tw[(j * s) % N];
  const cplx* uvp = u_v + (long long)z * plane + (long long)row * N + j;
  cplx nxt[8];
  if (row_on) {
#pragma unroll
    for (int q = 0; q < 8; q++) nxt[q] = uvp[q * R2];
  }
  __syncthreads();
  const int J = nk1 * nk2;
  for (int v = 0; v < nvb; v++) {
    cplx* cb = cb0 + (v & 1) * nk2 * P;
    // ---- rows: product + pass A
    if (row_on) {
      cplx x[8];
#pragma unroll
      for (int q = 0; q < 8; q++) {
        cplx a = nxt[q], b = sc[row * P + j + q * R2];
        x[q] = make_double2(a.x * b.x + a.y * b.y, a.x * b.y - a.y * b.x);   // conj(u_v) u_c
      }
      if (v + 1 < nvb) {
        const cplx* nx = uvp + (long long)(v + 1) * n_r;
#pragma unroll
        for (int q = 0; q < 8; q++) nxt[q] = nx[q * R2];
      }
      fftsm::bfly8<false>(x);
      wk[row * P + j] = x[0];
#pragma unroll
      for (int s = 1; s < 8; s++) wk[row * P + s * R2 + j] = fftsm::cmul(x[s], twj[s]);
    }
    __syncwarp();
    // ---- rows: pass B on the kept y-frequencies, transposed into cb[i2][x]
    for (int idx = lane; idx < RW * nk2; idx += 32) {
      const int xr = idx % RW, i2 = idx / RW;
      if (xr < nrow) {
        const int ss = s_k2[i2], s = ss & 255, s2 = ss >> 8;
        const cplx* zrow = wk + (r0 + xr) * P + s * R2;
        cplx acc = zrow[0];
#pragma unroll
        for (int q = 1; q < R2; q++) {
          cplx w = root[(q * s2) % R2], zz = zrow[q];
          acc.x += zz.x * w.x - zz.y * w.y;
          acc.y += zz.x * w.y + zz.y * w.x;
        }
        cb[i2 * P + r0 + xr] = acc;
      }
    }
    __syncthreads();
    // ---- kept columns: pass A (in place in cb)
    if (col_on) {
      cplx x[8];
      cplx* line = cb + col * P + j;
#pragma unroll
      for (int q = 0; q < 8; q++) x[q] = line[q * R2];
      fftsm::bfly8<false>(x);
      line[0] = x[0];
#pragma unroll
      for (int s = 1; s < 8; s++) line[s * R2] = fftsm::cmul(x[s], twj[s]);
    }
    __syncthreads();
    // ---- kept columns: pass B on the kept x-frequencies -> T
    cplx* dst = T + (((long long)v * ncc + c) * N3 + z) * J;
    for (int idx = tid; idx < J; idx += NTHR) {
      const int i1 = idx / nk2, i2 = idx - i1 * nk2;
      const int ss = s_k1[i1], s = ss & 255, s2 = ss >> 8;
      const cplx* zc = cb + i2 * P + s * R2;
      cplx acc = zc[0];
#pragma unroll
      for (int q = 1; q < R2; q++) {
        cplx w = root[(q * s2) % R2], zz = zc[q];
        acc.x += zz.x * w.x - zz.y * w.y;
        acc.y += zz.x * w.y + zz.y * w.x;
      }
      dst[idx] = acc;
    }
  }
}

template <int N>
size_t smem_bytes(int nk1, int nk2) {
  return ((size_t)2 * N * Geo<N>::P + (size_t)2 * nk2 * Geo<N>::P + Geo<N>::R2) * sizeof(cplx) + (size_t)(nk1 + nk2) * sizeof(int);
}

}  // namespace fft8
