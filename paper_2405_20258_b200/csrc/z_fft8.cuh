// z_fft8_scatter_kernel<N3>: the z transform + sphere gather of MTXEL for N3 = 8 * R3 (40, 120, 160: every config of
// BASELINE.json); same result as fft_axis_kernel<false,1> (mtxel.cu), written to stream T at HBM speed:
//
//   M[(v*nc + c0 + cl)*n_g + g] = (1/N_r) sum_z T[pair][z][j] e^{-2 pi i k z / N3},   g = inv_map[j*nk3 + i3] >= 0
//
// (eq. 3, last axis, evaluated on the kept k_z only).  Persistent CTAs take tiles of 32 consecutive lines (a line = one kept
// (k_x,k_y) column j of one pair); lane = line, so every global load of a warp is one contiguous 512-byte run.
//   pass A: thread (line, j3), j3 < R3 = warp index, loads z = j3 + q R3, q < 8, straight from global memory into
//           registers (8 independent loads in flight), does the radix-8 butterfly, multiplies by w_N3^{j3 s} (uniform
//           per warp) and stores y_s[j3] to shared memory.
//   pass B: task (residue s, two of its kept frequencies k = s + 8 s2), dealt to the warps, lane = line: direct sums over
//           j3 with warp-uniform twiddles w_R3^{j3 s2} (the pruning), scaled and scattered onto the epsilon sphere.
// The loads of the next tile are issued into registers before pass B of the current one, so HBM latency hides behind it.
#pragma once
#include "fft_smem.cuh"

namespace zfft8 {

using fftsm::cplx;
constexpr int MAXO = 8;   // kept frequencies per residue class s (host falls back to the generic kernel beyond)

struct Args {
  const cplx* T; long long n_lines; int J;
  const cplx* tw;          // [N3] exp(-2 pi i k / N3)
  const int* kfreq3; int nk3;
  const int* inv_map; cplx* M; int ncc, nc, c0, n_g; double scale;
};

constexpr int MAXT = 8 * ((MAXO + 1) / 2);   // pass-B tasks (at least 2 kept outputs per task)

// N3 = 120: two CTAs per SM (64 registers per thread; the pass-A twiddles are read from shared memory, warp-uniform, instead
// of living in 28 registers) -- with one CTA the only latency hiding is the prefetch of the next tile behind pass B.
template <int N3>
__global__ void __launch_bounds__(32 * (N3 / 8), N3 == 120 ? 2 : 0) z_fft8_scatter_kernel(Args a) {
  constexpr int R3 = N3 / 8, P = N3 | 1, NTHR = 32 * R3;
  constexpr int OG = R3 >= 20 ? 3 : 2;                  // kept outputs per pass-B task: about one round of tasks per tile
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx* y = reinterpret_cast<cplx*>(smem_raw);          // [32][P]   y_s[j3] at s*R3 + j3
  cplx* twb = y + 32 * P;                               // [8][MAXO][R3]  w_R3^{j3 s2} of the kept outputs of residue s
  int* oidx = reinterpret_cast<int*>(twb + 8 * MAXO * R3);   // [8][MAXO] index into the kept list, or -1
  cplx* twa_s = reinterpret_cast<cplx*>(oidx + 8 * MAXO);    // [R3][8] w_N3^{j3 s} (pass A), used when TWA_SMEM
  __shared__ long long s_row[32];
  __shared__ int s_j[32];
  __shared__ int t_s[MAXT], t_o0[MAXT], n_task;         // pass-B tasks: residue s, outputs o0 .. o0 + OG - 1 of it
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  for (int i = tid; i < 8 * MAXO; i += NTHR) oidx[i] = -1;
  __syncthreads();
  if (tid < 8) {
    int cnt = 0;
    for (int i = 0; i < a.nk3; i++)
      if ((a.kfreq3[i] & 7) == tid && cnt < MAXO) oidx[tid * MAXO + cnt++] = i;
  }
  __syncthreads();
  if (tid == 0) {
    int nt = 0;
    for (int o0 = 0; o0 < MAXO; o0 += OG)               // outputs-major: consecutive tasks hit different residues
      for (int s8 = 0; s8 < 8; s8++)
        if (oidx[s8 * MAXO + o0] >= 0) { t_s[nt] = s8; t_o0[nt] = o0; nt++; }
    n_task = nt;
  }
  for (int i = tid; i < 8 * MAXO * R3; i += NTHR) {
    const int j3 = i % R3, so = i / R3, o = oidx[so];
    cplx w = make_double2(1.0, 0.0);
    if (o >= 0) { const int s2 = a.kfreq3[o] >> 3; w = a.tw[(8 * ((j3 * s2) % R3)) % N3]; }
    twb[i] = w;
  }
  const int j3 = warp;                                   // pass A role
  constexpr bool TWA_SMEM = N3 == 120;
  cplx twa[TWA_SMEM ? 1 : 8];
  if (TWA_SMEM) {
    for (int i = tid; i < R3 * 8; i += NTHR) twa_s[i] = a.tw[((i >> 3) * (i & 7)) % N3];
  } else {
#pragma unroll
    for (int sA = 1; sA < 8; sA++) twa[sA] = a.tw[(j3 * sA) % N3];
  }
  const long long n_tiles = (a.n_lines + 31) / 32;
  // prefetch of the first tile
  long long tile = blockIdx.x;
  cplx x[8];
  long long row_n = 0; int j_n = -1;
  auto fetch = [&](long long t) {
    const long long line = t * 32 + lane;
    const bool on = t < n_tiles && line < a.n_lines;
    const long long pair = on ? line / a.J : 0;
    const int jj = on ? (int)(line - pair * a.J) : 0;
    const long long v = pair / a.ncc;
    const int cl = (int)(pair - v * a.ncc);
    row_n = (v * a.nc + a.c0 + cl) * a.n_g;
    j_n = on ? jj : -1;
    const cplx* src = a.T + (pair * N3 + j3) * a.J + jj;
#pragma unroll
    for (int q = 0; q < 8; q++) x[q] = on ? src[(long long)q * R3 * a.J] : make_double2(0.0, 0.0);
  };
  fetch(tile);
  __syncthreads();
  for (; tile < n_tiles; tile += gridDim.x) {
    // pass A on the prefetched tile
    fftsm::bfly8<false>(x);
    cplx* dst = y + lane * P + j3;
    dst[0] = x[0];
#pragma unroll
    for (int sA = 1; sA < 8; sA++) dst[sA * R3] = fftsm::cmul(x[sA], TWA_SMEM ? twa_s[j3 * 8 + sA] : twa[sA]);
    if (warp == 0) { s_row[lane] = row_n; s_j[lane] = j_n; }
    __syncthreads();
    fetch(tile + gridDim.x);                             // next tile's loads fly while pass B runs
    // pass B: task = (residue s, up to OG of its kept outputs), lane = line
    const int jl = s_j[lane];
    for (int t = warp; t < n_task; t += R3) {
      const int sB = t_s[t], o0 = t_o0[t];
      const cplx* ys = y + lane * P + sB * R3;
      const cplx* tw_s = twb + (sB * MAXO + o0) * R3;
      const int* oi = oidx + sB * MAXO + o0;
      // sphere indices of this task's outputs first: their (dependent) loads fly during the sums
      int g[OG];
#pragma unroll
      for (int o = 0; o < OG; o++) {
        const int i3 = (o0 + o < MAXO) ? oi[o] : -1;
        g[o] = (i3 >= 0 && jl >= 0) ? a.inv_map[jl * a.nk3 + i3] : -1;
      }
      cplx acc[OG];
#pragma unroll
      for (int o = 0; o < OG; o++) acc[o] = make_double2(0.0, 0.0);
#pragma unroll 5
      for (int k3 = 0; k3 < R3; k3++) {
        const cplx v = ys[k3];
#pragma unroll
        for (int o = 0; o < OG; o++) {
          const cplx w = tw_s[o * R3 + k3];
          acc[o].x += v.x * w.x - v.y * w.y;
          acc[o].y += v.x * w.y + v.y * w.x;
        }
      }
#pragma unroll
      for (int o = 0; o < OG; o++)
        if (g[o] >= 0) a.M[s_row[lane] + g[o]] = make_double2(acc[o].x * a.scale, acc[o].y * a.scale);
    }
    __syncthreads();                                     // y, s_row, s_j are free again
  }
}

template <int N3>
size_t smem_bytes() {
  constexpr int R3 = N3 / 8, P = N3 | 1;
  return ((size_t)32 * P + (size_t)8 * MAXO * R3) * sizeof(cplx) + 8 * MAXO * sizeof(int) + (size_t)R3 * 8 * sizeof(cplx);
}

}  // namespace zfft8
