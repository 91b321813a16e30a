// pair_plane_fft8_kernel<N>: the hot kernel of MTXEL for square xy planes with N = 8 * R2 (N = 24, 40, 48, 64: every
// config of BASELINE.json).  Same role as the generic pair_plane_kernel (see mtxel.cu): for one (conduction band c,
// plane z) and every valence band v of the block,
//
//   T[v][c][z][i2][i1] = sum_{x,y} conj(u_v(x,y,z)) u_c(x,y,z) e^{-2 pi i (k1[i1] x + k2[i2] y)/N}
//
// on the kept (epsilon-sphere) frequencies only -- PAPER.md:52 eq. 3 before the z transform.  Each 1-D transform is a
// two-pass decimation-in-frequency FFT, N = 8 x R2:
//
//   pass A (radix 8):  thread (line, j), j < R2, holds x[j + q R2], q < 8, in registers, does an 8-point butterfly and
//                      multiplies by w_N^{j s}; y_s goes to shared memory at position s G + j of the line (G = R2 or
//                      R2 + 1: an odd group pitch keeps pass B bank-conflict free).
//   pass B (radix R2): task (line, s) loads the R2 values of group s, does an R2-point butterfly in registers and
//                      stores only the kept frequencies k = s + 8 s2 (the pruning to the epsilon sphere).
//
// Rows (y transforms) are private to a warp: product fused into the pass-A loads, passes A and B separated by
// __syncwarp() only; pass B writes the kept y-frequencies transposed (x contiguous) into a double-buffered column
// buffer.  Bands are taken VB at a time: the x transforms of the previous VB bands run in the same loop iteration as the
// rows of the current VB bands (software pipeline), on the other half of the buffer, again warp-private -- so there is
// ONE block barrier per VB valence bands, and the VB x nk2 kept columns are dealt to the warps in full batches.  The twiddles
// w_N^{j s} live in registers for the whole valence loop and the next band's u_v elements are prefetched into
// registers while the current band is transformed.
#pragma once
#include "fft_smem.cuh"

namespace fft8 {

using fftsm::cplx;

constexpr int up_mod8(int x, int r) { return x + (((r - x) % 8) + 8) % 8; }   // smallest y >= x with y = r (mod 8)

template <int N>
struct Geo {
  static constexpr int R2 = N / 8;            // lanes per line in pass A
#ifndef RPA_PLANE48_RW
#define RPA_PLANE48_RW 4
#endif
  // lines per warp: as many as have R2 lanes each -- except N = 48, where 5 lines would leave the second pass (8 tasks
  // per line, one lane each) with 40 tasks for 32 lanes, i.e. a second, quarter-full sweep of the most expensive code
  static constexpr int RW = N == 48 ? RPA_PLANE48_RW : 32 / R2;
  static constexpr int NWARP = (N + RW - 1) / RW;
  // register cap (__maxnreg__) where a whole number of CTAs per SM needs one: 5 CTAs of 96 threads (N = 24), 2 of 224
  // (N = 40), 1 of 512 (N = 64); 0 = plain __launch_bounds__ (N = 48: 1 CTA of 320 threads, no cap needed)
  static constexpr int MAXREG = N <= 24 ? 128 : (N <= 40 ? 128 : (N <= 48 ? 0 : 128));
  // valence bands per loop iteration: one block barrier per VB bands, and the VB x nk2 kept columns of an iteration
  // fill whole warps of the x transforms (bounded by shared memory: 2 CTAs/SM at N = 40, 1 at N = 48, 64)
  static constexpr int VB = N <= 24 ? 4 : (N <= 48 ? 3 : 1);
  // Valence planes are read in LANE ORDER (uv_lane_order_kernel): warp w owns a region of 8 QS elements at w 8 QS of
  // the plane, and inside it element q of lane l sits at q QS + l -- so each of the 8 loads a lane issues per band is
  // one contiguous, 512-byte aligned run per warp (4 L1 wavefronts) instead of RW runs of R2 x 16 B in RW different
  // rows (~9 wavefronts: the LSU data pipe is this kernel's limiter).  PP = plane pitch in that layout (lanes that
  // hold no element leave holes that are never read).
  static constexpr int QS = 32;
  static constexpr int PP = NWARP * 8 * QS;
  static constexpr int G = (R2 & 1) ? R2 : R2 + 1;   // pitch of an s-group in a pass-A output line (odd)
  static constexpr int LW = 8 * G;                   // length of a pass-A output line
  // pitches in 16-byte elements.  P = R2 (mod 8) makes (line, j) -> bank group linear in the lane index, so the
  // 128-bit pass-A accesses are conflict free; an odd pitch makes the transposed stores of pass B conflict free.
  static constexpr int PS = up_mod8(N, R2);          // u_c plane
  static constexpr int PW = up_mod8(LW, R2);         // row work lines
  // column lines.  R2 odd: = R2 (mod 8) is odd too and serves both access patterns.  R2 = 8: a line's 8 lanes are one
  // quarter-warp, any pitch is conflict-free in pass A, so the odd pitch the transposed stores want.  R2 = 6: no pitch
  // serves both; = 6 (mod 8) keeps the 16 pass-A accesses of the columns conflict-free and leaves the transposed stores
  // of the rows with 2-way conflicts (480 instead of 576 wavefronts per band for the three patterns together)
  static constexpr int PC = ((R2 & 1) || R2 == 6) ? up_mod8(LW > N ? LW : N, R2) : ((LW > N ? LW : N) | 1);
};

// natural-order R-point DFT in registers (forward)
template <int R>
__device__ __forceinline__ void dft_small(cplx* z) {
  if (R == 3) fftsm::bfly3<false>(z);
  else if (R == 5) fftsm::bfly5<false>(z);
  else if (R == 8) fftsm::bfly8<false>(z);
  else if (R == 6) {
    cplx e[3] = {z[0], z[2], z[4]}, o[3] = {z[1], z[3], z[5]};
    fftsm::bfly3<false>(e);
    fftsm::bfly3<false>(o);
    const double h = 0.5, s = 0.86602540378443864676;
    cplx o1 = make_double2(h * o[1].x + s * o[1].y, h * o[1].y - s * o[1].x);      // w6   = ( 1/2, -sqrt3/2)
    cplx o2 = make_double2(-h * o[2].x + s * o[2].y, -h * o[2].y - s * o[2].x);    // w6^2 = (-1/2, -sqrt3/2)
    z[0] = fftsm::cadd(e[0], o[0]); z[3] = fftsm::csub(e[0], o[0]);
    z[1] = fftsm::cadd(e[1], o1);   z[4] = fftsm::csub(e[1], o1);
    z[2] = fftsm::cadd(e[2], o2);   z[5] = fftsm::csub(e[2], o2);
  }
}

// Outputs 0 and 5 only of the 6-point forward DFT: the second pass of a 48-point transform whose kept frequencies are
// |k| <= 7 needs, of the group k = s + 8 s2, only s2 = 0 (k >= 0) and s2 = 5 (k < 0).  With w = e^{+i pi/3} (= w6^5),
// w^3 = -1:  X5 = (z0 - z3) + w (z1 - z4) + w^2 (z2 - z5);  X0 = (z0 + z3) + (z1 + z4) + (z2 + z5).  24 FP64
// instructions instead of the ~55 of the full butterfly.
__device__ __forceinline__ void dft6_ends(const cplx* z, cplx& x0, cplx& x5) {
  const double h = 0.5, s = 0.86602540378443864676;
  const cplx a0 = fftsm::cadd(z[0], z[3]), a1 = fftsm::cadd(z[1], z[4]), a2 = fftsm::cadd(z[2], z[5]);
  const cplx d0 = fftsm::csub(z[0], z[3]), d1 = fftsm::csub(z[1], z[4]), d2 = fftsm::csub(z[2], z[5]);
  x0 = fftsm::cadd(fftsm::cadd(a0, a1), a2);
  const cplx p = fftsm::csub(d1, d2), r = fftsm::cadd(d1, d2);
  x5 = make_double2(fma(-s, r.y, fma(h, p.x, d0.x)), fma(s, r.x, fma(h, p.y, d0.y)));
}

template <int N>
__device__ __forceinline__ void pair_plane_fft8_body(const cplx* __restrict__ u_v, const cplx* __restrict__ u_c, int nvb, int ncc, int N3,
                       const cplx* __restrict__ tw /* [N] exp(-2 pi i k/N) */, const int* __restrict__ kfreq1,
                       const int* __restrict__ kfreq2, int nk1, int nk2, cplx* __restrict__ T) {
  using GE = Geo<N>;
  constexpr int R2 = GE::R2, RW = GE::RW, NWARP = GE::NWARP, G = GE::G, PS = GE::PS, PW = GE::PW, PC = GE::PC, VB = GE::VB;
  constexpr int NTHR = NWARP * 32;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx* sc = reinterpret_cast<cplx*>(smem_raw);   // [N][PS]  u_c plane
  cplx* wk = sc + N * PS;                         // [N][PW]  pass-A output of the rows (warp-private rows)
  cplx* cb0 = wk + N * PW;                        // 2 x [VB][nk2][PC] kept y-frequencies, x contiguous
  unsigned long long* slot2 = reinterpret_cast<unsigned long long*>(cb0 + 2 * VB * nk2 * PC);   // [8]: byte s2 = i2 or 0xff
  unsigned long long* slot1 = slot2 + 8;                                                   // [8]: byte s2 = i1 or 0xff
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int z = blockIdx.x / ncc, c = blockIdx.x - z * ncc;
  constexpr int plane = N * N;
  const long long n_r = (long long)plane * N3;
  const long long n_rp = (long long)GE::PP * N3;   // one valence band in lane order
  const cplx* ucp = u_c + (long long)c * n_r + (long long)z * plane;
  for (int idx = tid; idx < plane; idx += NTHR) {
    int x = idx / N, y = idx - x * N;
    sc[x * PS + y] = ucp[idx];
  }
  if (tid < 16) {
    // slot tables: which frequencies k = s + 8 s2 of group s are kept, and where they go
    const int* kf = tid < 8 ? kfreq2 : kfreq1;
    const int nk = tid < 8 ? nk2 : nk1, s = tid & 7;
    unsigned long long m = ~0ull;
    for (int i = 0; i < nk; i++) {
      const int k = kf[i];
      if ((k & 7) == s) { const int sh = 8 * (k >> 3); m = (m & ~(0xffull << sh)) | ((unsigned long long)i << sh); }
    }
    (tid < 8 ? slot2 : slot1)[s] = m;
  }

  // role of this lane in pass A: line slot ls (row r0 + ls, or line l0 + ls of the column buffer), position j
  const int ls = lane / R2, j = lane - ls * R2;
  const bool lane_on = lane < RW * R2;
  const int r0 = warp * RW;                       // first row of this warp
  const int row = r0 + ls;
  const bool row_on = lane_on && row < N;
  const int nrow = min(RW, N - r0);               // > 0 for every warp by construction
  cplx twj[8];
#pragma unroll
  for (int s = 1; s < 8; s++) twj[s] = tw[(j * s) % N];
  const cplx* uvp = u_v + (long long)z * GE::PP + warp * (8 * GE::QS) + lane;   // lane order, see Geo
  cplx nxt[8];
  if (row_on) {
#pragma unroll
    for (int q = 0; q < 8; q++) nxt[q] = uvp[q * GE::QS];
  }
  __syncthreads();
  const long long J = (long long)nk1 * nk2;
  const int cbsz = VB * nk2 * PC;                 // one half of the column buffer: VB bands x nk2 lines
  const int n_it = (nvb + VB - 1) / VB;
  for (int it = 0; it <= n_it; it++) {
    // ---------------- rows of bands it VB .. it VB + VB - 1 -> cb[it & 1]
    if (it < n_it) {
      const int v0 = it * VB, nb = min(VB, nvb - v0);
      for (int u = 0; u < nb; u++) {
        cplx* cb = cb0 + (it & 1) * cbsz + u * nk2 * PC;
        if (row_on) {
          cplx x[8];
#pragma unroll
          for (int q = 0; q < 8; q++) {
            cplx a = nxt[q], b = sc[row * PS + j + q * R2];
            x[q] = make_double2(a.x * b.x + a.y * b.y, a.x * b.y - a.y * b.x);   // conj(u_v) u_c
          }
          if (v0 + u + 1 < nvb) {
            const cplx* nx = uvp + (long long)(v0 + u + 1) * n_rp;
#pragma unroll
            for (int q = 0; q < 8; q++) nxt[q] = nx[q * GE::QS];
          }
          fftsm::bfly8<false>(x);
          cplx* line = wk + row * PW + j;
          line[0] = x[0];
#pragma unroll
          for (int s = 1; s < 8; s++) line[s * G] = fftsm::cmul(x[s], twj[s]);
        }
        __syncwarp();
        for (int t = lane; t < nrow * 8; t += 32) {
          const int l = t >> 3, s = t & 7;
          const cplx* grp = wk + (r0 + l) * PW + s * G;
          cplx zz[R2];
#pragma unroll
          for (int q = 0; q < R2; q++) zz[q] = grp[q];
          dft_small<R2>(zz);
          const unsigned long long sl = slot2[s];
          cplx* dst = cb + r0 + l;
#pragma unroll
          for (int s2 = 0; s2 < R2; s2++) {
            const int i2 = (int)((sl >> (8 * s2)) & 0xff);
            if (i2 != 0xff) dst[i2 * PC] = zz[s2];
          }
        }
        __syncwarp();                               // wk rows are reused by the next band of this iteration
      }
    }
    // ---------------- x transforms of the kept columns of the previous iteration's bands <- cb[(it - 1) & 1]
    // The nbp * nk2 lines of that half are one flat list, dealt to the warps in batches of RW lines.
    if (it > 0) {
      const int v0 = (it - 1) * VB, nbp = min(VB, nvb - v0);
      cplx* cb = cb0 + ((it - 1) & 1) * cbsz;
      const int nline = nbp * nk2;
      for (int l0 = (NWARP - 1 - warp) * RW; l0 < nline; l0 += NWARP * RW) {
        const int nl = min(RW, nline - l0);
        const bool col_on = lane_on && ls < nl;
        cplx x[8];
        cplx* line = cb + (l0 + ls) * PC;
        if (col_on) {
#pragma unroll
          for (int q = 0; q < 8; q++) x[q] = line[j + q * R2];
          fftsm::bfly8<false>(x);
        }
        __syncwarp();                               // pass A is in place with a different layout: read all, then write
        if (col_on) {
          line[j] = x[0];
#pragma unroll
          for (int s = 1; s < 8; s++) line[s * G + j] = fftsm::cmul(x[s], twj[s]);
        }
        __syncwarp();
        for (int t = lane; t < nl * 8; t += 32) {
          const int l = l0 + (t >> 3), s = t & 7;
          const cplx* grp = cb + l * PC + s * G;
          cplx zz[R2];
#pragma unroll
          for (int q = 0; q < R2; q++) zz[q] = grp[q];
          dft_small<R2>(zz);
          const unsigned long long sl = slot1[s];
          const int u = l / nk2, i2 = l - u * nk2;
          cplx* dst = T + (((long long)(v0 + u) * ncc + c) * N3 + z) * J + (long long)i2 * nk1;
#pragma unroll
          for (int s2 = 0; s2 < R2; s2++) {
            const int i1 = (int)((sl >> (8 * s2)) & 0xff);
            if (i1 != 0xff) dst[i1] = zz[s2];
          }
        }
        __syncwarp();
      }
    }
    __syncthreads();
  }
}

// ---------------------------------------------------------------------------------------------------------------
// Ring variant of the same kernel (used where only ONE CTA fits per SM: N = 48, 64).  There is no block barrier in the
// band loop: the column buffer is a ring of D = RingDepth<N>::value bands guarded by mbarriers (full[b]: all warps have written their rows
// of the band into cb[b]; empty[b]: the x transforms of that band are done and cb[b] may be overwritten).  The x
// transforms of band v are dealt, in batches of RW kept columns, to ncb warps that rotate with v, and a warp takes that
// duty one band late -- so a warp with column duty falls behind by one duty and catches up while the others carry the
// next bands, instead of every warp idling at a barrier while ncb of them transform columns.
// ring depth: 3 bands; 4 where shared memory allows it next to two u_c planes (N = 48: -1 % time), not at N = 64 (227 KB)
template <int N> struct RingDepth { static constexpr int value = N == 48 ? 4 : 3; };

__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned long long* bar) {
  asm volatile("{\n .reg .b64 st;\n mbarrier.arrive.shared::cta.b64 st, [%0];\n}\n" ::"r"((unsigned)__cvta_generic_to_shared(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity) {
  const unsigned a = (unsigned)__cvta_generic_to_shared(bar);
  unsigned ok;
  do {
    asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}\n"
                 : "=r"(ok) : "r"(a), "r"(parity) : "memory");
  } while (!ok);
}

// ENDS (N = 48 only): every kept frequency of both axes has s2 = 0 or s2 = R2 - 1 (the host checks), so the second passes
// form just those two outputs (dft6_ends) instead of the full R2-point butterfly.
// Pass-A output twiddles w_N^{j s}, s = 1..7.  TW3 (N = 64, where 512 threads cap the kernel at 128 registers and the
// seven values of the plain form spill -- and a spill is one more access on the LSU data pipe that already bounds the
// kernel): only s = 1, 2, 4 live in registers, the other four are their products (16 FP64 instructions per pass A on a pipe
// that is 37 % busy; each product adds one rounding, far inside the 1e-12 of M).
template <bool TW3>
struct Twid {
  cplx w[TW3 ? 3 : 8];
  __device__ __forceinline__ void init(const cplx* __restrict__ tw, int j, int n) {
    if (TW3) { w[0] = tw[j % n]; w[1] = tw[(2 * j) % n]; w[2] = tw[(4 * j) % n]; }
    else {
#pragma unroll
      for (int s = 1; s < 8; s++) w[s] = tw[(j * s) % n];
    }
  }
  __device__ __forceinline__ void apply(cplx* x) const {   // x[s] *= w^{j s}, s = 1..7
    if (TW3) {
      const cplx w3 = fftsm::cmul(w[0], w[1]);
      x[1] = fftsm::cmul(x[1], w[0]); x[2] = fftsm::cmul(x[2], w[1]); x[3] = fftsm::cmul(x[3], w3);
      x[4] = fftsm::cmul(x[4], w[2]); x[5] = fftsm::cmul(x[5], fftsm::cmul(w[0], w[2]));
      x[6] = fftsm::cmul(x[6], fftsm::cmul(w[1], w[2])); x[7] = fftsm::cmul(x[7], fftsm::cmul(w3, w[2]));
    } else {
#pragma unroll
      for (int s = 1; s < 8; s++) x[s] = fftsm::cmul(x[s], w[s]);
    }
  }
};

// CB conduction bands per CTA (N = 48: 2, where two u_c planes fit): the band loop runs over the nvb CB (valence band,
// conduction band) pairs of the CTA, so every u_v element fetched from L2 is used CB times.
template <int N, bool ENDS, int CB>
__device__ __forceinline__ void pair_plane_fft8_ring_body(const cplx* __restrict__ u_v, const cplx* __restrict__ u_c, int nvb, int ncc,
                                                          int N3, const cplx* __restrict__ tw, const int* __restrict__ kfreq1,
                                                          const int* __restrict__ kfreq2, int nk1, int nk2, cplx* __restrict__ T) {
  using GE = Geo<N>;
  constexpr int R2 = GE::R2, RW = GE::RW, NWARP = GE::NWARP, G = GE::G, PS = GE::PS, PW = GE::PW, PC = GE::PC, D = RingDepth<N>::value;
  constexpr int NTHR = NWARP * 32;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx* sc = reinterpret_cast<cplx*>(smem_raw);   // [CB][N][PS]  u_c planes
  cplx* wk = sc + CB * N * PS;                    // [N][PW]  pass-A output of the rows (warp-private rows)
  cplx* cb0 = wk + N * PW;                        // D x [nk2][PC] kept y-frequencies, x contiguous
  unsigned long long* slot2 = reinterpret_cast<unsigned long long*>(cb0 + D * nk2 * PC);
  unsigned long long* slot1 = slot2 + 8;
  unsigned long long* full = slot1 + 8;           // [D]
  unsigned long long* empty = full + D;           // [D]
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int ncg = (ncc + CB - 1) / CB;            // conduction-band groups of the launch
  const int z = blockIdx.x / ncg, c = (blockIdx.x - z * ncg) * CB;
  const int ncb_here = CB == 1 ? 1 : min(CB, ncc - c);   // conduction bands of this CTA (the last group may be short)
  constexpr int plane = N * N;
  const long long n_r = (long long)plane * N3;
  const long long n_rp = (long long)GE::PP * N3;   // one valence band in lane order
  for (int cs = 0; cs < ncb_here; cs++) {
    const cplx* ucp = u_c + (long long)(c + cs) * n_r + (long long)z * plane;
    for (int idx = tid; idx < plane; idx += NTHR) {
      int x = idx / N, y = idx - x * N;
      sc[(cs * N + x) * PS + y] = ucp[idx];
    }
  }
  const int ncb = (nk2 + RW - 1) / RW;            // column batches per band (host guarantees ncb <= NWARP)
  if (tid < 16) {
    const int* kf = tid < 8 ? kfreq2 : kfreq1;
    const int nk = tid < 8 ? nk2 : nk1, s = tid & 7;
    unsigned long long m = ~0ull;
    for (int i = 0; i < nk; i++) {
      const int k = kf[i];
      if ((k & 7) == s) { const int sh = 8 * (k >> 3); m = (m & ~(0xffull << sh)) | ((unsigned long long)i << sh); }
    }
    (tid < 8 ? slot2 : slot1)[s] = m;
  }
  if (tid == 32) {
    for (int b = 0; b < D; b++) { mbar_init(full + b, NWARP); mbar_init(empty + b, ncb); }
  }
  const int ls = lane / R2, j = lane - ls * R2;
  const bool lane_on = lane < RW * R2;
  const int r0 = warp * RW, row = r0 + ls;
  const bool row_on = lane_on && row < N;
  const int nrow = min(RW, N - r0);
#ifndef RPA_TW3
#define RPA_TW3 1
#endif
  Twid<N == 64 && RPA_TW3> twj;
  twj.init(tw, j, N);
  const cplx* uvp = u_v + (long long)z * GE::PP + warp * (8 * GE::QS) + lane;   // lane order, see Geo
  cplx nxt[8];
  if (row_on) {
#pragma unroll
    for (int q = 0; q < 8; q++) nxt[q] = uvp[q * GE::QS];
  }
  __syncthreads();
  const long long J = (long long)nk1 * nk2;

  auto cols = [&](int band) {   // this warp's share of the x transforms of `band`, if it has one
    int k = warp - (int)(((long long)band * ncb) % NWARP);
    if (k < 0) k += NWARP;
    if (k >= ncb) return;
    const int b = band % D;
    mbar_wait(full + b, (band / D) & 1);
    cplx* cb = cb0 + b * nk2 * PC;
    const int l0 = k * RW, nl = min(RW, nk2 - l0);
    const bool col_on = lane_on && ls < nl;
    cplx x[8];
    cplx* line = cb + (l0 + ls) * PC;
    if (col_on) {
#pragma unroll
      for (int q = 0; q < 8; q++) x[q] = line[j + q * R2];
      fftsm::bfly8<false>(x);
    }
    __syncwarp();
    if (col_on) {
      twj.apply(x);
#pragma unroll
      for (int s = 0; s < 8; s++) line[s * G + j] = x[s];
    }
    __syncwarp();
    const int bv = band / ncb_here, bc = band - bv * ncb_here;   // valence band, conduction band of the CTA
    cplx* dstT = T + (((long long)bv * ncc + c + bc) * N3 + z) * J;
    for (int t = lane; t < nl * 8; t += 32) {
      const int l = l0 + (t >> 3), s = t & 7;
      const cplx* grp = cb + l * PC + s * G;
      cplx zz[R2];
#pragma unroll
      for (int q = 0; q < R2; q++) zz[q] = grp[q];
      const unsigned long long sl = slot1[s];
      cplx* dst = dstT + (long long)l * nk1;
      if (ENDS && R2 == 6) {
        cplx x0, x5;
        dft6_ends(zz, x0, x5);
        const int ia = (int)(sl & 0xff), ib = (int)((sl >> 40) & 0xff);
        if (ia != 0xff) dst[ia] = x0;
        if (ib != 0xff) dst[ib] = x5;
      } else {
        dft_small<R2>(zz);
#pragma unroll
        for (int s2 = 0; s2 < R2; s2++) {
          const int i1 = (int)((sl >> (8 * s2)) & 0xff);
          if (i1 != 0xff) dst[i1] = zz[s2];
        }
      }
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(empty + b);
  };

  const int n_it = nvb * ncb_here;                // (valence band, conduction band) pairs, conduction band fastest
  int iv_run = 0, ic_run = 0;                     // valence band / conduction band of iteration it
  for (int it = 0; it < n_it; it++) {
    const int iv = CB == 1 ? it : iv_run, ic = CB == 1 ? 0 : ic_run;
    const int b = it % D;
    if (it >= D) mbar_wait(empty + b, ((it / D) - 1) & 1);   // the x transforms of band it - D have left cb[b]
    cplx* cb = cb0 + b * nk2 * PC;
    if (row_on) {
      cplx x[8];
#pragma unroll
      for (int q = 0; q < 8; q++) {
        cplx a = nxt[q], bb = sc[(ic * N + row) * PS + j + q * R2];
        x[q] = make_double2(a.x * bb.x + a.y * bb.y, a.x * bb.y - a.y * bb.x);   // conj(u_v) u_c
      }
      if (ic + 1 == ncb_here && iv + 1 < nvb) {   // last use of this valence band: fetch the next one
        const cplx* nx = uvp + (long long)(iv + 1) * n_rp;
#pragma unroll
        for (int q = 0; q < 8; q++) nxt[q] = nx[q * GE::QS];
      }
      fftsm::bfly8<false>(x);
      twj.apply(x);
      cplx* line = wk + row * PW + j;
#pragma unroll
      for (int s = 0; s < 8; s++) line[s * G] = x[s];
    }
    __syncwarp();
    for (int t = lane; t < nrow * 8; t += 32) {
      const int l = t >> 3, s = t & 7;
      const cplx* grp = wk + (r0 + l) * PW + s * G;
      cplx zz[R2];
#pragma unroll
      for (int q = 0; q < R2; q++) zz[q] = grp[q];
      const unsigned long long sl = slot2[s];
      cplx* dst = cb + r0 + l;
      if (ENDS && R2 == 6) {
        cplx x0, x5;
        dft6_ends(zz, x0, x5);
        const int ia = (int)(sl & 0xff), ib = (int)((sl >> 40) & 0xff);
        if (ia != 0xff) dst[ia * PC] = x0;
        if (ib != 0xff) dst[ib * PC] = x5;
      } else {
        dft_small<R2>(zz);
#pragma unroll
        for (int s2 = 0; s2 < R2; s2++) {
          const int i2 = (int)((sl >> (8 * s2)) & 0xff);
          if (i2 != 0xff) dst[i2 * PC] = zz[s2];
        }
      }
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(full + b);
    if (it >= 1) cols(it - 1);
    if (CB > 1 && ++ic_run == ncb_here) { ic_run = 0; iv_run++; }
  }
  cols(n_it - 1);
}

// u_nat[v][z][x][y] (plane-major, as the wavefunction transforms leave it) -> u_lane[v][z][PP] in the lane order of the
// plane kernels (Geo<N>::QS, PP).  One CTA of NWARP warps per (z, v) plane, the same lane roles as in the plane kernels.
template <int N>
__global__ void __launch_bounds__(Geo<N>::NWARP * 32) uv_lane_order_kernel(const cplx* __restrict__ u_nat, cplx* __restrict__ u_lane, int N3) {
  using GE = Geo<N>;
  constexpr int R2 = GE::R2, RW = GE::RW;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int ls = lane / R2, j = lane - ls * R2, r0 = warp * RW, row = r0 + ls;
  if (lane >= RW * R2 || row >= N) return;
  const long long pl = (long long)blockIdx.y * N3 + blockIdx.x;
  const cplx* src = u_nat + pl * (N * N) + (long long)row * N + j;
  cplx* dst = u_lane + pl * GE::PP + warp * (8 * GE::QS) + lane;
#pragma unroll
  for (int q = 0; q < 8; q++) dst[q * GE::QS] = src[q * R2];
}

#define RPA_FFT8_ARGS                                                                                              \
  const cplx *__restrict__ u_v, const cplx *__restrict__ u_c, int nvb, int ncc, int N3, const cplx *__restrict__ tw, \
      const int *__restrict__ kfreq1, const int *__restrict__ kfreq2, int nk1, int nk2, cplx *__restrict__ T
template <int N>
__global__ void __maxnreg__(Geo<N>::MAXREG > 0 ? Geo<N>::MAXREG : 255) pair_plane_fft8_kernel_r(RPA_FFT8_ARGS) {
  pair_plane_fft8_body<N>(u_v, u_c, nvb, ncc, N3, tw, kfreq1, kfreq2, nk1, nk2, T);
}
template <int N>
__global__ void __launch_bounds__(Geo<N>::NWARP * 32) pair_plane_fft8_kernel_b(RPA_FFT8_ARGS) {
  pair_plane_fft8_body<N>(u_v, u_c, nvb, ncc, N3, tw, kfreq1, kfreq2, nk1, nk2, T);
}
template <int N, bool ENDS, int CB>
__global__ void __launch_bounds__(Geo<N>::NWARP * 32) pair_plane_fft8_kernel_ring(RPA_FFT8_ARGS) {
  pair_plane_fft8_ring_body<N, ENDS, CB>(u_v, u_c, nvb, ncc, N3, tw, kfreq1, kfreq2, nk1, nk2, T);
}
#undef RPA_FFT8_ARGS

template <int N>
size_t smem_bytes(int nk1, int nk2) {
  (void)nk1;
  return ((size_t)N * Geo<N>::PS + (size_t)N * Geo<N>::PW + (size_t)2 * Geo<N>::VB * nk2 * Geo<N>::PC) * sizeof(cplx) + 16 * sizeof(unsigned long long);
}

}  // namespace fft8

namespace fft8 {
template <int N>
size_t smem_bytes_ring(int nk2, int cb = 1) {
  return ((size_t)cb * N * Geo<N>::PS + (size_t)N * Geo<N>::PW + (size_t)RingDepth<N>::value * nk2 * Geo<N>::PC) * sizeof(cplx) +
         (16 + 2 * RingDepth<N>::value) * sizeof(unsigned long long);
}
}  // namespace fft8
