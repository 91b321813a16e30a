// In-place mixed-radix (8,4,2,3,5) decimation-in-frequency FFT on lines held in shared memory (complex FP64).
//
// A pass of radix r on sub-length L (m = L/r) maps, for every block b and j < m,
//   x[bL + j + q m], q < r   ->   y_s = (sum_q x_q w_r^{qs}) w_L^{js}  stored at  bL + j + s m.
// After all passes the value X[k] sits at position perm[k] (mixed-radix digit reversal, computed on the host), so a
// caller that needs only a few frequencies (the pruned epsilon box of MTXEL, eq. 3 restricted to the
// epsilon sphere) just reads those positions.  Consecutive threads work on consecutive LINES, and the caller gives
// lines an odd pitch (in 16-byte elements), so every 128-bit shared-memory access is bank-conflict free in every pass.
#pragma once
#include <cuda_runtime.h>

namespace fftsm {

typedef double2 cplx;
constexpr int MAX_PASS = 12;

struct Plan {            // passed by value to kernels
  int n;
  int n_pass;
  int radix[MAX_PASS];
  const cplx* tw;        // dev [n]: exp(-+ 2 pi i k / n) for the direction the plan is used in
  const int* perm;       // dev [n]: position of frequency k after the in-place passes
};

__device__ __forceinline__ cplx cadd(cplx a, cplx b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ cplx csub(cplx a, cplx b) { return make_double2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ cplx cmul(cplx a, cplx b) {
  return make_double2(fma(a.x, b.x, -a.y * b.y), fma(a.x, b.y, a.y * b.x));
}
// multiply by -i (forward) or +i (inverse)
template <bool INV>
__device__ __forceinline__ cplx mul_mi(cplx a) { return INV ? make_double2(-a.y, a.x) : make_double2(a.y, -a.x); }

template <bool INV>
__device__ __forceinline__ void bfly2(cplx* x) {
  cplx a = x[0], b = x[1];
  x[0] = cadd(a, b); x[1] = csub(a, b);
}
template <bool INV>
__device__ __forceinline__ void bfly4(cplx& x0, cplx& x1, cplx& x2, cplx& x3) {
  cplx t0 = cadd(x0, x2), t1 = csub(x0, x2), t2 = cadd(x1, x3), t3 = mul_mi<INV>(csub(x1, x3));
  x0 = cadd(t0, t2); x2 = csub(t0, t2); x1 = cadd(t1, t3); x3 = csub(t1, t3);
}
template <bool INV>
__device__ __forceinline__ void bfly3(cplx* x) {
  const double s = 0.86602540378443864676;  // sqrt(3)/2
  cplx t1 = cadd(x[1], x[2]);
  cplx m1 = make_double2(x[0].x - 0.5 * t1.x, x[0].y - 0.5 * t1.y);
  cplx d = csub(x[1], x[2]);
  cplx m2 = mul_mi<INV>(make_double2(s * d.x, s * d.y));
  x[0] = cadd(x[0], t1); x[1] = cadd(m1, m2); x[2] = csub(m1, m2);
}
template <bool INV>
__device__ __forceinline__ void bfly5(cplx* x) {
  const double c1 = 0.30901699437494742410, c2 = -0.80901699437494742410;   // cos(2pi/5), cos(4pi/5)
  const double s1 = 0.95105651629515357212, s2 = 0.58778525229247312917;    // sin(2pi/5), sin(4pi/5)
  cplx a1 = cadd(x[1], x[4]), a2 = cadd(x[2], x[3]), b1 = csub(x[1], x[4]), b2 = csub(x[2], x[3]);
  cplx p1 = make_double2(x[0].x + c1 * a1.x + c2 * a2.x, x[0].y + c1 * a1.y + c2 * a2.y);
  cplx p2 = make_double2(x[0].x + c2 * a1.x + c1 * a2.x, x[0].y + c2 * a1.y + c1 * a2.y);
  cplx q1 = mul_mi<INV>(make_double2(s1 * b1.x + s2 * b2.x, s1 * b1.y + s2 * b2.y));
  cplx q2 = mul_mi<INV>(make_double2(s2 * b1.x - s1 * b2.x, s2 * b1.y - s1 * b2.y));
  x[0] = make_double2(x[0].x + a1.x + a2.x, x[0].y + a1.y + a2.y);
  x[1] = cadd(p1, q1); x[4] = csub(p1, q1);
  x[2] = cadd(p2, q2); x[3] = csub(p2, q2);
}
template <bool INV>
__device__ __forceinline__ void bfly8(cplx* x) {
  const double h = 0.70710678118654752440;
  bfly4<INV>(x[0], x[2], x[4], x[6]);  // E_s in x[0],x[2],x[4],x[6] (s = 0..3)
  bfly4<INV>(x[1], x[3], x[5], x[7]);  // O_s in x[1],x[3],x[5],x[7]
  // w8^s O_s : w8 = (1 -+ i)/sqrt2
  cplx o1 = x[3], o2 = x[5], o3 = x[7];
  cplx w1 = INV ? make_double2(h * (o1.x - o1.y), h * (o1.x + o1.y)) : make_double2(h * (o1.x + o1.y), h * (o1.y - o1.x));
  cplx w2 = mul_mi<INV>(o2);
  cplx w3 = INV ? make_double2(-h * (o3.x + o3.y), h * (o3.x - o3.y)) : make_double2(h * (o3.y - o3.x), -h * (o3.x + o3.y));
  cplx e0 = x[0], e1 = x[2], e2 = x[4], e3 = x[6], o0 = x[1];
  x[0] = cadd(e0, o0); x[4] = csub(e0, o0);
  x[1] = cadd(e1, w1); x[5] = csub(e1, w1);
  x[2] = cadd(e2, w2); x[6] = csub(e2, w2);
  x[3] = cadd(e3, w3); x[7] = csub(e3, w3);
}

template <int R, bool INV>
__device__ __forceinline__ void bfly(cplx* x) {
  if (R == 2) bfly2<INV>(x);
  else if (R == 3) bfly3<INV>(x);
  else if (R == 4) bfly4<INV>(x[0], x[1], x[2], x[3]);
  else if (R == 5) bfly5<INV>(x);
  else bfly8<INV>(x);
}

// One pass of radix R over n_lines lines.  Line l starts at base + line_pos(l) * line_pitch; elements of a line
// are elem_pitch apart.  line_idx (optional, shared or global memory) selects which lines take part (pruning).
template <int R, bool INV>
__device__ __forceinline__ void pass(cplx* base, int n, int L, const cplx* __restrict__ tw, int n_lines,
                                     const int* line_idx, int line_pitch, int elem_pitch, int tid, int nthr) {
  const int m = L / R;
  const int per_line = n / R;
  const int total = n_lines * per_line;
  const int tw_step = n / L;
  for (int idx = tid; idx < total; idx += nthr) {
    const int l = idx % n_lines;
    const int bj = idx / n_lines;
    const int b = bj / m, j = bj - b * m;
    cplx* p = base + (line_idx ? line_idx[l] : l) * line_pitch + (b * L + j) * elem_pitch;
    cplx x[R];
#pragma unroll
    for (int q = 0; q < R; q++) x[q] = p[q * m * elem_pitch];
    bfly<R, INV>(x);
    if (m > 1 && j > 0) {
#pragma unroll
      for (int s = 1; s < R; s++) x[s] = cmul(x[s], tw[j * s * tw_step]);
    }
#pragma unroll
    for (int q = 0; q < R; q++) p[q * m * elem_pitch] = x[q];
  }
}

// Full in-place transform of n_lines lines.  WARP = false: all threads of the CTA take part (tid/nthr = thread index
// and count), every pass ends with __syncthreads().  WARP = true: one warp transforms its own lines (tid = lane,
// nthr = 32) and only __syncwarp() separates the passes, so warps run unsynchronised with each other.
template <bool INV, bool WARP = false>
__device__ __forceinline__ void fft_lines(cplx* base, const Plan& pl, int n_lines, const int* line_idx, int line_pitch,
                                          int elem_pitch, int tid, int nthr) {
  int L = pl.n;
  for (int ps = 0; ps < pl.n_pass; ps++) {
    const int r = pl.radix[ps];
    switch (r) {
      case 8: pass<8, INV>(base, pl.n, L, pl.tw, n_lines, line_idx, line_pitch, elem_pitch, tid, nthr); break;
      case 4: pass<4, INV>(base, pl.n, L, pl.tw, n_lines, line_idx, line_pitch, elem_pitch, tid, nthr); break;
      case 2: pass<2, INV>(base, pl.n, L, pl.tw, n_lines, line_idx, line_pitch, elem_pitch, tid, nthr); break;
      case 3: pass<3, INV>(base, pl.n, L, pl.tw, n_lines, line_idx, line_pitch, elem_pitch, tid, nthr); break;
      default: pass<5, INV>(base, pl.n, L, pl.tw, n_lines, line_idx, line_pitch, elem_pitch, tid, nthr); break;
    }
    L /= r;
    if (WARP) __syncwarp(); else __syncthreads();
  }
}

}  // namespace fftsm
