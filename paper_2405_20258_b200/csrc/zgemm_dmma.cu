// Complex-FP64 GEMM / HERK on the FP64 tensor-core path of sm_100a (mma.sync.m8n8k4.f64 -> SASS DMMA.8x8x4).
//
// Serves CHI_SUM (PAPER.md:75 eq. 6, :127 eq. 13, :152 eq. 15), the projection M_s = M C_s (eq. 7),
// chi_s = M_s^H Delta M_s (eq. 8) and the dense products of the subspace iteration.
//
//   C[m][n] (+)= alpha rs[m] cs[n] sum_k w_k A^(m,k) opB(B^(n,k))
//
// One complex MAC = 4 real DMMAs on (re, im) fragments:  Cre += Ar Br + Ai Bi ; Cim += Ai Br - Ar Bi  (opB = conj).
// The diagonal weight w_k (Delta of eq. 5 in the D(i omega) form, written once per block by pair_weights) rides the
// cp.async ring with the operand tiles and is fused into the A fragment after it is read
// from shared memory; v^1/2 is fused into the epilogue (rs, cs).  Operand tiles are staged global -> shared with
// cp.async (16 B = one complex element) in a 2-3 stage ring, in their native interleaved layout; padding makes the
// 128-bit fragment loads bank-conflict free (leading dimension = 2 mod 8 elements for [k][m], 4 mod 8 for [m][k]).
#include <algorithm>

#include <cuda.h>
#include <cudaTypedefs.h>

#include "rpa_internal.h"

namespace {

constexpr int BM = 64, BN = 64, BK = 16;
constexpr int NTHREADS = 128;          // 4 warps, 2 x 2, warp tile 32 x 32 complex
constexpr int LD_KM = BM + 2;          // [k][m] layout: elements per k row
constexpr int LD_MK = BK + 4;          // [m][k] layout: elements per m row
constexpr int TILE_KM = BK * LD_KM;    // 1056 elements
constexpr int TILE_MK = BM * LD_MK;    // 1280 elements

__device__ __forceinline__ void dmma(double& d0, double& d1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
               : "+d"(d0), "+d"(d1)
               : "d"(a), "d"(b));
}
__device__ __forceinline__ void cp_async16(void* smem, const void* gmem, bool valid) {
  unsigned s = (unsigned)__cvta_generic_to_shared(smem);
  int sz = valid ? 16 : 0;
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(s), "l"(gmem), "r"(sz));
}
__device__ __forceinline__ void cp_async8(void* smem, const void* gmem, bool valid) {   // one double, zero-filled if !valid
  unsigned s = (unsigned)__cvta_generic_to_shared(smem);
  int sz = valid ? 8 : 0;
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;\n" ::"r"(s), "l"(gmem), "r"(sz));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N)); }

struct KArgs {
  const cplx* A; long long lda;
  const cplx* B; long long ldb;
  cplx* C; long long ldc;
  int M, N, K;
  int herm, accumulate, atomic;
  double alpha;
  const double* rs; const double* cs;
  const double* wk; long long strideW;
  long long strideA, strideB, strideC;
  int tiles_n, kt_per_split, n_kt;
  int batch_fastest;   // zherk_tma_kernel only: grid = (batch, tiles, split) instead of (tiles, split, batch)
};

template <bool KM>
__device__ __forceinline__ void load_tile(cplx* s, const cplx* g, long long ld, int r0, int rmax, int k0, int kmax,
                                          int tid) {
  // r = the m (or n) index, k = contraction index.  8 x 16-byte cp.async per thread.
#pragma unroll
  for (int i = 0; i < (BM * BK) / NTHREADS; i++) {
    int idx = tid + i * NTHREADS;
    int r, k;
    if (KM) { k = idx / BM; r = idx % BM; } else { r = idx / BK; k = idx % BK; }
    bool ok = (r0 + r < rmax) && (k0 + k < kmax);
    const cplx* src = g;
    if (ok) src = KM ? g + (long long)(k0 + k) * ld + (r0 + r) : g + (long long)(r0 + r) * ld + (k0 + k);
    cplx* dst = KM ? s + k * LD_KM + r : s + r * LD_MK + k;
    cp_async16(dst, src, ok);
  }
}

// The DMMAs of one warp on one staged k-tile.  TRI = false: an NI x NJ block of 8 x 8 fragments at (mb, nb) -- 4 x 4 is
// the 32 x 32 warp tile, 3 x 4 / 2 x 4 / 1 x 4 the warp's share of a ragged last tile row, 3 x 3 a share of a diagonal
// Hermitian tile.  TRI = true: three 2 x 2 lower fragment triangles on the diagonal at 0, 24, 48 (slot [t][0] =
// (24t, 24t), [t][1] = (24t+8, 24t), [t][2] = (24t+8, 24t+8)).  3 x 3 x 3 + TRI tile the 36 fragments on or below the
// diagonal of a diagonal Hermitian tile, 9 per warp (see the kernel).
template <bool A_KM, bool B_KN, bool CONJ_B, int NI, int NJ, bool TRI, int BOX = 0, bool HASW = true>
__device__ __forceinline__ void mma_ktile(const cplx* __restrict__ a_s, const cplx* __restrict__ b_s,
                                          const double* __restrict__ w_s, int g, int q, int mb, int nb,
                                          double (&cre)[4][4][2], double (&cim)[4][4][2], bool skip_upper = false) {
  constexpr int NA = TRI ? 6 : NI, NB = TRI ? 6 : NJ;   // fragments loaded per operand
#pragma unroll
  for (int k4 = 0; k4 < BK / 4; k4++) {
    const int k = k4 * 4 + q;
    const double w = HASW ? w_s[k] : 1.0;
    double ar[NA], ai[NA], br[NB], bi[NB];
#pragma unroll
    for (int i = 0; i < NA; i++) {
      const int m = TRI ? 24 * (i >> 1) + 8 * (i & 1) + g : mb + i * 8 + g;
      // BOX: the TMA layout of a [k][m] tile, 8 boxes of [16 k][8 m] with the 128-byte swizzle: element (k, m) sits in box
      // m >> 3, row k, 16-byte chunk (m & 7) ^ (k & 7).  The caller passes g already permuted (see zherk_tma_kernel).
      // BOX 2: the TMA layout of an [m][k] tile, 2 boxes of [64 m][8 k], swizzled: element (m, k) in box k >> 3, row m, chunk (k & 7) ^ (m & 7)
      cplx a = BOX == 1 ? a_s[((m >> 3) << 7) + k * 8 + ((m & 7) ^ (k & 7))]
             : BOX == 2 ? a_s[((k >> 3) << 9) + m * 8 + ((k & 7) ^ (m & 7))]
             : A_KM ? a_s[k * LD_KM + m] : a_s[m * LD_MK + k];
      ar[i] = HASW ? a.x * w : a.x; ai[i] = HASW ? a.y * w : a.y;
    }
#pragma unroll
    for (int j = 0; j < NB; j++) {
      const int n = TRI ? 24 * (j >> 1) + 8 * (j & 1) + g : nb + j * 8 + g;
      cplx b = BOX == 1 ? b_s[((n >> 3) << 7) + k * 8 + ((n & 7) ^ (k & 7))]
             : BOX == 2 ? b_s[((k >> 3) << 9) + n * 8 + ((k & 7) ^ (n & 7))]
             : B_KN ? b_s[k * LD_KM + n] : b_s[n * LD_MK + k];
      br[j] = b.x; bi[j] = b.y;
    }
    // a conj(b): re += ar br + ai bi, im += ai br - ar bi;  a b: re += ar br - ai bi, im += ai br + ar bi.  The sign is
    // a compile-time negation of the A operand, which DMMA takes as an operand modifier (no FP64 instruction).
#pragma unroll
    for (int i = 0; i < NI; i++)
#pragma unroll
      for (int j = 0; j < NJ; j++) {
        const int ia = TRI ? 2 * i + (j >= 1) : i, jb = TRI ? 2 * i + (j == 2) : j;
        if (skip_upper && j > i) continue;
        dmma(cre[i][j][0], cre[i][j][1], ar[ia], br[jb]);
        dmma(cim[i][j][0], cim[i][j][1], ai[ia], br[jb]);
      }
#pragma unroll
    for (int i = 0; i < NI; i++)
#pragma unroll
      for (int j = 0; j < NJ; j++) {
        const int ia = TRI ? 2 * i + (j >= 1) : i, jb = TRI ? 2 * i + (j == 2) : j;
        if (skip_upper && j > i) continue;
        dmma(cre[i][j][0], cre[i][j][1], CONJ_B ? ai[ia] : -ai[ia], bi[jb]);
        dmma(cim[i][j][0], cim[i][j][1], CONJ_B ? -ar[ia] : ar[ia], bi[jb]);
      }
  }
}

// HERM: compiled for Hermitian updates (p.herm set): only then do the diagonal-tile modes exist in the main loop.
template <bool A_KM, bool B_KN, bool CONJ_B, int STAGES, bool HERM>
__global__ void __launch_bounds__(NTHREADS, 2) zgemm_dmma_kernel(KArgs p) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  constexpr int TA = A_KM ? TILE_KM : TILE_MK;
  constexpr int TB = B_KN ? TILE_KM : TILE_MK;
  cplx* sA = reinterpret_cast<cplx*>(smem_raw);
  cplx* sB = sA + STAGES * TA;
  double* sW = reinterpret_cast<double*>(sB + STAGES * TB);

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int wm = warp >> 1, wn = warp & 1;
  const int g = lane >> 2, q = lane & 3;

  // tile coordinates
  int tm, tn;
  if (p.herm) {
    int t = blockIdx.x;
    tm = (int)((sqrt(8.0 * t + 1.0) - 1.0) * 0.5);
    while ((tm + 1) * (tm + 2) / 2 <= t) tm++;
    while (tm * (tm + 1) / 2 > t) tm--;
    tn = t - tm * (tm + 1) / 2;
  } else {
    tm = blockIdx.x / p.tiles_n;
    tn = blockIdx.x % p.tiles_n;
  }
  const int m0 = tm * BM, n0 = tn * BN;
  const int batch = blockIdx.z;
  const cplx* A = p.A + batch * p.strideA;
  const cplx* B = p.B + batch * p.strideB;
  cplx* C = p.C + batch * p.strideC;
  const int kt0 = blockIdx.y * p.kt_per_split;
  const int kt1 = min(p.n_kt, kt0 + p.kt_per_split);
  const int nkt = kt1 - kt0;
  if (nkt <= 0) return;
  const double* wk = p.wk ? p.wk + batch * p.strideW : nullptr;

  auto load_stage = [&](int stage, int kt) {
    const int k0 = kt * BK;
    load_tile<A_KM>(sA + stage * TA, A, p.lda, m0, p.M, k0, p.K, tid);
    load_tile<B_KN>(sB + stage * TB, B, p.ldb, n0, p.N, k0, p.K, tid);
    if (tid < BK) {   // the BK weights of this k-tile (zero beyond K, so ragged tiles add nothing)
      double* dst = sW + stage * BK + tid;
      const int kk = k0 + tid;
      if (wk) cp_async8(dst, kk < p.K ? wk + kk : wk, kk < p.K);
      else dst[0] = 1.0;   // operand tiles are zero-filled beyond K
    }
  };

  // A diagonal tile of a Hermitian update stores only its lower triangle: 36 of its 64 8 x 8 fragments (the upper ones
  // are mirrored in the epilogue).  Its four warps share them 9 each instead of keeping their 32 x 32 blocks, so the
  // CTA issues 9/16 of a full tile's DMMAs *and finishes in 9/16 of its time*: warp 0 takes the three 2 x 2 fragment
  // triangles on the diagonal (mode 2), warps 1-3 the 3 x 3 blocks at fragment rows 2-4 x columns 0-2, rows 5-7 x
  // columns 0-2 and rows 5-7 x columns 3-5 (mode 1).
  int mode = 0, mb = wm * 32, nb = wn * 32;
  if (HERM && tm == tn) {
    if (warp == 0) { mode = 2; mb = nb = 0; }
    else { mode = 1; mb = warp == 1 ? 16 : 40; nb = warp == 3 ? 24 : 0; }
  }
  // A ragged last tile row (M not a multiple of 64) has rv < 8 valid fragment rows: the two warp rows take ceil(rv / 2)
  // of them each instead of 4 (N_eig = 300: 3, N_eig = 2400: 2), the rest of the tile is zero and never stored.
  int ni = mode == 0 ? 4 : 3;
  // Never true in the kernels compiled without HERM (launch() sends every Hermitian update to the HERM kernels).  It
  // predicates the DMMAs above the fragment diagonal of the general 4 x 4 shape, as the first version of this kernel did
  // for diagonal tiles: ptxas schedules the main loop measurably better with the predicate in place (projection at
  // configs[2]: 1.76 s without, 1.72 s with), so it stays.
  const bool old_diag_warp = p.herm && tm == tn && wm == wn;
  if (HERM && mode == 0 && p.M - m0 < BM - 8) {
    ni = (((p.M - m0 + 7) >> 3) + 1) >> 1;
    mb = wm * ni * 8;
  }
  double cre[4][4][2], cim[4][4][2];
#pragma unroll
  for (int i = 0; i < 4; i++)
#pragma unroll
    for (int j = 0; j < 4; j++) { cre[i][j][0] = cre[i][j][1] = 0.0; cim[i][j][0] = cim[i][j][1] = 0.0; }

#pragma unroll
  for (int s = 0; s < STAGES - 1; s++) {
    if (s < nkt) load_stage(s, kt0 + s);
    cp_async_commit();
  }

  for (int it = 0; it < nkt; it++) {
    cp_async_wait<STAGES - 2>();
    __syncthreads();
    {
      int nx = it + STAGES - 1;
      if (nx < nkt) load_stage(nx % STAGES, kt0 + nx);
      cp_async_commit();
    }
    const int st = it % STAGES;
    const cplx* a_s = sA + st * TA;
    const cplx* b_s = sB + st * TB;
    const double* w_s = sW + st * BK;
    if (!HERM) mma_ktile<A_KM, B_KN, CONJ_B, 4, 4, false>(a_s, b_s, w_s, g, q, mb, nb, cre, cim, old_diag_warp);
    else if (mode == 0) {
      if (ni == 4) mma_ktile<A_KM, B_KN, CONJ_B, 4, 4, false>(a_s, b_s, w_s, g, q, mb, nb, cre, cim);
      else if (ni == 3) mma_ktile<A_KM, B_KN, CONJ_B, 3, 4, false>(a_s, b_s, w_s, g, q, mb, nb, cre, cim);
      else if (ni == 2) mma_ktile<A_KM, B_KN, CONJ_B, 2, 4, false>(a_s, b_s, w_s, g, q, mb, nb, cre, cim);
      else mma_ktile<A_KM, B_KN, CONJ_B, 1, 4, false>(a_s, b_s, w_s, g, q, mb, nb, cre, cim);
    } else if (mode == 1) mma_ktile<A_KM, B_KN, CONJ_B, 3, 3, false>(a_s, b_s, w_s, g, q, mb, nb, cre, cim);
    else mma_ktile<A_KM, B_KN, CONJ_B, 3, 3, true>(a_s, b_s, w_s, g, q, mb, nb, cre, cim);
  }
  cp_async_wait<0>();

  // epilogue: scale, (mirror,) store / accumulate
  const bool diag_tile = p.herm && (tm == tn);
#pragma unroll
  for (int i = 0; i < 4; i++) {
#pragma unroll
    for (int j = 0; j < 4; j++) {
      if (HERM && (i >= ni || (mode != 0 && j == 3))) continue;   // accumulator slots this warp does not use
      const int ro = HERM && mode == 2 ? 24 * i + (j >= 1 ? 8 : 0) : mb + i * 8;
      const int co = HERM && mode == 2 ? 24 * i + (j == 2 ? 8 : 0) : nb + j * 8;
      const int r = m0 + ro + g;
      if (r >= p.M) continue;
      const double sr = p.alpha * (p.rs ? p.rs[r] : 1.0);
#pragma unroll
      for (int e = 0; e < 2; e++) {
        const int c = n0 + co + 2 * q + e;
        if (c >= p.N) continue;
        const double sc = sr * (p.cs ? p.cs[c] : 1.0);
        double vr = sc * cre[i][j][e], vi = sc * cim[i][j][e];
        if (diag_tile && r == c) vi = 0.0;
        // Hermitian mode: the lower triangle (c <= r) is the truth, the upper one its exact conjugate mirror
        // (w_k is fused into the A side only, so (r,c) and (c,r) computed separately would differ in the last bit).
        if (p.herm && c > r) continue;
        cplx* dst = C + (long long)r * p.ldc + c;
        if (p.atomic) {
          // split-K: partial sums meet in global memory; herm_mirror_kernel fills the upper triangle afterwards
          atomicAdd(&dst->x, vr); atomicAdd(&dst->y, vi);
          continue;
        }
        if (p.accumulate) {
          cplx o = *dst; o.x += vr; o.y += vi; vr = o.x; vi = o.y;
        }
        *dst = make_double2(vr, vi);
        if (p.herm && c < r) C[(long long)c * p.ldc + r] = make_double2(vr, -vi);
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------------------------
// TMA-staged variant of the Hermitian [k][m] x [k][n] update (CHI_SUM, chi_s): the same tile, warp shares and epilogue
// as zgemm_dmma_kernel<1,1,1,3,1>, but the operand panels arrive by cp.async.bulk.tensor (one elected thread issues
// 8 + 8 box loads and one weight row per k-tile) into a 3-stage ring guarded by mbarriers: full[s] (transaction bytes)
// and empty[s] (one arrival per warp) -- no per-thread address arithmetic, no cp.async groups and no block barrier in the
// main loop.  A [k][64] panel is loaded as 8 boxes of [16 k][8 m] complex (128-byte rows) with the 128-byte swizzle, and the
// fragment row g of the MMA is mapped to row rho(g) = (g >> 1) + 4 (g & 1) of its 8-row group: a quarter-warp (two g, four
// k) then touches 8 different 16-byte bank groups -- conflict-free without padding.  (Unswizzled boxes are 4-way
// conflicted: all rows of a box share their bank alignment; the swizzle alone still pairs g = 2a, 2a + 1 in one half.)
constexpr int TMA_STAGES = 3;
constexpr int TMA_TILE = BK * BM;   // 1024 complex per operand tile

__device__ __forceinline__ void tma_mbar_init(unsigned long long* bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void tma_mbar_arrive(unsigned long long* bar) {
  asm volatile("{\n .reg .b64 st;\n mbarrier.arrive.shared::cta.b64 st, [%0];\n}\n" ::"r"((unsigned)__cvta_generic_to_shared(bar)) : "memory");
}
__device__ __forceinline__ void tma_mbar_expect(unsigned long long* bar, unsigned bytes) {
  asm volatile("{\n .reg .b64 st;\n mbarrier.arrive.expect_tx.shared::cta.b64 st, [%0], %1;\n}\n" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void tma_mbar_wait(unsigned long long* bar, unsigned parity) {
  const unsigned a = (unsigned)__cvta_generic_to_shared(bar);
  unsigned ok;
  do {
    asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}\n"
                 : "=r"(ok) : "r"(a), "r"(parity) : "memory");
  } while (!ok);
}
__device__ __forceinline__ void tma_load_2d(void* smem, const CUtensorMap* map, int x, int y, unsigned long long* bar) {
  asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];\n" ::
               "r"((unsigned)__cvta_generic_to_shared(smem)), "l"(map), "r"(x), "r"(y), "r"((unsigned)__cvta_generic_to_shared(bar)) : "memory");
}

struct TmaMaps { CUtensorMap a; CUtensorMap w; };   // operand [K][2 M doubles], weights [batch][K doubles]

__global__ void __launch_bounds__(NTHREADS, 2) zherk_tma_kernel(KArgs p, const __grid_constant__ TmaMaps maps) {
  extern __shared__ __align__(1024) unsigned char smem_tma[];
  cplx* sA = reinterpret_cast<cplx*>(smem_tma);
  cplx* sB = sA + TMA_STAGES * TMA_TILE;
  double* sW = reinterpret_cast<double*>(sB + TMA_STAGES * TMA_TILE);
  unsigned long long* full = reinterpret_cast<unsigned long long*>(sW + TMA_STAGES * BK);
  unsigned long long* empty = full + TMA_STAGES;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int wm = warp >> 1, wn = warp & 1;
  const int q = lane & 3;
  const int g = ((lane >> 2) >> 1) + 4 * ((lane >> 2) & 1);   // rho(fragment row): the tile row this lane's fragment row maps to
  int tm, tn;
  {
    const int t = p.batch_fastest ? blockIdx.y : blockIdx.x;
    tm = (int)((sqrt(8.0 * t + 1.0) - 1.0) * 0.5);
    while ((tm + 1) * (tm + 2) / 2 <= t) tm++;
    while (tm * (tm + 1) / 2 > t) tm--;
    tn = t - tm * (tm + 1) / 2;
  }
  const int m0 = tm * BM, n0 = tn * BN;
  const bool diag = tm == tn;
  // batch_fastest (chi_s: one operand, n_w weight rows): the CTAs of one tile and all frequencies are neighbours in the
  // launch order, so the CTAs resident together read the SAME operand panels at the same pace -- L2 serves 15 of 16
  const int batch = p.batch_fastest ? blockIdx.x : blockIdx.z;
  cplx* C = p.C + batch * p.strideC;
  const int kt0 = (p.batch_fastest ? blockIdx.z : blockIdx.y) * p.kt_per_split;
  const int kt1 = min(p.n_kt, kt0 + p.kt_per_split);
  const int nkt = kt1 - kt0;
  if (nkt <= 0) return;
  if (tid == 0) {
    for (int s = 0; s < TMA_STAGES; s++) { tma_mbar_init(full + s, 1); tma_mbar_init(empty + s, NTHREADS / 32); }
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
  }
  __syncthreads();
  const unsigned stage_bytes = (unsigned)((diag ? 1 : 2) * TMA_TILE * sizeof(cplx) + BK * sizeof(double));
  auto issue = [&](int stage, int kt) {   // one thread
    const int k0 = kt * BK;
    tma_mbar_expect(full + stage, stage_bytes);
#pragma unroll
    for (int b = 0; b < 8; b++) tma_load_2d(sA + stage * TMA_TILE + b * 128, &maps.a, 2 * (m0 + 8 * b), k0, full + stage);
    if (!diag) {
#pragma unroll
      for (int b = 0; b < 8; b++) tma_load_2d(sB + stage * TMA_TILE + b * 128, &maps.a, 2 * (n0 + 8 * b), k0, full + stage);
    }
    tma_load_2d(sW + stage * BK, &maps.w, k0, batch, full + stage);
  };

  int mode = 0, mb = wm * 32, nb = wn * 32;
  if (diag) {
    if (warp == 0) { mode = 2; mb = nb = 0; }
    else { mode = 1; mb = warp == 1 ? 16 : 40; nb = warp == 3 ? 24 : 0; }
  }
  int ni = mode == 0 ? 4 : 3;
  if (mode == 0 && p.M - m0 < BM - 8) {
    ni = (((p.M - m0 + 7) >> 3) + 1) >> 1;
    mb = wm * ni * 8;
  }
  double cre[4][4][2], cim[4][4][2];
#pragma unroll
  for (int i = 0; i < 4; i++)
#pragma unroll
    for (int j = 0; j < 4; j++) { cre[i][j][0] = cre[i][j][1] = 0.0; cim[i][j][0] = cim[i][j][1] = 0.0; }

  if (tid == 0)
    for (int s = 0; s < TMA_STAGES - 1 && s < nkt; s++) issue(s, kt0 + s);

  // Full off-diagonal tiles (the great majority) run a loop of their own with the one 4 x 4 warp shape and no shape
  // dispatch inside (a CTA-uniform choice, made once): its body holds exactly one DMMA schedule, and the kernel is 2-3 %
  // faster for it (CHI_SUM(0) 2.738 -> 2.679 s, chi_s 4.264 -> 4.149 s per step at configs[2]).  Diagonal and ragged
  // tiles take the general loop below; hoisting their shapes out as well was no further gain (more registers).
  const bool plain_tile = !diag && p.M - m0 >= BM - 8;
  if (plain_tile) {
    for (int it = 0; it < nkt; it++) {
      const int st = it % TMA_STAGES;
      if (tid == 0) {
        const int nx = it + TMA_STAGES - 1;
        if (nx < nkt) {
          const int sx = nx % TMA_STAGES;
          if (nx >= TMA_STAGES) tma_mbar_wait(empty + sx, (unsigned)(((nx / TMA_STAGES) - 1) & 1));
          issue(sx, kt0 + nx);
        }
      }
      __syncwarp();
      tma_mbar_wait(full + st, (unsigned)((it / TMA_STAGES) & 1));
      mma_ktile<true, true, true, 4, 4, false, 1>(sA + st * TMA_TILE, sB + st * TMA_TILE, sW + st * BK, g, q, mb, nb, cre, cim);
      __syncwarp();
      if (lane == 0) tma_mbar_arrive(empty + st);
    }
  } else
  for (int it = 0; it < nkt; it++) {
    const int st = it % TMA_STAGES;
    if (tid == 0) {   // refill the stage all warps left one iteration ago
      const int nx = it + TMA_STAGES - 1;
      if (nx < nkt) {
        const int sx = nx % TMA_STAGES;
        if (nx >= TMA_STAGES) tma_mbar_wait(empty + sx, (unsigned)(((nx / TMA_STAGES) - 1) & 1));
        issue(sx, kt0 + nx);
      }
    }
    __syncwarp();
    tma_mbar_wait(full + st, (unsigned)((it / TMA_STAGES) & 1));
    const cplx* a_s = sA + st * TMA_TILE;
    const cplx* b_s = diag ? a_s : sB + st * TMA_TILE;
    const double* w_s = sW + st * BK;
    if (mode == 0) {
      if (ni == 4) mma_ktile<true, true, true, 4, 4, false, 1>(a_s, b_s, w_s, g, q, mb, nb, cre, cim);
      else if (ni == 3) mma_ktile<true, true, true, 3, 4, false, 1>(a_s, b_s, w_s, g, q, mb, nb, cre, cim);
      else if (ni == 2) mma_ktile<true, true, true, 2, 4, false, 1>(a_s, b_s, w_s, g, q, mb, nb, cre, cim);
      else mma_ktile<true, true, true, 1, 4, false, 1>(a_s, b_s, w_s, g, q, mb, nb, cre, cim);
    } else if (mode == 1) mma_ktile<true, true, true, 3, 3, false, 1>(a_s, b_s, w_s, g, q, mb, nb, cre, cim);
    else mma_ktile<true, true, true, 3, 3, true, 1>(a_s, b_s, w_s, g, q, mb, nb, cre, cim);
    __syncwarp();
    if (lane == 0) tma_mbar_arrive(empty + st);
  }

#pragma unroll
  for (int i = 0; i < 4; i++) {
#pragma unroll
    for (int j = 0; j < 4; j++) {
      if (i >= ni || (mode != 0 && j == 3)) continue;
      const int ro = mode == 2 ? 24 * i + (j >= 1 ? 8 : 0) : mb + i * 8;
      const int co = mode == 2 ? 24 * i + (j == 2 ? 8 : 0) : nb + j * 8;
      const int r = m0 + ro + g;
      if (r >= p.M) continue;
      const double sr = p.alpha * (p.rs ? p.rs[r] : 1.0);
#pragma unroll
      for (int e = 0; e < 2; e++) {
        const int cf = 2 * q + e;                                    // fragment column -> tile column, same rho
        const int c = n0 + co + (cf >> 1) + 4 * (cf & 1);
        if (c >= p.N || c > r) continue;
        const double sc = sr * (p.cs ? p.cs[c] : 1.0);
        double vr = sc * cre[i][j][e], vi = sc * cim[i][j][e];
        if (r == c) vi = 0.0;
        cplx* dst = C + (long long)r * p.ldc + c;
        if (p.atomic) { atomicAdd(&dst->x, vr); atomicAdd(&dst->y, vi); continue; }
        if (p.accumulate) { cplx o = *dst; vr += o.x; vi += o.y; }
        *dst = make_double2(vr, vi);
        if (c < r) C[(long long)c * p.ldc + r] = make_double2(vr, -vi);
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------------------------
// TMA-staged general product for operands stored [m][k] and [n][k] (k contiguous): the projection B_vc = C^H v^1/2 M_vc
// (eq. 7), C[m][n] = sum_k w_k A[m][k] conj(B[n][k]).  Same ring, barriers and warp tiles as
// zherk_tma_kernel; a 64 x 16 operand tile arrives as two boxes of [64 rows][8 k] (128-byte rows, 128-byte swizzle), and
// with the same fragment-row map rho a quarter-warp's fragment load touches 8 different bank groups.  One k-split, plain
// stores (the projection has tens of thousands of tiles), rows / columns / k beyond the matrix are zero-filled by TMA.
struct TmaMapsMK { CUtensorMap a; CUtensorMap b; CUtensorMap w; };

template <bool HASW>
__global__ void __launch_bounds__(NTHREADS, 2) zgemm_tma_mk_kernel(KArgs p, const __grid_constant__ TmaMapsMK maps) {
  extern __shared__ __align__(1024) unsigned char smem_tma[];
  cplx* sA = reinterpret_cast<cplx*>(smem_tma);
  cplx* sB = sA + TMA_STAGES * TMA_TILE;
  double* sW = reinterpret_cast<double*>(sB + TMA_STAGES * TMA_TILE);
  unsigned long long* full = reinterpret_cast<unsigned long long*>(sW + TMA_STAGES * BK);
  unsigned long long* empty = full + TMA_STAGES;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int wm = warp >> 1, wn = warp & 1;
  const int q = lane & 3;
  const int g = ((lane >> 2) >> 1) + 4 * ((lane >> 2) & 1);   // rho(fragment row), see zherk_tma_kernel
  const int tm = blockIdx.x / p.tiles_n, tn = blockIdx.x % p.tiles_n;
  const int m0 = tm * BM, n0 = tn * BN;
  const int nkt = p.n_kt;
  if (tid == 0) {
    for (int s = 0; s < TMA_STAGES; s++) { tma_mbar_init(full + s, 1); tma_mbar_init(empty + s, NTHREADS / 32); }
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
  }
  __syncthreads();
  constexpr unsigned stage_bytes = (unsigned)(2 * TMA_TILE * sizeof(cplx) + (HASW ? BK * sizeof(double) : 0));
  auto issue = [&](int stage, int kt) {   // one thread
    const int k0 = kt * BK;
    tma_mbar_expect(full + stage, stage_bytes);
#pragma unroll
    for (int b = 0; b < 2; b++) {
      tma_load_2d(sA + stage * TMA_TILE + b * 512, &maps.a, 2 * (k0 + 8 * b), m0, full + stage);
      tma_load_2d(sB + stage * TMA_TILE + b * 512, &maps.b, 2 * (k0 + 8 * b), n0, full + stage);
    }
    if (HASW) tma_load_2d(sW + stage * BK, &maps.w, k0, 0, full + stage);
  };
  const int mb = wm * 32, nb = wn * 32;
  double cre[4][4][2], cim[4][4][2];
#pragma unroll
  for (int i = 0; i < 4; i++)
#pragma unroll
    for (int j = 0; j < 4; j++) { cre[i][j][0] = cre[i][j][1] = 0.0; cim[i][j][0] = cim[i][j][1] = 0.0; }

  if (tid == 0)
    for (int s = 0; s < TMA_STAGES - 1 && s < nkt; s++) issue(s, s);
  for (int it = 0; it < nkt; it++) {
    const int st = it % TMA_STAGES;
    if (tid == 0) {   // refill the stage all warps left one iteration ago
      const int nx = it + TMA_STAGES - 1;
      if (nx < nkt) {
        const int sx = nx % TMA_STAGES;
        if (nx >= TMA_STAGES) tma_mbar_wait(empty + sx, (unsigned)(((nx / TMA_STAGES) - 1) & 1));
        issue(sx, nx);
      }
    }
    __syncwarp();
    tma_mbar_wait(full + st, (unsigned)((it / TMA_STAGES) & 1));
    mma_ktile<false, false, true, 4, 4, false, 2, HASW>(sA + st * TMA_TILE, sB + st * TMA_TILE, sW + st * BK, g, q, mb, nb, cre, cim);
    __syncwarp();
    if (lane == 0) tma_mbar_arrive(empty + st);
  }
#pragma unroll
  for (int i = 0; i < 4; i++) {
    const int r = m0 + mb + i * 8 + g;
    if (r >= p.M) continue;
#pragma unroll
    for (int j = 0; j < 4; j++) {
#pragma unroll
      for (int e = 0; e < 2; e++) {
        const int cf = 2 * q + e;                                    // fragment column -> tile column, same rho
        const int c = n0 + nb + j * 8 + (cf >> 1) + 4 * (cf & 1);
        if (c >= p.N) continue;
        p.C[(long long)r * p.ldc + c] = make_double2(p.alpha * cre[i][j][e], p.alpha * cim[i][j][e]);
      }
    }
  }
}

// C[c][r] = conj(C[r][c]) for c > r (after a split-K Hermitian accumulation)
__global__ void herm_mirror_kernel(cplx* C, long long ldc, long long strideC, int n) {
  cplx* c = C + blockIdx.z * strideC;
  const int col = blockIdx.x * blockDim.x + threadIdx.x, row = blockIdx.y;   // row < col: upper element
  if (col < n && col > row) {
    cplx v = c[(long long)col * ldc + row];
    c[(long long)row * ldc + col] = make_double2(v.x, -v.y);
  }
}

template <bool A_KM, bool B_KN, bool CONJ_B, bool HERM>
int launch_h(rpa_ctx* ctx, const KArgs& ka, dim3 grid) {
  constexpr int STAGES = (A_KM || B_KN) ? 3 : 2;
  constexpr int TA = A_KM ? TILE_KM : TILE_MK;
  constexpr int TB = B_KN ? TILE_KM : TILE_MK;
  constexpr size_t smem = (size_t)STAGES * (TA + TB) * sizeof(cplx) + STAGES * BK * sizeof(double);
  auto kern = zgemm_dmma_kernel<A_KM, B_KN, CONJ_B, STAGES, HERM>;
  if (ctx->attr_once(RPA_ATTR_ZGEMM + (A_KM ? 1 : 0) + (B_KN ? 2 : 0) + (CONJ_B ? 4 : 0) + (HERM ? 8 : 0)))
    RPA_CUDA(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  kern<<<grid, NTHREADS, smem, ctx->stream>>>(ka);
  RPA_LAUNCH_CHECK(ctx);
  return RPA_OK;
}

// Tensor maps for zherk_tma_kernel.  Returns RPA_OK and sets *ok = false when the operands do not meet TMA's alignment
// rules (the caller then takes the cp.async kernel).
int launch_tma(rpa_ctx* ctx, const KArgs& ka, dim3 grid, int batch, bool* ok) {
  *ok = false;
  if (!ctx->tma_encode) {
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn) { (void)cudaGetLastError(); return RPA_OK; }
    ctx->tma_encode = fn;
  }
  auto encode = reinterpret_cast<PFN_cuTensorMapEncodeTiled>(ctx->tma_encode);
  if (!ka.wk || ((uintptr_t)ka.A & 15) || ((uintptr_t)ka.wk & 15) || (ka.strideW * 8) % 16 != 0 || (batch > 1 && ka.strideA != 0)) return RPA_OK;
  TmaMaps maps;
  {
    cuuint64_t dims[2] = {(cuuint64_t)2 * ka.M, (cuuint64_t)ka.K};
    cuuint64_t strides[1] = {(cuuint64_t)ka.lda * sizeof(cplx)};
    cuuint32_t box[2] = {16, (cuuint32_t)BK};
    cuuint32_t es[2] = {1, 1};
    if (encode(&maps.a, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, (void*)ka.A, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
               CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS) return RPA_OK;
  }
  {
    cuuint64_t dims[2] = {(cuuint64_t)ka.K, (cuuint64_t)batch};
    cuuint64_t strides[1] = {(cuuint64_t)(batch > 1 ? ka.strideW : ka.K + (ka.K & 1)) * sizeof(double)};
    cuuint32_t box[2] = {(cuuint32_t)BK, 1};
    cuuint32_t es[2] = {1, 1};
    if (encode(&maps.w, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, (void*)ka.wk, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
               CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS) return RPA_OK;
  }
  constexpr size_t smem = (size_t)TMA_STAGES * 2 * TMA_TILE * sizeof(cplx) + TMA_STAGES * BK * sizeof(double) + 2 * TMA_STAGES * sizeof(unsigned long long) + 128;
  static_assert((TMA_TILE * sizeof(cplx)) % 1024 == 0, "swizzled boxes need 1024-byte aligned stages");
  if (ctx->attr_once(RPA_ATTR_ZHERK_TMA))
    RPA_CUDA(ctx, cudaFuncSetAttribute(zherk_tma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  KArgs kb = ka;
  kb.batch_fastest = batch > 1 && ka.strideA == 0 && grid.x <= 65535 ? 1 : 0;
  if (kb.batch_fastest) grid = dim3(grid.z, grid.x, grid.y);
  zherk_tma_kernel<<<grid, NTHREADS, smem, ctx->stream>>>(kb, maps);
  RPA_LAUNCH_CHECK(ctx);
  *ok = true;
  return RPA_OK;
}

// Tensor maps + launch of zgemm_tma_mk_kernel; *ok = false (and nothing launched) when TMA's rules are not met.
int launch_tma_mk(rpa_ctx* ctx, const KArgs& ka, dim3 grid, bool* ok) {
  *ok = false;
  if (!ctx->tma_encode) {
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn) { (void)cudaGetLastError(); return RPA_OK; }
    ctx->tma_encode = fn;
  }
  auto encode = reinterpret_cast<PFN_cuTensorMapEncodeTiled>(ctx->tma_encode);
  if (((uintptr_t)ka.A & 15) || ((uintptr_t)ka.B & 15) || ((uintptr_t)ka.wk & 15)) return RPA_OK;
  const bool hasw = ka.wk != nullptr;
  TmaMapsMK maps;
  auto operand = [&](CUtensorMap* m, const cplx* base, long long ld, int rows) {
    cuuint64_t dims[2] = {(cuuint64_t)2 * ka.K, (cuuint64_t)rows};
    cuuint64_t strides[1] = {(cuuint64_t)ld * sizeof(cplx)};
    cuuint32_t box[2] = {16, (cuuint32_t)BM};
    cuuint32_t es[2] = {1, 1};
    return encode(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, (void*)base, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                  CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
  };
  if (!operand(&maps.a, ka.A, ka.lda, ka.M) || !operand(&maps.b, ka.B, ka.ldb, ka.N)) return RPA_OK;
  maps.w = maps.a;   // unused without weights
  if (hasw) {
    cuuint64_t dims[2] = {(cuuint64_t)ka.K, 1};
    cuuint64_t strides[1] = {(cuuint64_t)(ka.K + (ka.K & 1)) * sizeof(double)};
    cuuint32_t box[2] = {(cuuint32_t)BK, 1};
    cuuint32_t es[2] = {1, 1};
    if (encode(&maps.w, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, (void*)ka.wk, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
               CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS) return RPA_OK;
  }
  constexpr size_t smem = (size_t)TMA_STAGES * 2 * TMA_TILE * sizeof(cplx) + TMA_STAGES * BK * sizeof(double) + 2 * TMA_STAGES * sizeof(unsigned long long) + 128;
  if (ctx->attr_once(RPA_ATTR_ZGEMM_TMA_MK)) {
    RPA_CUDA(ctx, cudaFuncSetAttribute(zgemm_tma_mk_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    RPA_CUDA(ctx, cudaFuncSetAttribute(zgemm_tma_mk_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  }
  if (hasw) zgemm_tma_mk_kernel<true><<<grid, NTHREADS, smem, ctx->stream>>>(ka, maps);
  else zgemm_tma_mk_kernel<false><<<grid, NTHREADS, smem, ctx->stream>>>(ka, maps);
  RPA_LAUNCH_CHECK(ctx);
  *ok = true;
  return RPA_OK;
}

template <bool A_KM, bool B_KN, bool CONJ_B>
int launch(rpa_ctx* ctx, const KArgs& ka, dim3 grid) {
  if (ka.herm) {
    // Hermitian updates come in two operand layouts only (CHI_SUM / chi_s: [k][m] x [k][n]; Gram matrices: [m][k] x [m][k])
    if constexpr (A_KM == B_KN && CONJ_B) return launch_h<A_KM, B_KN, CONJ_B, true>(ctx, ka, grid);
    else return rpa_fail(ctx, RPA_ERR_INVALID, "zgemm_dmma: Hermitian update in an operand layout not instantiated");
  }
  return launch_h<A_KM, B_KN, CONJ_B, false>(ctx, ka, grid);
}

}  // namespace

int zgemm_dmma(rpa_ctx* ctx, const ZgemmParams& p) {
  if (p.M <= 0 || p.N <= 0 || p.batch <= 0) return RPA_OK;
  if (p.herm && p.M != p.N) return rpa_fail(ctx, RPA_ERR_INVALID, "zgemm_dmma: herm needs M == N");
  KArgs ka;
  ka.A = p.A; ka.lda = p.lda; ka.B = p.B; ka.ldb = p.ldb; ka.C = p.C; ka.ldc = p.ldc;
  ka.M = p.M; ka.N = p.N; ka.K = p.K;
  ka.herm = p.herm; ka.accumulate = p.accumulate;
  ka.alpha = p.alpha; ka.rs = p.rs; ka.cs = p.cs;
  ka.wk = p.wk; ka.strideW = p.strideW;
  ka.strideA = p.strideA; ka.strideB = p.strideB; ka.strideC = p.strideC;
  ka.batch_fastest = 0;
  const int tiles_m = (p.M + BM - 1) / BM, tiles_n = (p.N + BN - 1) / BN;
  ka.tiles_n = tiles_n;
  const long long tiles = p.herm ? (long long)tiles_m * (tiles_m + 1) / 2 : (long long)tiles_m * tiles_n;
  const int n_kt = (p.K + BK - 1) / BK;
  ka.n_kt = n_kt;
  int split = p.split_k;
  // the projection's TMA kernel takes one k-split and plain stores: with several waves of tiles that beats trimming the last
  // partial wave by a split (which would send it to the cp.async kernel and its atomics)
  if (split <= 0 && p.tma_mk && ctx->opt.zgemm_tma && !p.herm && p.batch == 1 && tiles >= 4LL * 2 * ctx->sm_count) split = 1;
  if (split <= 0) {
    // pick the split that fills whole waves of (2 CTAs per SM): maximise CTAs / (waves * slots)
    const long long slots = 2LL * ctx->sm_count;
    const long long base = tiles * p.batch;
    split = 1;
    int max_split = n_kt / 8;  // at least 8 k-tiles (128 k) per split
    if (base >= 8 * slots) max_split = std::min(max_split, 4);   // many waves already: only trim the last partial wave
    if (max_split > 1 && base < 8 * slots) {
      // Few tiles (the contractions of the small configs, the Gram matrices of the basis stage): cut K finely and let the
      // block scheduler balance.  Cost model in k-tiles of a full tile: the diagonal tiles of a Hermitian update issue
      // 9/16 of the DMMAs, a CTA pays ~EPI k-tiles for the pipeline fill and the atomic epilogue, and the last CTAs to
      // finish leave about 0.6 of a chunk idle.  (A single wave of equal CTAs would idle the slots it does not fill and
      // those whose diagonal tiles finish early: 77 % -> 8x % of the DMMA peak for CHI_SUM at configs[1].)
      const double EPI = 6.0;
      const double w_tiles = p.herm ? (double)(tiles - tiles_m) + 0.5625 * tiles_m : (double)tiles;
      const double W = w_tiles * p.batch * n_kt;
      double best = 1e300;
      for (int s = 1; s <= max_split && s <= 512; s++) {
        const long long chunk = (n_kt + s - 1) / s;
        const long long s_eff = (n_kt + chunk - 1) / chunk;
        const long long ctas = base * s_eff;
        double t = ctas <= slots ? (double)chunk : W / (double)slots + 0.6 * (double)chunk;
        t += EPI * (double)((ctas + slots - 1) / slots);
        if (t < best * (1.0 - 1e-3)) { best = t; split = s; }
      }
    } else if (max_split > 1 && base < 64 * slots) {
      double best = 0.0;
      for (int s = 1; s <= max_split && s <= 64; s++) {
        const long long ctas = base * s;
        const long long waves = (ctas + slots - 1) / slots;
        double eff = (double)ctas / (double)(waves * slots);
        eff -= 0.002 * s;  // mild preference for fewer splits (less atomic traffic)
        if (eff > best + 1e-9) { best = eff; split = s; }
      }
    }
  }
  if (n_kt == 0) split = 1;
  ka.kt_per_split = n_kt > 0 ? (n_kt + split - 1) / split : 1;
  split = n_kt > 0 ? (n_kt + ka.kt_per_split - 1) / ka.kt_per_split : 1;
  ka.atomic = split > 1;
  if (n_kt == 0 || (ka.atomic && !p.accumulate)) {
    // zero C first (K == 0 gives C = 0 when not accumulating)
    if (!p.accumulate) {
      if (p.ldc == p.N && (p.batch == 1 || p.strideC == (long long)p.M * p.N)) {   // one contiguous slab
        RPA_CUDA(ctx, cudaMemsetAsync(p.C, 0, (size_t)p.batch * p.M * p.N * sizeof(cplx), ctx->stream));
      } else {
        for (int b = 0; b < p.batch; b++)
          RPA_CUDA(ctx, cudaMemset2DAsync(p.C + b * p.strideC, p.ldc * sizeof(cplx), 0, (size_t)p.N * sizeof(cplx), p.M,
                                          ctx->stream));
      }
    }
    if (n_kt == 0) return RPA_OK;
  }
  if (tiles > 2147483647LL || p.batch > 65535 || split > 65535)
    return rpa_fail(ctx, RPA_ERR_INVALID, "zgemm_dmma: grid too large");
  dim3 grid((unsigned)tiles, (unsigned)split, (unsigned)p.batch);
  int rc;
  // the combinations the library uses: [k][m] x [k][n] conj (CHI_SUM, chi_s), [m][k] x [m][k] conj (projection, Gram,
  // Cholesky updates), [m][k] x [k][n] conj / plain (subspace iteration, rotations, triangular solves)
  bool tma_done = false;
  if (ctx->opt.zgemm_tma && p.herm && p.a_km && p.b_kn && p.conj_b && p.A == p.B && p.lda == p.ldb && p.strideA == p.strideB) {
    if ((rc = launch_tma(ctx, ka, grid, p.batch, &tma_done))) return rc;
  }
#ifndef RPA_PROJ_TMA
#define RPA_PROJ_TMA 1
#endif
  // the projection shape: [m][k] x [n][k] conj, weights along k, one split, plain store of alpha * sum
  if (RPA_PROJ_TMA && p.tma_mk && ctx->opt.zgemm_tma && !tma_done && !p.a_km && !p.b_kn && p.conj_b && !p.herm && p.batch == 1 && !ka.atomic && !p.accumulate &&
      !p.rs && !p.cs && (p.lda * (long long)sizeof(cplx)) % 16 == 0) {
    if ((rc = launch_tma_mk(ctx, ka, grid, &tma_done))) return rc;
  }
  if (tma_done) rc = RPA_OK;
  else if (p.a_km && p.b_kn && p.conj_b) rc = launch<true, true, true>(ctx, ka, grid);
  else if (!p.a_km && !p.b_kn && p.conj_b) rc = launch<false, false, true>(ctx, ka, grid);
  else if (!p.a_km && p.b_kn && p.conj_b) rc = launch<false, true, true>(ctx, ka, grid);
  else if (!p.a_km && p.b_kn && !p.conj_b) rc = launch<false, true, false>(ctx, ka, grid);
  else return rpa_fail(ctx, RPA_ERR_INVALID, "zgemm_dmma: operand layout combination not instantiated");
  if (rc) return rc;
  if (ka.atomic && p.herm) {
    dim3 mg((p.N + 255) / 256, p.N, p.batch);
    herm_mirror_kernel<<<mg, 256, 0, ctx->stream>>>(p.C, p.ldc, p.strideC, p.N);
    RPA_LAUNCH_CHECK(ctx);
  }
  return RPA_OK;
}

namespace {
__global__ void pair_weights_kernel(const double* __restrict__ e_v, const double* __restrict__ e_c, int nc, long long P,
                                    const double* __restrict__ omega, const double* __restrict__ f_v,
                                    const double* __restrict__ f_c, double* __restrict__ out) {
  const double w = omega ? omega[blockIdx.y] : 0.0, w2 = w * w;
  double* o = out + blockIdx.y * P;
  for (long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x; k < P; k += (long long)gridDim.x * blockDim.x) {
    const int v = (int)(k / nc), c = (int)(k - (long long)v * nc);
    const double d = e_c[c] - e_v[v];
    const double den = d * d + w2;
    double x = den > 0.0 ? 2.0 * d / den : 0.0;
    if (f_v) x *= fmax(f_v[v] - f_c[c], 0.0);   // partial occupations (reading R21): every unordered pair once, f_v > f_c
    o[k] = x;
  }
}
}  // namespace

int pair_weights(rpa_ctx* ctx, const double* e_v, const double* e_c, int nvb, int nc, const double* omega, int n_w, double* out,
                 const double* f_v, const double* f_c) {
  const long long P = (long long)nvb * nc;
  dim3 grid((unsigned)std::min<long long>((P + 255) / 256, 4096), omega ? n_w : 1);
  pair_weights_kernel<<<grid, 256, 0, ctx->stream>>>(e_v, e_c, nc, P, omega, f_v, f_c, out);
  RPA_LAUNCH_CHECK(ctx);
  return RPA_OK;
}

// ---------------------------------------------------------------------------------------------
// Register-only FP64 peak microbenchmarks (rpa_fp64_peak): the roofline denominators for CHI_SUM (DMMA) and the
// FFT butterflies (DFMA).  MEASURED_PEAKS.json has no FP64 entry, so bench.py measures these on the box.
namespace {
constexpr int PEAK_ITERS = 4096;
__global__ void __launch_bounds__(256) dmma_peak_kernel(double* out) {
  double acc[16][2];
#pragma unroll
  for (int i = 0; i < 16; i++) acc[i][0] = acc[i][1] = 0.0;
  double a = 1.0 + threadIdx.x * 1e-9, b = 1.0 - threadIdx.x * 1e-9;
  for (int it = 0; it < PEAK_ITERS; it++) {
#pragma unroll
    for (int i = 0; i < 16; i++) dmma(acc[i][0], acc[i][1], a, b);
  }
  double s = 0;
#pragma unroll
  for (int i = 0; i < 16; i++) s += acc[i][0] + acc[i][1];
  if (s == 123.456) out[0] = s;
}
// kind 2: the instruction mix a 3-multiply complex product would run per k-step and warp -- 24 DMMAs and 14 independent
// DADDs -- to show that plain FP64 instructions share the pipe with the DMMAs.  Counts DMMA FLOPs only.
__global__ void __launch_bounds__(256) dmma_dadd_mix_kernel(double* out) {
  double acc[24][2], s[14];
#pragma unroll
  for (int i = 0; i < 24; i++) acc[i][0] = acc[i][1] = 0.0;
#pragma unroll
  for (int i = 0; i < 14; i++) s[i] = threadIdx.x * 1e-3 + i;
  double a = 1.0 + threadIdx.x * 1e-9, b = 1.0 - threadIdx.x * 1e-9;
  for (int it = 0; it < PEAK_ITERS; it++) {
#pragma unroll
    for (int i = 0; i < 24; i++) dmma(acc[i][0], acc[i][1], a, b);
#pragma unroll
    for (int i = 0; i < 14; i++) s[i] += a;
  }
  double t = 0;
#pragma unroll
  for (int i = 0; i < 24; i++) t += acc[i][0] + acc[i][1];
#pragma unroll
  for (int i = 0; i < 14; i++) t += s[i];
  if (t == 123.456) out[0] = t;
}
__global__ void __launch_bounds__(256) dfma_peak_kernel(double* out) {
  double acc[16];
#pragma unroll
  for (int i = 0; i < 16; i++) acc[i] = threadIdx.x * 1e-3 + i;
  double a = 1.0 + threadIdx.x * 1e-12, b = 1e-9;
  for (int it = 0; it < PEAK_ITERS; it++) {
#pragma unroll
    for (int i = 0; i < 16; i++) acc[i] = fma(acc[i], a, b);
  }
  double s = 0;
#pragma unroll
  for (int i = 0; i < 16; i++) s += acc[i];
  if (s == 123.456) out[0] = s;
}
}  // namespace

int fp64_peak_kernel(rpa_ctx* ctx, int kind, int iters, double* tflops) {
  if (!ctx->ws || ctx->ws_bytes < 8) return rpa_fail(ctx, RPA_ERR_WORKSPACE, "rpa_fp64_peak needs a workspace");
  if (iters < 1) iters = 1;
  const int blocks = ctx->sm_count * 8;
  cudaEvent_t e0, e1;
  RPA_CUDA(ctx, cudaEventCreate(&e0));
  RPA_CUDA(ctx, cudaEventCreate(&e1));
  for (int rep = 0; rep < 2; rep++) {  // rep 0 = warm-up
    RPA_CUDA(ctx, cudaEventRecord(e0, ctx->stream));
    for (int i = 0; i < iters; i++) {
      if (kind == 0) dmma_peak_kernel<<<blocks, 256, 0, ctx->stream>>>((double*)ctx->ws);
      else if (kind == 2) dmma_dadd_mix_kernel<<<blocks, 256, 0, ctx->stream>>>((double*)ctx->ws);
      else dfma_peak_kernel<<<blocks, 256, 0, ctx->stream>>>((double*)ctx->ws);
      ctx->launches++;
    }
    RPA_CUDA(ctx, cudaEventRecord(e1, ctx->stream));
    RPA_CUDA(ctx, cudaEventSynchronize(e1));
  }
  float ms = 0;
  RPA_CUDA(ctx, cudaEventElapsedTime(&ms, e0, e1));
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  const double warps = (double)blocks * 8;
  const double flops = kind == 0 ? warps * PEAK_ITERS * 16.0 * (2.0 * 8 * 8 * 4) : kind == 2 ? warps * PEAK_ITERS * 24.0 * (2.0 * 8 * 8 * 4)
                                                                                             : warps * 32.0 * PEAK_ITERS * 16.0 * 2.0;
  *tflops = flops * iters / (ms * 1e-3) / 1e12;
  return RPA_OK;
}
