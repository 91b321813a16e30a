// MTXEL (step a1): M[v][c][G] = (1/N_r) sum_r conj(u_v(r)) u_c(r) e^{-iG.r}, G on the epsilon sphere.
// PAPER.md:52 eq. 3, :96, :104-110 ("batched FFT algorithm"); readings R7/R8 of DESIGN.md.
//
// B200 design (differs from the paper's vendor-FFT offload):
//   * real-space functions u_n are stored plane-major [z][x][y] so one z-plane is contiguous;
//   * pair_plane_kernel: one CTA per (conduction band c, plane z) keeps u_c(:,:,z) in shared memory and loops over
//     the valence bands of the block: product, y-FFT, x-FFT restricted to the kept y-frequencies, and writes only
//     the nk1 x nk2 kept (x,y)-frequencies: an ~11x data reduction before anything goes back to global memory;
//   * z_fft_scatter: the remaining 1-D transforms along z on the pruned columns, fused with the gather onto the
//     epsilon sphere and the 1/N_r normalisation.
// All transforms are the hand-written shared-memory radix-8/4/2/3/5 FFT of fft_smem.cuh.
#include <algorithm>
#include <cmath>
#include <cstdlib>

#include "fft_smem.cuh"
#include "pair_plane_fft8.cuh"
#include "z_fft8.cuh"
#include "rpa_internal.h"

using fftsm::Plan;

struct AxisPlan {
  int n = 0, n_pass = 0;
  int radix[fftsm::MAX_PASS];
  cplx* d_tw_fwd = nullptr;
  cplx* d_tw_inv = nullptr;
  int* d_perm = nullptr;
  int nk = 0;            // number of distinct epsilon-sphere Miller indices on this axis
  int* d_kpos = nullptr; // [nk] position (after the in-place passes) of each kept frequency
  int* d_kfreq = nullptr; // [nk] the kept frequencies themselves, in 0..n-1
  int max_res8 = 0;       // largest number of kept frequencies in one residue class mod 8
  bool ends_only = false; // n = 8 R: every kept frequency k = s + 8 s2 has s2 = 0 or s2 = R - 1
  Plan fwd() const { Plan p; p.n = n; p.n_pass = n_pass; for (int i = 0; i < n_pass; i++) p.radix[i] = radix[i]; p.tw = d_tw_fwd; p.perm = d_perm; return p; }
  Plan inv() const { Plan p = fwd(); p.tw = d_tw_inv; return p; }
};

struct MtxelPlan {
  AxisPlan ax[3];        // 0: x (N1), 1: y (N2), 2: z (N3)
  int* d_wfn_box = nullptr;  // [n_pw] index of each wavefunction G in the [z][x][y] box
  int* d_wx = nullptr; int n_wx = 0;   // distinct x (axis 0) box indices of the wavefunction sphere
  int* d_wz = nullptr; int n_wz = 0;   // distinct z (axis 2) box indices of the wavefunction sphere
  int* d_inv_map = nullptr;  // [nk2*nk1*nk3] epsilon-sphere index of pruned-box point ((i2*nk1+i1)*nk3+i3), or -1
};

static bool factorize(int n, AxisPlan& ap) {
  ap.n = n; ap.n_pass = 0;
  const int rad[5] = {8, 4, 2, 3, 5};
  for (int f : rad)
    while (n % f == 0) {
      if (ap.n_pass >= fftsm::MAX_PASS) return false;
      ap.radix[ap.n_pass++] = f; n /= f;
    }
  return n == 1;
}

static int upload(rpa_ctx* ctx, void** dst, const void* src, size_t bytes) {
  RPA_CUDA(ctx, cudaMalloc(dst, bytes ? bytes : 16));
  if (bytes) RPA_CUDA(ctx, cudaMemcpy(*dst, src, bytes, cudaMemcpyHostToDevice));
  return RPA_OK;
}

int mtxel_plan_create(rpa_ctx* ctx, const int32_t* g_eps, const int32_t* g_wfn) {
  MtxelPlan* mp = new MtxelPlan();
  ctx->mtxel = mp;
  const int N[3] = {ctx->fft[0], ctx->fft[1], ctx->fft[2]};
  std::vector<int> kidx[3];  // sorted distinct Miller indices per axis
  for (int a = 0; a < 3; a++) {
    AxisPlan& ap = mp->ax[a];
    if (N[a] < 1 || N[a] > 1024 || !factorize(N[a], ap))
      return rpa_fail(ctx, RPA_ERR_INVALID, "fft axis %d = %d must factor into 2,3,5 and be <= 1024", a, N[a]);
    const int n = N[a];
    std::vector<cplx> twf(n), twi(n);
    for (int k = 0; k < n; k++) {
      long double ang = 2.0L * 3.14159265358979323846264338327950288L * (long double)k / (long double)n;
      twf[k] = make_double2((double)cosl(ang), (double)(-sinl(ang)));
      twi[k] = make_double2((double)cosl(ang), (double)sinl(ang));
    }
    std::vector<int> perm(n);
    for (int k = 0; k < n; k++) {
      int kk = k, nn = n, pos = 0;
      for (int ps = 0; ps < ap.n_pass; ps++) { int r = ap.radix[ps]; pos += (kk % r) * (nn / r); kk /= r; nn /= r; }
      perm[k] = pos;
    }
    for (int g = 0; g < ctx->n_g; g++) {
      int m = g_eps[3 * g + a];
      if (2 * std::abs(m) >= n) return rpa_fail(ctx, RPA_ERR_INVALID, "g_eps[%d] axis %d index %d outside the grid", g, a, m);
      kidx[a].push_back(m);
    }
    std::sort(kidx[a].begin(), kidx[a].end());
    kidx[a].erase(std::unique(kidx[a].begin(), kidx[a].end()), kidx[a].end());
    ap.nk = (int)kidx[a].size();
    std::vector<int> kpos(ap.nk);
    std::vector<int> kfreq(ap.nk);
    for (int i = 0; i < ap.nk; i++) { kfreq[i] = ((kidx[a][i] % n) + n) % n; kpos[i] = perm[kfreq[i]]; }
    { int cnt[8] = {0}; for (int i = 0; i < ap.nk; i++) ap.max_res8 = std::max(ap.max_res8, ++cnt[kfreq[i] & 7]); }
    ap.ends_only = n % 8 == 0;
    for (int i = 0; i < ap.nk && ap.ends_only; i++) ap.ends_only = (kfreq[i] >> 3) == 0 || (kfreq[i] >> 3) == n / 8 - 1;
    int rc;
    if ((rc = upload(ctx, (void**)&ap.d_tw_fwd, twf.data(), n * sizeof(cplx)))) return rc;
    if ((rc = upload(ctx, (void**)&ap.d_tw_inv, twi.data(), n * sizeof(cplx)))) return rc;
    if ((rc = upload(ctx, (void**)&ap.d_perm, perm.data(), n * sizeof(int)))) return rc;
    if ((rc = upload(ctx, (void**)&ap.d_kpos, kpos.data(), ap.nk * sizeof(int)))) return rc;
    if ((rc = upload(ctx, (void**)&ap.d_kfreq, kfreq.data(), ap.nk * sizeof(int)))) return rc;
  }
  std::vector<int> box(ctx->n_pw), wxs, wzs;
  for (int g = 0; g < ctx->n_pw; g++) {
    int i[3];
    for (int a = 0; a < 3; a++) {
      int m = g_wfn[3 * g + a];
      if (2 * std::abs(m) >= N[a]) return rpa_fail(ctx, RPA_ERR_INVALID, "g_wfn[%d] axis %d index %d outside the grid", g, a, m);
      i[a] = ((m % N[a]) + N[a]) % N[a];
    }
    box[g] = (i[2] * N[0] + i[0]) * N[1] + i[1];
    wxs.push_back(i[0]); wzs.push_back(i[2]);
  }
  for (auto* w : {&wxs, &wzs}) { std::sort(w->begin(), w->end()); w->erase(std::unique(w->begin(), w->end()), w->end()); }
  mp->n_wx = (int)wxs.size(); mp->n_wz = (int)wzs.size();
  const int nk1 = mp->ax[0].nk, nk2 = mp->ax[1].nk, nk3 = mp->ax[2].nk;
  std::vector<int> inv((size_t)nk1 * nk2 * nk3, -1);
  for (int g = 0; g < ctx->n_g; g++) {
    int i[3];
    for (int a = 0; a < 3; a++)
      i[a] = (int)(std::lower_bound(kidx[a].begin(), kidx[a].end(), g_eps[3 * g + a]) - kidx[a].begin());
    size_t pb = ((size_t)i[1] * nk1 + i[0]) * nk3 + i[2];
    if (inv[pb] >= 0) return rpa_fail(ctx, RPA_ERR_INVALID, "g_eps has a duplicate entry at %d", g);
    inv[pb] = g;
  }
  int rc;
  if ((rc = upload(ctx, (void**)&mp->d_wfn_box, box.data(), box.size() * sizeof(int)))) return rc;
  if ((rc = upload(ctx, (void**)&mp->d_wx, wxs.data(), wxs.size() * sizeof(int)))) return rc;
  if ((rc = upload(ctx, (void**)&mp->d_wz, wzs.data(), wzs.size() * sizeof(int)))) return rc;
  if ((rc = upload(ctx, (void**)&mp->d_inv_map, inv.data(), inv.size() * sizeof(int)))) return rc;
  return RPA_OK;
}

void mtxel_plan_destroy(rpa_ctx* ctx) {
  MtxelPlan* mp = ctx->mtxel;
  if (!mp) return;
  for (int a = 0; a < 3; a++) {
    cudaFree(mp->ax[a].d_tw_fwd); cudaFree(mp->ax[a].d_tw_inv); cudaFree(mp->ax[a].d_perm); cudaFree(mp->ax[a].d_kpos); cudaFree(mp->ax[a].d_kfreq);
  }
  cudaFree(mp->d_wfn_box); cudaFree(mp->d_inv_map); cudaFree(mp->d_wx); cudaFree(mp->d_wz);
  delete mp;
  ctx->mtxel = nullptr;
}

// ---------------------------------------------------------------------------------------------
// kernels
namespace {

// psi [nb][n_pw] -> zero-initialised boxes [nb][N_r] at box[g]
__global__ void scatter_wfn_kernel(const cplx* __restrict__ psi, const int* __restrict__ box, int n_pw, long long n_r,
                                   cplx* __restrict__ u) {
  const int b = blockIdx.y;
  for (int g = blockIdx.x * blockDim.x + threadIdx.x; g < n_pw; g += gridDim.x * blockDim.x)
    u[(long long)b * n_r + box[g]] = psi[(long long)b * n_pw + g];
}

// Batched 1-D transform along one axis of data viewed as [outer][n][inner], TL lines per CTA in shared memory.
// MODE 0: in place, natural-order write-back (inverse transforms of the wavefunctions).
// MODE 1: forward along z of T[pair][z][J]; writes only the kept k3 and scatters them onto the epsilon sphere:
//         M[(v*nc + c0 + cl)*n_g + g] = X * scale, pair = v*ncc + cl.
struct ZScatter {
  const int* kpos3; int nk3; const int* inv_map; cplx* M; int ncc, nc, c0, n_g; double scale;
  // MODE 0 only, optional pruning of the wavefunction transforms (lines that hold nothing but zeros are skipped):
  //   sel 1 (y pass, inner == 1):  line = (band, iz < nz, ix < nx) -> box line (band, zl[iz], xl[ix])
  //   sel 2 (x pass, inner == N2): line = (band, iz < nz, y < N2)   -> box plane (band, zl[iz]), column y
  int sel; const int* zl; int nz; const int* xl; int nx; int N1, N3;
};
template <bool INV, int MODE>
__global__ void fft_axis_kernel(cplx* __restrict__ data, Plan pl, long long n_lines, int inner, int TL, ZScatter zs) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx* s = reinterpret_cast<cplx*>(smem_raw);
  __shared__ long long s_base[64];   // per line of the tile (TL <= 64): element offset of its first element ...
  __shared__ long long s_row[64];    // ... MODE 1: offset of the M row of its pair
  __shared__ int s_j[64];            // ... MODE 1: its kept (k_x, k_y) column
  const int n = pl.n, pitch = n | 1;
  const int tid = threadIdx.x, nthr = blockDim.x;
  const long long line0 = (long long)blockIdx.x * TL;
  const int nl = (int)min((long long)TL, n_lines - line0);
  if (tid < nl) {   // the 64-bit divisions are done once per line, not once per element
    const long long line = line0 + tid, o = line / inner;
    const int i = (int)(line - o * inner);
    if (MODE == 0 && zs.sel == 1) {
      const long long band = line / ((long long)zs.nz * zs.nx);
      const int r = (int)(line - band * zs.nz * zs.nx), iz = r / zs.nx, ix = r - iz * zs.nx;
      s_base[tid] = ((band * zs.N3 + zs.zl[iz]) * zs.N1 + zs.xl[ix]) * (long long)n;
    } else if (MODE == 0 && zs.sel == 2) {
      const long long band = line / ((long long)zs.nz * inner);
      const int r = (int)(line - band * zs.nz * inner), iz = r / inner, yy = r - iz * inner;
      s_base[tid] = (band * zs.N3 + zs.zl[iz]) * (long long)n * inner + yy;
    } else {
      s_base[tid] = inner == 1 ? line * n : o * n * inner + i;
    }
    if (MODE == 1) {
      const long long v = o / zs.ncc;
      const int cl = (int)(o - v * zs.ncc);
      s_row[tid] = (v * zs.nc + zs.c0 + cl) * zs.n_g;
      s_j[tid] = i;
    }
  }
  __syncthreads();
  if (inner == 1) {
    for (int idx = tid; idx < nl * n; idx += nthr) {
      int l = idx / n, e = idx - l * n;
      s[l * pitch + e] = data[s_base[l] + e];
    }
  } else {
    for (int idx = tid; idx < nl * n; idx += nthr) {
      int e = idx / nl, l = idx - e * nl;
      s[l * pitch + e] = data[s_base[l] + (long long)e * inner];
    }
  }
  __syncthreads();
  fftsm::fft_lines<INV>(s, pl, nl, nullptr, pitch, 1, tid, nthr);
  if (MODE == 0) {
    if (inner == 1) {
      for (int idx = tid; idx < nl * n; idx += nthr) {
        int l = idx / n, e = idx - l * n;
        data[s_base[l] + e] = s[l * pitch + pl.perm[e]];
      }
    } else {
      for (int idx = tid; idx < nl * n; idx += nthr) {
        int e = idx / nl, l = idx - e * nl;
        data[s_base[l] + (long long)e * inner] = s[l * pitch + pl.perm[e]];
      }
    }
  } else {
    for (int idx = tid; idx < nl * zs.nk3; idx += nthr) {
      int l = idx / zs.nk3, i3 = idx - l * zs.nk3;
      int g = zs.inv_map[s_j[l] * zs.nk3 + i3];
      if (g >= 0) {
        cplx x = s[l * pitch + zs.kpos3[i3]];
        zs.M[s_row[l] + g] = make_double2(x.x * zs.scale, x.y * zs.scale);
      }
    }
  }
}

// One CTA per (c, z): the u_c plane stays in shared memory while the CTA loops over the valence bands of the block.
//   T[((v*ncc + c)*N3 + z)*J + i2*nk1 + i1] = sum_{x,y} conj(u_v) u_c e^{-2 pi i (k1 x/N1 + k2 y/N2)}
// Warp-private rows: warp w owns rows [w*LW, (w+1)*LW) of the plane; it forms the product for them, transforms them
// along y and copies the nk2 kept y-frequencies into the (double-buffered, transposed) column buffer -- with only
// __syncwarp() in between.  One __syncthreads() per valence band then separates that from the x transforms, which are
// again distributed over the warps (LX kept columns each).  u_v rows of the next band are prefetched into registers.
template <int EPT>
__global__ void pair_plane_kernel(const cplx* __restrict__ u_v, const cplx* __restrict__ u_c, int nvb, int ncc, int N1,
                                  int N2, int N3, Plan px, Plan py, const int* __restrict__ kpos1,
                                  const int* __restrict__ kpos2, int nk1, int nk2, cplx* __restrict__ T) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int P1 = N1 | 1, P2 = N2 | 1;
  cplx* sc = reinterpret_cast<cplx*>(smem_raw);       // [N1][P2] u_c plane
  cplx* wk = sc + N1 * P2;                            // [N1][P2] work plane (rows private to their warp)
  cplx* cb0 = wk + N1 * P2;                           // 2 x [nk2][P1] kept y-frequencies, x contiguous
  int* s_k1 = reinterpret_cast<int*>(cb0 + 2 * nk2 * P1);  // [nk1]
  int* s_k2 = s_k1 + nk1;                             // [nk2]
  const int tid = threadIdx.x, nthr = blockDim.x, lane = tid & 31, warp = tid >> 5, nwarp = nthr >> 5;
  const int z = blockIdx.x / ncc, c = blockIdx.x - z * ncc;
  const int plane = N1 * N2;
  const long long n_r = (long long)plane * N3;
  const cplx* ucp = u_c + (long long)c * n_r + (long long)z * plane;
  for (int idx = tid; idx < plane; idx += nthr) {
    int x = idx / N2, y = idx - x * N2;
    sc[x * P2 + y] = ucp[idx];
  }
  for (int i = tid; i < nk1; i += nthr) s_k1[i] = kpos1[i];
  for (int i = tid; i < nk2; i += nthr) s_k2[i] = kpos2[i];
  // this warp's rows (y transforms) and kept columns (x transforms)
  const int LW = (N1 + nwarp - 1) / nwarp;
  const int r0 = min(N1, warp * LW), r1 = min(N1, r0 + LW), nrow = r1 - r0;
  const int LX = (nk2 + nwarp - 1) / nwarp;
  const int j0 = min(nk2, warp * LX), j1 = min(nk2, j0 + LX), ncol = j1 - j0;
  const int nel = nrow * N2;                          // contiguous elements of the plane owned by this warp
  const cplx* uvp = u_v + (long long)z * plane + (long long)r0 * N2;
  cplx nxt[EPT > 0 ? EPT : 1];
  if (EPT > 0) {
#pragma unroll
    for (int e = 0; e < EPT; e++) {
      int idx = lane + e * 32;
      if (idx < nel) nxt[e] = uvp[idx];
    }
  }
  __syncthreads();
  const int J = nk1 * nk2;
  for (int v = 0; v < nvb; v++) {
    cplx* cb = cb0 + (v & 1) * nk2 * P1;
    if (nrow > 0) {
      // (a) product on the warp's rows
      if (EPT > 0) {
#pragma unroll
        for (int e = 0; e < EPT; e++) {
          int idx = lane + e * 32;
          if (idx < nel) {
            int x = r0 + idx / N2, y = idx % N2;
            cplx a = nxt[e], b = sc[x * P2 + y];
            wk[x * P2 + y] = make_double2(a.x * b.x + a.y * b.y, a.x * b.y - a.y * b.x);
          }
        }
        if (v + 1 < nvb) {
          const cplx* nx = uvp + (long long)(v + 1) * n_r;
#pragma unroll
          for (int e = 0; e < EPT; e++) {
            int idx = lane + e * 32;
            if (idx < nel) nxt[e] = nx[idx];
          }
        }
      } else {
        const cplx* cur = uvp + (long long)v * n_r;
        for (int idx = lane; idx < nel; idx += 32) {
          int x = r0 + idx / N2, y = idx % N2;
          cplx a = cur[idx], b = sc[x * P2 + y];
          wk[x * P2 + y] = make_double2(a.x * b.x + a.y * b.y, a.x * b.y - a.y * b.x);
        }
      }
      __syncwarp();
      // (b) y transforms of the warp's rows, then keep the nk2 needed y-frequencies (transposed: x contiguous)
      fftsm::fft_lines<false, true>(wk + r0 * P2, py, nrow, nullptr, P2, 1, lane, 32);
      for (int idx = lane; idx < nrow * nk2; idx += 32) {
        int xr = idx % nrow, i2 = idx / nrow;
        cb[i2 * P1 + r0 + xr] = wk[(r0 + xr) * P2 + s_k2[i2]];
      }
    }
    __syncthreads();
    if (ncol > 0) {
      // (c) x transforms on the warp's kept columns, then write the nk1 kept x-frequencies
      fftsm::fft_lines<false, true>(cb + j0 * P1, px, ncol, nullptr, P1, 1, lane, 32);
      cplx* dst = T + (((long long)v * ncc + c) * N3 + z) * J;
      for (int idx = lane; idx < ncol * nk1; idx += 32) {
        int i1 = idx % nk1, jc = idx / nk1;
        dst[(j0 + jc) * nk1 + i1] = cb[(j0 + jc) * P1 + s_k1[i1]];
      }
    }
  }
}

}  // namespace

// ---------------------------------------------------------------------------------------------
// host side
namespace {

struct MtxelSizes {
  int ncc;             // conduction bands per chunk
  size_t u_v, u_vp, u_c, t;  // bytes
};

int fft8_plane_size(const rpa_ctx* ctx);
size_t fft8_lane_plane(int n8);

MtxelSizes mtxel_sizes(const rpa_ctx* ctx, int nvb, int nc) {
  const MtxelPlan* mp = ctx->mtxel;
  const size_t n_r = (size_t)ctx->n_r;
  const size_t J = (size_t)mp->ax[0].nk * mp->ax[1].nk;
  const size_t per_c = n_r * sizeof(cplx) + (size_t)nvb * ctx->fft[2] * J * sizeof(cplx);
  size_t budget = (size_t)1536 << 20;  // chunk the conduction bands so that u_c + T stay near 1.5 GB
  int ncc = (int)std::max<size_t>(16, budget / per_c);
  if (ncc > nc) ncc = nc;
  else {
    // the plane kernel launches one CTA per (conduction band or pair of bands, plane) and one CTA per SM is resident: take
    // the chunk, not more than a quarter below the budget, whose CTAs come closest to whole waves
    const int per_cta = (ctx->fft[0] == 48 && ctx->fft[1] == 48) ? 2 : 1;
    double best = -1.0; int best_ncc = ncc;
#ifndef RPA_WAVE_CHUNK
#define RPA_WAVE_CHUNK 1
#endif
    for (int cand = ncc; RPA_WAVE_CHUNK && cand >= std::max(16, ncc - ncc / 4); cand--) {
      const long long ctas = (long long)((cand + per_cta - 1) / per_cta) * ctx->fft[2];
      const long long waves = (ctas + ctx->sm_count - 1) / ctx->sm_count;
      const double eff = (double)ctas / (double)(waves * ctx->sm_count);
      if (eff > best + 1e-9) { best = eff; best_ncc = cand; }
    }
    ncc = best_ncc;
  }
  MtxelSizes s;
  s.ncc = ncc;
  s.u_v = ws_round((size_t)nvb * n_r * sizeof(cplx));
  // the valence functions once more, in the lane order of the fft8 plane kernels (pair_plane_fft8.cuh)
  s.u_vp = ws_round((size_t)nvb * ctx->fft[2] * fft8_lane_plane(fft8_plane_size(ctx)) * sizeof(cplx));
  s.u_c = ws_round((size_t)ncc * n_r * sizeof(cplx));
  s.t = ws_round((size_t)nvb * ncc * ctx->fft[2] * J * sizeof(cplx));
  return s;
}

int axis_tile_lines(int n) {
  int pitch = n | 1;
  int tl = (int)((64 * 1024) / (pitch * sizeof(cplx)));
  tl &= ~7;
  if (tl < 8) tl = 8;
  if (tl > 64) tl = 64;
  return tl;
}

template <bool INV, int MODE>
int launch_axis(rpa_ctx* ctx, cplx* data, const Plan& pl, long long n_lines, int inner, const ZScatter& zs) {
  const int tl = axis_tile_lines(pl.n);
  const size_t smem = (size_t)tl * (pl.n | 1) * sizeof(cplx);
  auto kern = fft_axis_kernel<INV, MODE>;
  if (ctx->attr_once(RPA_ATTR_AXIS + (INV ? 1 : 0) + 2 * MODE))
    RPA_CUDA(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024));
  const long long blocks = (n_lines + tl - 1) / tl;
  if (blocks > 2147483647LL) return rpa_fail(ctx, RPA_ERR_INVALID, "fft grid too large");
  kern<<<(unsigned)blocks, 256, smem, ctx->stream>>>(data, pl, n_lines, inner, tl, zs);
  RPA_LAUNCH_CHECK(ctx);
  return RPA_OK;
}

// psi [nb][n_pw] -> u [nb][z][x][y]
int wfn_to_realspace(rpa_ctx* ctx, const cplx* psi, int nb, cplx* u) {
  const MtxelPlan* mp = ctx->mtxel;
  const int N1 = ctx->fft[0], N2 = ctx->fft[1], N3 = ctx->fft[2];
  const long long n_r = ctx->n_r;
  RPA_CUDA(ctx, cudaMemsetAsync(u, 0, (size_t)nb * n_r * sizeof(cplx), ctx->stream));
  dim3 grid((ctx->n_pw + 255) / 256, nb);
  scatter_wfn_kernel<<<grid, 256, 0, ctx->stream>>>(psi, mp->d_wfn_box, ctx->n_pw, n_r, u);
  RPA_LAUNCH_CHECK(ctx);
  ZScatter zs{};
  int rc;
  // y and x passes only on the lines that hold coefficients (the others are zero and stay zero); z pass on all
  zs.zl = mp->d_wz; zs.nz = mp->n_wz; zs.xl = mp->d_wx; zs.nx = mp->n_wx; zs.N1 = N1; zs.N3 = N3;
  zs.sel = 1;
  if ((rc = launch_axis<true, 0>(ctx, u, mp->ax[1].inv(), (long long)nb * mp->n_wz * mp->n_wx, 1, zs))) return rc;    // y
  zs.sel = 2;
  if ((rc = launch_axis<true, 0>(ctx, u, mp->ax[0].inv(), (long long)nb * mp->n_wz * N2, N2, zs))) return rc;         // x
  zs.sel = 0;
  if ((rc = launch_axis<true, 0>(ctx, u, mp->ax[2].inv(), (long long)nb * N1 * N2, N1 * N2, zs))) return rc;  // z
  return RPA_OK;
}

template <int N>
int launch_fft8(rpa_ctx* ctx, const cplx* u_v, const cplx* u_c, int nvb, int ncc, int N3, const MtxelPlan* mp, cplx* T) {
  const int nk1 = mp->ax[0].nk, nk2 = mp->ax[1].nk;
  // ring variant (no block barrier in the band loop) where one CTA fits per SM anyway (N = 48, 64)
  const size_t smem_ring = fft8::smem_bytes_ring<N>(nk2);
  const bool ring_ok = smem_ring <= 227 * 1024 && (nk2 + fft8::Geo<N>::RW - 1) / fft8::Geo<N>::RW <= fft8::Geo<N>::NWARP;
  const bool ring = ring_ok && N >= 48;
  // N = 48: second passes that form only the two outputs the pruning keeps, when the kept sets allow it; and two
  // conduction bands per CTA (two u_c planes fit next to the ring), which halves the u_v traffic from L2
  const bool ends = N == 48 && mp->ax[0].ends_only && mp->ax[1].ends_only;
  const bool two = N == 48 && ring && fft8::smem_bytes_ring<N>(nk2, 2) <= 227 * 1024 && ncc >= 2;
  const size_t smem = ring ? fft8::smem_bytes_ring<N>(nk2, two ? 2 : 1) : fft8::smem_bytes<N>(nk1, nk2);
  constexpr int CB2 = N == 48 ? 2 : 1;   // the two-band form is compiled for N = 48 only
  auto kern = ring ? (two ? (ends ? fft8::pair_plane_fft8_kernel_ring<N, true, CB2> : fft8::pair_plane_fft8_kernel_ring<N, false, CB2>)
                          : (ends ? fft8::pair_plane_fft8_kernel_ring<N, true, 1> : fft8::pair_plane_fft8_kernel_ring<N, false, 1>))
                   : (fft8::Geo<N>::MAXREG > 0 ? fft8::pair_plane_fft8_kernel_r<N> : fft8::pair_plane_fft8_kernel_b<N>);
  if (ctx->attr_once(RPA_ATTR_FFT8 + (N == 24 ? 0 : N == 40 ? 1 : N == 48 ? 2 : 3))) {
    RPA_CUDA(ctx, cudaFuncSetAttribute(fft8::pair_plane_fft8_kernel_ring<N, false, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024));
    RPA_CUDA(ctx, cudaFuncSetAttribute(fft8::pair_plane_fft8_kernel_ring<N, true, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024));
    RPA_CUDA(ctx, cudaFuncSetAttribute(fft8::pair_plane_fft8_kernel_ring<N, false, CB2>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024));
    RPA_CUDA(ctx, cudaFuncSetAttribute(fft8::pair_plane_fft8_kernel_ring<N, true, CB2>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024));
    RPA_CUDA(ctx, cudaFuncSetAttribute(fft8::pair_plane_fft8_kernel_r<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024));
    RPA_CUDA(ctx, cudaFuncSetAttribute(fft8::pair_plane_fft8_kernel_b<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024));
    if (ctx->opt.verbose) {
      cudaFuncAttributes fa;
      cudaFuncGetAttributes(&fa, kern);
      fprintf(stderr, "[rpa] pair_plane_fft8_kernel<%d>: %d regs, max %d threads/block, launching %d threads, %zu B smem\n", N,
              fa.numRegs, fa.maxThreadsPerBlock, fft8::Geo<N>::NWARP * 32, smem);
    }
  }
  const int ctas_c = two ? (ncc + 1) / 2 : ncc;
  kern<<<(unsigned)(ctas_c * N3), fft8::Geo<N>::NWARP * 32, smem, ctx->stream>>>(u_v, u_c, nvb, ncc, N3, mp->ax[0].d_tw_fwd,
                                                                                mp->ax[0].d_kfreq, mp->ax[1].d_kfreq, nk1, nk2, T);
  RPA_LAUNCH_CHECK(ctx);
  return RPA_OK;
}

// 0 = no specialised kernel for this plane size (or it does not fit): use the generic pair_plane_kernel
int fft8_plane_size(const rpa_ctx* ctx) {
  const int N1 = ctx->fft[0], N2 = ctx->fft[1];
  if (N1 != N2) return 0;
  const int nk1 = ctx->mtxel->ax[0].nk, nk2 = ctx->mtxel->ax[1].nk;
  size_t smem = 0;
  switch (N1) {
    case 24: smem = fft8::smem_bytes<24>(nk1, nk2); break;
    case 40: smem = fft8::smem_bytes<40>(nk1, nk2); break;
    case 48: smem = fft8::smem_bytes<48>(nk1, nk2); break;
    case 64: smem = fft8::smem_bytes<64>(nk1, nk2); break;
    default: return 0;
  }
  return smem <= 227 * 1024 ? N1 : 0;
}

// elements of one valence plane in lane order (0 = no fft8 kernel)
size_t fft8_lane_plane(int n8) {
  switch (n8) {
    case 24: return fft8::Geo<24>::PP;
    case 40: return fft8::Geo<40>::PP;
    case 48: return fft8::Geo<48>::PP;
    case 64: return fft8::Geo<64>::PP;
    default: return 0;
  }
}

template <int N>
int launch_lane_order(rpa_ctx* ctx, const cplx* u_nat, cplx* u_lane, int nvb, int N3) {
  fft8::uv_lane_order_kernel<N><<<dim3((unsigned)N3, (unsigned)nvb), fft8::Geo<N>::NWARP * 32, 0, ctx->stream>>>(u_nat, u_lane, N3);
  RPA_LAUNCH_CHECK(ctx);
  return RPA_OK;
}

}  // namespace

size_t mtxel_workspace_bytes(const rpa_ctx* ctx, int nvb, int nc) {
  MtxelSizes s = mtxel_sizes(ctx, nvb, nc);
  return s.u_v + s.u_vp + s.u_c + s.t;
}

int mtxel_run(rpa_ctx* ctx, WsAlloc& ws, const cplx* psi_v, int nvb, const cplx* psi_c, int nc, cplx* M) {
  const MtxelPlan* mp = ctx->mtxel;
  const int N1 = ctx->fft[0], N2 = ctx->fft[1], N3 = ctx->fft[2];
  const long long n_r = ctx->n_r;
  const MtxelSizes sz = mtxel_sizes(ctx, nvb, nc);
  cplx* u_v = ws.get<cplx>((size_t)nvb * n_r);
  const int n8 = ctx->opt.generic_fft ? 0 : fft8_plane_size(ctx);
  cplx* u_vp = n8 ? ws.get<cplx>((size_t)nvb * N3 * fft8_lane_plane(n8)) : nullptr;
  cplx* u_c = ws.get<cplx>((size_t)sz.ncc * n_r);
  const int nk1 = mp->ax[0].nk, nk2 = mp->ax[1].nk, nk3 = mp->ax[2].nk, J = nk1 * nk2;
  cplx* T = ws.get<cplx>((size_t)nvb * sz.ncc * N3 * J);
  if (!ws.ok) return rpa_fail(ctx, RPA_ERR_WORKSPACE, "rpa_mtxel: workspace too small (need %zu bytes)", ws.off);

  const int plane = N1 * N2, P1 = N1 | 1, P2 = N2 | 1;
  const size_t smem = ((size_t)2 * N1 * P2 + (size_t)2 * nk2 * P1) * sizeof(cplx) + (size_t)(nk1 + nk2) * sizeof(int);
  if (n8 == 0 && smem > 227 * 1024)
    return rpa_fail(ctx, RPA_ERR_INVALID, "rpa_mtxel: an xy plane of %d x %d does not fit in shared memory", N1, N2);
  // warps: about 32 lanes' worth of butterflies per warp in a radix-8 pass over its rows
  int nwarp = (plane / 8 + 31) / 32;
  nwarp = std::max(2, std::min(16, nwarp));
  if (nwarp > N1) nwarp = N1;
  const int nthr = nwarp * 32;
  const int LW = (N1 + nwarp - 1) / nwarp;
  const bool prefetch = LW * N2 <= 8 * 32;
  auto kern = prefetch ? pair_plane_kernel<8> : pair_plane_kernel<0>;
  if (n8 == 0) RPA_CUDA(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));

  int rc;
  {
    ProfScope ps(ctx, RPA_PROF_MTXEL_WFN);
    rc = wfn_to_realspace(ctx, psi_v, nvb, u_v);
    if (!rc) switch (n8) {
      case 24: rc = launch_lane_order<24>(ctx, u_v, u_vp, nvb, N3); break;
      case 40: rc = launch_lane_order<40>(ctx, u_v, u_vp, nvb, N3); break;
      case 48: rc = launch_lane_order<48>(ctx, u_v, u_vp, nvb, N3); break;
      case 64: rc = launch_lane_order<64>(ctx, u_v, u_vp, nvb, N3); break;
      default: break;
    }
  }
  if (rc) return rc;
  cplx* const u_c_scratch = u_c;
  const bool have_cache = ctx->uc_cache && ctx->uc_cache_src == psi_c && ctx->uc_cache_nc == nc;
  const int n_cached = have_cache ? ctx->uc_cache_rows : 0;   // the first n_cached conduction bands live in the cache
  for (int c0 = 0, ncc = 0; c0 < nc; c0 += ncc) {
    ncc = std::min(sz.ncc, nc - c0);
    if (c0 < n_cached && c0 + ncc > n_cached) ncc = n_cached - c0;   // a chunk is either all cached or all scratch
    const bool cached = c0 < n_cached;
    u_c = cached ? ctx->uc_cache + (long long)c0 * n_r : u_c_scratch;
    if (!cached || !ctx->uc_cache_filled) {
      ProfScope ps(ctx, RPA_PROF_MTXEL_WFN);
      rc = wfn_to_realspace(ctx, psi_c + (long long)c0 * ctx->n_pw, ncc, u_c);
    }
    if (rc) return rc;
    ProfScope* pp = new ProfScope(ctx, RPA_PROF_MTXEL_PLANE);
    switch (n8) {
      case 24: rc = launch_fft8<24>(ctx, u_vp, u_c, nvb, ncc, N3, mp, T); break;
      case 40: rc = launch_fft8<40>(ctx, u_vp, u_c, nvb, ncc, N3, mp, T); break;
      case 48: rc = launch_fft8<48>(ctx, u_vp, u_c, nvb, ncc, N3, mp, T); break;
      case 64: rc = launch_fft8<64>(ctx, u_vp, u_c, nvb, ncc, N3, mp, T); break;
      default:
        kern<<<(unsigned)(ncc * N3), nthr, smem, ctx->stream>>>(u_v, u_c, nvb, ncc, N1, N2, N3, mp->ax[0].fwd(),
                                                                mp->ax[1].fwd(), mp->ax[0].d_kpos, mp->ax[1].d_kpos, nk1,
                                                                nk2, T);
        RPA_LAUNCH_CHECK(ctx);
        rc = RPA_OK;
    }
    delete pp;
    if (rc) return rc;
    ZScatter zs{};
    zs.kpos3 = mp->ax[2].d_kpos; zs.nk3 = nk3; zs.inv_map = mp->d_inv_map; zs.M = M;
    zs.ncc = ncc; zs.nc = nc; zs.c0 = c0; zs.n_g = ctx->n_g; zs.scale = 1.0 / (double)n_r;
    {
      ProfScope ps(ctx, RPA_PROF_MTXEL_Z);
      const long long n_lines = (long long)nvb * ncc * J;
      const bool z8 = !ctx->opt.generic_fft && (N3 == 40 || N3 == 120 || N3 == 160) && mp->ax[2].max_res8 <= zfft8::MAXO &&
                      (n_lines + 31) / 32 <= 2147483647LL;
      if (z8) {
        zfft8::Args za;
        za.T = T; za.n_lines = n_lines; za.J = J; za.tw = mp->ax[2].d_tw_fwd; za.kfreq3 = mp->ax[2].d_kfreq; za.nk3 = nk3;
        za.inv_map = mp->d_inv_map; za.M = M; za.ncc = ncc; za.nc = nc; za.c0 = c0; za.n_g = ctx->n_g; za.scale = zs.scale;
        int* per_sm = ctx->z_per_sm;   // resident CTAs per SM of the three instantiations (persistent grid)
        if (ctx->attr_once(RPA_ATTR_ZFFT8)) {
          RPA_CUDA(ctx, cudaFuncSetAttribute(zfft8::z_fft8_scatter_kernel<40>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)zfft8::smem_bytes<40>()));
          RPA_CUDA(ctx, cudaFuncSetAttribute(zfft8::z_fft8_scatter_kernel<120>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)zfft8::smem_bytes<120>()));
          RPA_CUDA(ctx, cudaFuncSetAttribute(zfft8::z_fft8_scatter_kernel<160>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)zfft8::smem_bytes<160>()));
          cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm[0], zfft8::z_fft8_scatter_kernel<40>, 32 * 5, zfft8::smem_bytes<40>());
          cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm[1], zfft8::z_fft8_scatter_kernel<120>, 32 * 15, zfft8::smem_bytes<120>());
          cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm[2], zfft8::z_fft8_scatter_kernel<160>, 32 * 20, zfft8::smem_bytes<160>());
        }
        const int occ = std::max(1, per_sm[N3 == 40 ? 0 : (N3 == 120 ? 1 : 2)]);
        const unsigned zb = (unsigned)std::min<long long>((n_lines + 31) / 32, (long long)ctx->sm_count * occ);
        if (N3 == 40) zfft8::z_fft8_scatter_kernel<40><<<zb, 32 * 5, zfft8::smem_bytes<40>(), ctx->stream>>>(za);
        else if (N3 == 120) zfft8::z_fft8_scatter_kernel<120><<<zb, 32 * 15, zfft8::smem_bytes<120>(), ctx->stream>>>(za);
        else zfft8::z_fft8_scatter_kernel<160><<<zb, 32 * 20, zfft8::smem_bytes<160>(), ctx->stream>>>(za);
        RPA_LAUNCH_CHECK(ctx);
        rc = RPA_OK;
      } else {
        rc = launch_axis<false, 1>(ctx, T, mp->ax[2].fwd(), n_lines, J, zs);
      }
    }
    if (rc) return rc;
  }
  if (ctx->uc_cache && ctx->uc_cache_src == psi_c && ctx->uc_cache_nc == nc) ctx->uc_cache_filled = true;
  return RPA_OK;
}
