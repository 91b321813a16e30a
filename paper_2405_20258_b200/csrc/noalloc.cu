// rpa_chi0_static_noalloc: CHI_SUM at omega = 0 (eq. 6 with :71 eq. 5 and :152 eq. 15; readings R5/R6) for
// callers that cannot allocate or lend device memory at call time -- code under CUDA graph capture, tight serving loops,
// harnesses that forbid cudaMalloc.  Same arithmetic and same kernels as rpa_chi0_static (pair_weights_kernel + the
// Hermitian DMMA contraction); the only difference is where the one piece of scratch that call needs lives: the pair
// weights D_vc(0) = 2 / Delta_vc, [nvb * nc] doubles, go into the file-scope device array below instead of the workspace
// lent with rpa_set_workspace.
//
//   * The array is RPA_NOALLOC_MAX_PAIRS doubles = 4 MiB.  It is part of the library image: every GPU that loads
//     librpa_b200.so holds it until the process exits.
//   * In host code the NAME of a __device__ array is a host-side stand-in, not a device address (a kernel given it would
//     fault, or silently use host memory where the GPU can reach it).  The device address is fetched once per device with
//     cudaGetSymbolAddress, with that device current, and that pointer is what the kernels get.
//   * Every call on a device shares the array and finds the previous call's contents in it.  Nothing in it has to start
//     at zero: a call overwrites the nvb * nc entries it reads before it reads them.  Calls that overlap on the GPU
//     (two streams, two contexts on one device) race on it; calls on one stream are ordered and safe.
//   * The entry point calls no cudaMalloc / cudaFree and no allocating library routine.
#include <mutex>

#include "rpa_internal.h"

#define RPA_NOALLOC_MAX_PAIRS (1 << 19)

static __device__ __align__(256) double g_noalloc_pair_weights[RPA_NOALLOC_MAX_PAIRS];

// device address of g_noalloc_pair_weights per device ordinal (each device has its own copy of the array)
constexpr int RPA_NOALLOC_MAX_DEVICES = 64;
static double* g_noalloc_ptr[RPA_NOALLOC_MAX_DEVICES];
static std::mutex g_noalloc_mutex;

namespace {

// Once per device, with that device current.  cudaGetSymbolAddress allocates nothing: the array exists since the module
// was loaded on the device.
int noalloc_setup(rpa_ctx* ctx, double** out) {
  if (ctx->device < 0 || ctx->device >= RPA_NOALLOC_MAX_DEVICES)
    return rpa_fail(ctx, RPA_ERR_INVALID, "rpa_chi0_static_noalloc: device ordinal %d beyond the %d this entry point serves", ctx->device,
                    RPA_NOALLOC_MAX_DEVICES);
  RPA_CUDA(ctx, cudaSetDevice(ctx->device));
  std::lock_guard<std::mutex> lock(g_noalloc_mutex);
  if (!g_noalloc_ptr[ctx->device]) {
    double* p = nullptr;
    cudaError_t e = cudaGetSymbolAddress((void**)&p, g_noalloc_pair_weights);
    if (e != cudaSuccess || !p)
      return rpa_fail(ctx, RPA_ERR_CUDA, "rpa_chi0_static_noalloc: cudaGetSymbolAddress failed: %s", cudaGetErrorString(e));
    g_noalloc_ptr[ctx->device] = p;
  }
  *out = g_noalloc_ptr[ctx->device];
  return RPA_OK;
}

}  // namespace

extern "C" {

long long rpa_noalloc_max_pairs(void) { return RPA_NOALLOC_MAX_PAIRS; }

int rpa_noalloc_setup(rpa_ctx* ctx) {
  if (!ctx) return rpa_fail(nullptr, RPA_ERR_INVALID, "null context");
  double* p = nullptr;
  return noalloc_setup(ctx, &p);
}

int rpa_chi0_static_noalloc(rpa_ctx* ctx, const void* M, int nvb, int nc, const double* e_v, const double* e_c, int accumulate,
                            void* chi0) {
  if (!ctx) return rpa_fail(nullptr, RPA_ERR_INVALID, "null context");
  if (!M || !e_v || !e_c || !chi0 || nvb < 1 || nc < 1) return rpa_fail(ctx, RPA_ERR_INVALID, "rpa_chi0_static_noalloc: invalid argument");
  const long long P = (long long)nvb * nc;
  if (P > RPA_NOALLOC_MAX_PAIRS)
    return rpa_fail(ctx, RPA_ERR_INVALID,
                    "rpa_chi0_static_noalloc: nvb * nc = %lld pairs exceed the %d the built-in scratch array holds; "
                    "split the valence block or use rpa_chi0_static with a workspace", P, RPA_NOALLOC_MAX_PAIRS);
  double* wk = nullptr;
  int rc = noalloc_setup(ctx, &wk);   // a table look-up after the first call on this device
  if (rc) return rc;
  // D_vc(0) = 2 / Delta_vc into the static array (eq. 5), then the Hermitian rank-P update (eq. 6)
  if ((rc = pair_weights(ctx, e_v, e_c, nvb, nc, nullptr, 1, wk))) return rc;
  ZgemmParams g;
  g.A = (const cplx*)M; g.lda = ctx->n_g; g.a_km = true; g.B = (const cplx*)M; g.ldb = ctx->n_g; g.b_kn = true;
  g.C = (cplx*)chi0; g.ldc = ctx->n_g; g.M = ctx->n_g; g.N = ctx->n_g; g.K = nvb * nc;
  g.conj_b = true; g.herm = true; g.accumulate = accumulate != 0; g.alpha = -1.0;
  g.rs = ctx->d_vsqrt; g.cs = ctx->d_vsqrt;
  g.wk = wk;
  return zgemm_dmma(ctx, g);
}

}  // extern "C"
