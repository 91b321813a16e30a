// Internal declarations shared by the translation units of librpa_b200.so (not part of the C-ABI).
#pragma once
#include <cuda_runtime.h>
#include <cstdarg>
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <string>
#include <vector>

#include "rpa_b200.h"

typedef double2 cplx;  // interleaved (re, im), same bytes as cuDoubleComplex / torch.complex128

struct rpa_ctx {
  int device = 0;
  cudaStream_t stream = nullptr;
  std::string err;
  long long launches = 0;
  int sm_count = 148;

  // Diagnostic switches, read ONCE from the environment by rpa_create (listed under "Diagnostics" in rpa_b200.h); the
  // tests use them to force the routes that the default size rules would not take on small test inputs.
  struct Options {
    bool generic_fft = false;      // RPA_GENERIC_FFT=1: generic mixed-radix MTXEL kernels instead of the radix-8 x R ones
    bool verbose = false;          // RPA_VERBOSE=1: route decisions and kernel resources on stderr
    bool no_tridiag = false;       // RPA_NO_TRIDIAG=1: a3 skips the tridiagonalisation route (block iteration / Jacobi run)
    int jacobi_block_min = 1024;   // RPA_JACOBI_BLOCK_MIN: smallest matrix that takes the GEMM block Jacobi
    int hetrd_mode = -1;           // RPA_HETRD_MODE=0..2: force a large-matrix variant of the tridiagonalisation kernel
    int hetrd_threads = 0;         // RPA_HETRD_THREADS: its CTA size
    bool zgemm_tma = true;         // RPA_ZGEMM_TMA=0: Hermitian [k][m] updates staged by cp.async + block barrier instead of TMA + mbarriers
  } opt;

  // Kernel function attributes (dynamic shared memory > 48 KB) are per device: each launch site sets them the first time
  // THIS context reaches it (attr_once), never once per process.  Resident-CTA counts queried with them live here too.
  unsigned long long attr_mask = 0;
  bool attr_once(int id) { const unsigned long long b = 1ull << id; if (attr_mask & b) return false; attr_mask |= b; return true; }
  int z_per_sm[3] = {0, 0, 0};     // z_fft8_scatter_kernel<40/120/160>
  void* tma_encode = nullptr;      // cuTensorMapEncodeTiled, fetched through the runtime (no link against libcuda)

  // problem statement
  double cell[9];
  int fft[3];
  int n_r = 0, n_g = 0, n_pw = 0;

  // plans (device, owned)
  struct MtxelPlan* mtxel = nullptr;  // FFT plans, index maps (mtxel.cu)
  double* d_vsqrt = nullptr;           // [n_g]  v^1/2

  // workspace lent by the caller
  char* ws = nullptr;
  size_t ws_bytes = 0;

  // real-space conduction functions u_c kept across the valence blocks of one rpa_energy_* call when HBM allows
  // (set by the driver in api.cu, used by mtxel_run): the first uc_cache_rows of the uc_cache_nc bands of coefficient
  // array uc_cache_src, [uc_cache_rows][n_r]
  cplx* uc_cache = nullptr; const cplx* uc_cache_src = nullptr; int uc_cache_nc = 0, uc_cache_rows = 0; bool uc_cache_filled = false;

  // the two-pass loop between rpa_pass_begin and rpa_pass_end (api.cu): caller's inputs, the persistent part of the
  // workspace (chi~0, C, lambda, chi_s, the M block or all of M) and the stage timers
  struct PassState {
    bool active = false, keep_all = false, timing = false;
    int stage = 0;   // 0 begun, 1 pass 1 done, 2 basis set, 3 pass 2 done, 4 energy done
    const cplx* psi_v = nullptr; const cplx* psi_c = nullptr; const double* e_v = nullptr; const double* e_c = nullptr; const double* omega = nullptr;
    int nv = 0, nc = 0, nvb = 0, n_eig = 0, n_w = 0, nblocks = 0;
    cplx* chi0 = nullptr; cplx* C = nullptr; cplx* chi_s = nullptr; cplx* Mbuf = nullptr; double* lam = nullptr;
    char* scratch = nullptr; size_t scratch_bytes = 0;
    std::vector<cudaEvent_t> evs; std::vector<int> ev_stage;
  } pass;

  // last direct Jacobi eigen-decomposition of the basis stage: matrix size, sweeps, 0 = vector iteration / 1 = block
  int jac_n = 0, jac_sweeps = 0, jac_kind = 0;
  // what the last basis stage measured on its result: max_i ||chi0 c_i - lambda_i c_i|| / |lambda_1| and max|C C^H - 1|
  double basis_residual = -1.0, basis_ortho = -1.0;

  // per-kernel-class device timers (rpa_profile_begin / rpa_profile_end): event pairs around the launches of a class
  bool prof = false;
  struct ProfRec { int cls; cudaEvent_t a, b; };
  std::vector<ProfRec> prof_recs;
  std::vector<cudaEvent_t> prof_pool;
};

// attr_once ids
enum { RPA_ATTR_ZGEMM = 0 /* + 16 layout/HERM combinations */, RPA_ATTR_AXIS = 16 /* + 4 */, RPA_ATTR_FFT8 = 20 /* + 4 */,
       RPA_ATTR_ZFFT8 = 24, RPA_ATTR_POTRF = 25, RPA_ATTR_TRSM = 26, RPA_ATTR_JACOBI = 27, RPA_ATTR_PLANE_GENERIC = 28 /* + 2 */,
       RPA_ATTR_WFN = 30 /* + 4 */, RPA_ATTR_ZHERK_TMA = 34, RPA_ATTR_ZGEMM_TMA_MK = 35 };

int rpa_fail(rpa_ctx* ctx, int code, const char* fmt, ...);
#define RPA_CUDA(ctx, call)                                                              \
  do {                                                                                   \
    cudaError_t e__ = (call);                                                            \
    if (e__ != cudaSuccess)                                                              \
      return rpa_fail(ctx, RPA_ERR_CUDA, "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e__), \
                      __FILE__, __LINE__);                                               \
  } while (0)
#define RPA_LAUNCH_CHECK(ctx)                                                            \
  do {                                                                                   \
    (ctx)->launches++;                                                                   \
    cudaError_t e__ = cudaGetLastError();                                                \
    if (e__ != cudaSuccess)                                                              \
      return rpa_fail(ctx, RPA_ERR_CUDA, "kernel launch failed: %s (%s:%d)", cudaGetErrorString(e__), \
                      __FILE__, __LINE__);                                               \
  } while (0)

// Times the launches enqueued during its lifetime under class `cls` (RPA_PROF_* of rpa_b200.h) when profiling is on.
struct ProfScope {
  rpa_ctx* ctx; bool on; rpa_ctx::ProfRec rec;
  static cudaEvent_t get(rpa_ctx* c) {
    cudaEvent_t e;
    if (!c->prof_pool.empty()) { e = c->prof_pool.back(); c->prof_pool.pop_back(); }
    else cudaEventCreate(&e);
    return e;
  }
  ProfScope(rpa_ctx* c, int cls) : ctx(c), on(c->prof) {
    if (!on) return;
    rec.cls = cls; rec.a = get(c); rec.b = get(c);
    cudaEventRecord(rec.a, c->stream);
  }
  ~ProfScope() {
    if (!on) return;
    cudaEventRecord(rec.b, ctx->stream);
    ctx->prof_recs.push_back(rec);
  }
};

// bump allocator over the caller's workspace (256-byte aligned)
struct WsAlloc {
  char* base;
  size_t cap, off = 0;
  bool ok = true;
  WsAlloc(char* b, size_t c) : base(b), cap(c) {}
  template <class T>
  T* get(size_t n) {
    size_t bytes = (n * sizeof(T) + 255) & ~size_t(255);
    if (!base || off + bytes > cap) { ok = false; off += bytes; return nullptr; }
    T* p = reinterpret_cast<T*>(base + off);
    off += bytes;
    return p;
  }
};
static inline size_t ws_round(size_t bytes) { return (bytes + 255) & ~size_t(255); }

// ---------------------------------------------------------------------------------------------
// Complex FP64 GEMM on the DMMA (mma.sync m8n8k4 f64) path -- zgemm_dmma.cu
//   C[m][n] (+)= alpha * rs[m] * cs[n] * sum_k w_k * A^(m,k) * opB(B^(n,k)),  opB = conj or identity.
struct ZgemmParams {
  const cplx* A = nullptr; long long lda = 0; bool a_km = false;  // a_km: A stored [k][m] (m fastest) else [m][k]
  const cplx* B = nullptr; long long ldb = 0; bool b_kn = false;
  cplx* C = nullptr; long long ldc = 0;
  int M = 0, N = 0, K = 0;
  bool conj_b = true;
  bool herm = false;          // A^ == B^ rows: compute tiles with tile_m >= tile_n only, mirror the rest
  bool accumulate = false;
  double alpha = 1.0;
  const double* rs = nullptr; // [M] optional
  const double* cs = nullptr; // [N] optional
  // k weights: wk == nullptr none, else w_k = wk[batch * strideW + k] (the pair weights D_vc(i omega) of eq. 5 written
  // by pair_weights(), or v^1/2 for the projection)
  const double* wk = nullptr; long long strideW = 0;
  int batch = 1; long long strideA = 0, strideB = 0, strideC = 0;
  int split_k = 0;            // 0 = choose automatically
  bool tma_mk = false;        // [m][k] x [n][k] product that may take the TMA-staged kernel (the projection asks for it)
};
int zgemm_dmma(rpa_ctx* ctx, const ZgemmParams& p);
// out[k][v * nc + c] = 2 D/(D^2 + omega_k^2), D = e_c[c] - e_v[v]  (eq. 5 in the reading R6); omega == nullptr: one
// row with omega = 0
int pair_weights(rpa_ctx* ctx, const double* e_v, const double* e_c, int nvb, int nc, const double* omega, int n_w, double* out,
                 const double* f_v = nullptr, const double* f_c = nullptr);   // f given: times max(f_v - f_c, 0)
int fp64_peak_kernel(rpa_ctx* ctx, int kind, int iters, double* tflops);

// mtxel.cu
int mtxel_plan_create(rpa_ctx* ctx, const int32_t* g_eps, const int32_t* g_wfn);
void mtxel_plan_destroy(rpa_ctx* ctx);
size_t mtxel_workspace_bytes(const rpa_ctx* ctx, int nvb, int nc);
int mtxel_run(rpa_ctx* ctx, WsAlloc& ws, const cplx* psi_v, int nvb, const cplx* psi_c, int nc, cplx* M);

// basis.cu
size_t basis_workspace_bytes(const rpa_ctx* ctx, int n, int n_eig);
int basis_run(rpa_ctx* ctx, WsAlloc& ws, const cplx* chi0, int n, int n_eig, double tol, cplx* C, double* lambda,
              int* iters_out);

// tridiag_eig.cu
size_t tridiag_workspace_bytes(int n, int n_eig);
int tridiag_eigh_lowest(rpa_ctx* ctx, WsAlloc& ws, const cplx* H, long long ld, int n, int n_eig, cplx* Abuf, cplx* Vbuf, cplx* C,
                        double* lambda);

// energy.cu
size_t energy_workspace_bytes(const rpa_ctx* ctx, int n_eig, int n_w);
int energy_run(rpa_ctx* ctx, WsAlloc& ws, const cplx* chi_s, int n_eig, const double* weight, int n_w, double* e_c,
               double* per_freq);

size_t epsinv_workspace_bytes(const rpa_ctx* ctx, int n_eig, int n_w);
int epsinv_run(rpa_ctx* ctx, WsAlloc& ws, const cplx* chi_s, int n_eig, int n_w, cplx* eps_inv);

// chol.cu
int zpotrf_batched(rpa_ctx* ctx, cplx* A, int n, long long lda, int batch, long long stride, int* d_info, int shift = 0,
                   double* dvec = nullptr);
int ztrsm_left_lower(rpa_ctx* ctx, const cplx* L, long long ldl, int p, cplx* X, long long ldx, int ncols);
