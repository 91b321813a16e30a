// C-ABI of librpa_b200.so (include/rpa_b200.h): argument checking, workspace carving and the NV-block two-pass driver
// (PAPER.md:139-158).  All arithmetic of the hot path runs in the CUDA kernels of the other translation units.
#include <algorithm>
#include <cmath>
#include <cstdlib>

#include "rpa_internal.h"

static thread_local std::string g_null_err;

int rpa_fail(rpa_ctx* ctx, int code, const char* fmt, ...) {
  char buf[512];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof(buf), fmt, ap);
  va_end(ap);
  if (ctx) ctx->err = buf; else g_null_err = buf;
  return code;
}

namespace {

// Cs[i][G] = C[i][G] v^1/2(G): the Coulomb factor of the projection (eq. 7) folded into the basis once per call,
// so that the projection GEMM multiplies no weights in its main loop
__global__ void scale_basis_kernel(const cplx* __restrict__ C, const double* __restrict__ vsqrt, int n_g, long long total,
                                   cplx* __restrict__ out) {
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < total; i += (long long)gridDim.x * blockDim.x) {
    const double s = vsqrt[i % n_g];
    const cplx c = C[i];
    out[i] = make_double2(c.x * s, c.y * s);
  }
}

__global__ void sqrt_kernel(const double* __restrict__ v, int n, double* __restrict__ out) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) out[i] = sqrt(v[i]);
}

size_t chi_freq_vchunk(const rpa_ctx* ctx, int nvb, int nc, int n_eig) {
  (void)ctx;
  const size_t per_v = (size_t)nc * n_eig * sizeof(cplx);
  size_t budget = (size_t)4 << 30;
  size_t vc = std::max<size_t>(1, budget / std::max<size_t>(per_v, 1));
  return std::min<size_t>(vc, (size_t)nvb);
}
size_t chi_freq_workspace(const rpa_ctx* ctx, int nvb, int nc, int n_eig, int n_w) {
  return ws_round(chi_freq_vchunk(ctx, nvb, nc, n_eig) * nc * n_eig * sizeof(cplx)) + ws_round((size_t)n_w * nvb * nc * sizeof(double)) +
         ws_round((size_t)n_eig * ctx->n_g * sizeof(cplx));
}
size_t chi0_static_workspace(int nvb, int nc) { return ws_round((size_t)nvb * nc * sizeof(double)); }

int do_chi0_static(rpa_ctx* ctx, WsAlloc& ws, const cplx* M, int nvb, int nc, const double* e_v, const double* e_c,
                   int accumulate, cplx* chi0, const double* f_v = nullptr, const double* f_c = nullptr) {
  double* wk = ws.get<double>((size_t)nvb * nc);
  if (!ws.ok) return rpa_fail(ctx, RPA_ERR_WORKSPACE, "rpa_chi0_static: workspace too small (need %zu bytes)", ws.off);
  int rc = pair_weights(ctx, e_v, e_c, nvb, nc, nullptr, 1, wk, f_v, f_c);   // D_vc(0) = 2/Delta_vc  (eq. 5)
  if (rc) return rc;
  ZgemmParams g;
  g.A = M; g.lda = ctx->n_g; g.a_km = true; g.B = M; g.ldb = ctx->n_g; g.b_kn = true;
  g.C = chi0; g.ldc = ctx->n_g; g.M = ctx->n_g; g.N = ctx->n_g; g.K = nvb * nc;
  g.conj_b = true; g.herm = true; g.accumulate = accumulate != 0; g.alpha = -1.0;
  g.rs = ctx->d_vsqrt; g.cs = ctx->d_vsqrt;
  g.wk = wk;
  ProfScope ps(ctx, RPA_PROF_CHI0);
  return zgemm_dmma(ctx, g);
}

int do_chi_freq(rpa_ctx* ctx, WsAlloc& ws, const cplx* M, int nvb, int nc, const double* e_v, const double* e_c, const cplx* C,
                int n_eig, const double* omega, int n_w, int accumulate, cplx* chi_s, const double* f_v = nullptr,
                const double* f_c = nullptr) {
  const int n_g = ctx->n_g;
  const long long Pall = (long long)nvb * nc;
  double* wk = ws.get<double>((size_t)n_w * Pall);   // D_vc(i omega_k) for the whole block, [k][v * nc + c]
  if (!ws.ok) return rpa_fail(ctx, RPA_ERR_WORKSPACE, "rpa_chi_subspace_freq: workspace too small (need %zu bytes)", ws.off);
  int rc = pair_weights(ctx, e_v, e_c, nvb, nc, omega, n_w, wk, f_v, f_c);
  if (rc) return rc;
  if (!C) {  // full basis: chi~0(i w_k) directly from M
    ZgemmParams g;
    g.A = M; g.lda = n_g; g.a_km = true; g.B = M; g.ldb = n_g; g.b_kn = true;
    g.C = chi_s; g.ldc = n_g; g.M = n_g; g.N = n_g; g.K = nvb * nc;
    g.conj_b = true; g.herm = true; g.accumulate = accumulate != 0; g.alpha = -1.0;
    g.rs = ctx->d_vsqrt; g.cs = ctx->d_vsqrt;
    g.wk = wk; g.strideW = Pall;
    g.batch = n_w; g.strideC = (long long)n_g * n_g;
    ProfScope ps(ctx, RPA_PROF_CHIS);
    return zgemm_dmma(ctx, g);
  }
  const int vchunk = (int)chi_freq_vchunk(ctx, nvb, nc, n_eig);
  cplx* Bp = ws.get<cplx>((size_t)vchunk * nc * n_eig);
  cplx* Cs = ws.get<cplx>((size_t)n_eig * n_g);
  if (!ws.ok) return rpa_fail(ctx, RPA_ERR_WORKSPACE, "rpa_chi_subspace_freq: workspace too small (need %zu bytes)", ws.off);
  {
    const long long total = (long long)n_eig * n_g;
    scale_basis_kernel<<<(unsigned)std::min<long long>((total + 255) / 256, 8192), 256, 0, ctx->stream>>>(C, ctx->d_vsqrt, n_g, total, Cs);
    RPA_LAUNCH_CHECK(ctx);
  }
  for (int v0 = 0; v0 < nvb; v0 += vchunk) {
    const int nv = std::min(vchunk, nvb - v0);
    const int P = nv * nc;
    // projection  Bp[p][i] = sum_G M[p][G] v^1/2(G) conj(C[i][G])        (eq. 7)
    ZgemmParams g;
    g.A = M + (long long)v0 * nc * n_g; g.lda = n_g; g.a_km = false;
    g.B = Cs; g.ldb = n_g; g.b_kn = false;                                // v^1/2 sits in Cs: no k weights
    g.C = Bp; g.ldc = n_eig; g.M = P; g.N = n_eig; g.K = n_g; g.conj_b = true; g.tma_mk = true;
    { ProfScope ps(ctx, RPA_PROF_PROJ); rc = zgemm_dmma(ctx, g); }
    if (rc) return rc;
    // chi_s[k] (+)= - sum_p Bp[p][:] D_p(w_k) Bp[p][:]^H                   (eq. 8)
    ZgemmParams h;
    h.A = Bp; h.lda = n_eig; h.a_km = true; h.B = Bp; h.ldb = n_eig; h.b_kn = true;
    h.C = chi_s; h.ldc = n_eig; h.M = n_eig; h.N = n_eig; h.K = P;
    h.conj_b = true; h.herm = true; h.accumulate = (accumulate != 0) || v0 > 0; h.alpha = -1.0;
    h.wk = wk + (long long)v0 * nc; h.strideW = Pall;
    h.batch = n_w; h.strideC = (long long)n_eig * n_eig;
    { ProfScope ps(ctx, RPA_PROF_CHIS); rc = zgemm_dmma(ctx, h); }
    if (rc) return rc;
  }
  return RPA_OK;
}

bool bad_ctx(rpa_ctx* ctx) { return ctx == nullptr; }

}  // namespace

extern "C" {

int rpa_create(rpa_ctx** out, const double cell[9], const int fft[3], int n_g, const int32_t* g_eps, const double* vcoul,
               int n_pw, const int32_t* g_wfn, int device, void* cuda_stream) {
  if (!out) return rpa_fail(nullptr, RPA_ERR_INVALID, "rpa_create: out is null");
  *out = nullptr;
  if (!cell || !fft || !g_eps || !vcoul || !g_wfn) return rpa_fail(nullptr, RPA_ERR_INVALID, "rpa_create: null argument");
  if (n_g <= 0 || n_pw <= 0) return rpa_fail(nullptr, RPA_ERR_INVALID, "rpa_create: n_g and n_pw must be positive");
  for (int i = 0; i < n_g; i++)
    if (!(vcoul[i] >= 0.0) || !std::isfinite(vcoul[i]))
      return rpa_fail(nullptr, RPA_ERR_INVALID, "rpa_create: vcoul[%d] is negative or not finite", i);
  int ndev = 0;
  cudaError_t e = cudaGetDeviceCount(&ndev);
  if (e != cudaSuccess || ndev <= 0)
    return rpa_fail(nullptr, RPA_ERR_CUDA, "rpa_create: no CUDA device (%s); there is no CPU fallback",
                    e == cudaSuccess ? "device count 0" : cudaGetErrorString(e));
  if (device < 0 || device >= ndev) return rpa_fail(nullptr, RPA_ERR_INVALID, "rpa_create: device %d out of range", device);
  rpa_ctx* ctx = new rpa_ctx();
  ctx->device = device;
  ctx->stream = (cudaStream_t)cuda_stream;
  memcpy(ctx->cell, cell, sizeof(ctx->cell));
  for (int a = 0; a < 3; a++) ctx->fft[a] = fft[a];
  ctx->n_g = n_g; ctx->n_pw = n_pw;
  {  // diagnostic switches (rpa_b200.h "Diagnostics"): read here, once, never on the launch paths
    auto on = [](const char* k) { const char* e = getenv(k); return e && e[0] == '1'; };
    auto num = [](const char* k, int dflt) { const char* e = getenv(k); return e && *e ? atoi(e) : dflt; };
    ctx->opt.generic_fft = on("RPA_GENERIC_FFT");
    ctx->opt.verbose = on("RPA_VERBOSE");
    ctx->opt.no_tridiag = on("RPA_NO_TRIDIAG");
    ctx->opt.jacobi_block_min = std::max(2, num("RPA_JACOBI_BLOCK_MIN", 1024));
    ctx->opt.hetrd_mode = num("RPA_HETRD_MODE", -1);
    ctx->opt.hetrd_threads = num("RPA_HETRD_THREADS", 0);
    { const char* e = getenv("RPA_ZGEMM_TMA"); ctx->opt.zgemm_tma = !(e && e[0] == '0'); }
  }
  auto fail = [&](int rc) { g_null_err = ctx->err; rpa_destroy(ctx); return rc; };
  if ((e = cudaSetDevice(device)) != cudaSuccess) return fail(rpa_fail(ctx, RPA_ERR_CUDA, "cudaSetDevice: %s", cudaGetErrorString(e)));
  cudaDeviceProp prop;
  if ((e = cudaGetDeviceProperties(&prop, device)) != cudaSuccess)
    return fail(rpa_fail(ctx, RPA_ERR_CUDA, "cudaGetDeviceProperties: %s", cudaGetErrorString(e)));
  ctx->sm_count = prop.multiProcessorCount;
  if (prop.major != 10 || prop.minor != 0)   // the .so holds sm_100a SASS only (arch-specific: no PTX JIT to other parts)
    return fail(rpa_fail(ctx, RPA_ERR_CUDA, "device %d is sm_%d%d; this library is built for sm_100a (compute capability 10.0) only", device, prop.major, prop.minor));
  long long nr = 1;
  for (int a = 0; a < 3; a++) {
    if (fft[a] < 1) return fail(rpa_fail(ctx, RPA_ERR_INVALID, "rpa_create: fft[%d] = %d", a, fft[a]));
    nr *= fft[a];
  }
  if (nr > 2147483647LL) return fail(rpa_fail(ctx, RPA_ERR_INVALID, "rpa_create: fft grid too large"));
  ctx->n_r = (int)nr;
  int rc = mtxel_plan_create(ctx, g_eps, g_wfn);
  if (rc) return fail(rc);
  double* d_v = nullptr;
  if (cudaMalloc(&d_v, n_g * sizeof(double)) != cudaSuccess || cudaMalloc(&ctx->d_vsqrt, n_g * sizeof(double)) != cudaSuccess)
    return fail(rpa_fail(ctx, RPA_ERR_CUDA, "rpa_create: cudaMalloc failed"));
  e = cudaMemcpy(d_v, vcoul, n_g * sizeof(double), cudaMemcpyHostToDevice);
  if (e == cudaSuccess) {
    sqrt_kernel<<<(n_g + 255) / 256, 256, 0, ctx->stream>>>(d_v, n_g, ctx->d_vsqrt);
    ctx->launches++;
    e = cudaGetLastError();
  }
  if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
  cudaFree(d_v);
  if (e != cudaSuccess) return fail(rpa_fail(ctx, RPA_ERR_CUDA, "rpa_create: upload of v(G): %s", cudaGetErrorString(e)));
  *out = ctx;
  return RPA_OK;
}

int rpa_destroy(rpa_ctx* ctx) {
  if (!ctx) return RPA_OK;
  cudaSetDevice(ctx->device);
  for (auto e : ctx->pass.evs) cudaEventDestroy(e);
  ctx->pass.evs.clear();
  mtxel_plan_destroy(ctx);
  cudaFree(ctx->d_vsqrt);
  for (auto& r : ctx->prof_recs) { cudaEventDestroy(r.a); cudaEventDestroy(r.b); }
  for (auto e : ctx->prof_pool) cudaEventDestroy(e);
  delete ctx;
  return RPA_OK;
}

const char* rpa_last_error(const rpa_ctx* ctx) { return ctx ? ctx->err.c_str() : g_null_err.c_str(); }

long long rpa_launch_count(const rpa_ctx* ctx) { return ctx ? ctx->launches : 0; }

int rpa_basis_info(const rpa_ctx* ctx, int* n, int* sweeps, int* kind) {
  if (!ctx || !n || !sweeps || !kind) return RPA_ERR_INVALID;
  *n = ctx->jac_n; *sweeps = ctx->jac_sweeps; *kind = ctx->jac_kind;
  return RPA_OK;
}

int rpa_basis_quality(const rpa_ctx* ctx, double* residual, double* orthogonality) {
  if (!ctx || !residual || !orthogonality) return RPA_ERR_INVALID;
  *residual = ctx->basis_residual; *orthogonality = ctx->basis_ortho;
  return RPA_OK;
}

int rpa_profile_begin(rpa_ctx* ctx) {
  if (bad_ctx(ctx)) return rpa_fail(nullptr, RPA_ERR_INVALID, "null context");
  for (auto& r : ctx->prof_recs) { ctx->prof_pool.push_back(r.a); ctx->prof_pool.push_back(r.b); }
  ctx->prof_recs.clear();
  ctx->prof = true;
  return RPA_OK;
}

int rpa_profile_end(rpa_ctx* ctx, double* ms, long long* launches) {
  if (bad_ctx(ctx)) return rpa_fail(nullptr, RPA_ERR_INVALID, "null context");
  if (!ms || !launches) return rpa_fail(ctx, RPA_ERR_INVALID, "rpa_profile_end: null argument");
  ctx->prof = false;
  RPA_CUDA(ctx, cudaSetDevice(ctx->device));
  RPA_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
  for (int c = 0; c < RPA_PROF_NCLASS; c++) { ms[c] = 0.0; launches[c] = 0; }
  for (auto& r : ctx->prof_recs) {
    float t = 0.f;
    if (cudaEventElapsedTime(&t, r.a, r.b) == cudaSuccess && r.cls >= 0 && r.cls < RPA_PROF_NCLASS) { ms[r.cls] += t; launches[r.cls]++; }
    ctx->prof_pool.push_back(r.a); ctx->prof_pool.push_back(r.b);
  }
  ctx->prof_recs.clear();
  return RPA_OK;
}

size_t rpa_workspace_bytes(const rpa_ctx* ctx, int nvb, int nc, int n_eig, int n_w) {
  if (!ctx || nvb < 1 || nc < 1 || n_eig < 1 || n_w < 1) return 0;
  size_t need = mtxel_workspace_bytes(ctx, nvb, nc);
  need = std::max(need, basis_workspace_bytes(ctx, ctx->n_g, n_eig));
  need = std::max(need, chi_freq_workspace(ctx, nvb, nc, n_eig, n_w));
  need = std::max(need, chi0_static_workspace(nvb, nc));
  need = std::max(need, energy_workspace_bytes(ctx, n_eig, n_w));
  return need + 4096;
}

int rpa_set_workspace(rpa_ctx* ctx, void* dev_ptr, size_t bytes) {
  if (bad_ctx(ctx)) return rpa_fail(nullptr, RPA_ERR_INVALID, "null context");
  if (dev_ptr && ((uintptr_t)dev_ptr & 255)) return rpa_fail(ctx, RPA_ERR_INVALID, "workspace must be 256-byte aligned");
  if (ctx->pass.active) rpa_pass_end(ctx);   // an open pass sequence lives in the old workspace
  ctx->ws = (char*)dev_ptr;
  ctx->ws_bytes = dev_ptr ? bytes : 0;
  return RPA_OK;
}

int rpa_mtxel(rpa_ctx* ctx, const void* psi_v, int nvb, const void* psi_c, int nc, void* M) {
  if (bad_ctx(ctx)) return rpa_fail(nullptr, RPA_ERR_INVALID, "null context");
  if (!psi_v || !psi_c || !M || nvb < 1 || nc < 1) return rpa_fail(ctx, RPA_ERR_INVALID, "rpa_mtxel: invalid argument");
  if ((long long)nvb * nc > 2147483647LL) return rpa_fail(ctx, RPA_ERR_INVALID, "rpa_mtxel: too many pairs in one block");
  RPA_CUDA(ctx, cudaSetDevice(ctx->device));
  WsAlloc ws(ctx->ws, ctx->ws_bytes);
  return mtxel_run(ctx, ws, (const cplx*)psi_v, nvb, (const cplx*)psi_c, nc, (cplx*)M);
}

int rpa_chi0_static(rpa_ctx* ctx, const void* M, int nvb, int nc, const double* e_v, const double* e_c, int accumulate,
                    void* chi0) {
  if (bad_ctx(ctx)) return rpa_fail(nullptr, RPA_ERR_INVALID, "null context");
  if (!M || !e_v || !e_c || !chi0 || nvb < 1 || nc < 1) return rpa_fail(ctx, RPA_ERR_INVALID, "rpa_chi0_static: invalid argument");
  if ((long long)nvb * nc > 2147483647LL) return rpa_fail(ctx, RPA_ERR_INVALID, "rpa_chi0_static: too many pairs");
  RPA_CUDA(ctx, cudaSetDevice(ctx->device));
  WsAlloc ws(ctx->ws, ctx->ws_bytes);
  return do_chi0_static(ctx, ws, (const cplx*)M, nvb, nc, e_v, e_c, accumulate, (cplx*)chi0);
}

int rpa_subspace_basis(rpa_ctx* ctx, const void* chi0, int n_eig, double tol, void* C, double* lambda, int* iters_out) {
  if (bad_ctx(ctx)) return rpa_fail(nullptr, RPA_ERR_INVALID, "null context");
  if (!chi0 || !C || !lambda) return rpa_fail(ctx, RPA_ERR_INVALID, "rpa_subspace_basis: null argument");
  if (n_eig < 1 || n_eig > ctx->n_g) return rpa_fail(ctx, RPA_ERR_INVALID, "rpa_subspace_basis: n_eig = %d not in 1..n_g = %d", n_eig, ctx->n_g);
  RPA_CUDA(ctx, cudaSetDevice(ctx->device));
  WsAlloc ws(ctx->ws, ctx->ws_bytes);
  return basis_run(ctx, ws, (const cplx*)chi0, ctx->n_g, n_eig, tol, (cplx*)C, lambda, iters_out);
}

int rpa_chi_subspace_freq(rpa_ctx* ctx, const void* M, int nvb, int nc, const double* e_v, const double* e_c, const void* C,
                          int n_eig, const double* omega, int n_w, int accumulate, void* chi_s) {
  if (bad_ctx(ctx)) return rpa_fail(nullptr, RPA_ERR_INVALID, "null context");
  if (!M || !e_v || !e_c || !omega || !chi_s || nvb < 1 || nc < 1 || n_w < 1)
    return rpa_fail(ctx, RPA_ERR_INVALID, "rpa_chi_subspace_freq: invalid argument");
  if (n_eig < 1 || n_eig > ctx->n_g || (!C && n_eig != ctx->n_g))
    return rpa_fail(ctx, RPA_ERR_INVALID, "rpa_chi_subspace_freq: n_eig = %d invalid (n_g = %d, C %s)", n_eig, ctx->n_g, C ? "given" : "null");
  if ((long long)nvb * nc > 2147483647LL) return rpa_fail(ctx, RPA_ERR_INVALID, "rpa_chi_subspace_freq: too many pairs");
  RPA_CUDA(ctx, cudaSetDevice(ctx->device));
  WsAlloc ws(ctx->ws, ctx->ws_bytes);
  return do_chi_freq(ctx, ws, (const cplx*)M, nvb, nc, e_v, e_c, (const cplx*)C, n_eig, omega, n_w, accumulate, (cplx*)chi_s);
}

int rpa_chi0_static_occ(rpa_ctx* ctx, const void* M, int nvb, int nc, const double* e_v, const double* e_c, const double* f_v,
                        const double* f_c, int accumulate, void* chi0) {
  if (bad_ctx(ctx)) return rpa_fail(nullptr, RPA_ERR_INVALID, "null context");
  if (!M || !e_v || !e_c || !f_v || !f_c || !chi0 || nvb < 1 || nc < 1)
    return rpa_fail(ctx, RPA_ERR_INVALID, "rpa_chi0_static_occ: invalid argument");
  if ((long long)nvb * nc > 2147483647LL) return rpa_fail(ctx, RPA_ERR_INVALID, "rpa_chi0_static_occ: too many pairs");
  RPA_CUDA(ctx, cudaSetDevice(ctx->device));
  WsAlloc ws(ctx->ws, ctx->ws_bytes);
  return do_chi0_static(ctx, ws, (const cplx*)M, nvb, nc, e_v, e_c, accumulate, (cplx*)chi0, f_v, f_c);
}

int rpa_chi_subspace_freq_occ(rpa_ctx* ctx, const void* M, int nvb, int nc, const double* e_v, const double* e_c, const double* f_v,
                              const double* f_c, const void* C, int n_eig, const double* omega, int n_w, int accumulate,
                              void* chi_s) {
  if (bad_ctx(ctx)) return rpa_fail(nullptr, RPA_ERR_INVALID, "null context");
  if (!M || !e_v || !e_c || !f_v || !f_c || !omega || !chi_s || nvb < 1 || nc < 1 || n_w < 1)
    return rpa_fail(ctx, RPA_ERR_INVALID, "rpa_chi_subspace_freq_occ: invalid argument");
  if (n_eig < 1 || n_eig > ctx->n_g || (!C && n_eig != ctx->n_g))
    return rpa_fail(ctx, RPA_ERR_INVALID, "rpa_chi_subspace_freq_occ: n_eig = %d invalid (n_g = %d)", n_eig, ctx->n_g);
  if ((long long)nvb * nc > 2147483647LL) return rpa_fail(ctx, RPA_ERR_INVALID, "rpa_chi_subspace_freq_occ: too many pairs");
  RPA_CUDA(ctx, cudaSetDevice(ctx->device));
  WsAlloc ws(ctx->ws, ctx->ws_bytes);
  return do_chi_freq(ctx, ws, (const cplx*)M, nvb, nc, e_v, e_c, (const cplx*)C, n_eig, omega, n_w, accumulate, (cplx*)chi_s, f_v,
                     f_c);
}

int rpa_correlation_energy(rpa_ctx* ctx, const void* chi_s, int n_eig, const double* weight, int n_w, double* e_c,
                           double* per_freq) {
  if (bad_ctx(ctx)) return rpa_fail(nullptr, RPA_ERR_INVALID, "null context");
  if (!chi_s || !weight || !e_c || n_eig < 1 || n_w < 1) return rpa_fail(ctx, RPA_ERR_INVALID, "rpa_correlation_energy: invalid argument");
  RPA_CUDA(ctx, cudaSetDevice(ctx->device));
  WsAlloc ws(ctx->ws, ctx->ws_bytes);
  return energy_run(ctx, ws, (const cplx*)chi_s, n_eig, weight, n_w, e_c, per_freq);
}

size_t rpa_epsilon_inverse_workspace_bytes(const rpa_ctx* ctx, int n_eig, int n_w) {
  if (!ctx || n_eig < 1 || n_w < 1) return 0;
  return epsinv_workspace_bytes(ctx, n_eig, n_w) + 4096;
}

int rpa_epsilon_inverse(rpa_ctx* ctx, const void* chi_s, int n_eig, int n_w, void* eps_inv) {
  if (bad_ctx(ctx)) return rpa_fail(nullptr, RPA_ERR_INVALID, "null context");
  if (!chi_s || !eps_inv || n_eig < 1 || n_w < 1) return rpa_fail(ctx, RPA_ERR_INVALID, "rpa_epsilon_inverse: invalid argument");
  RPA_CUDA(ctx, cudaSetDevice(ctx->device));
  WsAlloc ws(ctx->ws, ctx->ws_bytes);
  return epsinv_run(ctx, ws, (const cplx*)chi_s, n_eig, n_w, (cplx*)eps_inv);
}

int rpa_fp64_peak(rpa_ctx* ctx, int kind, int iters, double* tflops) {
  if (bad_ctx(ctx)) return rpa_fail(nullptr, RPA_ERR_INVALID, "null context");
  if (!tflops || kind < 0 || kind > 2) return rpa_fail(ctx, RPA_ERR_INVALID, "rpa_fp64_peak: invalid argument");
  RPA_CUDA(ctx, cudaSetDevice(ctx->device));
  return fp64_peak_kernel(ctx, kind, iters, tflops);
}

// ------------------------------------------------------------------------------------------------
// whole path
static size_t energy_persistent_bytes(const rpa_ctx* ctx, int nv, int nc, int nvb, int n_eig, int n_w, bool keep_all) {
  const size_t n_g = ctx->n_g;
  size_t b = ws_round(n_g * n_g * sizeof(cplx)) + ws_round((size_t)n_eig * n_g * sizeof(cplx)) + ws_round(n_eig * sizeof(double)) +
             ws_round((size_t)n_w * n_eig * n_eig * sizeof(cplx));
  b += ws_round((size_t)(keep_all ? nv : nvb) * nc * n_g * sizeof(cplx));
  return b;
}

size_t rpa_energy_workspace_bytes(const rpa_ctx* ctx, int nv, int nc, int nvb, int n_eig, int n_w) {
  if (!ctx || nv < 1 || nc < 1 || n_eig < 1 || n_w < 1) return 0;
  if (nvb < 1 || nvb > nv) nvb = nv;
  const size_t inputs = ws_round((size_t)nv * ctx->n_pw * sizeof(cplx)) + ws_round((size_t)nc * ctx->n_pw * sizeof(cplx)) +
                        ws_round(nv * sizeof(double)) + ws_round(nc * sizeof(double)) + 2 * ws_round(n_w * sizeof(double));
  return inputs + energy_persistent_bytes(ctx, nv, nc, nvb, n_eig, n_w, false) + rpa_workspace_bytes(ctx, nvb, nc, n_eig, n_w);
}

// The two-pass loop, split at the points where a multi-GPU run exchanges data (rpa_b200.h "Pass-level calls").  The state
// lives in ctx->pass between rpa_pass_begin and rpa_pass_end; rpa_energy_device is these calls in sequence.
namespace {

void pass_tic(rpa_ctx* ctx, int stage) {
  rpa_ctx::PassState& ps = ctx->pass;
  if (!ps.timing) return;
  cudaEvent_t a; cudaEventCreate(&a); cudaEventRecord(a, ctx->stream); ps.evs.push_back(a); ps.ev_stage.push_back(stage);
}
void pass_toc(rpa_ctx* ctx) {
  rpa_ctx::PassState& ps = ctx->pass;
  if (!ps.timing) return;
  cudaEvent_t b; cudaEventCreate(&b); cudaEventRecord(b, ctx->stream); ps.evs.push_back(b); ps.ev_stage.push_back(-1);
}
void pass_reset(rpa_ctx* ctx) {
  rpa_ctx::PassState& ps = ctx->pass;
  for (auto e : ps.evs) cudaEventDestroy(e);
  ps = rpa_ctx::PassState();
  ctx->uc_cache = nullptr; ctx->uc_cache_filled = false; ctx->uc_cache_rows = 0;
}
int pass_need(rpa_ctx* ctx, const char* who, int stage) {
  if (bad_ctx(ctx)) return rpa_fail(nullptr, RPA_ERR_INVALID, "null context");
  if (!ctx->pass.active) return rpa_fail(ctx, RPA_ERR_INVALID, "%s: no pass sequence is open (call rpa_pass_begin first)", who);
  if (ctx->pass.stage != stage)
    return rpa_fail(ctx, RPA_ERR_INVALID, "%s: called out of order (the sequence is begin, pass1, basis, pass2, energy, end)", who);
  return RPA_OK;
}

}  // namespace

int rpa_pass_begin(rpa_ctx* ctx, const void* psi_v, int nv, const void* psi_c, int nc, const double* e_v, const double* e_c, int nvb,
                   int n_eig, const double* omega, int n_w, int keep_m, int timing) {
  if (bad_ctx(ctx)) return rpa_fail(nullptr, RPA_ERR_INVALID, "null context");
  if (!psi_v || !psi_c || !e_v || !e_c || !omega || nv < 1 || nc < 1 || n_w < 1) return rpa_fail(ctx, RPA_ERR_INVALID, "rpa_pass_begin: invalid argument");
  if (n_eig < 1 || n_eig > ctx->n_g) return rpa_fail(ctx, RPA_ERR_INVALID, "rpa_pass_begin: n_eig = %d not in 1..%d", n_eig, ctx->n_g);
  if (nvb < 1 || nvb > nv) nvb = nv;
  if ((long long)nvb * nc > 2147483647LL) return rpa_fail(ctx, RPA_ERR_INVALID, "rpa_pass_begin: too many pairs in one block");
  RPA_CUDA(ctx, cudaSetDevice(ctx->device));
  pass_reset(ctx);
  rpa_ctx::PassState& ps = ctx->pass;
  const int n_g = ctx->n_g;
  ps.psi_v = (const cplx*)psi_v; ps.psi_c = (const cplx*)psi_c; ps.e_v = e_v; ps.e_c = e_c; ps.omega = omega;
  ps.nv = nv; ps.nc = nc; ps.nvb = nvb; ps.n_eig = n_eig; ps.n_w = n_w; ps.timing = timing != 0;
  ps.nblocks = (nv + nvb - 1) / nvb;
  const size_t stage_need = rpa_workspace_bytes(ctx, nvb, nc, n_eig, n_w);
  ps.keep_all = keep_m && energy_persistent_bytes(ctx, nv, nc, nvb, n_eig, n_w, true) + stage_need <= ctx->ws_bytes;
  if (ps.nblocks == 1) ps.keep_all = true;
  WsAlloc ws(ctx->ws, ctx->ws_bytes);
  ps.chi0 = ws.get<cplx>((size_t)n_g * n_g);
  ps.C = ws.get<cplx>((size_t)n_eig * n_g);
  ps.lam = ws.get<double>(n_eig);
  ps.chi_s = ws.get<cplx>((size_t)n_w * n_eig * n_eig);
  ps.Mbuf = ws.get<cplx>((size_t)(ps.keep_all ? nv : nvb) * nc * n_g);
  if (!ws.ok || ws.off + stage_need > ctx->ws_bytes) {
    const size_t need = ws.off + stage_need;
    pass_reset(ctx);
    return rpa_fail(ctx, RPA_ERR_WORKSPACE, "rpa_energy: workspace too small (need %zu bytes, have %zu)", need, ctx->ws_bytes);
  }
  // several MTXEL calls on the same conduction bands: keep their real-space functions too if there is room
  const int n_mtxel = ps.keep_all ? ps.nblocks : 2 * ps.nblocks;
  const size_t per_band = (size_t)ctx->n_r * sizeof(cplx);
  if (keep_m && n_mtxel > 1 && ws.off + stage_need + 256 < ctx->ws_bytes) {
    const size_t room = ctx->ws_bytes - ws.off - stage_need - 256;
    const int rows = (int)std::min<size_t>((size_t)nc, room / per_band);   // as many bands as fit: the rest is recomputed
    if (rows >= 64 || rows == nc) {
      ctx->uc_cache = ws.get<cplx>((size_t)rows * ctx->n_r);
      ctx->uc_cache_src = ps.psi_c; ctx->uc_cache_nc = nc; ctx->uc_cache_rows = rows;
    }
  }
  ps.scratch = ctx->ws + ws.off;
  ps.scratch_bytes = ctx->ws_bytes - ws.off;
  ps.active = true; ps.stage = 0;
  return RPA_OK;
}

int rpa_pass1_chi0(rpa_ctx* ctx, void** chi0_out) {   // MTXEL + static CHI_SUM over all valence blocks (eq. 15)
  int rc = pass_need(ctx, "rpa_pass1_chi0", 0);
  if (rc) return rc;
  RPA_CUDA(ctx, cudaSetDevice(ctx->device));
  rpa_ctx::PassState& ps = ctx->pass;
  const int n_g = ctx->n_g, n_pw = ctx->n_pw;
  for (int b = 0; b < ps.nblocks && !rc; b++) {
    const int v0 = b * ps.nvb, nb = std::min(ps.nvb, ps.nv - v0);
    cplx* M = ps.keep_all ? ps.Mbuf + (size_t)v0 * ps.nc * n_g : ps.Mbuf;
    WsAlloc s1(ps.scratch, ps.scratch_bytes);
    pass_tic(ctx, 0); rc = mtxel_run(ctx, s1, ps.psi_v + (size_t)v0 * n_pw, nb, ps.psi_c, ps.nc, M); pass_toc(ctx);
    if (rc) break;
    WsAlloc s2(ps.scratch, ps.scratch_bytes);
    pass_tic(ctx, 1); rc = do_chi0_static(ctx, s2, M, nb, ps.nc, ps.e_v + v0, ps.e_c, b > 0, ps.chi0); pass_toc(ctx);
  }
  if (rc) return rc;
  ps.stage = 1;
  if (chi0_out) *chi0_out = ps.chi0;
  return RPA_OK;
}

int rpa_pass_basis(rpa_ctx* ctx, double tol, int compute, void** C_out, double** lambda_out) {
  int rc = pass_need(ctx, "rpa_pass_basis", 1);
  if (rc) return rc;
  RPA_CUDA(ctx, cudaSetDevice(ctx->device));
  rpa_ctx::PassState& ps = ctx->pass;
  if (compute) {
    WsAlloc s2(ps.scratch, ps.scratch_bytes);
    pass_tic(ctx, 2); rc = basis_run(ctx, s2, ps.chi0, ctx->n_g, ps.n_eig, tol, ps.C, ps.lam, nullptr); pass_toc(ctx);
    if (rc) return rc;
  }
  ps.stage = 2;
  if (C_out) *C_out = ps.C;
  if (lambda_out) *lambda_out = ps.lam;
  return RPA_OK;
}

int rpa_pass2_chis(rpa_ctx* ctx, void** chi_s_out) {   // (MTXEL again) + projected chi_s(i w) over all valence blocks
  int rc = pass_need(ctx, "rpa_pass2_chis", 2);
  if (rc) return rc;
  RPA_CUDA(ctx, cudaSetDevice(ctx->device));
  rpa_ctx::PassState& ps = ctx->pass;
  const int n_g = ctx->n_g, n_pw = ctx->n_pw;
  for (int b = 0; b < ps.nblocks && !rc; b++) {
    const int v0 = b * ps.nvb, nb = std::min(ps.nvb, ps.nv - v0);
    cplx* M = ps.keep_all ? ps.Mbuf + (size_t)v0 * ps.nc * n_g : ps.Mbuf;
    if (!ps.keep_all) {
      WsAlloc s1(ps.scratch, ps.scratch_bytes);
      pass_tic(ctx, 0); rc = mtxel_run(ctx, s1, ps.psi_v + (size_t)v0 * n_pw, nb, ps.psi_c, ps.nc, M); pass_toc(ctx);
      if (rc) break;
    }
    WsAlloc s3(ps.scratch, ps.scratch_bytes);
    pass_tic(ctx, 3); rc = do_chi_freq(ctx, s3, M, nb, ps.nc, ps.e_v + v0, ps.e_c, ps.C, ps.n_eig, ps.omega, ps.n_w, b > 0, ps.chi_s); pass_toc(ctx);
  }
  if (rc) return rc;
  ps.stage = 3;
  if (chi_s_out) *chi_s_out = ps.chi_s;
  return RPA_OK;
}

int rpa_pass_energy(rpa_ctx* ctx, const double* weight, double* e_c_out, double* lambda_out, double* per_freq, double* stage_ms) {
  int rc = pass_need(ctx, "rpa_pass_energy", 3);
  if (rc) return rc;
  if (!weight || !e_c_out) return rpa_fail(ctx, RPA_ERR_INVALID, "rpa_pass_energy: null argument");
  RPA_CUDA(ctx, cudaSetDevice(ctx->device));
  rpa_ctx::PassState& ps = ctx->pass;
  {
    WsAlloc s4(ps.scratch, ps.scratch_bytes);
    pass_tic(ctx, 4); rc = energy_run(ctx, s4, ps.chi_s, ps.n_eig, weight, ps.n_w, e_c_out, per_freq); pass_toc(ctx);
  }
  if (rc) return rc;
  if (lambda_out) RPA_CUDA(ctx, cudaMemcpyAsync(lambda_out, ps.lam, ps.n_eig * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
  RPA_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
  if (stage_ms) {
    for (int s = 0; s < 5; s++) stage_ms[s] = 0.0;
    for (size_t i = 0; i + 1 < ps.evs.size(); i += 2) {
      float ms = 0.f;
      cudaEventElapsedTime(&ms, ps.evs[i], ps.evs[i + 1]);
      stage_ms[ps.ev_stage[i]] += ms;
    }
  }
  ps.stage = 4;
  return RPA_OK;
}

int rpa_pass_end(rpa_ctx* ctx) {
  if (bad_ctx(ctx)) return rpa_fail(nullptr, RPA_ERR_INVALID, "null context");
  cudaSetDevice(ctx->device);
  pass_reset(ctx);
  return RPA_OK;
}

int rpa_energy_device(rpa_ctx* ctx, const void* psi_v, int nv, const void* psi_c, int nc, const double* e_v, const double* e_c,
                      int nvb, int n_eig, double tol, const double* omega, const double* weight, int n_w, int keep_m,
                      double* e_c_out, double* lambda_out, double* per_freq, double* stage_ms) {
  if (bad_ctx(ctx)) return rpa_fail(nullptr, RPA_ERR_INVALID, "null context");
  if (!psi_v || !psi_c || !e_v || !e_c || !omega || !weight || !e_c_out || nv < 1 || nc < 1 || n_w < 1)
    return rpa_fail(ctx, RPA_ERR_INVALID, "rpa_energy: invalid argument");
  int rc = rpa_pass_begin(ctx, psi_v, nv, psi_c, nc, e_v, e_c, nvb, n_eig, omega, n_w, keep_m, stage_ms != nullptr);
  if (!rc) rc = rpa_pass1_chi0(ctx, nullptr);
  if (!rc) rc = rpa_pass_basis(ctx, tol, 1, nullptr, nullptr);
  if (!rc) rc = rpa_pass2_chis(ctx, nullptr);
  if (!rc) rc = rpa_pass_energy(ctx, weight, e_c_out, lambda_out, per_freq, stage_ms);
  const std::string err = ctx->err;
  rpa_pass_end(ctx);
  if (rc) ctx->err = err;
  return rc;
}

int rpa_energy_host(rpa_ctx* ctx, const void* psi_v, int nv, const void* psi_c, int nc, const double* e_v, const double* e_c,
                    int nvb, int n_eig, double tol, const double* omega, const double* weight, int n_w, int keep_m,
                    double* e_c_out, double* lambda_out, double* per_freq, double* stage_ms) {
  if (bad_ctx(ctx)) return rpa_fail(nullptr, RPA_ERR_INVALID, "null context");
  if (!psi_v || !psi_c || !e_v || !e_c || !omega || !weight || !e_c_out || nv < 1 || nc < 1 || n_w < 1)
    return rpa_fail(ctx, RPA_ERR_INVALID, "rpa_energy_host: invalid argument");
  RPA_CUDA(ctx, cudaSetDevice(ctx->device));
  WsAlloc ws(ctx->ws, ctx->ws_bytes);
  cplx* d_pv = ws.get<cplx>((size_t)nv * ctx->n_pw);
  cplx* d_pc = ws.get<cplx>((size_t)nc * ctx->n_pw);
  double* d_ev = ws.get<double>(nv);
  double* d_ec = ws.get<double>(nc);
  double* d_om = ws.get<double>(n_w);
  double* d_wt = ws.get<double>(n_w);
  if (!ws.ok) return rpa_fail(ctx, RPA_ERR_WORKSPACE, "rpa_energy_host: workspace too small for the inputs (%zu bytes)", ws.off);
  RPA_CUDA(ctx, cudaMemcpyAsync(d_pv, psi_v, (size_t)nv * ctx->n_pw * sizeof(cplx), cudaMemcpyHostToDevice, ctx->stream));
  RPA_CUDA(ctx, cudaMemcpyAsync(d_pc, psi_c, (size_t)nc * ctx->n_pw * sizeof(cplx), cudaMemcpyHostToDevice, ctx->stream));
  RPA_CUDA(ctx, cudaMemcpyAsync(d_ev, e_v, nv * sizeof(double), cudaMemcpyHostToDevice, ctx->stream));
  RPA_CUDA(ctx, cudaMemcpyAsync(d_ec, e_c, nc * sizeof(double), cudaMemcpyHostToDevice, ctx->stream));
  RPA_CUDA(ctx, cudaMemcpyAsync(d_om, omega, n_w * sizeof(double), cudaMemcpyHostToDevice, ctx->stream));
  RPA_CUDA(ctx, cudaMemcpyAsync(d_wt, weight, n_w * sizeof(double), cudaMemcpyHostToDevice, ctx->stream));
  // run on the remainder of the workspace
  char* save_ws = ctx->ws; size_t save_bytes = ctx->ws_bytes;
  ctx->ws = save_ws + ws.off; ctx->ws_bytes = save_bytes - ws.off;
  int rc = rpa_energy_device(ctx, d_pv, nv, d_pc, nc, d_ev, d_ec, nvb, n_eig, tol, d_om, d_wt, n_w, keep_m, e_c_out, lambda_out,
                             per_freq, stage_ms);
  ctx->ws = save_ws; ctx->ws_bytes = save_bytes;
  return rc;
}

}  // extern "C"
