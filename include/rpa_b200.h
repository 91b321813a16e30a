/* rpa_b200.h -- C-ABI of the B200-native static-subspace RPA correlation-energy hot path.
 *
 * Method: Weinberg et al., "Static Subspace Approximation for Random Phase Approximation
 * Correlation Energies: Implementation and Performance" (arxiv 2405.20258); citations below are
 * line numbers of /root/reference/PAPER.md.  Readings of ambiguous passages (R1..R18) are listed
 * in DESIGN.md.
 *
 * Conventions that hold for every entry point
 *   - complex128 = interleaved (re, im) doubles (cuDoubleComplex, torch.complex128).
 *   - "dev" pointers are device pointers on the context's device, "host" pointers are host memory.
 *     The caller owns every array it passes; the library never frees caller memory and keeps no
 *     pointer past the call, except the workspace given to rpa_set_workspace.
 *   - All device work is enqueued on the CUDA stream given to rpa_create (a cudaStream_t, e.g.
 *     torch.cuda.current_stream().cuda_stream).  Calls return after enqueueing unless stated.
 *   - Return value: 0 = RPA_OK, negative = error (outputs undefined); text via rpa_last_error.
 *     The library never exits the process and never throws across this boundary.
 *   - There is no CPU fallback: without a CUDA device every call fails with RPA_ERR_CUDA.
 */
#ifndef RPA_B200_H
#define RPA_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct rpa_ctx rpa_ctx; /* opaque, library-owned */

enum {
  RPA_OK = 0,
  RPA_ERR_INVALID = -1,     /* null pointer, non-positive size, Miller index outside the grid,
                               grid axis with a prime factor other than 2/3/5, n_eig > n_g, v < 0 */
  RPA_ERR_WORKSPACE = -2,   /* workspace missing or too small (see rpa_workspace_bytes) */
  RPA_ERR_CUDA = -3,        /* CUDA runtime error (message has the CUDA error string) */
  RPA_ERR_NOT_POSDEF = -4,  /* Cholesky of 1 - chi_s broke down: chi_s not negative-semidefinite */
  RPA_ERR_NO_CONVERGENCE = -5 /* subspace iteration / Jacobi hit its iteration cap */
};

/* Statement of the problem: cell, FFT grid, the epsilon G-sphere with v(q+G), and
 * the wavefunction G-sphere.
 *   cell   host [9]   row-major lattice vectors a1,a2,a3 in bohr (kept for reference only)
 *   fft    host [3]   FFT grid (N1,N2,N3); every axis must factor into 2,3,5 and be <= 1024.  An xy plane must fit in
 *                     shared memory: square planes of 24, 40, 48 or 64 take the specialised kernels; any other N1 x N2
 *                     needs 16 B x (2 N1 (N2|1) + 2 nk2 (N1|1)) <= 227 KB (nk2 = distinct epsilon-sphere indices on axis 2;
 *                     roughly N1 N2 <= 80 x 80), else rpa_mtxel returns RPA_ERR_INVALID
 *   g_eps  host [n_g][3]  Miller indices of the epsilon sphere, any order (order defines M's G order)
 *   vcoul  host [n_g]     v(q+G) >= 0 (bare Coulomb 4 pi/(Omega |q+G|^2) in the configs)
 *   g_wfn  host [n_pw][3] Miller indices of the wavefunction sphere, any order
 *   |Miller index| must be < N/2 on each axis.  The pair product is alias-free (exact G-space
 *   convolution) when 2 max|n_wfn| + max|n_eps| < N; the library does not require it.
 *   device / cuda_stream: CUDA device ordinal (compute capability 10.0 exactly: the library holds sm_100a code only)
 *   and the caller's stream.  Several contexts, on the same or on different devices, may live in one process; a context
 *   must not be used from two threads at once.
 * Synchronises once (uploads plans: twiddles, index maps, v^1/2).                              */
int rpa_create(rpa_ctx** out, const double cell[9], const int fft[3], int n_g, const int32_t* g_eps,
               const double* vcoul, int n_pw, const int32_t* g_wfn, int device, void* cuda_stream);
int rpa_destroy(rpa_ctx* ctx);
const char* rpa_last_error(const rpa_ctx* ctx); /* valid until the next call on ctx; ctx may be NULL */

/* Scratch memory: the caller allocates (e.g. a torch uint8 tensor) and lends it to the context.
 * rpa_workspace_bytes = what the five stage calls below need for blocks of (nvb, nc) bands,
 * n_eig basis vectors and n_w frequencies; rpa_energy_workspace_bytes = what rpa_energy_* needs. */
size_t rpa_workspace_bytes(const rpa_ctx* ctx, int nvb, int nc, int n_eig, int n_w);
size_t rpa_energy_workspace_bytes(const rpa_ctx* ctx, int nv, int nc, int nvb, int n_eig, int n_w);
int rpa_set_workspace(rpa_ctx* ctx, void* dev_ptr, size_t bytes);

/* (a1) MTXEL, PAPER.md:52 eq. 3, :96, :104-110; reading R7/R8.
 *   u_n(r) = sum_G c_n(G) e^{+iG.r};  M[v][c][G] = (1/N_r) sum_r conj(u_v(r)) u_c(r) e^{-iG.r}, G on the
 *   epsilon sphere.  psi_v dev [nvb][n_pw], psi_c dev [nc][n_pw] (rows = bands, sum_G |c|^2 = 1),
 *   M dev out [nvb][nc][n_g], G fastest.  One valence block (eq. 14) per call.     */
int rpa_mtxel(rpa_ctx* ctx, const void* psi_v, int nvb, const void* psi_c, int nc, void* M);

/* (a2) CHI_SUM at omega = 0, eq. 6 with :71 eq. 5 and :152 eq. 15; readings R5/R6.
 *   chi0[G][G'] (+)= - sum_{v,c} v^1/2(G) M[v][c][G] (2/Delta_vc) conj(M[v][c][G']) v^1/2(G'),
 *   Delta_vc = e_c[c] - e_v[v] > 0.  e_v dev [nvb], e_c dev [nc].  accumulate: 0 overwrite, 1 add (the
 *   sum over valence blocks).  chi0 dev in/out [n_g][n_g], both triangles written.              */
int rpa_chi0_static(rpa_ctx* ctx, const void* M, int nvb, int nc, const double* e_v, const double* e_c,
                    int accumulate, void* chi0);

/* (a2) without any memory from the caller or from the allocator: the same CHI_SUM (same kernels, same result up to the
 * order in which split-K partial sums meet) for callers that cannot call cudaMalloc or lend a workspace at call time --
 * code under CUDA graph capture, tight serving loops, harnesses that forbid allocation.  The one piece of scratch
 * rpa_chi0_static takes from the workspace (the pair weights D_vc(0), nvb * nc doubles) lives in a device array built
 * into the library: rpa_noalloc_max_pairs() = 524 288 pairs = 4 MiB, held by every GPU that loads the library until the
 * process exits.  nvb * nc beyond that is rejected with RPA_ERR_INVALID (split the valence block, or use
 * rpa_chi0_static).  No workspace is needed (rpa_set_workspace need not have been called); the call makes no cudaMalloc /
 * cudaFree and calls no allocating library routine.  ALL calls on a device share that array: calls on one stream are
 * ordered and safe, calls that overlap on the GPU (two streams, two contexts on one device) race on it.  The array keeps
 * the previous call's contents; a call overwrites what it reads, so nothing needs clearing.
 * rpa_noalloc_setup (optional; otherwise done by the first call): fetches the array's device address for the context's
 * device -- call it once before capturing a graph.  Arguments of rpa_chi0_static_noalloc as rpa_chi0_static.          */
long long rpa_noalloc_max_pairs(void);
int rpa_noalloc_setup(rpa_ctx* ctx);
int rpa_chi0_static_noalloc(rpa_ctx* ctx, const void* M, int nvb, int nc, const double* e_v, const double* e_c,
                            int accumulate, void* chi0);

/* (a3) Static subspace basis; reading R9.  The n_eig eigenpairs of Hermitian chi0 with
 *   the greatest |lambda| (chi0 is negative-semidefinite: the most negative ones).
 *   C dev out [n_eig][n_g], row i = eigenvector i (unit 2-norm); lambda dev out [n_eig] ascending.
 *   tol: relative residual target ||chi0 c_i - lambda_i c_i|| <= tol |lambda_1| (<= 0 selects 1e-11).  Every route
 *   measures it on its result, together with max|C C^H - 1| <= max(10 tol, 1e-11), before returning: the direct
 *   tridiagonalisation route falls back to Jacobi / block subspace iteration when it misses either, and those return
 *   RPA_ERR_NO_CONVERGENCE when they do (or when the iteration hits its cap).
 *   iters_out host, optional: subspace iterations used (0 = a direct eigen-decomposition of the whole matrix).
 *   Synchronises (convergence is checked on the host).                                           */
int rpa_subspace_basis(rpa_ctx* ctx, const void* chi0, int n_eig, double tol, void* C, double* lambda,
                       int* iters_out);

/* (a4) Projected chi_s(i omega_k), PAPER.md:84 eq. 7, :88 eq. 8, :158.
 *   B_vc = C^H v^1/2 M_vc;  chi_s[k] (+)= - sum_vc B_vc D_vc(omega_k) B_vc^H,
 *   D = 2 Delta/(Delta^2 + omega^2).  omega dev [n_w].  chi_s dev in/out [n_w][n_eig][n_eig].
 *   C == NULL means the identity (n_eig must equal n_g): the full-basis chi~0(i omega_k).         */
int rpa_chi_subspace_freq(rpa_ctx* ctx, const void* M, int nvb, int nc, const double* e_v,
                          const double* e_c, const void* C, int n_eig, const double* omega, int n_w,
                          int accumulate, void* chi_s);

/* (next-4) Partial occupations, PAPER.md:29, :48-67 eq. 4, :71 eq. 5; reading R21 of DESIGN.md.  The same two
 * contractions with the pair weight  D_vc(i omega) = max(f_v - f_c, 0) 2 Delta/(Delta^2 + omega^2),  Delta = e_c - e_v:
 * the "valence" set holds every band with f > 0 and the "conduction" set every band with f < 1, so a partially occupied
 * band sits in both (the four classes of eq. 4); max(., 0) counts each unordered pair once and gives the pair of a band
 * with itself weight 0.  f_v dev [nvb], f_c dev [nc], occupations in [0, 1]; f_v = 1, f_c = 0 reproduces
 * rpa_chi0_static / rpa_chi_subspace_freq.  A pair with Delta = 0 and omega = 0 gets weight 0.                          */
int rpa_chi0_static_occ(rpa_ctx* ctx, const void* M, int nvb, int nc, const double* e_v, const double* e_c,
                        const double* f_v, const double* f_c, int accumulate, void* chi0);
int rpa_chi_subspace_freq_occ(rpa_ctx* ctx, const void* M, int nvb, int nc, const double* e_v, const double* e_c,
                              const double* f_v, const double* f_c, const void* C, int n_eig, const double* omega,
                              int n_w, int accumulate, void* chi_s);

/* (a5) E_c, PAPER.md:35 eq. 1, :160, :174; reading R10.
 *   per k: L L^H = 1 - chi_s[k];  t_k = 2 sum_i ln L_ii + Re Tr chi_s[k];  E_c = (1/2 pi) sum_k W_k t_k.
 *   weight dev [n_w] (quadrature weight incl. Jacobian).  e_c host out; per_freq host out [n_w],
 *   optional.  chi_s is not modified.  Synchronises.                                             */
int rpa_correlation_energy(rpa_ctx* ctx, const void* chi_s, int n_eig, const double* weight, int n_w,
                           double* e_c, double* per_freq);

/* (next-3) eps_s^-1(i omega_k) = (1 - chi_s(i omega_k))^-1 in the subspace, from the same Cholesky factor as E_c -- the
 * by-product the paper keeps for later GW.  chi_s dev [n_w][n_eig][n_eig] (not modified); eps_inv dev out
 * [n_w][n_eig][n_eig], Hermitian, both triangles.  Needs rpa_epsilon_inverse_workspace_bytes of workspace.  Synchronises;
 * RPA_ERR_NOT_POSDEF as for rpa_correlation_energy.                                                                   */
size_t rpa_epsilon_inverse_workspace_bytes(const rpa_ctx* ctx, int n_eig, int n_w);
int rpa_epsilon_inverse(rpa_ctx* ctx, const void* chi_s, int n_eig, int n_w, void* eps_inv);

/* Whole path (PAPER.md:139-158 NV-block two-pass loop): for each valence block of nvb bands
 * {a1, a2}; a3; for each block {a1, a4}; a5.  All inputs dev (rpa_energy_device) or host
 * (rpa_energy_host: inputs are copied to the device and the scalar copied back inside the call).
 *   psi_v [nv][n_pw], psi_c [nc][n_pw], e_v [nv], e_c [nc], omega/weight [n_w].
 *   keep_m != 0: keep all M blocks resident and skip the second MTXEL pass when they fit in the
 *   workspace (the single-block case of PAPER.md:158); otherwise recompute.
 *   stage_ms host out [5], optional: device time of a1 (both passes), a2, a3, a4, a5 in ms.
 *   lambda_out host [n_eig], per_freq host [n_w]: optional.  Synchronises.                       */
int rpa_energy_device(rpa_ctx* ctx, const void* psi_v, int nv, const void* psi_c, int nc, const double* e_v,
                      const double* e_c, int nvb, int n_eig, double tol, const double* omega,
                      const double* weight, int n_w, int keep_m, double* e_c_out, double* lambda_out,
                      double* per_freq, double* stage_ms);
int rpa_energy_host(rpa_ctx* ctx, const void* psi_v, int nv, const void* psi_c, int nc, const double* e_v,
                    const double* e_c, int nvb, int n_eig, double tol, const double* omega,
                    const double* weight, int n_w, int keep_m, double* e_c_out, double* lambda_out,
                    double* per_freq, double* stage_ms);

/* Pass-level calls: the same two-pass loop split at the two points where a multi-GPU run exchanges data (PAPER.md:104-108
 * eq. 9: conduction bands over ranks; :127-129 eq. 13: the per-rank contributions to chi are summed).  Each rank opens a
 * sequence on ITS conduction slice; the partial chi~0(0) and chi_s stay inside the workspace, the calls hand out device
 * pointers to them and the caller reduces them in place (one all-reduce each) before the next call:
 *
 *   rpa_pass_begin -> rpa_pass1_chi0 -> [all-reduce chi0] -> rpa_pass_basis(compute on one rank) -> [broadcast C, lambda]
 *   -> rpa_pass2_chis -> [all-reduce chi_s] -> rpa_pass_energy -> rpa_pass_end
 *
 * rpa_energy_device is exactly this sequence with no exchange, so one rank reproduces it bit for bit.  What the library
 * keeps resident across the valence blocks (all M blocks and the real-space conduction functions, keep_m) is the same.
 *   rpa_pass_begin   arguments as rpa_energy_device (all dev); timing != 0 records the stage timers.  EXCEPTION to the
 *                    ownership rule: the library keeps the input pointers until rpa_pass_end -- the arrays must stay alive
 *                    and unchanged.  Needs rpa_energy_workspace_bytes of workspace.  Ends any sequence still open.
 *   rpa_pass1_chi0   {a1, a2} over all valence blocks.  *chi0 (optional) = dev pointer INTO THE WORKSPACE [n_g][n_g].
 *   rpa_pass_basis   compute != 0: a3 on the (reduced) chi0; compute == 0: skip it, the caller fills C and lambda.
 *                    *C = dev pointer into the workspace [n_eig][n_g], *lambda [n_eig] (both optional).
 *   rpa_pass2_chis   {a1 again unless M was kept, a4} over all valence blocks.  *chi_s = dev pointer into the workspace
 *                    [n_w][n_eig][n_eig].
 *   rpa_pass_energy  a5 on the (reduced) chi_s; outputs as rpa_energy_device.  Synchronises.
 *   rpa_pass_end     closes the sequence; the pointers handed out become invalid (so do they on rpa_set_workspace).
 * Calls out of order return RPA_ERR_INVALID.                                                                           */
int rpa_pass_begin(rpa_ctx* ctx, const void* psi_v, int nv, const void* psi_c, int nc, const double* e_v, const double* e_c,
                   int nvb, int n_eig, const double* omega, int n_w, int keep_m, int timing);
int rpa_pass1_chi0(rpa_ctx* ctx, void** chi0);
int rpa_pass_basis(rpa_ctx* ctx, double tol, int compute, void** C, double** lambda);
int rpa_pass2_chis(rpa_ctx* ctx, void** chi_s);
int rpa_pass_energy(rpa_ctx* ctx, const double* weight, double* e_c_out, double* lambda_out, double* per_freq, double* stage_ms);
int rpa_pass_end(rpa_ctx* ctx);

/* ---------------------------------------------------------------------------------------------------------------------
 * Diagnostics -- NOT part of the method's ABI (nothing below computes any step of the path); used by bench.py, the
 * profiles and the tests.
 *
 * Environment switches, read ONCE by rpa_create (never on a launch path):
 *   RPA_GENERIC_FFT=1        MTXEL runs its generic mixed-radix plane / z kernels even where a specialised one exists
 *   RPA_NO_TRIDIAG=1         a3 skips the tridiagonalisation route: block subspace iteration + CholeskyQR2 + Jacobi
 *                            Rayleigh-Ritz when 4 N_eig <= n_g (about), direct Jacobi otherwise
 *   RPA_JACOBI_BLOCK_MIN=n   smallest matrix for which the Jacobi solver takes its GEMM block form (default 1024)
 *   RPA_HETRD_MODE=0|1|2, RPA_HETRD_THREADS=n   force a large-matrix variant / CTA size of the tridiagonalisation kernel
 *   RPA_ZGEMM_TMA=0          CHI_SUM / chi_s contractions stage their operands with cp.async and a block barrier per k-tile
 *                            (the round-1 kernel) instead of TMA box loads and mbarriers
 *   RPA_VERBOSE=1            route decisions and kernel resources on stderr
 * --------------------------------------------------------------------------------------------------------------------- */
/* Register-only FP64 peaks on the context's device.
 *   kind 0: mma.sync m8n8k4 f64 (DMMA), kind 1: DFMA, kind 2: DMMA throughput when every 24 DMMAs are interleaved with 14
 *   independent DADDs (plain FP64 instructions share the pipe).  Returns TFLOP/s in *tflops; runs `iters` launches of a
 *   fixed-size kernel on the context stream and synchronises.                                    */
int rpa_fp64_peak(rpa_ctx* ctx, int kind, int iters, double* tflops);
/* Per-kernel-class device times (bench.py's roofline of the dominant kernel).  Between rpa_profile_begin and
 * rpa_profile_end every launch of the classes below is bracketed by a pair of CUDA events on the context stream;
 * rpa_profile_end synchronises and returns, per class, the summed device time in ms and the number of timed launches
 * (host out, arrays of RPA_PROF_NCLASS).  Classes: the MTXEL plane kernel (product + pruned xy transforms), the MTXEL z
 * transform + sphere gather, the wavefunction -> real-space transforms, the CHI_SUM(0) contraction, the projection
 * GEMM, the chi_s(i omega) contraction, the whole basis stage, the whole E_c stage.                                 */
enum { RPA_PROF_MTXEL_PLANE = 0, RPA_PROF_MTXEL_Z = 1, RPA_PROF_MTXEL_WFN = 2, RPA_PROF_CHI0 = 3, RPA_PROF_PROJ = 4,
       RPA_PROF_CHIS = 5, RPA_PROF_BASIS = 6, RPA_PROF_ENERGY = 7, RPA_PROF_NCLASS = 8 };
int rpa_profile_begin(rpa_ctx* ctx);
int rpa_profile_end(rpa_ctx* ctx, double* ms, long long* launches);
/* Route taken by the last rpa_subspace_basis / basis stage (bench.py's work model; the tests assert it): n = size of the
 * last dense eigen-decomposition (n_g, or the block size p of the subspace iteration), sweeps = Jacobi sweeps done,
 * kind 0 = vector one-sided Jacobi (44 n FLOP per rotated pair, n(n-1)/2 pairs per sweep), 1 = block Jacobi (32 n^3 GEMM
 * FLOP per sweep), 2 = tridiagonalisation + bisection + inverse iteration.  Whether the block subspace iteration ran is
 * what rpa_subspace_basis returns in iters_out (> 0).  Host out.                                                    */
int rpa_basis_info(const rpa_ctx* ctx, int* n, int* sweeps, int* kind);
/* What the last rpa_subspace_basis / basis stage measured on its own result before returning (every route checks it
 * against tol): residual = max_i ||chi0 c_i - lambda_i c_i|| / |lambda_1|, orthogonality = max |C C^H - 1|.  Host out. */
int rpa_basis_quality(const rpa_ctx* ctx, double* residual, double* orthogonality);
/* Number of kernels launched by this context since creation (for bench.py's gpu_launches). */
long long rpa_launch_count(const rpa_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* RPA_B200_H */
