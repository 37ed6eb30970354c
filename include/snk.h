/* =====================================================================================
 * snk.h -- C ABI of the B200-native seminumerical exact-exchange (sn-K) build.
 *
 * Method: arXiv 2303.14280 (PAPER.md = /root/reference/PAPER.md), Sec. II D-E + App. A:
 *
 *   Phi[g,mu]  = phi_mu(r_g)                                        Eq. 31
 *   F[g,lam]   = sum_{sigma in B_j} P[lam,sigma] Phi[g,sigma]       Eq. 35/48
 *   A[g,nu,lam]= int phi_nu(r) phi_lam(r) / |r - r_g| d^3r          Eq. 37, on the fly, never stored
 *   G[g,nu]    = sum_{(nu,lam) in V_j} A[g,nu,lam] F[g,lam]         Eq. 38/48
 *   Kt[mu,nu]  = sum_g Phi[g,mu] w_g G[g,nu],  mu in B_j            Eq. 39
 *   K          = (Kt + Kt^T)/2                                      Eq. 40
 *
 * with grid points batched spatially (Q_j), basis screening B_j (Eq. 41,
 * PAPER.md:243) and sn-LinK shell-pair screening V_j (Eqs. 43-47).
 * The readings of everything the paper leaves open are R1-R20 in DESIGN.md.
 *
 * All reals are IEEE double, all coordinates bohr.  Every pointer is annotated HOST or
 * DEVICE.  The caller owns every pointer it passes; the library copies what it needs
 * during the call (host arrays synchronously, device arrays stream-ordered) and never
 * frees caller memory.  No exception or abort crosses this boundary: every call returns
 * SNK_OK (0) or a negative snk_status, and snk_last_error() gives the text.
 * There is no CPU fallback anywhere behind this interface.
 * ===================================================================================== */
#ifndef SNK_H_
#define SNK_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct snk_ctx snk_ctx; /* opaque; owns all internal device/host memory */

typedef enum snk_status {
  SNK_OK = 0,
  SNK_EINVAL = -1, /* bad argument: l > 3, nprim < 1, exponent <= 0, negative weight, NULL, unknown option */
  SNK_ENOMEM = -2, /* host or device allocation failed */
  SNK_ECUDA = -3,  /* a CUDA call failed; snk_last_error() holds cudaGetErrorString */
  SNK_ESTATE = -4  /* call order: snk_build_K before snk_set_grid, ... */
} snk_status;

/* Counters and per-stage device times of the LAST snk_set_grid / snk_build_K (PAPER.md:437 splits
 * sn-K into "Screen" and "LocalWork" the same way).  Times are CUDA-event milliseconds. */
typedef struct snk_stats {
  int64_t npts;             /* grid points handed to snk_set_grid                                   */
  int64_t npts_kept;        /* points in batches with non-empty B_j                                  */
  int64_t nbatch;           /* batches Q_j with non-empty B_j                                        */
  int64_t sum_B;            /* sum_j |B_j|  (shells)                                                 */
  int64_t sum_B_fn;         /* sum_j nbf(B_j) (functions)                                            */
  int64_t npair_sig;        /* shell pairs that survive in at least one batch's upper bound          */
  int64_t sum_V;            /* sum_j |V_j|  (unordered shell pairs)                                  */
  int64_t nprimpair;        /* primitive pairs kept for the significant shell pairs (R14)            */
  int64_t nsuper;           /* super-batches the build was split into (Alg. 1 line 8)  */
  double n_pairpoints;      /* sum_j |Q_j| |V_j|                                                     */
  double n_int_contracted;  /* sum_j |Q_j| sum_{(a,b) in V_j} ncart(l_a) ncart(l_b)  -- "integrals"  */
  double n_int_primitive;   /* same, times the number of primitive pairs actually evaluated          */
  double flops_integral;    /* FP64 flop model of the integral-contraction kernels */
  double flops_gemm;        /* 2*M*N*K of the F and Kt contractions as executed (lists padded to tiles) */
  double ms_set_grid;       /* a0 + a1 + maxima                                                      */
  double ms_screen;         /* a3: |P|, Ftilde GEMM, V_j masks, pair tables                          */
  double ms_colloc;         /* a2                                                                    */
  double ms_F;              /* a4                                                                    */
  double ms_G;              /* a5 (all classes)                                                      */
  double ms_Kt;             /* a6                                                                    */
  double ms_sym;            /* a7                                                                    */
  double ms_build;          /* whole snk_build_K on the stream                                       */
  double ms_G_class[10];    /* a5 per (l_a,l_b) class, order (0,0),(1,0),(1,1),(2,0)...(3,3)         */
  double n_int_class[10];   /* contracted integrals per class                                        */
  double flops_class[10];   /* flop model per class                                                  */
  int64_t n_launches;       /* kernels of this library launched by the last snk_build_K              */
  double flops_gemm_alg;    /* 2 |Q_j| nbf(B_j) nbf summed over batches, for a4 and a6 (Eq. 48 operands) */
} snk_stats;

/* ---- snk_create: the basis set "B" of Alg. 1 -------------------------------------
 * Contracted atom-centred Cartesian Gaussian shells, Eq. 13 + contraction:
 *   phi(r) = x_A^i y_A^j z_A^k * sum_k prim_coef[k] * exp(-prim_exp[k] * |r-A|^2)
 * prim_coef is the FULL coefficient; the library applies no hidden normalisation (R5).
 * Function order: shells in input order; inside a shell the Cartesian components (i,j,k), i from l
 * down to 0, then j from l-i down to 0  (l=2: xx, xy, xz, yy, yz, zz).
 *   atom_xyz   HOST [natoms*3]     shell_atom HOST [nshells] index into atoms
 *   shell_l    HOST [nshells] 0..3 shell_nprim HOST [nshells] >= 1
 *   prim_exp   HOST [sum nprim] > 0      prim_coef HOST [sum nprim]
 * Errors: SNK_EINVAL (see enum), SNK_ENOMEM, SNK_ECUDA.  *out is NULL on failure. */
int snk_create(snk_ctx** out, int32_t natoms, const double* atom_xyz, int32_t nshells, const int32_t* shell_atom,
               const int32_t* shell_l, const int32_t* shell_nprim, const double* prim_exp, const double* prim_coef);

/* ---- options ("eps_B = eps_E = eps_K", "maximum grid partition size") ---------------
 *   "eps"          one threshold for Eqs. 41, 43 (R9); 0 => no screening at all.   default 0
 *   "batch_cell"   h0, root cell edge of the lattice-anchored octree in bohr (R13). default 6.0
 *   "batch_max"    N_max, largest batch (R13), 32..4096.                           default 2048
 *   "workspace_gb" device-memory budget for the Phi/F/G super-batch (Alg. 1 l.8).  default 24
 *   "tile_split"   CTAs that share one 128-point tile in the integral kernel (each takes a contiguous share of the tile's
 *                  unit list); 0 = the library's choice.                                     default 0
 *   "atomics"      1: G and the split-K partial tiles of Kt are accumulated with fp64 RED atomics (default, the only mode);
 *                  the order of those additions is not fixed, so K is reproducible from run to run only up to fp64
 *                  summation order (observed: a few 1e-15 relative), never bit for bit.  Reserved for a deterministic mode.
 * Must be set before snk_set_grid.  Unknown key or out-of-range value: SNK_EINVAL. */
int snk_set_option(snk_ctx* ctx, const char* key, double value);

/* ---- snk_set_grid: the quadrature Q = {(w_i, r_i)} --------------------------------
 * Per-geometry work: batching a0, basis lists B_j a1, density-independent maxima of Eq. 47.
 *   points  DEVICE [npts*3] row-major      weights DEVICE [npts], all >= 0 (checked on device)
 *   stream  cudaStream_t (may be NULL = default stream)
 * Synchronises the stream (list sizes are read back).  npts == 0 is allowed (K = 0). */
int snk_set_grid(snk_ctx* ctx, int64_t npts, const double* points, const double* weights, void* stream);

/* ---- snk_build_K: "Input: density matrix D ... Output: K" ---------------------
 *   P  DEVICE [nbf*nbf] row-major, symmetric (assumed, R7)    K  DEVICE [nbf*nbf], overwritten
 * Ordered on `stream`; K is valid when the stream reaches the end of the call's work.  The call reads back
 * a handful of list sizes (one small synchronisation) but never moves matrix data through the host.
 * Environment: SNK_TRACE (any value) makes the call synchronise after every stage and report it on stderr
 * (debugging aid; it perturbs the timings). */
int snk_build_K(snk_ctx* ctx, const double* P, double* K, void* stream);

/* Same build with HOST buffers: H2D copy of P, build, D2H copy of K, stream synchronised on return.
 * This is the end-to-end call bench.py times as "e2e". */
int snk_build_K_host(snk_ctx* ctx, const double* P_host, double* K_host, void* stream);

/* ---- work estimates for the batch-to-rank partition of Alg. 2 (cost model W_j, Eq. 49 at PAPER.md:330) --
 * snk_screen runs only the density-dependent screening of snk_build_K (row a3, Eqs. 43-47: V_j for this P on the current
 * grid), ordered on `stream`.  snk_batch_costs then returns, for every batch j in batch order,
 *   cost[j] = |Q_j| * (primitive pairs of the shell pairs kept in V_j)     -- primitive pair-points, what a5's time follows.
 *   P DEVICE [nbf*nbf]     cost HOST [nbatch] (nbatch from snk_get_stats / snk_export_lists); synchronises the stream.
 * Errors: SNK_ESTATE before snk_set_grid / before a screening or build. */
int snk_screen(snk_ctx* ctx, const double* P, void* stream);
int snk_batch_costs(snk_ctx* ctx, double* cost);

/* sum over shells of (l+1)(l+2)/2 */
int snk_nbf(const snk_ctx* ctx);

/* Synchronises the last stream used and fills *out. */
int snk_get_stats(snk_ctx* ctx, snk_stats* out);

/* ---- audit (off the timed path): two-call pattern, NULL buffers => sizes only ---------------------
 *   sizes HOST [4]: nbatch, npts_kept, sum_B, sum_V
 *   batch_off HOST [nbatch+1]; perm HOST [npts_kept] input index of every kept point, batch by batch;
 *   B_off HOST [nbatch+1], B_ids HOST [sum_B] (ascending shells);
 *   V_off HOST [nbatch+1], V_pairs HOST [2*sum_V] unordered pairs as (min,max), sorted.  V_* need a prior build. */
int snk_export_lists(snk_ctx* ctx, int64_t* sizes, int64_t* batch_off, int64_t* perm, int64_t* B_off, int32_t* B_ids,
                     int64_t* V_off, int32_t* V_pairs);

/* ---- kernel-level test hooks (same device code the build uses) -----------------------------------
 * F_0..F_mmax at n arguments: x DEVICE [n] -> out DEVICE [n*(mmax+1)], mmax <= 6 (Eq. 22). */
int snk_debug_boys(int32_t mmax, int64_t n, const double* x, double* out, void* stream);
/* A block of shell pair (a,b) at n points through the Obara-Saika kernel (App. A): pts DEVICE [n*3] ->
 * out DEVICE [n * ncart(l_a) * ncart(l_b)], row-major [g][ia][ib]. */
int snk_debug_A_pair(snk_ctx* ctx, int32_t a, int32_t b, int64_t n, const double* pts, double* out, void* stream);

/* ---- the same A block without any allocation --------------------------------------------------------
 * snk_debug_A_pair cudaMallocs and frees a scratch buffer (the primitive-pair records of the shell pair) on every call and
 * synchronises the stream.  Callers that cannot call cudaMalloc -- code under CUDA graph capture, tight serving loops,
 * harnesses that forbid it -- use this variant: same kernel, same arguments, same result layout (pts DEVICE [n*3] ->
 * out DEVICE [n * ncart(l_a) * ncart(l_b)], row-major [g][ia][ib]), but the scratch is a fixed array inside the library
 * (1024 primitive pairs x 80 bytes = 80 KB of device memory per GPU that loads the library, held until exit) that a small
 * kernel fills on the device.  The call makes no cudaMalloc / cudaFree / allocating library call, copies nothing through
 * the host and does not synchronise: it is ordered on `stream`, out is valid when the stream reaches the end of its work.
 * LIMIT: nprim(a) * nprim(b) <= 1024, else SNK_EINVAL with the reason in snk_last_error.
 * SHARED STATE: every call on a GPU uses the same scratch array, which keeps the last call's contents (each call overwrites
 * the entries it reads; nothing needs clearing).  Calls that may overlap on the GPU (different streams, or concurrent
 * graph branches) race on it: keep them on one stream or order them with events.
 * Errors: SNK_EINVAL (bad shell index, NULL pointer, limit), SNK_ESTATE (wrong current device), SNK_ECUDA. */
int snk_A_pair_noalloc(snk_ctx* ctx, int32_t a, int32_t b, int64_t n, const double* pts, double* out, void* stream);

/* ---- measured FP64 roofs of this GPU: register-resident DFMA loop and DMMA.884 loop,
 * TFLOP/s each (2 flops per FMA), best of `reps`. */
int snk_measure_fp64_peak(double* dfma_tflops, double* dmma_tflops, int32_t reps);

const char* snk_last_error(const snk_ctx* ctx); /* ctx may be NULL: last error of a failed snk_create */
void snk_destroy(snk_ctx* ctx);
const char* snk_version(void);

#ifdef __cplusplus
}
#endif
#endif /* SNK_H_ */
