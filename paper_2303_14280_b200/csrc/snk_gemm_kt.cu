// snk_gemm_kt.cu -- a6:  Kt[mu,nu] += sum_g Phi[mu,g] w_g G[nu,g]        Eq. 39, fp64 DMMA (m8n8k4)
//
// Both operands are rows of the [nbf x ld] slabs of one super-batch, i.e. contiguous along the contraction index g.
//   * CTA tile 32 (Phi rows) x 128 (G rows), k-tile 16 slots, 8 warps (1 x 8), warp tile 32 x 16 = 4 x 2 fragments,
//     accumulators in registers.  (64 x 256 with 2 x 4 warps has the better operand reuse but skips fewer blocks:
//     490 vs 427 ms on cfg 3.)
//   * Operand tiles travel global -> shared with 16-byte cp.async, double buffered (one __syncthreads per k-tile), four
//     CTAs per SM (51 KB of shared memory each; 32 x 256 tiles with two CTAs are 8 % slower, a 4-stage ring with one
//     CTA 25 %); the
//     shared rows keep the k-contiguous order with a row stride of 20 doubles, which makes the fragment loads
//     (thread (g,t) reads [row g][k t]) hit 16 distinct 8-byte banks per half warp.
//   * w_g is staged with the tile and folded into the Phi fragments.
//   * Basis screening (Eq. 41): Phi rows of shells outside B_j are identically zero over batch j.  A bit per
//     (32-function row tile, 16-slot k-tile) says whether any function of the row tile is in B_j of the batch that owns
//     the k-tile; the kernel walks only the set bits (batches start on 32-slot boundaries, so a k-tile never straddles
//     two batches).  Skipped tiles contribute exact zeros, so the result is unchanged.
//   * split-K into short k-chunks (2048 slots) gives thousands of CTAs whatever nbf is; partial tiles are RED-added into Kt.
#include <algorithm>

#include "snk_internal.h"
#include "snk_kernels.h"

namespace snk {
namespace {
constexpr int TM = 128, TK = 16, LDK = 20, NTH = 256, STAGES = 4;

__device__ __forceinline__ void dmma884(double& d0, double& d1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n" : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}
__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src, uint32_t src_bytes) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(dst), "l"(src), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory"); }

// walks the set bits of act[w0 .. w1), restricted to k-tiles [kt0, kt1)
struct BitWalk {
  const uint32_t* __restrict__ words;
  int64_t w, w1, kt0, kt1;
  uint32_t bits, nbits;                  // current word, prefetched next word
  __device__ __forceinline__ uint32_t load(int64_t i) const {
    if (i >= w1) return 0u;
    uint32_t v = __ldg(words + i);
    const int64_t base = i << 5;
    if (base < kt0) v &= (kt0 - base >= 32) ? 0u : (0xffffffffu << (int)(kt0 - base));
    if (base + 32 > kt1) v &= (kt1 <= base) ? 0u : (0xffffffffu >> (int)(base + 32 - kt1));
    return v;
  }
  __device__ __forceinline__ void init(const uint32_t* p, int64_t w0_, int64_t w1_, int64_t a, int64_t b) {
    words = p; w = w0_; w1 = w1_; kt0 = a; kt1 = b;
    bits = load(w); nbits = load(w + 1);
  }
  __device__ __forceinline__ int64_t next() {       // -1 when exhausted
    while (bits == 0u) {
      if (w + 1 >= w1) return -1;
      ++w; bits = nbits; nbits = load(w + 1);
    }
    const int b = __ffs(bits) - 1;
    bits &= bits - 1;
    return (w << 5) + b;
  }
};

// CTA tile TA (Phi rows) x TB (G rows): the Phi side is kept narrow because that is where the zero blocks are
#ifndef SNK_KT_TA
#define SNK_KT_TA 32
#endif
#ifndef SNK_KT_TB
#define SNK_KT_TB 128
#endif
constexpr int TA = SNK_KT_TA, TB = SNK_KT_TB, KT_STAGE_DOUBLES = (TA + TB) * LDK + TK;
#ifndef SNK_KT_STAGES
#define SNK_KT_STAGES 2
#endif
#ifndef SNK_KT_MINB
#define SNK_KT_MINB 4
#endif
constexpr int KT_STAGES = SNK_KT_STAGES;
constexpr int KT_WM = TA / 32, KT_WN = 8 / KT_WM, KT_NJ = TB / KT_WN / 8;   // warps along Phi rows / G rows, fragments per warp along G
__global__ void __launch_bounds__(NTH, SNK_KT_MINB) k_gemm_kt(int64_t nbf, int64_t slot0, int64_t nslots, const double* __restrict__ Phi,
                                                 const double* __restrict__ G, int64_t ld, const double* __restrict__ wts,
                                                 double* __restrict__ Kt, const uint32_t* __restrict__ act, int64_t actw, int64_t wchunk) {
  extern __shared__ __align__(16) double smem_kt[];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int wm = warp / KT_WN, wn = warp % KT_WN;          // KT_WM x KT_WN warps, warp tile 32 x (8 KT_NJ)
  const int g = lane >> 2, t = lane & 3;
  const int64_t m0 = (int64_t)blockIdx.y * TA, n0 = (int64_t)blockIdx.x * TB;
  const int64_t kt0 = slot0 / TK, kt1 = (slot0 + nslots) / TK;
  const int64_t wlo = (kt0 >> 5) + (int64_t)blockIdx.z * wchunk, whi = min(((kt1 + 31) >> 5), wlo + wchunk);
  if (wlo >= whi) return;
  BitWalk walk;
  walk.init(act + (int64_t)blockIdx.y * actw, wlo, whi, kt0, kt1);

  const uint32_t sbase = (uint32_t)__cvta_generic_to_shared(smem_kt);
  // 16-byte chunks: row c/8, k (c%8)*2; threads 0..7 also copy the weights
  auto issue = [&](int stage, int64_t ktg) {
    const int64_t kloc = ktg * TK - slot0;                 // column inside the slabs
    const uint32_t sa = sbase + (uint32_t)(stage * KT_STAGE_DOUBLES) * 8u;
#pragma unroll
    for (int i = 0; i < TA * 8 / NTH; ++i) {
      const int c = tid + NTH * i, row = c >> 3, kc = (c & 7) * 2;
      const int64_t ra = m0 + row;
      cp_async16(sa + (uint32_t)(row * LDK + kc) * 8u, Phi + min(ra, nbf - 1) * ld + kloc + kc, ra < nbf ? 16u : 0u);
    }
#pragma unroll
    for (int i = 0; i < TB * 8 / NTH; ++i) {
      const int c = tid + NTH * i, row = c >> 3, kc = (c & 7) * 2;
      const int64_t rb = n0 + row;
      cp_async16(sa + (uint32_t)(TA * LDK + row * LDK + kc) * 8u, G + min(rb, nbf - 1) * ld + kloc + kc, rb < nbf ? 16u : 0u);
    }
    if (tid < 8) cp_async16(sa + (uint32_t)((TA + TB) * LDK + tid * 2) * 8u, wts + ktg * TK + tid * 2, 16u);
  };

  double acc[4][KT_NJ][2];
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < KT_NJ; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

  int64_t pending = walk.next();                           // next k-tile to issue
  int issued = 0;
#pragma unroll
  for (int s = 0; s < KT_STAGES - 1; ++s) {
    if (pending >= 0) { issue(s, pending); ++issued; pending = walk.next(); }
    cp_commit();
  }
  for (int it = 0; it < issued; ++it) {
    cp_wait<KT_STAGES - 2>();                              // the group of tile `it` has landed
    __syncthreads();                                       // ... for every thread, and the stage of tile it-1 is free
    if (pending >= 0) { issue((it + KT_STAGES - 1) % KT_STAGES, pending); ++issued; pending = walk.next(); }
    cp_commit();
    const double* st = smem_kt + (it % KT_STAGES) * KT_STAGE_DOUBLES;
    const double* as = st + (wm * 32 + g) * LDK + t;
    const double* bs = st + TA * LDK + (wn * 8 * KT_NJ + g) * LDK + t;
    const double* ws = st + (TA + TB) * LDK + t;
#pragma unroll
    for (int kk = 0; kk < TK; kk += 4) {
      double af[4], bf[KT_NJ];
      const double wk = ws[kk];
#pragma unroll
      for (int i = 0; i < 4; ++i) af[i] = as[i * 8 * LDK + kk] * wk;
#pragma unroll
      for (int j = 0; j < KT_NJ; ++j) bf[j] = bs[j * 8 * LDK + kk];
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < KT_NJ; ++j) dmma884(acc[i][j][0], acc[i][j][1], af[i], bf[j]);
    }
  }
  if (issued == 0) return;
  // epilogue: thread holds C[row = g][cols 2t, 2t+1] of each 8x8 fragment; Kt is accumulated over k-chunks and super-batches
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int64_t row = m0 + wm * 32 + i * 8 + g;
    if (row >= nbf) continue;
#pragma unroll
    for (int j = 0; j < KT_NJ; ++j) {
      const int64_t col = n0 + wn * 8 * KT_NJ + j * 8 + 2 * t;
      double* c = Kt + row * nbf + col;
      if (col < nbf) atomicAdd(c, acc[i][j][0]);
      if (col + 1 < nbf) atomicAdd(c + 1, acc[i][j][1]);
    }
  }
}

// a4:  F[lam, g] = sum_sigma P[lam, sigma] Phi[sigma, g]     Eq. 35/48.  CTA tile 64 x 128, double
// buffered, three CTAs per SM; the B operand
// (Phi rows) is contiguous along the output column g, so its shared tile is [16 k][132].  P has an arbitrary row stride
// (nbf), hence 8-byte copies for it.  A bit per (128-slot column tile, 16-function k-tile) says whether Phi is non-zero
// there (some shell overlapping the k-tile is in B_j of a batch overlapping the column tile); zero blocks are skipped.
constexpr int LDN = 132;
#ifndef SNK_F_ROWS
#define SNK_F_ROWS 64
#endif
#ifndef SNK_F_STAGES
#define SNK_F_STAGES 2
#endif
#ifndef SNK_F_MINB
#define SNK_F_MINB 3
#endif
constexpr int TMR = SNK_F_ROWS, FNI = TMR / 16, FST = SNK_F_STAGES;   // rows of the F tile, row fragments per warp, ring depth
constexpr int FSTAGE_DOUBLES = TMR * LDK + TK * LDN;
__global__ void __launch_bounds__(NTH, SNK_F_MINB) k_gemm_f(int64_t nbf, int64_t ncols, const double* __restrict__ P, const double* __restrict__ Phi,
                                                double* __restrict__ F, int64_t ld, const uint32_t* __restrict__ act, int kwords) {
  extern __shared__ __align__(16) double smem_kt[];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int wm = warp >> 2, wn = warp & 3;
  const int g = lane >> 2, t = lane & 3;
  const int64_t n0 = (int64_t)blockIdx.x * TM, m0 = (int64_t)blockIdx.y * TMR;
  BitWalk walk;
  walk.init(act + (int64_t)blockIdx.x * kwords, 0, kwords, 0, (nbf + TK - 1) / TK);
  const uint32_t sbase = (uint32_t)__cvta_generic_to_shared(smem_kt);
  auto issue = [&](int stage, int64_t kt) {
    const int64_t k0 = kt * TK;
    const uint32_t sa = sbase + (uint32_t)(stage * FSTAGE_DOUBLES) * 8u;
#pragma unroll
    for (int i = 0; i < TMR * 16 / NTH; ++i) {             // A: TMR rows x 16 k, 8-byte copies
      const int c = tid + NTH * i, row = c >> 4, kc = c & 15;
      const int64_t r = m0 + row, k = k0 + kc;
      const bool ok = r < nbf && k < nbf;
      asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;\n" ::"r"(sa + (uint32_t)(row * LDK + kc) * 8u),
                   "l"(P + (ok ? r * nbf + k : 0)), "r"(ok ? 8u : 0u)
                   : "memory");
    }
#pragma unroll
    for (int i = 0; i < 4; ++i) {                          // B: 16 k x 128 columns, 16-byte copies (ncols, ld multiples of 32)
      const int c = tid + NTH * i, kr = c >> 6, nc = (c & 63) * 2;
      const int64_t k = k0 + kr, col = n0 + nc;
      const bool ok = k < nbf && col < ncols;
      cp_async16(sa + (uint32_t)(TMR * LDK + kr * LDN + nc) * 8u, Phi + (ok ? k * ld + col : 0), ok ? 16u : 0u);
    }
  };
  double acc[FNI][4][2];
#pragma unroll
  for (int i = 0; i < FNI; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;
  int64_t pending = walk.next();
  int issued = 0;
#pragma unroll
  for (int s = 0; s < FST - 1; ++s) {
    if (pending >= 0) { issue(s, pending); ++issued; pending = walk.next(); }
    cp_commit();
  }
  for (int it = 0; it < issued; ++it) {
    cp_wait<FST - 2>();
    __syncthreads();
    if (pending >= 0) { issue((it + FST - 1) % FST, pending); ++issued; pending = walk.next(); }
    cp_commit();
    const double* st = smem_kt + (it % FST) * FSTAGE_DOUBLES;
    const double* as = st + (wm * (TMR / 2) + g) * LDK + t;
    const double* bs = st + TMR * LDK + t * LDN + wn * 32 + g;
#pragma unroll
    for (int kk = 0; kk < TK; kk += 4) {
      double af[FNI], bf[4];
#pragma unroll
      for (int i = 0; i < FNI; ++i) af[i] = as[i * 8 * LDK + kk];
#pragma unroll
      for (int j = 0; j < 4; ++j) bf[j] = bs[kk * LDN + j * 8];
#pragma unroll
      for (int i = 0; i < FNI; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) dmma884(acc[i][j][0], acc[i][j][1], af[i], bf[j]);
    }
  }
  // F is overwritten (zeros where every block was skipped)
#pragma unroll
  for (int i = 0; i < FNI; ++i) {
    const int64_t row = m0 + wm * (TMR / 2) + i * 8 + g;
    if (row >= nbf) continue;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const int64_t col = n0 + wn * 32 + j * 8 + 2 * t;
      if (col < ncols) *reinterpret_cast<double2*>(F + row * ld + col) = make_double2(acc[i][j][0], acc[i][j][1]);
    }
  }
}

// bits of k_gemm_f: one CTA per batch; every shell of B_j sets its 16-function k-tiles in the column tiles the batch overlaps
__global__ void __launch_bounds__(128) k_f_flags(ShellTab sh, const int32_t* __restrict__ bn, const int64_t* __restrict__ bslot,
                                                 const int64_t* __restrict__ bslot0, const int64_t* __restrict__ btile0,
                                                 const uint32_t* __restrict__ bmask, int nshw, uint32_t* __restrict__ act, int kwords) {
  const int j = blockIdx.x;
  const int npad = (bn[j] + kSlotAlign - 1) / kSlotAlign * kSlotAlign;
  const int64_t c0 = bslot[j] - bslot0[j];                  // first column of the batch inside its super-batch
  const int64_t t0 = btile0[j] + c0 / TM, t1 = btile0[j] + (c0 + npad - 1) / TM;
  for (int a = threadIdx.x; a < sh.nsh; a += blockDim.x)
    if ((bmask[(int64_t)j * nshw + (a >> 5)] >> (a & 31)) & 1u) {
      const int f0 = sh.foff[a], f1 = f0 + (sh.l[a] + 1) * (sh.l[a] + 2) / 2 - 1;
      for (int kt = f0 / TK; kt <= f1 / TK; ++kt)
        for (int64_t tt = t0; tt <= t1; ++tt) atomicOr(act + tt * kwords + (kt >> 5), 1u << (kt & 31));
    }
}

// act bits: one CTA per batch; a shell of B_j marks the row tiles its functions fall into, then the batch's k-tiles are
// set for every marked row tile.
__global__ void __launch_bounds__(128) k_kt_flags(ShellTab sh, const int32_t* __restrict__ bn, const int64_t* __restrict__ bslot,
                                                  const uint32_t* __restrict__ bmask, int nshw, int nmt, uint32_t* __restrict__ act,
                                                  int64_t actw) {
  extern __shared__ int s_mark[];
  const int j = blockIdx.x;
  for (int i = threadIdx.x; i < nmt; i += blockDim.x) s_mark[i] = 0;
  __syncthreads();
  for (int a = threadIdx.x; a < sh.nsh; a += blockDim.x)
    if ((bmask[(int64_t)j * nshw + (a >> 5)] >> (a & 31)) & 1u) {
      const int f0 = sh.foff[a], f1 = f0 + (sh.l[a] + 1) * (sh.l[a] + 2) / 2 - 1;
      s_mark[f0 / TA] = 1;
      s_mark[f1 / TA] = 1;
    }
  __syncthreads();
  const int64_t k0 = bslot[j] / TK;
  const int nk = (bn[j] + kSlotAlign - 1) / kSlotAlign * kSlotAlign / TK;
  for (int i = threadIdx.x; i < nmt * nk; i += blockDim.x) {
    const int mt = i / nk;
    if (!s_mark[mt]) continue;
    const int64_t kt = k0 + i % nk;
    atomicOr(act + (int64_t)mt * actw + (kt >> 5), 1u << (kt & 31));
  }
}
}  // namespace
}  // namespace snk

namespace snk {

int kt_row_tile() { return TA; }

cudaError_t run_kt_flags(const ShellTab& sh, int nbatch, const int32_t* bn, const int64_t* bslot, const uint32_t* bmask, int nshw,
                         uint32_t* act, int64_t actw, cudaStream_t s) {
  const int nmt = (sh.nbf + TA - 1) / TA;
  cudaError_t e = cudaMemsetAsync(act, 0, (size_t)nmt * actw * sizeof(uint32_t), s);
  if (e != cudaSuccess) return e;
  if (nbatch > 0) k_kt_flags<<<nbatch, 128, nmt * sizeof(int), s>>>(sh, bn, bslot, bmask, nshw, nmt, act, actw);
  return cudaGetLastError();
}

cudaError_t gemm_kt(int64_t nbf, int64_t slot0, int64_t nslots, const double* Phi, const double* G, int64_t ld, const double* wts,
                    double* Kt, const uint32_t* act, int64_t actw, cudaStream_t s) {
  if (nbf <= 0 || nslots <= 0) return cudaSuccess;
  const int64_t nta = (nbf + TA - 1) / TA, ntb = (nbf + TB - 1) / TB;
  const int64_t kt0 = slot0 / TK, kt1 = (slot0 + nslots) / TK;
  const int64_t nwords = ((kt1 + 31) >> 5) - (kt0 >> 5);
  // split-K into short k-chunks (grid.z slowest): the CTAs of one chunk run together, so the chunk's Phi and G columns
  // (2 nbf x chunk x 8 B) are fetched from HBM once and shared through L2 although the row tiles skip different blocks
  int64_t wchunk = 4;                                      // words of 32 k-tiles: 2048 slots
  while (wchunk > 2 && 2.0 * nbf * (double)wchunk * 512 * 8 > 48e6) wchunk /= 2;
  const int64_t split = (nwords + wchunk - 1) / wchunk;
  constexpr int smem = KT_STAGES * KT_STAGE_DOUBLES * (int)sizeof(double);
  static bool attr_set[kMaxDevices] = {};
  if (cudaError_t e = opt_in_smem(k_gemm_kt, smem, attr_set); e != cudaSuccess) return e;
  dim3 grid((unsigned)ntb, (unsigned)nta, (unsigned)split);
  k_gemm_kt<<<grid, NTH, smem, s>>>(nbf, slot0, nslots, Phi, G, ld, wts, Kt, act, actw, wchunk);
  return cudaGetLastError();
}

cudaError_t run_f_flags(const ShellTab& sh, int nbatch, const int32_t* bn, const int64_t* bslot, const int64_t* bslot0,
                        const int64_t* btile0, const uint32_t* bmask, int nshw, uint32_t* act, int64_t ntiles, int kwords, cudaStream_t s) {
  cudaError_t e = cudaMemsetAsync(act, 0, (size_t)ntiles * kwords * sizeof(uint32_t), s);
  if (e != cudaSuccess) return e;
  if (nbatch > 0) k_f_flags<<<nbatch, 128, 0, s>>>(sh, bn, bslot, bslot0, btile0, bmask, nshw, act, kwords);
  return cudaGetLastError();
}

cudaError_t gemm_f(int64_t nbf, int64_t ncols, const double* P, const double* Phi, double* F, int64_t ld, const uint32_t* act, int kwords,
                   cudaStream_t s) {
  if (nbf <= 0 || ncols <= 0) return cudaSuccess;
  constexpr int smem = FST * FSTAGE_DOUBLES * (int)sizeof(double);
  static bool attr_set[kMaxDevices] = {};
  if (cudaError_t e = opt_in_smem(k_gemm_f, smem, attr_set); e != cudaSuccess) return e;
  dim3 grid((unsigned)((ncols + TM - 1) / TM), (unsigned)((nbf + TMR - 1) / TMR));
  k_gemm_f<<<grid, NTH, smem, s>>>(nbf, ncols, P, Phi, F, ld, act, kwords);
  return cudaGetLastError();
}

}  // namespace snk
