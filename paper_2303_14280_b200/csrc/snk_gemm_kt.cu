// snk_gemm_kt.cu -- the two DMMA contractions around the integral kernel, fp64 mma.sync.m8n8k4, packed to B_j (Eq. 42/48)
//   a4:  F[lam,g]  = sum_{sigma in B} P[lam,sigma] Phi[sigma,g]             Eq. 35/48
//   a6:  Kt[mu,nu] += sum_g Phi[mu,g] w_g G[nu,g],  mu in B                 Eq. 39
//
// Phi rows of shells outside B_j are identically zero over batch j (Eq. 41), and with the slab layout those rows would be
// multiplied all the same.  The grid's batches are therefore grouped, in order, into CHUNKS of up to 2048 slots (neighbouring
// batches: same or adjacent octree cells, nearly the same B_j), and every chunk carries the sorted list L of the functions in
// the union of its batches' B_j (k_chunk_rows, once per grid).  Both contractions address Phi through L -- the packed
// batch-local matrices of the paper (Eq. 42) without copying anything:
//   * a4: one CTA per (128-slot column tile of a chunk, 64 rows of F); the k loop runs over L in steps of 16 and gathers the
//     16 columns of P (8-byte cp.async, P has an arbitrary row stride anyway) and the 16 rows of Phi (1 KB each, 16-byte
//     cp.async) that L names; nothing outside L is loaded or multiplied.
//   * a6: one CTA per (chunk, 32 rows of L, 128 rows of G): the Phi operand rows are gathered through L (contiguous along
//     the contraction index g), the k loop runs over the chunk's slots, and the 32 x 128 partial tile is RED-added into the
//     rows of Kt that L names (split-K over chunks and super-batches).
//   * CTA tiles 64 x 128 (a4, three CTAs per SM) and 32 x 128 (a6, four CTAs per SM), k-tile 16, 8 warps, accumulators in
//     registers, operand tiles double buffered in shared memory (one __syncthreads per k-tile); shared row strides of 20
//     (k-contiguous tiles) and 132 (column-contiguous ones) make every m8n8k4 fragment load conflict free.
//   * w_g is staged with the a6 tile and folded into the Phi fragments.
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
__global__ void __launch_bounds__(NTH, SNK_KT_MINB) k_gemm_kt(int64_t nbf, int64_t slot0, const ChunkRec* __restrict__ chunks,
                                                 const int32_t* __restrict__ nrows, const int32_t* __restrict__ rowlist,
                                                 int64_t lstride, const double* __restrict__ Phi, const double* __restrict__ G,
                                                 int64_t ld, const double* __restrict__ wts, double* __restrict__ Kt) {
  extern __shared__ __align__(16) double smem_kt[];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int wm = warp / KT_WN, wn = warp % KT_WN;          // KT_WM x KT_WN warps, warp tile 32 x (8 KT_NJ)
  const int g = lane >> 2, t = lane & 3;
  const ChunkRec ch = chunks[blockIdx.z];
  const int nrow = nrows[blockIdx.z];
  const int r0 = blockIdx.y * TA;                          // first packed row of this CTA
  if (r0 >= nrow) return;
  const int32_t* __restrict__ L = rowlist + (int64_t)blockIdx.z * lstride;
  const int64_t n0 = (int64_t)blockIdx.x * TB;
  const int nkt = ch.nslots / TK;                          // chunks are whole batches: multiples of 32 slots
  const int64_t kbase = ch.slot0 - slot0;                  // first column of the chunk inside the slabs

  const uint32_t sbase = (uint32_t)__cvta_generic_to_shared(smem_kt);
  // the Phi rows this thread copies (through L); rows past the end of L are zero-filled
  int64_t arow[TA * 8 / NTH];
  bool aok[TA * 8 / NTH];
#pragma unroll
  for (int i = 0; i < TA * 8 / NTH; ++i) {
    const int row = (tid + NTH * i) >> 3;
    aok[i] = r0 + row < nrow;
    arow[i] = aok[i] ? (int64_t)__ldg(L + r0 + row) * ld : 0;
  }
  // 16-byte chunks: row c/8, k (c%8)*2; threads 0..7 also copy the weights
  auto issue = [&](int stage, int kt) {
    const int64_t kloc = kbase + (int64_t)kt * TK;         // column inside the slabs
    const uint32_t sa = sbase + (uint32_t)(stage * KT_STAGE_DOUBLES) * 8u;
#pragma unroll
    for (int i = 0; i < TA * 8 / NTH; ++i) {
      const int c = tid + NTH * i, row = c >> 3, kc = (c & 7) * 2;
      cp_async16(sa + (uint32_t)(row * LDK + kc) * 8u, Phi + arow[i] + kloc + kc, aok[i] ? 16u : 0u);
    }
#pragma unroll
    for (int i = 0; i < TB * 8 / NTH; ++i) {
      const int c = tid + NTH * i, row = c >> 3, kc = (c & 7) * 2;
      const int64_t rb = n0 + row;
      cp_async16(sa + (uint32_t)(TA * LDK + row * LDK + kc) * 8u, G + min(rb, nbf - 1) * ld + kloc + kc, rb < nbf ? 16u : 0u);
    }
    if (tid < 8) cp_async16(sa + (uint32_t)((TA + TB) * LDK + tid * 2) * 8u, wts + ch.slot0 + (int64_t)kt * TK + tid * 2, 16u);
  };

  double acc[4][KT_NJ][2];
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < KT_NJ; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

#pragma unroll
  for (int s = 0; s < KT_STAGES - 1; ++s) {
    if (s < nkt) issue(s, s);
    cp_commit();
  }
  for (int it = 0; it < nkt; ++it) {
    cp_wait<KT_STAGES - 2>();                              // the group of tile `it` has landed
    __syncthreads();                                       // ... for every thread, and the stage of tile it-1 is free
    if (it + KT_STAGES - 1 < nkt) issue((it + KT_STAGES - 1) % KT_STAGES, it + KT_STAGES - 1);
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
  // epilogue: thread holds C[row = g][cols 2t, 2t+1] of each 8x8 fragment; Kt is accumulated over chunks and super-batches
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int pr = r0 + wm * 32 + i * 8 + g;
    if (pr >= nrow) continue;
    const int64_t row = __ldg(L + pr);
#pragma unroll
    for (int j = 0; j < KT_NJ; ++j) {
      const int64_t col = n0 + wn * 8 * KT_NJ + j * 8 + 2 * t;
      double* c = Kt + row * nbf + col;
      if (col < nbf) atomicAdd(c, acc[i][j][0]);
      if (col + 1 < nbf) atomicAdd(c + 1, acc[i][j][1]);
    }
  }
}

// a4:  F[lam, g] = sum_{sigma in L} P[lam, sigma] Phi[sigma, g]     Eq. 35/48.  CTA tile 64 x 128, double
// buffered, three CTAs per SM; the B operand (Phi rows) is contiguous along the output column g, so its shared tile is
// [16 k][132].  Column tiles belong to one chunk each (ColTile); the k loop gathers through the chunk's list L.
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
__global__ void __launch_bounds__(NTH, SNK_F_MINB) k_gemm_f(int64_t nbf, int64_t slot0, const ColTile* __restrict__ tiles, int chunk0,
                                                const int32_t* __restrict__ nrows, const int32_t* __restrict__ rowlist, int64_t lstride,
                                                const double* __restrict__ P, const double* __restrict__ Phi, double* __restrict__ F,
                                                int64_t ld) {
  extern __shared__ __align__(16) double smem_kt[];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int wm = warp >> 2, wn = warp & 3;
  const int g = lane >> 2, t = lane & 3;
  const ColTile ct = tiles[blockIdx.x];
  const int64_t n0 = ct.slot - slot0, m0 = (int64_t)blockIdx.y * TMR;      // first column inside the slabs, first row of F
  const int ncols = ct.ncols;
  const int nrow = nrows[ct.chunk - chunk0];
  const int32_t* __restrict__ L = rowlist + (int64_t)(ct.chunk - chunk0) * lstride;
  const int nkt = (nrow + TK - 1) / TK;
  const uint32_t sbase = (uint32_t)__cvta_generic_to_shared(smem_kt);
  auto issue = [&](int stage, int kt) {
    const int k0 = kt * TK;
    const uint32_t sa = sbase + (uint32_t)(stage * FSTAGE_DOUBLES) * 8u;
#pragma unroll
    for (int i = 0; i < TMR * 16 / NTH; ++i) {             // A: TMR rows x 16 k, 8-byte copies, columns of P named by L
      const int c = tid + NTH * i, row = c >> 4, kc = c & 15;
      const int64_t r = m0 + row;
      const bool ok = r < nbf && k0 + kc < nrow;
      const int64_t k = ok ? __ldg(L + k0 + kc) : 0;
      asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;\n" ::"r"(sa + (uint32_t)(row * LDK + kc) * 8u),
                   "l"(P + (ok ? r * nbf + k : 0)), "r"(ok ? 8u : 0u)
                   : "memory");
    }
#pragma unroll
    for (int i = 0; i < 4; ++i) {                          // B: 16 k x 128 columns, 16-byte copies, rows of Phi named by L
      const int c = tid + NTH * i, kr = c >> 6, nc = (c & 63) * 2;
      const bool ok = k0 + kr < nrow && nc < ncols;
      const int64_t k = ok ? __ldg(L + k0 + kr) : 0;
      cp_async16(sa + (uint32_t)(TMR * LDK + kr * LDN + nc) * 8u, Phi + (ok ? k * ld + n0 + nc : 0), ok ? 16u : 0u);
    }
  };
  double acc[FNI][4][2];
#pragma unroll
  for (int i = 0; i < FNI; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;
#pragma unroll
  for (int s = 0; s < FST - 1; ++s) {
    if (s < nkt) issue(s, s);
    cp_commit();
  }
  for (int it = 0; it < nkt; ++it) {
    cp_wait<FST - 2>();
    __syncthreads();
    if (it + FST - 1 < nkt) issue((it + FST - 1) % FST, it + FST - 1);
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
  // F is overwritten (zeros where L is empty)
#pragma unroll
  for (int i = 0; i < FNI; ++i) {
    const int64_t row = m0 + wm * (TMR / 2) + i * 8 + g;
    if (row >= nbf) continue;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const int col = wn * 32 + j * 8 + 2 * t;
      if (col < ncols) *reinterpret_cast<double2*>(F + row * ld + n0 + col) = make_double2(acc[i][j][0], acc[i][j][1]);
    }
  }
}

// Row lists of the chunks: one CTA per chunk ORs the function ranges of the shells in B_j of its batches into a bit mask in
// shared memory and compacts it (ascending function index).
__global__ void __launch_bounds__(256) k_chunk_rows(ShellTab sh, const ChunkRec* __restrict__ chunks, const uint32_t* __restrict__ bmask,
                                                    int nshw, int32_t* __restrict__ rowlist, int64_t lstride, int32_t* __restrict__ nrows) {
  extern __shared__ uint32_t s_fm[];                       // nbf bits, then 8 warp sums
  const int nw = (sh.nbf + 31) / 32;
  int* wsum = reinterpret_cast<int*>(s_fm + nw);
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const ChunkRec ch = chunks[blockIdx.x];
  for (int i = tid; i < nw; i += 256) s_fm[i] = 0u;
  __syncthreads();
  for (int j = ch.b0; j < ch.b1; ++j)
    for (int a = tid; a < sh.nsh; a += 256)
      if ((bmask[(int64_t)j * nshw + (a >> 5)] >> (a & 31)) & 1u) {
        const int f0 = sh.foff[a], f1 = f0 + (sh.l[a] + 1) * (sh.l[a] + 2) / 2;
        for (int f = f0; f < f1; ++f) atomicOr(s_fm + (f >> 5), 1u << (f & 31));
      }
  __syncthreads();
  int32_t* __restrict__ out = rowlist + (int64_t)blockIdx.x * lstride;
  int running = 0;
  for (int wb = 0; wb < nw; wb += 256) {
    const int w = wb + tid;
    uint32_t word = w < nw ? s_fm[w] : 0u;
    const int n = __popc(word);
    int inc = n;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) { const int v = __shfl_up_sync(~0u, inc, d); if (lane >= d) inc += v; }
    if (lane == 31) wsum[warp] = inc;
    __syncthreads();
    int base = 0, total = 0;
#pragma unroll
    for (int k = 0; k < 8; ++k) { const int v = wsum[k]; if (k < warp) base += v; total += v; }
    int o = running + base + inc - n;
    while (word) { const int b = __ffs(word) - 1; word &= word - 1; out[o++] = (w << 5) + b; }
    running += total;
    __syncthreads();
  }
  if (tid == 0) nrows[blockIdx.x] = running;
}
}  // namespace
}  // namespace snk

namespace snk {

int kt_row_tile() { return TA; }
int f_k_tile() { return TK; }

cudaError_t run_chunk_rows(const ShellTab& sh, int nchunks, const ChunkRec* chunks, const uint32_t* bmask, int nshw, int32_t* rowlist,
                           int64_t lstride, int32_t* nrows, cudaStream_t s) {
  if (nchunks > 0) {
    const size_t smem = ((sh.nbf + 31) / 32) * sizeof(uint32_t) + 8 * sizeof(int);
    k_chunk_rows<<<nchunks, 256, smem, s>>>(sh, chunks, bmask, nshw, rowlist, lstride, nrows);
  }
  return cudaGetLastError();
}

cudaError_t gemm_kt(int64_t nbf, int64_t slot0, int nchunks, int max_nrow, const ChunkRec* chunks, const int32_t* nrows,
                    const int32_t* rowlist, int64_t lstride, const double* Phi, const double* G, int64_t ld, const double* wts, double* Kt,
                    cudaStream_t s) {
  if (nbf <= 0 || nchunks <= 0 || max_nrow <= 0) return cudaSuccess;
  constexpr int smem = KT_STAGES * KT_STAGE_DOUBLES * (int)sizeof(double);
  static bool attr_set[kMaxDevices] = {};
  if (cudaError_t e = opt_in_smem(k_gemm_kt, smem, attr_set); e != cudaSuccess) return e;
  for (int c0 = 0; c0 < nchunks; c0 += 65535) {            // grid.z limit
    const int nc = std::min(65535, nchunks - c0);
    dim3 grid((unsigned)((nbf + TB - 1) / TB), (unsigned)((max_nrow + TA - 1) / TA), (unsigned)nc);
    k_gemm_kt<<<grid, NTH, smem, s>>>(nbf, slot0, chunks + c0, nrows + c0, rowlist + (int64_t)c0 * lstride, lstride, Phi, G, ld, wts, Kt);
  }
  return cudaGetLastError();
}

cudaError_t gemm_f(int64_t nbf, int64_t slot0, int ntiles, const ColTile* tiles, int chunk0, const int32_t* nrows, const int32_t* rowlist,
                   int64_t lstride, const double* P, const double* Phi, double* F, int64_t ld, cudaStream_t s) {
  if (nbf <= 0 || ntiles <= 0) return cudaSuccess;
  constexpr int smem = FST * FSTAGE_DOUBLES * (int)sizeof(double);
  static bool attr_set[kMaxDevices] = {};
  if (cudaError_t e = opt_in_smem(k_gemm_f, smem, attr_set); e != cudaSuccess) return e;
  dim3 grid((unsigned)ntiles, (unsigned)((nbf + TMR - 1) / TMR));
  k_gemm_f<<<grid, NTH, smem, s>>>(nbf, slot0, tiles, chunk0, nrows, rowlist, lstride, P, Phi, F, ld);
  return cudaGetLastError();
}

}  // namespace snk
