// snk_gemm.cu -- fp64 tensor-core (DMMA m8n8k4) contraction used for
//   a4  F  = P * Phi                      Eq. 35/48
//   a6  Kt += Phi * diag(w) * G^T         Eq. 39
//   a3  Ftilde = |P| * PhiTilde           Eq. 46
// The paper runs these as MAGMA variable-size batched GEMMs; here the Phi/F/G of a whole
// super-batch are dense [nbf x slots] slabs, so each is ONE large GEMM.
//
// CTA tile 128 x 128 x 16, 8 warps (2 x 4), warp tile 64 x 32 = 8 x 4 m8n8 fragments, accumulators in registers.
// Shared tiles are stored k-major with row stride 132 doubles so that the m8n8k4 fragment loads
// (thread (g = lane/4, t = lane%4) reads [k = t][m = g]) hit 16 distinct 8-byte banks per half-warp.
#include <algorithm>

#include "snk_internal.h"

namespace snk {

namespace {
constexpr int BM = 128, BN = 128, BK = 16, LDS = 132, NT = 256;

__device__ __forceinline__ void dmma884(double& d0, double& d1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n" : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

// Loads one BK x 128 operand tile into registers (8 doubles per thread).
// kmajor_src: source element (r, k) at src[r*ld + k] (k contiguous)  -> thread reads 8 consecutive k of one row
// else      : source element (k, c) at src[k*ld + c] (c contiguous)  -> thread reads 8 c's strided by 16... (see below)
template <bool KCONTIG>
__device__ __forceinline__ void load_tile(double (&r)[8], const double* __restrict__ src, int64_t ld, int64_t r0, int64_t rmax,
                                          int64_t k0, int64_t kmax, const double* __restrict__ kscale, int tid) {
  if constexpr (KCONTIG) {
    // 128 rows x 16 k: thread -> row = tid/2, k-half = (tid&1)*8
    const int64_t row = r0 + (tid >> 1);
    const int64_t kb = k0 + (tid & 1) * 8;
    const bool rok = row < rmax;
    const double* s = src + row * ld + kb;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      double v = 0.0;
      if (rok && kb + i < kmax) { v = s[i]; if (kscale) v *= kscale[kb + i]; }
      r[i] = v;
    }
  } else {
    // 16 k x 128 cols: thread -> k = tid/16, cols = (tid%16) + 16*i  (coalesced across the 16 threads)
    const int64_t k = k0 + (tid >> 4);
    const bool kok = k < kmax;
    const double* s = src + k * ld + r0 + (tid & 15);
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      double v = 0.0;
      if (kok && r0 + (tid & 15) + 16 * i < rmax) v = s[16 * i];
      r[i] = v;
    }
  }
}

template <bool KCONTIG>
__device__ __forceinline__ void store_tile(const double (&r)[8], double* __restrict__ sm, int tid) {
  if constexpr (KCONTIG) {
    const int row = tid >> 1, kb = (tid & 1) * 8;
#pragma unroll
    for (int i = 0; i < 8; ++i) sm[(kb + i) * LDS + row] = r[i];
  } else {
    const int k = tid >> 4, c = tid & 15;
#pragma unroll
    for (int i = 0; i < 8; ++i) sm[k * LDS + c + 16 * i] = r[i];
  }
}

template <bool TRANSB>
__global__ void __launch_bounds__(NT) k_gemm_f64(int64_t M, int64_t N, int64_t K, const double* __restrict__ A, int64_t lda,
                                                 const double* __restrict__ B, int64_t ldb, double* __restrict__ C, int64_t ldc,
                                                 bool beta, const double* __restrict__ kscale, int64_t kchunk) {
  extern __shared__ __align__(16) double smem_gemm[];
  double (*As)[BK * LDS] = reinterpret_cast<double (*)[BK * LDS]>(smem_gemm);
  double (*Bs)[BK * LDS] = reinterpret_cast<double (*)[BK * LDS]>(smem_gemm + 2 * BK * LDS);
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int wm = warp >> 2, wn = warp & 3;            // 2 x 4 warps
  const int g = lane >> 2, t = lane & 3;
  const int64_t m0 = (int64_t)blockIdx.y * BM, n0 = (int64_t)blockIdx.x * BN;

  double acc[8][4][2];
#pragma unroll
  for (int i = 0; i < 8; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

  // split-K: this CTA contracts k in [kbeg, kend); partial results are RED-added (only used with beta = true)
  const int64_t kbeg = (int64_t)blockIdx.z * kchunk;
  const int64_t kend = min(K, kbeg + kchunk);
  const bool atomic_out = gridDim.z > 1;
  double ra[8], rb[8];
  const int64_t nk = kend > kbeg ? (kend - kbeg + BK - 1) / BK : 0;
  load_tile<true>(ra, A, lda, m0, M, kbeg, kend, kscale, tid);
  load_tile<TRANSB>(rb, B, ldb, n0, N, kbeg, kend, nullptr, tid);
  store_tile<true>(ra, As[0], tid);
  store_tile<TRANSB>(rb, Bs[0], tid);
  __syncthreads();

  for (int64_t kt = 0; kt < nk; ++kt) {
    const int cur = kt & 1;
    if (kt + 1 < nk) {
      load_tile<true>(ra, A, lda, m0, M, kbeg + (kt + 1) * BK, kend, kscale, tid);
      load_tile<TRANSB>(rb, B, ldb, n0, N, kbeg + (kt + 1) * BK, kend, nullptr, tid);
    }
    const double* as = As[cur] + wm * 64 + g;
    const double* bs = Bs[cur] + wn * 32 + g;
#pragma unroll
    for (int kk = 0; kk < BK; kk += 4) {
      double af[8], bf[4];
#pragma unroll
      for (int i = 0; i < 8; ++i) af[i] = as[(kk + t) * LDS + i * 8];
#pragma unroll
      for (int j = 0; j < 4; ++j) bf[j] = bs[(kk + t) * LDS + j * 8];
#pragma unroll
      for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) dmma884(acc[i][j][0], acc[i][j][1], af[i], bf[j]);
    }
    if (kt + 1 < nk) {
      store_tile<true>(ra, As[cur ^ 1], tid);
      store_tile<TRANSB>(rb, Bs[cur ^ 1], tid);
    }
    __syncthreads();
  }

  // epilogue: thread holds C[row = g][cols 2t, 2t+1] of each 8x8 fragment
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    const int64_t row = m0 + wm * 64 + i * 8 + g;
    if (row >= M) continue;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const int64_t col = n0 + wn * 32 + j * 8 + 2 * t;
      double* c = C + row * ldc + col;
      if (atomic_out) {
        if (col < N) atomicAdd(c, acc[i][j][0]);
        if (col + 1 < N) atomicAdd(c + 1, acc[i][j][1]);
      } else {
        if (col < N) c[0] = beta ? c[0] + acc[i][j][0] : acc[i][j][0];
        if (col + 1 < N) c[1] = beta ? c[1] + acc[i][j][1] : acc[i][j][1];
      }
    }
  }
}
}  // namespace

cudaError_t gemm_f64(bool transB, int64_t M, int64_t N, int64_t K, const double* A, int64_t lda, const double* B, int64_t ldb,
                     double* C, int64_t ldc, bool beta, const double* kscale, cudaStream_t s) {
  if (M <= 0 || N <= 0) return cudaSuccess;
  dim3 grid((unsigned)((N + BN - 1) / BN), (unsigned)((M + BM - 1) / BM));
  // split-K when the output is too small to fill the GPU (the Kt contraction: M = N = nbf, K = grid points)
  int64_t kchunk = K > 0 ? K : 1;
  if (beta && K > 0) {
    int sms = 0, dev = 0;
    cudaGetDevice(&dev); cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const int64_t ctas = (int64_t)grid.x * grid.y;
    int64_t split = (2 * sms + ctas - 1) / ctas;
    split = std::max<int64_t>(1, std::min<int64_t>(split, K / (8 * BK)));
    kchunk = ((K + split - 1) / split + BK - 1) / BK * BK;
    grid.z = (unsigned)((K + kchunk - 1) / kchunk);
  }
  constexpr int smem = 4 * BK * LDS * (int)sizeof(double);
  static bool attr_t[kMaxDevices] = {}, attr_n[kMaxDevices] = {};
  if (cudaError_t e = opt_in_smem(k_gemm_f64<true>, smem, attr_t); e != cudaSuccess) return e;
  if (cudaError_t e = opt_in_smem(k_gemm_f64<false>, smem, attr_n); e != cudaSuccess) return e;
  if (transB) k_gemm_f64<true><<<grid, NT, smem, s>>>(M, N, K, A, lda, B, ldb, C, ldc, beta, kscale, kchunk);
  else k_gemm_f64<false><<<grid, NT, smem, s>>>(M, N, K, A, lda, B, ldb, C, ldc, beta, kscale, kchunk);
  return cudaGetLastError();
}

}  // namespace snk
