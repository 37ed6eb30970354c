// snk_internal.h -- host-side context and kernel-launch prototypes of libsnk (not part of the public ABI).
#pragma once
#include <cuda_runtime.h>
#include <cstdint>
#include <string>
#include <vector>

#include "../../include/snk.h"

namespace snk {

constexpr int kTile = 128;          // grid points per CTA of the collocation / integral kernels
constexpr int kSlotAlign = 32;      // every batch starts on a warp boundary in the slot arrays
constexpr int kNumClasses = 10;     // (la,lb), la >= lb, la <= 3
constexpr int kMaxDepth = 20;       // R13

inline int class_id(int la, int lb) { return la * (la + 1) / 2 + lb; }   // (0,0)=0,(1,0)=1,(1,1)=2,(2,0)=3,...

struct PrimPair;   // snk_os.cuh

// ---- pair units ------------------------------------------------------------------------------------------------
// The significant shell pairs are streamed through shared memory (one bulk copy per unit) by the integral kernel.
// A "unit" is one shell pair (oriented so that l_a >= l_b, R6: a carries the VRR, the HRR shifts to b) with at most
// kUnitPrims of its primitive pairs; a pair with more primitive pairs is split into consecutive units.  Because the
// HRR (A2) and the F-contraction (Eq. 38) are linear in the contracted Theta (R4), the units of one pair simply add.
// Units are sorted by (class, a, b); V_j holds one bit per unit (all units of a pair share the pair's decision).
constexpr int kUnitPrims = 8;
struct __align__(16) UnitHdr {
  int32_t fa, fb;         // first basis-function index of shell a / b
  int32_t nprim;          // primitive pairs in this unit (R14 may leave 0: such a unit is never in V_j)
  int32_t first;          // 1 for the first unit of its pair
  double ABx, ABy, ABz;   // A - B
  int32_t sa, sb;         // shell ids
  int64_t offa, offb;     // fa * ld, fb * ld: element offsets of the shells' first rows in the F / G slabs
};
static_assert(sizeof(UnitHdr) == 64, "UnitHdr layout");
constexpr int kPrimBytes = 80;                                   // sizeof(PrimPair), snk_os.cuh
constexpr int kUnitBytes = 64 + kUnitPrims * kPrimBytes;         // 704: header + primitive pairs, contiguous in HBM
// what the screening kernels and the kernel's producer warp need, without touching the 704-byte records
struct __align__(8) UnitMeta {
  int32_t sa, sb;
  int32_t fb;
  int32_t nprim_first;    // nprim | first << 8
  double At;
};
static_assert(sizeof(UnitMeta) == 24, "UnitMeta layout");

// A chunk = consecutive whole batches of one super-batch, up to kChunkSlots slots: the unit of the packed DMMA contractions
// (snk_gemm_kt.cu).  Its row list (functions in the union of the batches' B_j) lives in a [nchunks x lstride] int table.
#ifndef SNK_CHUNK_SLOTS
#define SNK_CHUNK_SLOTS 2048
#endif
constexpr int kChunkSlots = SNK_CHUNK_SLOTS;
struct ChunkRec { int64_t slot0; int32_t nslots; int32_t b0, b1; int32_t pad; };
static_assert(sizeof(ChunkRec) == 24, "ChunkRec layout");
// 128-slot column tile of a4 (inside one chunk)
struct ColTile { int64_t slot; int32_t chunk; int32_t ncols; };

// One tile = up to kTile consecutive slots of one batch.
struct TileRec { int32_t batch; int32_t n; int64_t slot; };

// Device shell table (SoA)
struct ShellTab {
  const double* cx; const double* cy; const double* cz;
  const int32_t* l; const int32_t* foff; const int32_t* poff; const int32_t* nprim;
  const double* pexp; const double* pcoef;
  const double* rcut2;
  int nsh; int nbf;
};

template <class T>
struct DevBuf {           // grow-only device buffer
  T* p = nullptr;
  size_t cap = 0;         // elements
  cudaError_t reserve(size_t n) {
    if (n <= cap) return cudaSuccess;
    if (p) cudaFree(p);
    p = nullptr; cap = 0;
    cudaError_t e = cudaMalloc((void**)&p, n * sizeof(T));
    if (e == cudaSuccess) cap = n;
    return e;
  }
  void release() { if (p) cudaFree(p); p = nullptr; cap = 0; }
  DevBuf() = default;
  DevBuf(const DevBuf&) = delete;
  DevBuf& operator=(const DevBuf&) = delete;
  ~DevBuf() { release(); }
};

// cudaFuncSetAttribute is per device: one opt-in flag per (kernel, device).  `done` is the call site's static table.
constexpr int kMaxDevices = 64;
template <class Kern>
inline cudaError_t opt_in_smem(Kern kern, int bytes, bool (&done)[kMaxDevices]) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  const bool tracked = dev >= 0 && dev < kMaxDevices;
  if (tracked && done[dev]) return cudaSuccess;
  e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
  if (e == cudaSuccess && tracked) done[dev] = true;
  return e;
}

struct IntParams {
  const double* gx; const double* gy; const double* gz;
  const double* F; double* G;
  int64_t ld;              // leading dimension of F/G (slots of the super-batch, padded)
  int64_t slot0;           // first slot of the super-batch
  const TileRec* tiles; int ntiles;
  const int32_t* vlist; int64_t vlstride;   // kept unit ids of the super-batch's batches (k_vlist), ints per batch row
  const int32_t* vcnt;                      // [batches of the super-batch][kNumClasses] kept units per class
  int b0;                                   // first batch of the super-batch
  int cls;                                  // class of this launch
  int nsplit;                               // CTAs per tile: each takes every nsplit-th share of the tile's unit list
  int pbeg, pend;          // range of this class in the unit list
  const unsigned char* units;               // [nunit][kUnitBytes]
  const UnitMeta* meta;                     // [nunit]
  const double* boys;                       // Boys tables, all L (snk_os.cuh)
};

// ---- kernel launchers (each returns cudaGetLastError()) ----
cudaError_t launch_integrals(int cls, const IntParams& p, cudaStream_t s);
cudaError_t launch_debug_A(int la, int lb, bool transpose, const PrimPair* prims, int nprim, double ABx, double ABy, double ABz,
                           const double* pts, int64_t n, const double* boys, double* out, cudaStream_t s);
cudaError_t launch_debug_boys(int mmax, int64_t n, const double* x, const double* boys, double* out, cudaStream_t s);

// C[M x N] (beta ? += : =) A[M x K] * op(B);  A row-major lda;  transB=false: B[K x N] row-major ldb;
// transB=true: B given as [N x K] row-major ldb.  kscale (optional) multiplies A's column k.  fp64 DMMA.
cudaError_t gemm_f64(bool transB, int64_t M, int64_t N, int64_t K, const double* A, int64_t lda, const double* B, int64_t ldb,
                     double* C, int64_t ldc, bool beta, const double* kscale, cudaStream_t s);

}  // namespace snk
