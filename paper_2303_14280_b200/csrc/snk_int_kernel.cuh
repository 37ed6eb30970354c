// snk_int_kernel.cuh -- integral-contraction kernel (row a5):  G[nu][g] += sum_{(nu,lam) in V_j} A_{nu,lam}(g) F[lam][g]
// Eq. 38/48 via App. A.  One thread = one grid point, one CTA = one tile of
// kTile consecutive points of one batch; all threads of a CTA walk the same V_j bit mask, so control flow is uniform.
// The pair list of a class is sorted by (a, b): G_a / F_a stay in registers over a run of pairs sharing a.
// A is never stored.  Included once per (LA,LB) translation unit.
#pragma once
#include "snk_internal.h"
#include "snk_os.cuh"

namespace snk {

template <int LA, int LB>
__global__ void __launch_bounds__(kTile) k_integrals(IntParams p) {
  constexpr int NA = ncart(LA), NB = ncart(LB), L = LA + LB;
  const TileRec tile = p.tiles[blockIdx.x];
  const int t = threadIdx.x;
  const bool active = t < tile.n;
  const int64_t slot = tile.slot + (active ? t : tile.n - 1);
  const double gx = p.gx[slot], gy = p.gy[slot], gz = p.gz[slot];
  const int64_t col = slot - p.slot0;
  const double* __restrict__ Fc = p.F + col;
  double* __restrict__ Gc = p.G + col;
  const uint32_t* __restrict__ mask = p.vmask + (int64_t)tile.batch * p.vstride;

  int cur_fa = -1;
  double Fa[NA], Ga[NA];
#pragma unroll
  for (int i = 0; i < NA; ++i) { Fa[i] = 0.0; Ga[i] = 0.0; }

  const int w0 = p.pbeg >> 5, w1 = (p.pend + 31) >> 5;
  for (int w = w0; w < w1; ++w) {
    uint32_t bits = __ldg(mask + w);
    if (w == w0) bits &= 0xffffffffu << (p.pbeg & 31);
    if (w == w1 - 1 && (p.pend & 31)) bits &= 0xffffffffu >> (32 - (p.pend & 31));
    while (bits) {
      const int pid = (w << 5) + (__ffs(bits) - 1);
      bits &= bits - 1;
      const PairRec* __restrict__ pr = p.pairs + pid;
      const int fa = __ldg(&pr->fa), fb = __ldg(&pr->fb);
      if (fa != cur_fa) {
        if (cur_fa >= 0 && active) {
#pragma unroll
          for (int i = 0; i < NA; ++i) atomicAdd(Gc + (int64_t)(cur_fa + i) * p.ld, Ga[i]);
        }
        cur_fa = fa;
#pragma unroll
        for (int i = 0; i < NA; ++i) { Fa[i] = Fc[(int64_t)(fa + i) * p.ld]; Ga[i] = 0.0; }
      }
      double Fb[NB], Gb[NB];
#pragma unroll
      for (int k = 0; k < NB; ++k) { Fb[k] = Fc[(int64_t)(fb + k) * p.ld]; Gb[k] = 0.0; }

      double acc[nlev(LA, L)];
      theta_contracted<LA, LB>(p.prims + __ldg(&pr->prim_off), __ldg(&pr->nprim), gx, gy, gz, p.boys, acc);
      ContractSink<LA, LB> sink{Fa, Fb, Ga, Gb};
      HrrNode<LA, LB, 0, 0, 0, L>::run(acc, __ldg(&pr->ABx), __ldg(&pr->ABy), __ldg(&pr->ABz), sink);

      if (fa != fb && active) {      // a == b (same shell): one direction only
#pragma unroll
        for (int k = 0; k < NB; ++k) atomicAdd(Gc + (int64_t)(fb + k) * p.ld, Gb[k]);
      }
    }
  }
  if (cur_fa >= 0 && active) {
#pragma unroll
    for (int i = 0; i < NA; ++i) atomicAdd(Gc + (int64_t)(cur_fa + i) * p.ld, Ga[i]);
  }
}

template <int LA, int LB>
__global__ void __launch_bounds__(128) k_debug_A(const PrimPair* prims, int nprim, double ABx, double ABy, double ABz,
                                                 const double* pts, int64_t n, const double* boys_tab, double* out, bool transpose) {
  constexpr int NA = ncart(LA), NB = ncart(LB), L = LA + LB;
  const int64_t g = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= n) return;
  double acc[nlev(LA, L)];
  theta_contracted<LA, LB>(prims, nprim, pts[3 * g], pts[3 * g + 1], pts[3 * g + 2], boys_tab, acc);
  double blk[NA * NB];
  StoreSink<LA, LB> sink{blk};
  HrrNode<LA, LB, 0, 0, 0, L>::run(acc, ABx, ABy, ABz, sink);
  double* o = out + g * NA * NB;
#pragma unroll
  for (int i = 0; i < NA; ++i)
#pragma unroll
    for (int k = 0; k < NB; ++k) o[transpose ? k * NA + i : i * NB + k] = blk[i * NB + k];
}

template <int LA, int LB>
cudaError_t launch_class(const IntParams& p, cudaStream_t s) {
  if (p.ntiles > 0 && p.pend > p.pbeg) k_integrals<LA, LB><<<p.ntiles, kTile, 0, s>>>(p);
  return cudaGetLastError();
}
template <int LA, int LB>
cudaError_t launch_dbgA(bool tr, const PrimPair* prims, int nprim, double ABx, double ABy, double ABz, const double* pts, int64_t n,
                        const double* boys, double* out, cudaStream_t s) {
  if (n > 0) k_debug_A<LA, LB><<<(unsigned)((n + 127) / 128), 128, 0, s>>>(prims, nprim, ABx, ABy, ABz, pts, n, boys, out, tr);
  return cudaGetLastError();
}

#define SNK_DECLARE_CLASS(LA, LB)                                                                                              \
  cudaError_t launch_class_##LA##LB(const IntParams& p, cudaStream_t s);                                                       \
  cudaError_t launch_dbgA_##LA##LB(bool tr, const PrimPair* prims, int nprim, double ABx, double ABy, double ABz,               \
                                   const double* pts, int64_t n, const double* boys, double* out, cudaStream_t s);
#define SNK_DEFINE_CLASS(LA, LB)                                                                                               \
  cudaError_t launch_class_##LA##LB(const IntParams& p, cudaStream_t s) { return launch_class<LA, LB>(p, s); }                 \
  cudaError_t launch_dbgA_##LA##LB(bool tr, const PrimPair* prims, int nprim, double ABx, double ABy, double ABz,               \
                                   const double* pts, int64_t n, const double* boys, double* out, cudaStream_t s) {            \
    return launch_dbgA<LA, LB>(tr, prims, nprim, ABx, ABy, ABz, pts, n, boys, out, s);                                         \
  }

}  // namespace snk
