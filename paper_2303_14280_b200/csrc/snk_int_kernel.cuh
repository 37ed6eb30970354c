// snk_int_kernel.cuh -- integral-contraction kernel (row a5):  G[nu][g] += sum_{(nu,lam) in V_j} A_{nu,lam}(g) F[lam][g]
// Eq. 38/48 via App. A.  One consumer thread = one grid point, one CTA = one tile of
// up to kTile consecutive points of one batch.  A is never stored.
//
// B200 design (differs from the paper's A100 kernel):
//   * warp-specialised: warps 0..CW-1 are consumers (CW = 8, but 4 for L = 3 and L = 6), warp CW is a producer that walks the tile's V_j bit mask and streams
//     every kept pair unit -- header + primitive pairs (<= 704 B) and the F_b rows of this tile -- into a ring of
//     shared-memory slots with cp.async.bulk (TMA bulk copy) completing on an mbarrier; consumers never touch pair
//     data in global memory, so the recurrences run against broadcast LDS only;
//   * a consumer thread owns NP points of the tile (2 for L <= 1, else 1) and the warps that cover the same points
//     (4 of the 8 consumer warps for L <= 1, 2 for L = 2) split the unit stream dynamically (shared-memory ticket): the
//     point-independent work of a unit is paid once per 32 NP points and one staged unit feeds more resident chains;
//   * the unit list is sorted by (a, b): G_a / F_a stay in registers over a run of units sharing a; G_b goes out with
//     fire-and-forget RED.F64 (coalesced along the slot index);
//   * recurrence intermediates live in registers (compile-time unrolled VRR/HRR, snk_os.cuh).
// Included once per (LA,LB) translation unit.
#pragma once
#include "snk_internal.h"
#include "snk_os.cuh"

namespace snk {

// Work split inside a CTA (one tile of up to kTile points, four consumer warps + one producer warp).
// A consumer thread holds NP = int_npmax points of the tile (lane, lane + 32, ...): everything that does not depend on the grid
// point -- the broadcast LDS of the primitive pairs, the loop and barrier bookkeeping -- is paid once per NP points, and the
// NP recurrences are independent instruction streams.  The tile is therefore covered by G = 4 / NP point groups of NP warps
// each, and the warps of one group share the unit stream: each takes the next unit nobody of its group has taken yet.
#ifndef SNK_NP_L0
#define SNK_NP_L0 2
#endif
#ifndef SNK_NP_L1
#define SNK_NP_L1 2
#endif
#ifndef SNK_NP_L2
#define SNK_NP_L2 1
#endif
#ifndef SNK_NP_L3
#define SNK_NP_L3 1
#endif
__host__ __device__ constexpr int int_npmax(int LA, int LB) {
  const int L = LA + LB;
  return L == 0 ? SNK_NP_L0 : L == 1 ? SNK_NP_L1 : L == 2 ? SNK_NP_L2 : L == 3 ? SNK_NP_L3 : 1;
}
// resident CTAs per SM the register allocation is held to
#ifndef SNK_MB_L0
#define SNK_MB_L0 3
#endif
#ifndef SNK_MB_L1
#define SNK_MB_L1 2
#endif
#ifndef SNK_MB_L2
#define SNK_MB_L2 2
#endif
#ifndef SNK_MB_L4
#define SNK_MB_L4 1
#endif
#ifndef SNK_MB_L3
#define SNK_MB_L3 3
#endif
__host__ __device__ constexpr int int_minblocks(int LA, int LB) {
  const int L = LA + LB;
  return L == 0 ? SNK_MB_L0 : L == 1 ? SNK_MB_L1 : L == 2 ? SNK_MB_L2 : L == 3 ? SNK_MB_L3 : L == 4 ? SNK_MB_L4 : 1;
}
// consumer warps per CTA: NP per point group by default; more (SNK_CW_L*) let a group's unit stream be shared by more
// warps, i.e. more resident point chains per staged unit and per producer warp
#ifndef SNK_CW_L0
#define SNK_CW_L0 8
#endif
#ifndef SNK_CW_L1
#define SNK_CW_L1 8
#endif
#ifndef SNK_CW_L2
#define SNK_CW_L2 8
#endif
#ifndef SNK_CW_L3
#define SNK_CW_L3 4
#endif
#ifndef SNK_CW_L4
#define SNK_CW_L4 8
#endif
#ifndef SNK_CW_L5
#define SNK_CW_L5 8
#endif
#ifndef SNK_CW_L6
#define SNK_CW_L6 4
#endif
__host__ __device__ constexpr int int_cw(int LA, int LB) {
  const int L = LA + LB;
  return L == 0 ? SNK_CW_L0 : L == 1 ? SNK_CW_L1 : L == 2 ? SNK_CW_L2 : L == 3 ? SNK_CW_L3 : L == 4 ? SNK_CW_L4 : L == 5 ? SNK_CW_L5 : SNK_CW_L6;
}
__host__ __device__ constexpr int int_threads(int LA, int LB) { return 32 * int_cw(LA, LB) + 32; }

#ifndef SNK_NS_LB0
#define SNK_NS_LB0 8
#endif
#ifndef SNK_NS_LB1
#define SNK_NS_LB1 8
#endif
__host__ __device__ constexpr int int_nslots(int LA, int LB) { return (LA + LB >= 4 ? 4 : LB == 0 ? SNK_NS_LB0 : LB == 1 ? SNK_NS_LB1 : 8) * int_cw(LA, LB) / 4; }
__host__ __device__ constexpr int int_slot_bytes(int LB) { return kUnitBytes + ncart(LB) * kTile * 8; }
// ring slots, then full[NS] and empty[NS] mbarriers, then the per-group unit counters and the unit count
__host__ __device__ constexpr int int_smem_bytes(int LA, int LB) { return int_nslots(LA, LB) * int_slot_bytes(LB) + 2 * 8 * int_nslots(LA, LB) + 32; }

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "SNK_WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra SNK_DONE_%=;\n"
      "bra SNK_WAIT_%=;\n"
      "SNK_DONE_%=:\n"
      "}\n" ::"r"(bar),
      "r"(parity)
      : "memory");
}
// producer-side wait: try_wait suspends the lane in hardware until the phase completes or the time hint (ns) expires, so the
// waiting producer takes (almost) no issue slots from the consumer warps
__device__ __forceinline__ void mbar_wait_suspend(uint32_t bar, uint32_t parity) {
  uint32_t done;
  do {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n"
        : "=r"(done)
        : "r"(bar), "r"(parity), "r"(1000000u)
        : "memory");
  } while (!done);
}
// non-blocking probe (the consumer issues it one unit ahead, so the barrier round trip overlaps the recurrences)
__device__ __forceinline__ uint32_t mbar_test(uint32_t bar, uint32_t parity) {
  uint32_t done;
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "mbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n"
      "selp.u32 %0, 1, 0, p;\n"
      "}\n"
      : "=r"(done)
      : "r"(bar), "r"(parity)
      : "memory");
  return done;
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst), "l"(src), "r"(bytes),
               "r"(bar)
               : "memory");
}

// ---- consumer side: this warp's share of the unit stream for the points [pbase, pbase + 32 NP) of the tile, NP per thread ----
// s_next: shared counter of the warp's point group (next unit nobody of the group has taken); nunit: units of the tile's stream.
template <int LA, int LB, int NP>
__device__ __forceinline__ void consume_units(const IntParams& p, const unsigned char* smem_int, uint32_t s_full, uint32_t s_empty,
                                              int* s_next, int nunit, const TileRec& tile, int64_t col0, int pbase, int lane) {
  constexpr int NA = ncart(LA), NB = ncart(LB), L = LA + LB;
  constexpr int NS = int_nslots(LA, LB), SLOT = int_slot_bytes(LB);
  int pt[NP], ptc[NP];
  bool act[NP];
  double gx[NP], gy[NP], gz[NP];
#pragma unroll
  for (int s = 0; s < NP; ++s) {
    pt[s] = pbase + 32 * s + lane;
    act[s] = pt[s] < tile.n;
    ptc[s] = act[s] ? pt[s] : tile.n - 1;             // inactive lanes shadow the tile's last point and never write
    const int64_t slot = tile.slot + ptc[s];
    gx[s] = p.gx[slot]; gy[s] = p.gy[slot]; gz[s] = p.gz[slot];
  }
  const double* __restrict__ Fc = p.F + col0;
  double* __restrict__ Gc = p.G + col0;
  const int64_t ld = p.ld;

  int cur_fa = -1;
  int64_t cur_offa = 0;
  double Fa[NP][NA], Ga[NP][NA];
#pragma unroll
  for (int s = 0; s < NP; ++s)
#pragma unroll
    for (int i = 0; i < NA; ++i) { Fa[s][i] = 0.0; Ga[s][i] = 0.0; }

  auto flush_a = [&]() {
#pragma unroll
    for (int s = 0; s < NP; ++s)
      if (act[s]) {
#pragma unroll
        for (int i = 0; i < NA; ++i) atomicAdd(Gc + cur_offa + (int64_t)i * ld + pt[s], Ga[s][i]);
      }
  };

  auto take = [&]() {                                  // next unit of the group's stream
    int u = 0;
    if (lane == 0) u = atomicAdd(s_next, 1);
    return __shfl_sync(0xffffffffu, u, 0);
  };
  int u = take();
  while (u < nunit) {
    const uint32_t sl = (uint32_t)u % NS, phase = ((uint32_t)u / NS) & 1u;
    if (!mbar_test(s_full + 8 * sl, phase)) mbar_wait(s_full + 8 * sl, phase);
    const int unext = take();                          // the shared-memory round trip overlaps this unit's recurrences
    const unsigned char* rec = smem_int + sl * SLOT;
    const int4 h0 = *reinterpret_cast<const int4*>(rec);           // fa, fb, nprim, first
    const int fa = h0.x, fb = h0.y;
    const double2 ab0 = *reinterpret_cast<const double2*>(rec + 16);   // ABx, ABy
    const double ABz = *reinterpret_cast<const double*>(rec + 32);
    const longlong2 off = *reinterpret_cast<const longlong2*>(rec + 48);   // fa * ld, fb * ld
    if (fa != cur_fa) {
      if (cur_fa >= 0) flush_a();
      cur_fa = fa; cur_offa = off.x;
#pragma unroll
      for (int s = 0; s < NP; ++s)
#pragma unroll
        for (int i = 0; i < NA; ++i) { Fa[s][i] = Fc[off.x + (int64_t)i * ld + ptc[s]]; Ga[s][i] = 0.0; }
    }
    double Fb[NP][NB], Gb[NP][NB];
    const double* Fs = reinterpret_cast<const double*>(rec + kUnitBytes);
#pragma unroll
    for (int s = 0; s < NP; ++s)
#pragma unroll
      for (int k = 0; k < NB; ++k) { Fb[s][k] = Fs[k * kTile + ptc[s]]; Gb[s][k] = 0.0; }

    double acc[NP][nlev(LA, L)];
    theta_contracted<LA, LB, NP, true>(reinterpret_cast<const PrimPair*>(rec + 64), h0.z, gx, gy, gz, p.boys, acc);
#pragma unroll
    for (int s = 0; s < NP; ++s) {
      ContractSink<LA, LB> sink{Fa[s], Fb[s], Ga[s], Gb[s]};
      HrrNode<LA, LB, 0, 0, 0, L>::run(acc[s], ab0.x, ab0.y, ABz, sink);
    }

    __syncwarp();
    if (lane == 0) mbar_arrive(s_empty + 8 * sl);                  // slot may be refilled
    if (fa != fb) {                                                // a == b (same shell): one direction only
#pragma unroll
      for (int s = 0; s < NP; ++s)
        if (act[s]) {
#pragma unroll
          for (int k = 0; k < NB; ++k) atomicAdd(Gc + off.y + (int64_t)k * ld + pt[s], Gb[s][k]);
        }
    }
    u = unext;
  }
  if (cur_fa >= 0) flush_a();
}

template <int LA, int LB>
__global__ void __launch_bounds__(int_threads(LA, LB), int_minblocks(LA, LB)) k_integrals(IntParams p) {
  constexpr int NB = ncart(LB);
  constexpr int NPM = int_npmax(LA, LB), CW = int_cw(LA, LB);       // points per thread, consumer warps per CTA
  constexpr int WPG = CW * NPM * 32 / kTile;                         // consumer warps per point group
  static_assert(WPG >= 1 && WPG * (kTile / (32 * NPM)) == CW, "consumer warps: a whole number per point group");
  constexpr int NS = int_nslots(LA, LB), NG = NS / 2, SLOT = int_slot_bytes(LB);
  static_assert(NPM == 1 || NPM == 2 || NPM == 4, "points per thread");
  extern __shared__ __align__(128) unsigned char smem_int[];
  const uint32_t s_base = smem_u32(smem_int);
  const uint32_t s_full = s_base + NS * SLOT, s_empty = s_full + NS * 8;
  int* s_ctr = reinterpret_cast<int*>(smem_int + NS * SLOT + 16 * NS);   // [0..3] next unit of point group g, [4] units of the tile

  const TileRec tile = p.tiles[blockIdx.x];
  const int t = threadIdx.x, warp = t >> 5, lane = t & 31;
  const uint32_t* __restrict__ mask = p.vmask + (int64_t)tile.batch * p.vstride;
  const int w0 = p.pbeg >> 5, w1 = (p.pend + 31) >> 5;
  auto class_bits = [&](int w) {                           // V_j bits of word w that belong to this class
    uint32_t word = __ldg(mask + w);
    if (w == w0) word &= 0xffffffffu << (p.pbeg & 31);
    if (w == w1 - 1 && (p.pend & 31)) word &= 0xffffffffu >> (32 - (p.pend & 31));
    return word;
  };
  // length of the tile's unit stream
  int cnt = 0;
  for (int w = w0 + t; w < w1; w += int_threads(LA, LB)) cnt += __popc(class_bits(w));
  cnt = __reduce_add_sync(0xffffffffu, cnt);
  if (t < 8) s_ctr[t] = 0;
  __syncthreads();
  if (lane == 0 && cnt) atomicAdd(s_ctr + 4, cnt);
  const int nag = (tile.n + 32 * NPM - 1) / (32 * NPM);    // point groups that own at least one point
  if (t == 0) {
    for (int i = 0; i < NS; ++i) { mbar_init(s_full + 8 * i, 1); mbar_init(s_empty + 8 * i, nag); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  const int nunit = s_ctr[4];
  if (nunit == 0) return;
  const int64_t col0 = tile.slot - p.slot0;

  if (warp == CW) {
    // ------------------------------------------------ producer warp ------------------------------------------------
    const int npad = ((tile.n + 31) >> 5) << 5;
    const uint32_t frow = (uint32_t)npad * 8u;             // bytes of one staged F row
    uint32_t u = 0;                                        // units issued so far
    for (int wb = w0; wb < w1; wb += 32) {
      const int w = wb + lane;
      const uint32_t word = w < w1 ? class_bits(w) : 0u;
      uint32_t any = __ballot_sync(~0u, word != 0u);
      while (any) {
        const int src = __ffs(any) - 1;
        any &= any - 1;
        const uint32_t bits = __shfl_sync(~0u, word, src);
        const int n = __popc(bits);
        const int base_pid = (wb + src) << 5;
        for (int b0 = 0; b0 < n; b0 += NG) {               // NG units per step (half the ring): one lane per unit
          const int cnt_step = min(n, b0 + NG) - b0;
          if (lane >= b0 && lane < b0 + cnt_step) {
            const int pid = base_pid + (int)__fns(bits, 0, lane + 1);
            const UnitMeta m = p.meta[pid];                // in flight while we wait for the slot
            const uint32_t uu = u + (uint32_t)(lane - b0), slot = uu % NS;
            // the slot's previous unit is released by the one warp of every point group that processed it
            if (uu >= NS) mbar_wait_suspend(s_empty + 8 * slot, (uu / NS - 1) & 1);
            const uint32_t nb = 64u + (uint32_t)(m.nprim_first & 0xff) * (uint32_t)kPrimBytes;
            const uint32_t bar = s_full + 8 * slot, dst = s_base + slot * SLOT;
            mbar_arrive_expect_tx(bar, nb + NB * frow);
            bulk_g2s(dst, p.units + (size_t)pid * kUnitBytes, nb, bar);
            const double* __restrict__ Fsrc = p.F + (int64_t)m.fb * p.ld + col0;
#pragma unroll
            for (int k = 0; k < NB; ++k) bulk_g2s(dst + kUnitBytes + k * (kTile * 8), Fsrc + (int64_t)k * p.ld, frow, bar);
          }
          u += (uint32_t)cnt_step;
          __syncwarp();
        }
      }
    }
    return;
  }
  const int grp = warp / WPG, pbase = grp * 32 * NPM;
  if (pbase >= tile.n) return;
  const int need = min(NPM, (tile.n - pbase + 31) >> 5);   // point slots of the group that hold a point (ragged tiles)
  int* s_next = s_ctr + grp;
  if constexpr (NPM == 4) {
    if (need == 4) consume_units<LA, LB, 4>(p, smem_int, s_full, s_empty, s_next, nunit, tile, col0, pbase, lane);
    else if (need == 3) consume_units<LA, LB, 3>(p, smem_int, s_full, s_empty, s_next, nunit, tile, col0, pbase, lane);
    else if (need == 2) consume_units<LA, LB, 2>(p, smem_int, s_full, s_empty, s_next, nunit, tile, col0, pbase, lane);
    else consume_units<LA, LB, 1>(p, smem_int, s_full, s_empty, s_next, nunit, tile, col0, pbase, lane);
  } else if constexpr (NPM == 2) {
    if (need == 2) consume_units<LA, LB, 2>(p, smem_int, s_full, s_empty, s_next, nunit, tile, col0, pbase, lane);
    else consume_units<LA, LB, 1>(p, smem_int, s_full, s_empty, s_next, nunit, tile, col0, pbase, lane);
  } else {
    consume_units<LA, LB, 1>(p, smem_int, s_full, s_empty, s_next, nunit, tile, col0, pbase, lane);
  }
}

template <int LA, int LB>
__global__ void __launch_bounds__(128) k_debug_A(const PrimPair* prims, int nprim, double ABx, double ABy, double ABz,
                                                 const double* pts, int64_t n, const double* boys_tab, double* out, bool transpose) {
  constexpr int NA = ncart(LA), NB = ncart(LB), L = LA + LB;
  const int64_t g = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= n) return;
  const double gx[1] = {pts[3 * g]}, gy[1] = {pts[3 * g + 1]}, gz[1] = {pts[3 * g + 2]};
  double acc1[1][nlev(LA, L)];
  theta_contracted<LA, LB, 1, false>(prims, nprim, gx, gy, gz, boys_tab, acc1);
  double (&acc)[nlev(LA, L)] = acc1[0];
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
  if (p.ntiles > 0 && p.pend > p.pbeg) {
    constexpr int smem = int_smem_bytes(LA, LB);
    static bool attr_set[kMaxDevices] = {};
    if (cudaError_t e = opt_in_smem(k_integrals<LA, LB>, smem, attr_set); e != cudaSuccess) return e;
    k_integrals<LA, LB><<<p.ntiles, int_threads(LA, LB), smem, s>>>(p);
  }
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
