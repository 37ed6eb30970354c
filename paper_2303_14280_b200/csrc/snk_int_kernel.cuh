// snk_int_kernel.cuh -- integral-contraction kernel (row a5):  G[nu][g] += sum_{(nu,lam) in V_j} A_{nu,lam}(g) F[lam][g]
// Eq. 38/48 via App. A.  One consumer thread = NP grid points (PAPER.md:490 has one), one CTA = one tile of
// up to kTile consecutive points of one batch.  A is never stored.
//
// B200 design (differs from the paper's A100 kernel):
//   * the V_j bit masks are expanded once per super-batch into per-(batch, class) unit-id lists (k_vlist); the warps of a tile
//     that cover the same points (a point group: the 8 warps for s-s, the 4 warps for L = 1, 2 of 4 for L = 2, 3) take the list's
//     entries round robin; when a launch has few tiles, several CTAs share a tile and split its list the same way;
//   * every warp streams ITS units -- header + primitive pairs (<= 704 B) and the F_b row segments of its points -- through a
//     private ring of D shared-memory slots with 16-byte cp.async copies, one commit group per unit: the warp refills a slot as
//     soon as it has finished the unit in it, D units ahead, so the recurrences run against broadcast LDS only and never wait
//     for global memory.  No producer warp (a ninth warp costs every thread of the CTA a quarter of its registers: CTAs are
//     allocated in warp pairs), no tickets, no barrier shared between warps.  (Bulk copies completing on mbarriers were
//     measured first: one elected lane pays ~60 instructions per unit for the uniform-register set-up of 1 + ncart(l_b) copies;
//     the per-lane 16-byte copies cost a fifth of that and need no barrier objects.);
//   * a thread owns NP points of the tile (4 for L <= 1, 2 for L = 2, 3, else 1): the point-independent work of a unit is paid
//     once per 32 NP points and the NP recurrences are independent instruction streams;
//   * the unit list is sorted by (a, b): G_a / F_a stay in registers over a run of units sharing a; G_b goes out with
//     fire-and-forget RED.F64 (coalesced along the slot index);
//   * recurrence intermediates live in registers (compile-time unrolled VRR/HRR, snk_os.cuh).
// Included once per (LA,LB) translation unit.
#pragma once
#include "snk_internal.h"
#include "snk_os.cuh"

namespace snk {

// Work split inside a CTA (one tile of up to kTile points, CW warps).
// A thread holds NP = int_npmax points of the tile (lane, lane + 32, ...): everything that does not depend on the grid
// point -- the broadcast LDS of the primitive pairs, the loop and copy bookkeeping -- is paid once per NP points, and the
// NP recurrences are independent instruction streams.  The tile is therefore covered by 4 / NP point groups of
// WPG = CW NP / 4 warps each, and the warps of one group split the unit list round robin.
#ifndef SNK_NP_L0
#define SNK_NP_L0 4
#endif
#ifndef SNK_NP_L1
#define SNK_NP_L1 4
#endif
#ifndef SNK_NP_L2
#define SNK_NP_L2 2
#endif
#ifndef SNK_NP_L3
#define SNK_NP_L3 2
#endif
__host__ __device__ constexpr int int_npmax(int LA, int LB) {
  const int L = LA + LB;
  return L == 0 ? SNK_NP_L0 : L == 1 ? SNK_NP_L1 : L == 2 ? SNK_NP_L2 : L == 3 ? SNK_NP_L3 : 1;
}
// resident CTAs per SM the register allocation is held to (8 warps per CTA: 2 CTAs = 4 warps per sub-partition = 128 registers)
#ifndef SNK_MB_L0
#define SNK_MB_L0 2
#endif
#ifndef SNK_MB_L1
#define SNK_MB_L1 3
#endif
#ifndef SNK_MB_L2
#define SNK_MB_L2 3
#endif
#ifndef SNK_MB_L3
#define SNK_MB_L3 2
#endif
#ifndef SNK_MB_L4
#define SNK_MB_L4 1
#endif
__host__ __device__ constexpr int int_minblocks(int LA, int LB) {
  const int L = LA + LB;
  return L == 0 ? SNK_MB_L0 : L == 1 ? SNK_MB_L1 : L == 2 ? SNK_MB_L2 : L == 3 ? SNK_MB_L3 : L == 4 ? SNK_MB_L4 : 1;
}
// warps per CTA (all of them consume): NP per point group at least; more (SNK_CW_L*) let a group's unit stream be shared by
// more warps, i.e. more resident point chains per staged unit
#ifndef SNK_CW_L0
#define SNK_CW_L0 8
#endif
#ifndef SNK_CW_L1
#define SNK_CW_L1 4
#endif
#ifndef SNK_CW_L2
#define SNK_CW_L2 4
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
__host__ __device__ constexpr int int_threads(int LA, int LB) { return 32 * int_cw(LA, LB); }

// F_a of the current a-run: held in registers (0) or re-read through L1 when the unit's recurrences are done (1); the second
// takes ncart(l_a) NP doubles off the register budget of the primitive loop
#ifndef SNK_FA_RELOAD_L1
#define SNK_FA_RELOAD_L1 0
#endif
__host__ __device__ constexpr bool int_fa_reload(int LA, int LB) { return LA + LB == 1 && SNK_FA_RELOAD_L1 != 0; }
// depth of a warp's prefetch ring (a power of two): units in flight ahead of the one being evaluated
#ifndef SNK_D_L0
#define SNK_D_L0 8
#endif
#ifndef SNK_D_L1
#define SNK_D_L1 4
#endif
#ifndef SNK_D_L2
#define SNK_D_L2 4
#endif
#ifndef SNK_D_LHI
#define SNK_D_LHI 2
#endif
__host__ __device__ constexpr int int_depth(int LA, int LB) { return LA + LB == 0 ? SNK_D_L0 : LA + LB == 1 ? SNK_D_L1 : LA + LB == 2 ? SNK_D_L2 : SNK_D_LHI; }
// one ring slot of a warp: the unit record, then ncart(l_b) row segments of F for the 32 NP points of the warp
__host__ __device__ constexpr int int_slot_bytes(int LB, int NP) { return kUnitBytes + ncart(LB) * 32 * NP * 8; }
// per warp: D slots
__host__ __device__ constexpr int int_smem_bytes(int LA, int LB) { return int_cw(LA, LB) * int_depth(LA, LB) * int_slot_bytes(LB, int_npmax(LA, LB)); }

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void cp16(uint32_t dst, const void* src) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// ---- one warp: its share (entries rnk, rnk + WPG, ... of the list) of the tile's unit stream for the points
// [pbase, pbase + 32 NP) of the tile, NP per thread ----
// FULL: every lane of the warp owns NP points of the tile (no predicates, no clamped indices); ragged groups take FULL = false.
// Row addresses in the F / G slabs are base + row * ld8 with a 32-bit byte stride ld8 (the host keeps ld * 8 < 2^32): one
// 32 x 32 -> 64 bit multiply-add per address.
// The warp takes the list entries rnk, rnk + stride, ... (stride = warps of the point group x CTAs that share the tile).
template <int LA, int LB, int NP, bool FULL>
__device__ __forceinline__ void consume_units(const IntParams& p, const TileRec& tile, const int32_t* __restrict__ list, int cnt,
                                              unsigned char* ring, int pbase, int rnk, int stride, int lane) {
  constexpr int NA = ncart(LA), NB = ncart(LB), L = LA + LB;
  constexpr int D = int_depth(LA, LB), SLOT = int_slot_bytes(LB, int_npmax(LA, LB));
  constexpr uint32_t FROW = 32u * NP * 8u;             // bytes of one staged F row segment
  const int n_my = cnt > rnk ? (cnt - rnk + stride - 1) / stride : 0;
  if (n_my == 0) return;
  const uint32_t s_ring = smem_u32(ring);

  uint32_t pb[NP];                                     // byte offset of this thread's points inside a slab row of the tile
  bool act[NP];
  double gx[NP], gy[NP], gz[NP];
#pragma unroll
  for (int s = 0; s < NP; ++s) {
    const int pt = pbase + 32 * s + lane;
    act[s] = FULL || pt < tile.n;
    const int ptc = act[s] ? pt : tile.n - 1;         // inactive lanes shadow the tile's last point and never write
    pb[s] = (uint32_t)ptc * 8u;
    const int64_t slot = tile.slot + ptc;
    gx[s] = p.gx[slot]; gy[s] = p.gy[slot]; gz[s] = p.gz[slot];
  }
  const int64_t col0 = tile.slot - p.slot0;
  const uint32_t ld8 = (uint32_t)p.ld * 8u;
  const char* __restrict__ Fl = reinterpret_cast<const char*>(p.F + col0);
  char* __restrict__ Gl = reinterpret_cast<char*>(p.G + col0);
  auto F_at = [&](int row, int s) { return *reinterpret_cast<const double*>(Fl + (uint64_t)(uint32_t)row * ld8 + pb[s]); };
  auto G_add = [&](int row, int s, double v) { atomicAdd(reinterpret_cast<double*>(Gl + (uint64_t)(uint32_t)row * ld8 + pb[s]), v); };

  // unit ids and (fb | nprim << 24) of this warp's units [32 w, 32 w + 32): lane i holds unit 32 w + i; two windows in flight
  auto load_win = [&](int wb, int& e, int& m) {
    const int q = wb + lane;
    e = 0; m = 0;
    if (q < n_my) {
      e = __ldg(list + (int64_t)q * stride + rnk);
      const int2 mm = __ldg(reinterpret_cast<const int2*>(&p.meta[e].fb));   // fb, nprim | first << 8
      m = mm.x | (mm.y & 0xff) << 24;
    }
  };
  // stage this warp's k-th unit into slot k % D: 16-byte chunks, lane by lane (a unit record is at most 44 chunks, a row
  // segment of F 16 NP); k >= n_my only closes an (empty) commit group, which keeps "group k = unit k"
  const unsigned char* __restrict__ Ucp = p.units + lane * 16;
  const char* __restrict__ Fcp = Fl + (pbase * 8 + lane * 16);
  const uint32_t dst_lane = s_ring + lane * 16;
  // (no branch on k: the copies are predicated)
  auto issue = [&](int k, int e_w, int m_w) {
    const bool valid = k < n_my;
    const int e = __shfl_sync(0xffffffffu, e_w, k & 31), m = __shfl_sync(0xffffffffu, m_w, k & 31);
    const uint32_t dst = dst_lane + ((uint32_t)k % D) * SLOT;
    const int nb = valid ? 64 + (int)((uint32_t)m >> 24) * kPrimBytes : 0;
    const unsigned char* __restrict__ src = Ucp + (uint64_t)(uint32_t)e * (uint32_t)kUnitBytes;
    if (lane * 16 < nb) cp16(dst, src);
    if (512 + lane * 16 < nb) cp16(dst + 512, src + 512);
    const char* __restrict__ Fsrc = Fcp + (uint64_t)(uint32_t)(m & 0xffffff) * ld8;
#pragma unroll
    for (int k2 = 0; k2 < NB; ++k2)
#pragma unroll
      for (int c = 0; c < NP * 16; c += 32)
        if (valid && c + lane < NP * 16) cp16(dst + kUnitBytes + k2 * FROW + c * 16, Fsrc + (uint64_t)k2 * ld8 + c * 16);
    cp_commit();
  };
  int e0, m0, e1, m1;
  load_win(0, e0, m0);
  load_win(32, e1, m1);
  // units 0 .. D-2 are staged here; unit k+D-1 is staged at the top of iteration k, right after the one __syncwarp of the
  // iteration (every lane is then done with unit k-1, whose slot it takes)
#pragma unroll
  for (int k = 0; k < D - 1; ++k) issue(k, e0, m0);

  int cur_fa = -1;
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
        for (int i = 0; i < NA; ++i) G_add(cur_fa + i, s, Ga[s][i]);
      }
  };

  // windows of 32 units: the id registers move on between windows, not inside the unit loop
#pragma unroll 1
  for (int kw = 0; kw < n_my; kw += 32) {
    const int kend = min(kw + 32, n_my);
#pragma unroll 1
    for (int k = kw; k < kend; ++k) {
      cp_wait<D - 2>();                                            // this thread's copies of unit k have landed ...
      __syncwarp();                                                // ... and so have the other lanes'; all are done with unit k-1
      {
        const int kn = k + D - 1;                                  // kn's window is the current one or the next
        issue(kn, (kn & 32) == (kw & 32) ? e0 : e1, (kn & 32) == (kw & 32) ? m0 : m1);
      }
      const unsigned char* rec = ring + ((uint32_t)k % D) * SLOT;
      const int4 h0 = *reinterpret_cast<const int4*>(rec);         // fa, fb, nprim, first
      const int fa = h0.x, fb = h0.y;
      double ABx = 0.0, ABy = 0.0, ABz = 0.0;
      if constexpr (LB > 0) {
        const double2 ab0 = *reinterpret_cast<const double2*>(rec + 16);
        ABx = ab0.x; ABy = ab0.y; ABz = *reinterpret_cast<const double*>(rec + 32);
      }
      if (fa != cur_fa) {
        if (cur_fa >= 0) flush_a();
        cur_fa = fa;
#pragma unroll
        for (int s = 0; s < NP; ++s)
#pragma unroll
          for (int i = 0; i < NA; ++i) {
            if constexpr (!int_fa_reload(LA, LB)) Fa[s][i] = F_at(fa + i, s);
            Ga[s][i] = 0.0;
          }
      }
      double Fb[NP][NB], Gb[NP][NB];
      const double* Fs = reinterpret_cast<const double*>(rec + kUnitBytes);
#pragma unroll
      for (int s = 0; s < NP; ++s)
#pragma unroll
        for (int k2 = 0; k2 < NB; ++k2) { Fb[s][k2] = Fs[k2 * (32 * NP) + 32 * s + lane]; Gb[s][k2] = 0.0; }

      double acc[NP][nlev(LA, L)];
      theta_contracted<LA, LB, NP, true>(reinterpret_cast<const PrimPair*>(rec + 64), h0.z, gx, gy, gz, p.boys, acc);
      if constexpr (int_fa_reload(LA, LB)) {
#pragma unroll
        for (int s = 0; s < NP; ++s)
#pragma unroll
          for (int i = 0; i < NA; ++i) Fa[s][i] = F_at(cur_fa + i, s);
      }
#pragma unroll
      for (int s = 0; s < NP; ++s) {
        ContractSink<LA, LB> sink{Fa[s], Fb[s], Ga[s], Gb[s]};
        HrrNode<LA, LB, 0, 0, 0, L>::run(acc[s], ABx, ABy, ABz, sink);
      }
      const bool two_way = fa != fb;                               // a == b (same shell): one direction only
#pragma unroll
      for (int s = 0; s < NP; ++s)
#pragma unroll
        for (int k2 = 0; k2 < NB; ++k2)
          if (act[s] && two_way) G_add(fb + k2, s, Gb[s][k2]);
    }
    e0 = e1; m0 = m1;
    load_win(kw + 64, e1, m1);
  }
  if (cur_fa >= 0) flush_a();
}

template <int LA, int LB>
__global__ void __launch_bounds__(int_threads(LA, LB), int_minblocks(LA, LB)) k_integrals(IntParams p) {
  constexpr int NPM = int_npmax(LA, LB), CW = int_cw(LA, LB);       // points per thread, warps per CTA
  constexpr int WPG = CW * NPM * 32 / kTile;                         // warps per point group
  static_assert(WPG >= 1 && WPG * (kTile / (32 * NPM)) == CW, "warps: a whole number per point group");
  constexpr int D = int_depth(LA, LB), SLOT = int_slot_bytes(LB, NPM);
  static_assert((D & (D - 1)) == 0 && D >= 2 && D <= 32, "ring depth");
  static_assert(NPM == 1 || NPM == 2 || NPM == 4, "points per thread");
  extern __shared__ __align__(128) unsigned char smem_int[];

  // p.nsplit CTAs share a tile: CTA `part` takes the part-th contiguous range of the tile's unit list (contiguous, so that the
  // runs of units with the same shell a stay together; G is accumulated with REDs anyway).  The CTAs of a tile have
  // consecutive block indices, run at the same time and read the same F columns: fewer distinct tiles are resident, and the
  // F block of a tile (nbf x 1 KB) is fetched from HBM once and shared through the L2.
  const int tile_id = blockIdx.x / p.nsplit, part = blockIdx.x - tile_id * p.nsplit;
  const TileRec tile = p.tiles[tile_id];
  const int jj = tile.batch - p.b0;
  const int cnt_all = p.vcnt[jj * kNumClasses + p.cls];              // units of this class kept by the tile's batch
  const int lo = (int)((int64_t)cnt_all * part / p.nsplit), cnt = (int)((int64_t)cnt_all * (part + 1) / p.nsplit) - lo;
  if (cnt == 0) return;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int grp = warp / WPG, rnk = warp % WPG, stride = WPG, pbase = grp * 32 * NPM;
  if (pbase >= tile.n) return;
  const int32_t* __restrict__ list = p.vlist + (int64_t)jj * p.vlstride + p.pbeg + lo;
  unsigned char* ring = smem_int + warp * (D * SLOT);
  const int need = min(NPM, (tile.n - pbase + 31) >> 5);   // point slots of the group that hold a point (ragged tiles)
  if (tile.n - pbase >= 32 * NPM) { consume_units<LA, LB, NPM, true>(p, tile, list, cnt, ring, pbase, rnk, stride, lane); return; }
  if constexpr (NPM == 4) {
    if (need == 4) consume_units<LA, LB, 4, false>(p, tile, list, cnt, ring, pbase, rnk, stride, lane);
    else if (need == 3) consume_units<LA, LB, 3, false>(p, tile, list, cnt, ring, pbase, rnk, stride, lane);
    else if (need == 2) consume_units<LA, LB, 2, false>(p, tile, list, cnt, ring, pbase, rnk, stride, lane);
    else consume_units<LA, LB, 1, false>(p, tile, list, cnt, ring, pbase, rnk, stride, lane);
  } else if constexpr (NPM == 2) {
    if (need == 2) consume_units<LA, LB, 2, false>(p, tile, list, cnt, ring, pbase, rnk, stride, lane);
    else consume_units<LA, LB, 1, false>(p, tile, list, cnt, ring, pbase, rnk, stride, lane);
  } else {
    consume_units<LA, LB, 1, false>(p, tile, list, cnt, ring, pbase, rnk, stride, lane);
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
    k_integrals<LA, LB><<<p.ntiles * p.nsplit, int_threads(LA, LB), smem, s>>>(p);
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
