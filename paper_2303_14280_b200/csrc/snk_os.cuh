// snk_os.cuh -- device code of the 3c-CP integral kernel: Boys function + Obara-Saika recursions.
//
// App. A of arXiv 2303.14280, with the readings R1-R4 of DESIGN.md:
//   (A3) seed      Theta^n_0 = pref * F_n(p |P - r_g|^2),  pref = c_a c_b (2 pi / p) exp(-mu |A-B|^2)   (R1)
//   (A1) VRR       Theta^n_{a+1_q} = (P-A)_q Theta^n_a - (P-r_g)_q Theta^{n+1}_a
//                                    + a_q/(2p) (Theta^n_{a-1_q} - Theta^{n+1}_{a-1_q})                  (R3)
//   contraction    Theta^0_a summed over primitive pairs between VRR and HRR              (R4)
//   (A2) HRR       Xi_{a,b+1_q} = Xi_{a+1_q,b} + (A-B)_q Xi_{a,b}, built one b-column at a time and
//                  merged with the F-contraction so that A is never materialised
// Everything is compile-time unrolled (templates + constexpr index maps) so the
// recurrence intermediates live in registers.
#pragma once
#include <cuda_runtime.h>
#include <type_traits>

namespace snk {

__host__ __device__ constexpr int ncart(int l) { return (l + 1) * (l + 2) / 2; }
// index of component (i,j,k) inside level l=i+j+k; order: i from l down to 0, then j from l-i down to 0
__host__ __device__ constexpr int cidx(int i, int j, int k) { return (j + k) * (j + k + 1) / 2 + k; }
// inverse map
__host__ __device__ constexpr int comp_i(int l, int c) {
  int ip = 0;
  while ((ip + 1) * (ip + 2) / 2 <= c) ++ip;
  return l - ip;
}
__host__ __device__ constexpr int comp_k(int l, int c) {
  int ip = l - comp_i(l, c);
  return c - ip * (ip + 1) / 2;
}
__host__ __device__ constexpr int comp_j(int l, int c) { return l - comp_i(l, c) - comp_k(l, c); }
// number of components in levels [la, lb]
__host__ __device__ constexpr int nlev(int la, int lb) {
  int n = 0;
  for (int l = la; l <= lb; ++l) n += ncart(l);
  return n;
}

template <int B, int E, class F>
__device__ __forceinline__ void static_for(F&& f) {
  if constexpr (B < E) {
    f(std::integral_constant<int, B>{});
    static_for<B + 1, E>(f);
  }
}

// ------------------------------------------------------------------------------------------------
// Boys function, Eq. 22, reading R15:
//   x < xmax(L): 8-term Taylor about the nearest node x_i of a Delta = 1/16 grid at the top order m = L
//                (dF_m/dx = -F_{m+1}):  F_L(x) = sum_k [F_{L+k}(x_i)/k!] d^k,  d = x_i - x, |d| <= 1/32,
//                then downward recursion F_{m-1} = (2x F_m + e^{-x})/(2m-1) with
//                e^{-x} = e^{-x_i} e^{d}, e^{d} by its 8-term Taylor series (remainder < 3e-17).
//   x >= xmax(L): F_0 = sqrt(pi/x)/2 and upward F_{m+1} = (2m+1) F_m / (2x); the neglected e^{-x}
//                terms are < 4e-16 relative at xmax(L).
// Table layout (built on the host in snk_api.cu): one table per top order L = 0..kBoysLmax,
//   tab[(L*kBoysRows + i)*kBoysStride + k] = F_{L+k}(x_i)/k!  (k = 0..7),  [8] = e^{-x_i},  [9] = 0,
// so one evaluation is four (L = 0) or five 16-byte loads from an L1-resident 53-66 KB table.
// ------------------------------------------------------------------------------------------------
constexpr int kBoysStride = 10;
constexpr int kBoysLmax = 6;
constexpr double kBoysDelta = 1.0 / 16.0;
constexpr int kBoysRows = 52 * 16 + 2;
__host__ __device__ constexpr double boys_xmax(int L) {
  return L == 0 ? 34.0 : L == 1 ? 38.0 : L == 2 ? 40.0 : L == 3 ? 44.0 : L == 4 ? 46.0 : L == 5 ? 50.0 : 52.0;
}

// far field, x >= xmax(L)
template <int L>
__device__ __forceinline__ void boys_far(double x, double (&F)[L + 1]) {
  // 1/sqrt(x) for 34 <= x < inf: hardware seed (2^-22) + one third-order step; no special cases can occur here
  double y0;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y0) : "d"(x));
  const double e = fma(-x, y0 * y0, 1.0);
  const double r = fma(fma(e, 0.375, 0.5), y0 * e, y0);
  F[0] = 0.88622692545275801365 * r;               // sqrt(pi)/2
  if constexpr (L > 0) {
    const double h = 0.5 * r * r;                  // 1/(2x)
#pragma unroll
    for (int m = 0; m < L; ++m) F[m + 1] = (2 * m + 1) * F[m] * h;
  }
}

// near field, x < xmax(L); tab = base of the whole table set
template <int L>
__device__ __forceinline__ void boys_near(double x, const double* __restrict__ tab, double (&F)[L + 1]) {
  // nearest node without F2I/I2F (the conversion pipe is 4x slower than the FP64 pipe): adding 1.5*2^52 leaves
  // round-to-nearest(16 x) in the low mantissa bits
  const double tm = fma(x, 16.0, 6755399441055744.0);
  const int i = __double2loint(tm);
  const double d = fma(tm - 6755399441055744.0, kBoysDelta, -x);
  const double2* __restrict__ row = reinterpret_cast<const double2*>(tab + ((size_t)L * kBoysRows + i) * kBoysStride);
  const double2 t01 = __ldg(row), t23 = __ldg(row + 1), t45 = __ldg(row + 2), t67 = __ldg(row + 3);
  double s = fma(t67.y, d, t67.x);
  s = fma(s, d, t45.y);
  s = fma(s, d, t45.x);
  s = fma(s, d, t23.y);
  s = fma(s, d, t23.x);
  s = fma(s, d, t01.y);
  F[L] = fma(s, d, t01.x);
  if constexpr (L > 0) {
    const double2 e = __ldg(row + 4);
    double q = 1.0 / 5040.0;
    q = fma(q, d, 1.0 / 720.0);
    q = fma(q, d, 1.0 / 120.0);
    q = fma(q, d, 1.0 / 24.0);
    q = fma(q, d, 1.0 / 6.0);
    q = fma(q, d, 0.5);
    q = fma(q, d, 1.0);
    q = fma(q, d, 1.0);
    const double ex = e.x * q;
    const double x2 = x + x;
#pragma unroll
    for (int m = L; m >= 1; --m) F[m - 1] = fma(x2, F[m], ex) * (1.0 / (2 * m - 1));
  }
}

// Seeds (A3, R1) Theta^n_0 = pref F_n(x), n = 0..L, with the prefactor folded into the Boys evaluation.  The kernel carries
// x2 = 2x.  Far field: with r = 1/sqrt(x2), Theta^0_0 = cfar2 r (cfar2 = pref sqrt(pi/2)), 1/(2x) = r r, and
// Theta^{m+1}_0 = Theta^m_0 (2m+1)/(2x): the factors (2m+1) h are formed off the critical path; near field: pref scales F_L and
// e^{-x} once, the downward recursion is linear.
__host__ __device__ constexpr int boys_x2max_hi(int L) {       // high word of the double 2 xmax(L) (its low word is zero)
  const double v = 2.0 * boys_xmax(L);                         // 68, 76, 80, 88, 92, 100, 104: exact, exponent 6
  return (int)(0x40500000u + (unsigned)((v - 64.0) * 16384.0));  // 1.f * 2^6: mantissa bits (v/64 - 1) * 2^20
}
// x2 >= 2 xmax(L) for a non-negative finite double: an integer compare of the high words (the FP64 pipe is the scarce one)
template <int L>
__device__ __forceinline__ bool is_far(double x2) {
#ifdef SNK_KNOCKOUT_NEAR           // timing experiment only (wrong integrals): what the near-field branch costs
  return true;
#else
  return __double2hiint(x2) >= boys_x2max_hi(L);
#endif
}

template <int L>
__device__ __forceinline__ void seeds_far(double x2, double cfar2, double (&T)[L + 1]) {
  double y0;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y0) : "d"(x2));
  const double e = fma(-x2, y0 * y0, 1.0);
  const double r = fma(fma(e, 0.375, 0.5), y0 * e, y0);
  T[0] = cfar2 * r;
  if constexpr (L > 0) {
    const double h = r * r;                        // 1/(2x)
    T[1] = T[0] * h;
#pragma unroll
    for (int m = 1; m < L; ++m) T[m + 1] = T[m] * ((2 * m + 1) * h);
  }
}
// The same for N independent (primitive pair, point) arguments, written statement by statement across the N streams: the
// warp issues in order, so consecutive instructions must belong to different dependency chains to cover the 8-cycle FP64
// latency (a Newton step per point in sequence would stall on every instruction).
template <int L, int N>
__device__ __forceinline__ void seeds_far_v(const double (&x2)[N], const double (&cfar2)[N], double (&T)[N][L + 1]) {
  double y0[N], e[N], u[N], r[N];
#pragma unroll
  for (int i = 0; i < N; ++i) asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y0[i]) : "d"(x2[i]));
#pragma unroll
  for (int i = 0; i < N; ++i) u[i] = y0[i] * y0[i];
#pragma unroll
  for (int i = 0; i < N; ++i) e[i] = fma(-x2[i], u[i], 1.0);
#pragma unroll
  for (int i = 0; i < N; ++i) u[i] = y0[i] * e[i];
#pragma unroll
  for (int i = 0; i < N; ++i) e[i] = fma(e[i], 0.375, 0.5);
#pragma unroll
  for (int i = 0; i < N; ++i) r[i] = fma(e[i], u[i], y0[i]);
#pragma unroll
  for (int i = 0; i < N; ++i) T[i][0] = cfar2[i] * r[i];
  if constexpr (L > 0) {
    double h[N];
#pragma unroll
    for (int i = 0; i < N; ++i) h[i] = r[i] * r[i];            // 1/(2x)
#pragma unroll
    for (int i = 0; i < N; ++i) T[i][1] = T[i][0] * h[i];
#pragma unroll
    for (int m = 1; m < L; ++m) {
#pragma unroll
      for (int i = 0; i < N; ++i) T[i][m + 1] = T[i][m] * ((2 * m + 1) * h[i]);
    }
  }
}
// the same with the hardware seed y0 ~ 1/sqrt(x2) already formed (it is issued before the far/near vote, off the critical path)
template <int L, int N>
__device__ __forceinline__ void seeds_far_v_y0(const double (&x2)[N], const double (&y0)[N], const double (&cfar2)[N], double (&T)[N][L + 1]) {
  double e[N], u[N], r[N];
#pragma unroll
  for (int i = 0; i < N; ++i) u[i] = y0[i] * y0[i];
#pragma unroll
  for (int i = 0; i < N; ++i) e[i] = fma(-x2[i], u[i], 1.0);
#pragma unroll
  for (int i = 0; i < N; ++i) u[i] = y0[i] * e[i];
#pragma unroll
  for (int i = 0; i < N; ++i) e[i] = fma(e[i], 0.375, 0.5);
#pragma unroll
  for (int i = 0; i < N; ++i) r[i] = fma(e[i], u[i], y0[i]);
#pragma unroll
  for (int i = 0; i < N; ++i) T[i][0] = cfar2[i] * r[i];
  if constexpr (L > 0) {
    double h[N];
#pragma unroll
    for (int i = 0; i < N; ++i) h[i] = r[i] * r[i];
#pragma unroll
    for (int i = 0; i < N; ++i) T[i][1] = T[i][0] * h[i];
#pragma unroll
    for (int m = 1; m < L; ++m) {
#pragma unroll
      for (int i = 0; i < N; ++i) T[i][m + 1] = T[i][m] * ((2 * m + 1) * h[i]);
    }
  }
}
template <int L>
__device__ __forceinline__ void seeds_near(double x, double pref, const double* __restrict__ tab, double (&T)[L + 1]) {
  const double tm = fma(x, 16.0, 6755399441055744.0);
  const int i = __double2loint(tm);
  const double d = fma(tm - 6755399441055744.0, kBoysDelta, -x);
  const double2* __restrict__ row = reinterpret_cast<const double2*>(tab + ((size_t)L * kBoysRows + i) * kBoysStride);
  const double2 t01 = __ldg(row), t23 = __ldg(row + 1), t45 = __ldg(row + 2), t67 = __ldg(row + 3);
  double s = fma(t67.y, d, t67.x);
  s = fma(s, d, t45.y);
  s = fma(s, d, t45.x);
  s = fma(s, d, t23.y);
  s = fma(s, d, t23.x);
  s = fma(s, d, t01.y);
  s = fma(s, d, t01.x);
  T[L] = s * pref;
  if constexpr (L > 0) {
    const double2 e = __ldg(row + 4);
    const double ep = e.x * pref;
    double q = 1.0 / 5040.0;
    q = fma(q, d, 1.0 / 720.0);
    q = fma(q, d, 1.0 / 120.0);
    q = fma(q, d, 1.0 / 24.0);
    q = fma(q, d, 1.0 / 6.0);
    q = fma(q, d, 0.5);
    q = fma(q, d, 1.0);
    q = fma(q, d, 1.0);
    const double ex = ep * q;
    const double x2 = x + x;
#pragma unroll
    for (int m = L; m >= 1; --m) T[m - 1] = fma(x2, T[m], ex) * (1.0 / (2 * m - 1));
  }
}
template <int L>
__device__ __forceinline__ void seeds(double x2, double pref, double cfar2, const double* __restrict__ tab, double (&T)[L + 1]) {
  if (!is_far<L>(x2)) seeds_near<L>(0.5 * x2, pref, tab, T);
  else seeds_far<L>(x2, cfar2, T);
}

// per-lane dispatch (test hooks, divergent warps)
template <int L>
__device__ __forceinline__ void boys(double x, const double* __restrict__ tab, double (&F)[L + 1]) {
  if (x < boys_xmax(L)) boys_near<L>(x, tab, F);
  else boys_far<L>(x, F);
}

// ------------------------------------------------------------------------------------------------
// One primitive pair: everything that does not depend on the grid point.
// ------------------------------------------------------------------------------------------------
struct __align__(16) PrimPair {
  double p2;       // 2 (zeta_a + zeta_b): the kernel works with 2x = p2 |P - r_g|^2, whose inverse square root gives 1/(2x) in one multiply
  double inv2p;    // 1 / (2p)
  double Px, Py, Pz;
  double PAx, PAy, PAz;   // P - A, A = centre of the shell that carries the VRR (first of the pair, l_a >= l_b)
  double pref;     // c_a c_b (2 pi / p) exp(-zeta_a zeta_b / p |A-B|^2)
  double cfar2;    // pref * sqrt(pi/2): Theta^0_0 = cfar2 / sqrt(2x) in the far field
};
static_assert(sizeof(PrimPair) == 80, "PrimPair layout");

// offset of level l inside the flat VRR work array: level l holds Theta^n_a, |a| = l, n = 0..L-l, as [n][comp]
__host__ __device__ constexpr int vrr_off(int L, int l) {
  int o = 0;
  for (int m = 0; m < l; ++m) o += ncart(m) * (L - m + 1);
  return o;
}

// VRR (A1): acc[] (levels LA..L of Theta^0, contracted, R4) += this primitive pair's values.
// th0[n] = Theta^n_0 (seed already scaled by pref), n = 0..L.  The work array is flat with compile-time
// offsets; after unrolling the code is straight-line, so ptxas keeps only live values in registers.
template <int LA, int L>
__device__ __forceinline__ void vrr_accumulate(const double (&th0)[L + 1], double PAx, double PAy, double PAz, double PCx,
                                               double PCy, double PCz, double inv2p, double (&acc)[nlev(LA, L)]) {
  double v[vrr_off(L, L + 1)];
#pragma unroll
  for (int n = 0; n <= L; ++n) v[n] = th0[n];
  if constexpr (LA == 0) acc[0] += th0[0];
  static_for<0, L>([&](auto lc) {
    constexpr int l = decltype(lc)::value;                 // build level l+1 from levels l and l-1
    constexpr int nc1 = ncart(l + 1), nc0 = ncart(l), ncm = l > 0 ? ncart(l - 1) : 1;
    constexpr int o1 = vrr_off(L, l + 1), o0 = vrr_off(L, l), om = l > 0 ? vrr_off(L, l - 1) : 0;
    static_for<0, L - l>([&](auto nn) {
      constexpr int n = decltype(nn)::value;
      static_for<0, nc1>([&](auto cc) {
        constexpr int c = decltype(cc)::value;
        constexpr int i = comp_i(l + 1, c), j = comp_j(l + 1, c), k = comp_k(l + 1, c);
        constexpr int q = i > 0 ? 0 : (j > 0 ? 1 : 2);          // lower along the first non-zero direction
        constexpr int li = i - (q == 0), lj = j - (q == 1), lk = k - (q == 2);
        constexpr int cl = cidx(li, lj, lk);
        constexpr int aq = q == 0 ? li : (q == 1 ? lj : lk);     // a_q: quantum before raising
        const double PAq = q == 0 ? PAx : (q == 1 ? PAy : PAz);
        const double PCq = q == 0 ? PCx : (q == 1 ? PCy : PCz);
        if constexpr (l + 1 == L) {
          // top level: the value feeds nothing but the contraction sum (R4), so its terms go straight into acc
          double a = fma(PAq, v[o0 + n * nc0 + cl], acc[nlev(LA, l) + c]);
          a = fma(-PCq, v[o0 + (n + 1) * nc0 + cl], a);
          if constexpr (aq > 0) {
            constexpr int cll = cidx(li - (q == 0), lj - (q == 1), lk - (q == 2));
            a = fma((double)aq * inv2p, v[om + n * ncm + cll] - v[om + (n + 1) * ncm + cll], a);
          }
          acc[nlev(LA, l) + c] = a;
        } else {
          double t = fma(PAq, v[o0 + n * nc0 + cl], -PCq * v[o0 + (n + 1) * nc0 + cl]);
          if constexpr (aq > 0) {
            constexpr int cll = cidx(li - (q == 0), lj - (q == 1), lk - (q == 2));
            t = fma((double)aq * inv2p, v[om + n * ncm + cll] - v[om + (n + 1) * ncm + cll], t);
          }
          v[o1 + n * nc1 + c] = t;
          if constexpr (n == 0 && l + 1 >= LA) acc[nlev(LA, l) + c] += t;
        }
      });
    });
  });
}

// HRR (A2) tree, column by column, merged with the two contractions of Eq. 38 (both directions of the
// unordered pair, R8):   Ga[i] += A[i,b] Fb[b]     Gb[b] += sum_i A[i,b] Fa[i].
// W holds (a | b_partial) for a-levels LA..LTOP.
template <int LA, int LB, int BX, int BY, int BZ, int LTOP>
struct HrrNode {
  static constexpr int NA = ncart(LA);
  template <class Sink>
  static __device__ __forceinline__ void run(const double (&W)[nlev(LA, LTOP)], double ABx, double ABy, double ABz, Sink& sink) {
    if constexpr (BX + BY + BZ == LB) {
      static_assert(LTOP == LA, "HRR bookkeeping");
      sink.template column<cidx(BX, BY, BZ)>(W);
    } else {
      if constexpr (BY == 0 && BZ == 0) shift<0, BX + 1, BY, BZ>(W, ABx, ABx, ABy, ABz, sink);
      if constexpr (BZ == 0) shift<1, BX, BY + 1, BZ>(W, ABy, ABx, ABy, ABz, sink);
      shift<2, BX, BY, BZ + 1>(W, ABz, ABx, ABy, ABz, sink);
    }
  }
  template <int Q, int NX, int NY, int NZ, class Sink>
  static __device__ __forceinline__ void shift(const double (&W)[nlev(LA, LTOP)], double ABq, double ABx, double ABy, double ABz,
                                               Sink& sink) {
    double W2[nlev(LA, LTOP - 1)];
    static_for<LA, LTOP>([&](auto lc) {
      constexpr int l = decltype(lc)::value;
      static_for<0, ncart(l)>([&](auto cc) {
        constexpr int c = decltype(cc)::value;
        constexpr int i = comp_i(l, c), j = comp_j(l, c), k = comp_k(l, c);
        constexpr int cu = cidx(i + (Q == 0), j + (Q == 1), k + (Q == 2));    // a + 1_q, level l+1
        W2[nlev(LA, l - 1) + c] = fma(ABq, W[nlev(LA, l - 1) + c], W[nlev(LA, l) + cu]);
      });
    });
    HrrNode<LA, LB, NX, NY, NZ, LTOP - 1>::run(W2, ABx, ABy, ABz, sink);
  }
};

// Sink used by the build: contracts each finished column with F.
template <int LA, int LB>
struct ContractSink {
  static constexpr int NA = ncart(LA), NB = ncart(LB);
  const double (&Fa)[NA];
  const double (&Fb)[NB];
  double (&Ga)[NA];
  double (&Gb)[NB];
  template <int CB>
  __device__ __forceinline__ void column(const double (&col)[NA]) {
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < NA; ++i) {
      Ga[i] = fma(col[i], Fb[CB], Ga[i]);
      s = fma(col[i], Fa[i], s);
    }
    Gb[CB] += s;
  }
};

// Sink used by the test hook: stores the A block.
template <int LA, int LB>
struct StoreSink {
  static constexpr int NA = ncart(LA), NB = ncart(LB);
  double* out;   // [NA*NB] row-major for this thread
  template <int CB>
  __device__ __forceinline__ void column(const double (&col)[NA]) {
#pragma unroll
    for (int i = 0; i < NA; ++i) out[i * NB + CB] = col[i];
  }
};

// Contracted Theta^0 (levels LA..LA+LB) of one shell pair (unit) at NP grid points held by this thread.  pp points at
// the unit's primitive pairs: shared memory in the build kernel (every lane reads the same address: broadcast), global
// in the test hook.  NP = 2 gives two independent recurrence streams per thread (the kernel is latency bound) and
// halves the per-point cost of everything that does not depend on the point.
// WARP: all 32 lanes call together; when every point of the warp is in the far field of a primitive pair (the common
// case in the paper-shaped workloads) the Boys function runs without table loads or branches.
#ifndef SNK_KP2_MAXL
#define SNK_KP2_MAXL 1
#endif
#ifndef SNK_KP2_MAXNP
#define SNK_KP2_MAXNP 1
#endif
template <int LA, int LB, int NP, bool WARP>
__device__ __forceinline__ void theta_contracted(const PrimPair* __restrict__ pp, int nprim, const double (&gx)[NP], const double (&gy)[NP],
                                                 const double (&gz)[NP], const double* __restrict__ boys_tab,
                                                 double (&acc)[NP][nlev(LA, LA + LB)]) {
  constexpr int L = LA + LB;
  // KP primitive pairs are advanced together: with the NP points that is KP*NP independent dependency chains per thread
  // (the FP64 pipe has an 8-cycle latency, a warp issues in order); the far-field vote is taken once for the group.
  constexpr int KP = (WARP && L <= SNK_KP2_MAXL && NP <= SNK_KP2_MAXNP) ? 2 : 1;
#pragma unroll
  for (int s = 0; s < NP; ++s)
#pragma unroll
    for (int i = 0; i < nlev(LA, L); ++i) acc[s][i] = 0.0;

  auto step = [&](auto kpc, int k) {
    constexpr int K = decltype(kpc)::value, N = K * NP;
    double2 q0[K], q1[K], q2[K];
    double PCx[N], PCy[N], PCz[N], x[N], th0[N][L + 1];
#pragma unroll
    for (int j = 0; j < K; ++j) {
      const double2* __restrict__ q = reinterpret_cast<const double2*>(pp + k + j);
      q0[j] = q[0]; q1[j] = q[1]; q2[j] = q[2];     // (p2, inv2p) (Px, Py) (Pz, PAx)
    }
#pragma unroll
    for (int j = 0; j < K; ++j)
#pragma unroll
      for (int s = 0; s < NP; ++s) { PCx[j * NP + s] = q1[j].x - gx[s]; PCy[j * NP + s] = q1[j].y - gy[s]; PCz[j * NP + s] = q2[j].x - gz[s]; }
#pragma unroll
    for (int i = 0; i < N; ++i) x[i] = PCz[i] * PCz[i];
#pragma unroll
    for (int i = 0; i < N; ++i) x[i] = fma(PCy[i], PCy[i], x[i]);
#pragma unroll
    for (int i = 0; i < N; ++i) x[i] = fma(PCx[i], PCx[i], x[i]);
#pragma unroll
    for (int i = 0; i < N; ++i) x[i] *= q0[i / NP].x;
    // L <= 1: the hardware seed of 1/sqrt(2x) is issued before the far/near vote, so that its latency overlaps the vote's
    // (measured: ss and ps -1.5 %, pp and above +1 %, hence the condition); near-field lanes do not use it
    constexpr bool HOIST = WARP && L <= 1;
    [[maybe_unused]] double y0[HOIST ? N : 1];
    if constexpr (HOIST) {
#pragma unroll
      for (int i = 0; i < N; ++i) asm volatile("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y0[i]) : "d"(x[i]));
    }
    bool far = true;                                  // x[] holds 2x (p2 = 2p)
#pragma unroll
    for (int i = 0; i < N; ++i) far = far && is_far<L>(x[i]);
    bool allfar = false;
    if constexpr (WARP) allfar = __all_sync(0xffffffffu, far);
    double2 q4[K];                                    // (pref, cfar2)
#pragma unroll
    for (int j = 0; j < K; ++j) q4[j] = reinterpret_cast<const double2*>(pp + k + j)[4];
    if (allfar) {
      double cf[N];
#pragma unroll
      for (int i = 0; i < N; ++i) cf[i] = q4[i / NP].y;
      if constexpr (HOIST) seeds_far_v_y0<L, N>(x, y0, cf, th0);
      else seeds_far_v<L, N>(x, cf, th0);
    } else {
      // chain by chain: a chain whose 32 points are all far still runs without branches or table loads
#pragma unroll
      for (int i = 0; i < N; ++i) {
        bool cf = is_far<L>(x[i]);
        if constexpr (WARP) cf = __all_sync(0xffffffffu, cf);
        if (cf) seeds_far<L>(x[i], q4[i / NP].y, th0[i]);
        else seeds<L>(x[i], q4[i / NP].x, q4[i / NP].y, boys_tab, th0[i]);
      }
    }
#pragma unroll
    for (int j = 0; j < K; ++j) {
      if constexpr (L == 0) {
#pragma unroll
        for (int s = 0; s < NP; ++s) acc[s][0] += th0[j * NP + s][0];
      } else {
        const double2 q3 = reinterpret_cast<const double2*>(pp + k + j)[3];   // (PAy, PAz)
#pragma unroll
        for (int s = 0; s < NP; ++s)
          vrr_accumulate<LA, L>(th0[j * NP + s], q2[j].y, q3.x, q3.y, PCx[j * NP + s], PCy[j * NP + s], PCz[j * NP + s], q0[j].y, acc[s]);
      }
    }
  };
  int k = 0;
  if constexpr (KP > 1) {
#pragma unroll 1
    for (; k + KP <= nprim; k += KP) step(std::integral_constant<int, KP>{}, k);
  }
  if constexpr (WARP && KP == 1) {
    // the build kernel never sees a unit without primitive pairs (such units are not in V_j): no entry test
#pragma unroll 1
    do { step(std::integral_constant<int, 1>{}, k); } while (++k < nprim);
  } else {
#pragma unroll 1
    for (; k < nprim; ++k) step(std::integral_constant<int, 1>{}, k);
  }
}

}  // namespace snk
