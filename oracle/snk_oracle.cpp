// =====================================================================================
// snk_oracle.cpp  --  CPU ORACLE for the sn-K build.  TEST INFRASTRUCTURE ONLY.
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
// legs may build, link or call this file.  It shares NO code, header, table or constant
// generator with the CUDA path (paper_2303_14280_b200/csrc); neither includes the other.
//
// What it computes (PAPER.md = /root/reference/PAPER.md, arXiv 2303.14280):
//   Phi[g,mu] = phi_mu(r_g)                              Eq. 31, phi per Eq. 13
//   F[g,lam]  = sum_sigma P[lam,sigma] Phi[g,sigma]      Eq. 35, sigma in B_j (Eq. 48)
//   A[g,nu,lam] = int phi_nu phi_lam / |r - r_g| d3r     Eq. 37, analytic
//   G[g,nu]   = w_g sum_lam A[g,nu,lam] F[g,lam]         Eq. 38, (nu,lam) in V_j (Eq. 48)
//   Kt[mu,nu] = sum_g Phi[g,mu] G[g,nu]                  Eq. 39, mu in B_j
//   K         = (Kt + Kt^T)/2                            Eq. 40
// A is evaluated by the McMurchie-Davidson scheme of the paper's Sec. II B, Eqs. 15-24
// in the point-charge limit zeta_c -> infinity (rho -> zeta_p in Eq. 23,
// no (-1)^{l_c}); the GPU path uses Obara-Saika (App. A) -- two independent algorithms.
// Batching / screening follow DESIGN.md readings R8-R13 of Eqs. 41-47.
//
// Style: plain loops in the paper's order and notation; no blocking, fusion or reordering
// beyond what the equations state.  fp64, cross-batch accumulation in long double.
//
// Pins (tests/test_oracle_pins.py, all "-m 'not gpu'"):  Boys vs mpmath; s-type A closed form;
// A vs brute-force 3-D quadrature; Poisson / far-field / derivative relations; collocation vs
// closed-form overlap; K symmetry; sn-K -> analytic (ss|ss) exchange with grid refinement;
// linearity & invariances; screening error <= c*eps.  No function here is "parity unpinned",
// but NO value printed by the paper exists for K, A or F_m, so every pin is a
// closed form / invariant / brute force, not a paper number.
// =====================================================================================
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <limits>
#include <map>
#include <array>
#include <string>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

constexpr double kPi = 3.14159265358979323846264338327950288;
constexpr int kLmax = 3;          // per shell
constexpr int kMaxDepth = 20;     // R13

inline int ncart(int l) { return (l + 1) * (l + 2) / 2; }

struct Shell {
  int atom = 0, l = 0, nprim = 0, foff = 0;
  double A[3] = {0, 0, 0};
  std::vector<double> e, c;
  double rcut = std::numeric_limits<double>::infinity();
};

// Cartesian components in the library's order: i from l down to 0, j from l-i down to 0.
inline void cart_list(int l, int (*out)[3]) {
  int n = 0;
  for (int i = l; i >= 0; --i)
    for (int j = l - i; j >= 0; --j) { out[n][0] = i; out[n][1] = j; out[n][2] = l - i - j; ++n; }
}

// -------------------------------------------------------------------------------------
// Boys function F_m(x) = int_0^1 t^{2m} exp(-x t^2) dt      Eq. 22
//   x <= 35 : all-positive series  e^{-x} sum_k (2x)^k / [(2m+1)(2m+3)...(2m+2k+1)] at m = mmax,
//             then downward  F_{m-1} = (2x F_m + e^{-x})/(2m-1)
//   x  > 35 : F_0 = (1/2) sqrt(pi/x) erf(sqrt x), then upward  F_{m+1} = ((2m+1) F_m - e^{-x})/(2x)
// -------------------------------------------------------------------------------------
void boys(int mmax, double x, double* F) {
  const double ex = std::exp(-x);
  if (x <= 35.0) {
    double term = 1.0 / (2 * mmax + 1);
    double sum = term;
    for (int k = 1; k < 2000; ++k) {
      term *= 2.0 * x / (2 * mmax + 2 * k + 1);
      sum += term;
      if (term < 1e-18 * sum) break;
    }
    F[mmax] = ex * sum;
    for (int m = mmax; m >= 1; --m) F[m - 1] = (2.0 * x * F[m] + ex) / (2 * m - 1);
  } else {
    F[0] = 0.5 * std::sqrt(kPi / x) * std::erf(std::sqrt(x));
    for (int m = 0; m < mmax; ++m) F[m + 1] = ((2 * m + 1) * F[m] - ex) / (2.0 * x);
  }
}

// -------------------------------------------------------------------------------------
// 1-D Hermite expansion coefficients (E_x)^{t}_{ij}, Eq. 16; the recursion is
// the McMurchie-Davidson one the paper cites (Ref. 96):
//   E^{00}_0 = exp(-mu X_AB^2)
//   E^{i+1,j}_t = E^{ij}_{t-1}/(2p) + X_PA E^{ij}_t + (t+1) E^{ij}_{t+1}
//   E^{i,j+1}_t = E^{ij}_{t-1}/(2p) + X_PB E^{ij}_t + (t+1) E^{ij}_{t+1}
// E[i][j][t], zero outside 0 <= t <= i+j.
// -------------------------------------------------------------------------------------
struct E1D { double v[kLmax + 1][kLmax + 1][2 * kLmax + 2]; };

void hermite_E(int la, int lb, double a, double b, double Ax, double Bx, E1D& E) {
  std::memset(&E, 0, sizeof(E));
  const double p = a + b, mu = a * b / p;
  const double Px = (a * Ax + b * Bx) / p;
  const double XAB = Ax - Bx, XPA = Px - Ax, XPB = Px - Bx;
  E.v[0][0][0] = std::exp(-mu * XAB * XAB);
  for (int i = 0; i < la; ++i)        // raise i with j = 0
    for (int t = 0; t <= i + 1; ++t) {
      double s = XPA * E.v[i][0][t] + (t + 1) * E.v[i][0][t + 1];
      if (t > 0) s += E.v[i][0][t - 1] / (2.0 * p);
      E.v[i + 1][0][t] = s;
    }
  for (int i = 0; i <= la; ++i)       // raise j
    for (int j = 0; j < lb; ++j)
      for (int t = 0; t <= i + j + 1; ++t) {
        double s = XPB * E.v[i][j][t] + (t + 1) * E.v[i][j][t + 1];
        if (t > 0) s += E.v[i][j][t - 1] / (2.0 * p);
        E.v[i][j + 1][t] = s;
      }
}

// One primitive pair's combined Hermite coefficients E_ab^{p~} = prod_i (E_i) (Eq. 16) for all
// component pairs, with the primitive prefactor c_k c_l (2 pi / p) folded in.
struct PrimPair {
  double p, P[3];
  int L;
  // Etuv[(ca*nb + cb)*nherm + h], h indexes (t,u,v) with t<=L,u<=L,v<=L in a dense (L+1)^3 box
  std::vector<double> Etuv;
};

inline int hidx(int L, int t, int u, int v) { return (t * (L + 1) + u) * (L + 1) + v; }

void make_prim_pairs(const Shell& sa, const Shell& sb, std::vector<PrimPair>& out) {
  const int la = sa.l, lb = sb.l, L = la + lb, na = ncart(la), nb = ncart(lb);
  int ca[10][3], cb[10][3];
  cart_list(la, ca); cart_list(lb, cb);
  out.clear();
  for (int k = 0; k < sa.nprim; ++k)
    for (int l = 0; l < sb.nprim; ++l) {
      PrimPair pp;
      const double a = sa.e[k], b = sb.e[l];
      pp.p = a + b; pp.L = L;
      for (int q = 0; q < 3; ++q) pp.P[q] = (a * sa.A[q] + b * sb.A[q]) / pp.p;
      E1D Ex, Ey, Ez;
      hermite_E(la, lb, a, b, sa.A[0], sb.A[0], Ex);
      hermite_E(la, lb, a, b, sa.A[1], sb.A[1], Ey);
      hermite_E(la, lb, a, b, sa.A[2], sb.A[2], Ez);
      const double pref = sa.c[k] * sb.c[l] * 2.0 * kPi / pp.p;
      const int nh = (L + 1) * (L + 1) * (L + 1);
      pp.Etuv.assign((size_t)na * nb * nh, 0.0);
      for (int ia = 0; ia < na; ++ia)
        for (int ib = 0; ib < nb; ++ib)
          for (int t = 0; t <= ca[ia][0] + cb[ib][0]; ++t)
            for (int u = 0; u <= ca[ia][1] + cb[ib][1]; ++u)
              for (int v = 0; v <= ca[ia][2] + cb[ib][2]; ++v)
                pp.Etuv[((size_t)ia * nb + ib) * nh + hidx(L, t, u, v)] =
                    pref * Ex.v[ca[ia][0]][cb[ib][0]][t] * Ey.v[ca[ia][1]][cb[ib][1]][u] * Ez.v[ca[ia][2]][cb[ib][2]][v];
      out.push_back(std::move(pp));
    }
}

// Hermite Coulomb integrals R^0_{tuv} for a point charge at C (Eqs. 20, 21, 24 with zeta_c -> inf):
//   R^n_{000} = (-2p)^n F_n(p |P-C|^2),   R^n_{t+1,u,v} = t R^{n+1}_{t-1,u,v} + (P-C)_x R^{n+1}_{t,u,v}  (same in y, z)
// Rout[hidx(L,t,u,v)] for t+u+v <= L.
void hermite_R(int L, double p, const double* P, const double* C, double* Rout) {
  const double X = P[0] - C[0], Y = P[1] - C[1], Z = P[2] - C[2];
  double Fm[2 * kLmax + 2];
  boys(L, p * (X * X + Y * Y + Z * Z), Fm);
  const int n1 = L + 1;
  // R[n][t][u][v]
  static thread_local std::vector<double> R;
  R.assign((size_t)n1 * n1 * n1 * n1, 0.0);
  auto at = [&](int n, int t, int u, int v) -> double& { return R[(((size_t)n * n1 + t) * n1 + u) * n1 + v]; };
  double f = 1.0;
  for (int n = 0; n <= L; ++n) { at(n, 0, 0, 0) = f * Fm[n]; f *= -2.0 * p; }
  for (int tot = 1; tot <= L; ++tot)                 // total order t+u+v
    for (int t = 0; t <= tot; ++t)
      for (int u = 0; u <= tot - t; ++u) {
        const int v = tot - t - u;
        for (int n = 0; n <= L - tot; ++n) {
          double val;
          if (t > 0)      val = (t > 1 ? (t - 1) * at(n + 1, t - 2, u, v) : 0.0) + X * at(n + 1, t - 1, u, v);
          else if (u > 0) val = (u > 1 ? (u - 1) * at(n + 1, t, u - 2, v) : 0.0) + Y * at(n + 1, t, u - 1, v);
          else            val = (v > 1 ? (v - 1) * at(n + 1, t, u, v - 2) : 0.0) + Z * at(n + 1, t, u, v - 1);
          at(n, t, u, v) = val;
        }
      }
  for (int t = 0; t <= L; ++t)
    for (int u = 0; u <= L - t; ++u)
      for (int v = 0; v <= L - t - u; ++v) Rout[hidx(L, t, u, v)] = at(0, t, u, v);
}

// A block [na x nb] of one contracted shell pair at one point (Eq. 17 in the point-charge limit + contraction).
void A_block(const std::vector<PrimPair>& pps, int na, int nb, const double* C, double* A) {
  for (int i = 0; i < na * nb; ++i) A[i] = 0.0;
  double Rt[(2 * kLmax + 1) * (2 * kLmax + 1) * (2 * kLmax + 1)];
  for (const PrimPair& pp : pps) {
    const int L = pp.L, nh = (L + 1) * (L + 1) * (L + 1);
    for (int h = 0; h < nh; ++h) Rt[h] = 0.0;
    hermite_R(L, pp.p, pp.P, C, Rt);
    for (int ab = 0; ab < na * nb; ++ab) {
      const double* E = &pp.Etuv[(size_t)ab * nh];
      double s = 0.0;
      for (int h = 0; h < nh; ++h) s += E[h] * Rt[h];
      A[ab] += s;
    }
  }
}

// phi_mu(r) for every component of one shell (Eq. 13 + contraction)
void shell_values(const Shell& s, const double* r, double* out) {
  const double x = r[0] - s.A[0], y = r[1] - s.A[1], z = r[2] - s.A[2];
  const double r2 = x * x + y * y + z * z;
  double rad = 0.0;
  for (int k = 0; k < s.nprim; ++k) rad += s.c[k] * std::exp(-s.e[k] * r2);
  int comp[10][3];
  cart_list(s.l, comp);
  for (int i = 0; i < ncart(s.l); ++i)
    out[i] = std::pow(x, comp[i][0]) * std::pow(y, comp[i][1]) * std::pow(z, comp[i][2]) * rad;
}

// R10: cutoff radius on the 0.25-bohr ladder.  eps <= 0 -> infinity.
double shell_rcut(const Shell& s, double eps) {
  if (!(eps > 0.0)) return std::numeric_limits<double>::infinity();
  double zmin = s.e[0];
  for (double z : s.e) zmin = std::min(zmin, z);
  const double rmin = std::sqrt(s.l / (2.0 * zmin));
  for (int n = 1; n < 100000; ++n) {
    const double r = 0.25 * n;
    if (r < rmin) continue;
    double env = 0.0;
    for (int k = 0; k < s.nprim; ++k) env += std::fabs(s.c[k]) * std::exp(-s.e[k] * r * r);
    env *= std::pow(r, s.l);
    if (env < eps) return r;
  }
  return std::numeric_limits<double>::infinity();
}

// R11: rigorous point-independent bound  Atilde_ab >= max_g |A_{mu nu}(g)|, mu in a, nu in b.
double A_bound(const Shell& sa, const Shell& sb) {
  auto sgauss = [](const Shell& s, int k, double& c, double& z) {
    if (s.l == 0) { c = std::fabs(s.c[k]); z = s.e[k]; }
    else { z = 0.5 * s.e[k]; c = std::fabs(s.c[k]) * std::pow(s.l / (std::exp(1.0) * s.e[k]), 0.5 * s.l); }
  };
  double AB2 = 0.0;
  for (int q = 0; q < 3; ++q) AB2 += (sa.A[q] - sb.A[q]) * (sa.A[q] - sb.A[q]);
  double sum = 0.0;
  for (int k = 0; k < sa.nprim; ++k)
    for (int l = 0; l < sb.nprim; ++l) {
      double ca, za, cb, zb;
      sgauss(sa, k, ca, za); sgauss(sb, l, cb, zb);
      const double p = za + zb;
      sum += ca * cb * (2.0 * kPi / p) * std::exp(-(za * zb / p) * AB2);
    }
  return sum;
}

struct Batch {
  std::vector<int64_t> pts;          // indices into the input arrays, input order
  double lo[3], hi[3];               // tight bbox
  std::vector<int> B;                // shells (ascending)
  std::vector<double> PhiTilde;      // per shell of the basis (0 outside B)
  double phitilde = 0.0;
  std::vector<std::array<int, 2>> V; // unordered shell pairs a <= b
  int64_t root[3] = {0, 0, 0};
};

struct Ctx {
  std::vector<Shell> sh;
  int nbf = 0;
  std::vector<int> f2sh;
  // grid
  std::vector<double> pts, w;
  int64_t npts = 0;
  double eps = 0.0, h0 = 6.0;
  int nmax = 2048;
  std::vector<Batch> batches;
  std::vector<double> Abound;        // [nsh*nsh]
  bool extended = false;             // orc_set_extended
  // stats of the last build
  double n_int_contr = 0, n_int_prim = 0, n_pairpoints = 0;
  double t_build = 0;
  std::string err;
};

// R13: lattice-anchored octree.  Recursive, literal.
void split_node(const Ctx& c, const double* lo, const double* hi, std::vector<int64_t>& idx, int depth,
                const int64_t* root, std::vector<Batch>& out) {
  if ((int64_t)idx.size() <= c.nmax || depth >= kMaxDepth) {
    Batch b;
    b.pts = idx;
    for (int q = 0; q < 3; ++q) { b.lo[q] = std::numeric_limits<double>::infinity(); b.hi[q] = -b.lo[q]; b.root[q] = root[q]; }
    for (int64_t i : idx)
      for (int q = 0; q < 3; ++q) { b.lo[q] = std::min(b.lo[q], c.pts[3 * i + q]); b.hi[q] = std::max(b.hi[q], c.pts[3 * i + q]); }
    out.push_back(std::move(b));
    return;
  }
  double mid[3];
  for (int q = 0; q < 3; ++q) mid[q] = 0.5 * (lo[q] + hi[q]);
  std::vector<int64_t> child[8];
  for (int64_t i : idx) {
    const int k = 4 * (c.pts[3 * i + 0] >= mid[0]) + 2 * (c.pts[3 * i + 1] >= mid[1]) + (c.pts[3 * i + 2] >= mid[2]);
    child[k].push_back(i);     // points on a split plane go to the upper child
  }
  idx.clear(); idx.shrink_to_fit();
  for (int k = 0; k < 8; ++k) {
    if (child[k].empty()) continue;
    double clo[3], chi[3];
    for (int q = 0; q < 3; ++q) {
      const bool up = (k >> (2 - q)) & 1;
      clo[q] = up ? mid[q] : lo[q];
      chi[q] = up ? hi[q] : mid[q];
    }
    split_node(c, clo, chi, child[k], depth + 1, root, out);
  }
}

void do_batching(Ctx& c) {
  c.batches.clear();
  std::map<std::array<int64_t, 3>, std::vector<int64_t>> cells;   // lexicographic order of (ix,iy,iz)
  for (int64_t i = 0; i < c.npts; ++i) {
    std::array<int64_t, 3> key;
    for (int q = 0; q < 3; ++q) key[q] = (int64_t)std::floor(c.pts[3 * i + q] / c.h0);
    cells[key].push_back(i);
  }
  for (auto& kv : cells) {
    double lo[3], hi[3];
    for (int q = 0; q < 3; ++q) { lo[q] = (double)kv.first[q] * c.h0; hi[q] = (double)(kv.first[q] + 1) * c.h0; }
    split_node(c, lo, hi, kv.second, 0, kv.first.data(), c.batches);
  }
}

// R10 + R12 (density independent part): B_j, PhiTilde_a(j), phitilde(j)
void do_basis_screen(Ctx& c) {
  const int nsh = (int)c.sh.size();
  for (Shell& s : c.sh) s.rcut = shell_rcut(s, c.eps);
  std::vector<Batch> kept;
  for (Batch& b : c.batches) {
    b.B.clear();
    for (int a = 0; a < nsh; ++a) {
      const Shell& s = c.sh[a];
      double d2 = 0.0;
      for (int q = 0; q < 3; ++q) {
        const double d = std::max(0.0, std::max(b.lo[q] - s.A[q], s.A[q] - b.hi[q]));
        d2 += d * d;
      }
      if (d2 <= s.rcut * s.rcut) b.B.push_back(a);
    }
    if (b.B.empty()) continue;        // batches with empty B_j are dropped
    kept.push_back(std::move(b));
  }
  c.batches.swap(kept);
#pragma omp parallel for schedule(dynamic)
  for (int64_t j = 0; j < (int64_t)c.batches.size(); ++j) {
    Batch& b = c.batches[j];
    b.PhiTilde.assign(nsh, 0.0);
    b.phitilde = 0.0;
    double val[10];
    for (int64_t g : b.pts) {
      const double sw = std::sqrt(c.w[g]);
      double sumabs = 0.0;
      for (int a : b.B) {
        shell_values(c.sh[a], &c.pts[3 * g], val);
        for (int i = 0; i < ncart(c.sh[a].l); ++i) {
          const double v = std::fabs(val[i]);
          b.PhiTilde[a] = std::max(b.PhiTilde[a], sw * v);
          sumabs += v;
        }
      }
      b.phitilde = std::max(b.phitilde, sw * sumabs);
    }
  }
}

// R12: Ftilde_a(j) for every shell a; then V_j by Eqs. 43-45.
void do_pair_screen(Ctx& c, const double* P) {
  const int nsh = (int)c.sh.size(), nbf = c.nbf;
#pragma omp parallel for schedule(dynamic)
  for (int64_t j = 0; j < (int64_t)c.batches.size(); ++j) {
    Batch& b = c.batches[j];
    std::vector<double> Ft(nsh, 0.0);
    for (int a = 0; a < nsh; ++a) {
      const Shell& sa = c.sh[a];
      for (int i = 0; i < ncart(sa.l); ++i) {
        const int mu = sa.foff + i;
        double s = 0.0;
        for (int bsh : b.B) {
          const Shell& sb = c.sh[bsh];
          for (int k = 0; k < ncart(sb.l); ++k) s += std::fabs(P[(size_t)mu * nbf + sb.foff + k]) * b.PhiTilde[bsh];
        }
        Ft[a] = std::max(Ft[a], s);
      }
    }
    b.V.clear();
    for (int a = 0; a < nsh; ++a)
      for (int bb = a; bb < nsh; ++bb) {
        const double At = c.Abound[(size_t)a * nsh + bb];
        const double eE = Ft[a] * Ft[bb] * At;
        const double eK = std::max(Ft[a], Ft[bb]) * b.phitilde * At;
        if (eE >= c.eps || eK >= c.eps) b.V.push_back({a, bb});
      }
  }
}

}  // namespace

// =====================================================================================
// C entry points (ctypes).  All arrays host, row-major, double / int32 / int64 as named.
// =====================================================================================
// The batch loop of orc_build_K (Eqs. 31, 35/48, 37-39), with the accumulator type R of the three sums over sigma, lambda and
// g as a parameter.  R = double is the oracle proper.  R = long double evaluates the SAME terms in the SAME order with 64-bit
// mantissas: it changes rounding only and exists to tell which side owns a difference of the size of the fp64 summation error
// (DESIGN.md section 6); the A integrals and Phi stay fp64 in both.
template <class R>
static void build_batches(Ctx* c, const double* P, const std::vector<char>& insel, std::vector<std::vector<long double>>& Kacc,
                          std::vector<double>& st_contr, std::vector<double>& st_prim, std::vector<double>& st_pp) {
  const int nbf = c->nbf;
  const int64_t nb = (int64_t)c->batches.size();
#pragma omp parallel
  {
    int tid = 0;
#ifdef _OPENMP
    tid = omp_get_thread_num();
#endif
    std::vector<long double>& Kt = Kacc[tid];
    Kt.assign((size_t)nbf * nbf, 0.0L);
    std::vector<double> Phi, Ablk(100), val(10);
    std::vector<R> F, G, Kj;
    std::vector<PrimPair> pps;
#pragma omp for schedule(dynamic)
    for (int64_t j = 0; j < nb; ++j) {
      const Batch& b = c->batches[j];
      const int64_t nq = (int64_t)b.pts.size();
      // packed function list of B_j
      std::vector<int> bf;
      for (int a : b.B) for (int i = 0; i < ncart(c->sh[a].l); ++i) bf.push_back(c->sh[a].foff + i);
      const int nB = (int)bf.size();
      // Eq. 31 / 42: Phi^(j)[g, k], k over functions of B_j
      Phi.assign((size_t)nq * nB, 0.0);
      for (int64_t g = 0; g < nq; ++g) {
        int k = 0;
        for (int a : b.B) {
          shell_values(c->sh[a], &c->pts[3 * b.pts[g]], val.data());
          for (int i = 0; i < ncart(c->sh[a].l); ++i) Phi[(size_t)g * nB + k++] = val[i];
        }
      }
      // which functions lambda appear in V_j (as a partner we need F for)
      std::vector<char> needF(nbf, 0);
      for (auto& ab : b.V) {
        if (!(insel[ab[0]] || insel[ab[1]])) continue;
        for (int s2 = 0; s2 < 2; ++s2) for (int i = 0; i < ncart(c->sh[ab[s2]].l); ++i) needF[c->sh[ab[s2]].foff + i] = 1;
      }
      // Eq. 35 / 48: F[g, lam] = sum_{sigma in B_j} P[lam, sigma] Phi[g, sigma]
      F.assign((size_t)nq * nbf, R(0));
      for (int64_t g = 0; g < nq; ++g)
        for (int lam = 0; lam < nbf; ++lam) {
          if (!needF[lam]) continue;
          R s = 0;
          for (int k = 0; k < nB; ++k) s += (R)P[(size_t)lam * nbf + bf[k]] * (R)Phi[(size_t)g * nB + k];
          F[(size_t)g * nbf + lam] = s;
        }
      // Eq. 37 + 38: G[g, nu] = w_g sum_lam A[g, nu, lam] F[g, lam] over pairs in V_j (both directions, R8)
      G.assign((size_t)nq * nbf, R(0));
      for (auto& ab : b.V) {
        const int a = ab[0], bb = ab[1];
        if (!(insel[a] || insel[bb])) continue;
        const Shell& sa = c->sh[a]; const Shell& sb = c->sh[bb];
        const int na = ncart(sa.l), nbc = ncart(sb.l);
        make_prim_pairs(sa, sb, pps);
        st_contr[tid] += (double)nq * na * nbc;
        st_prim[tid] += (double)nq * na * nbc * sa.nprim * sb.nprim;
        st_pp[tid] += (double)nq;
        for (int64_t g = 0; g < nq; ++g) {
          const int64_t gi = b.pts[g];
          A_block(pps, na, nbc, &c->pts[3 * gi], Ablk.data());
          const double wg = c->w[gi];
          R* Gg = &G[(size_t)g * nbf];
          const R* Fg = &F[(size_t)g * nbf];
          if (insel[a])
            for (int i = 0; i < na; ++i) {
              R s = 0;
              for (int k = 0; k < nbc; ++k) s += (R)Ablk[i * nbc + k] * Fg[sb.foff + k];
              Gg[sa.foff + i] += (R)wg * s;
            }
          if (a != bb && insel[bb])
            for (int k = 0; k < nbc; ++k) {
              R s = 0;
              for (int i = 0; i < na; ++i) s += (R)Ablk[i * nbc + k] * Fg[sa.foff + i];
              Gg[sb.foff + k] += (R)wg * s;
            }
        }
      }
      // Eq. 39: Kt[mu, nu] += sum_g Phi[g, mu] G[g, nu],  mu in B_j
      Kj.assign((size_t)nB * nbf, R(0));
      for (int64_t g = 0; g < nq; ++g)
        for (int k = 0; k < nB; ++k) {
          const double ph = Phi[(size_t)g * nB + k];
          if (ph == 0.0) continue;
          R* row = &Kj[(size_t)k * nbf];
          const R* Gg = &G[(size_t)g * nbf];
          for (int nu = 0; nu < nbf; ++nu) row[nu] += (R)ph * Gg[nu];
        }
      for (int k = 0; k < nB; ++k)
        for (int nu = 0; nu < nbf; ++nu) Kt[(size_t)bf[k] * nbf + nu] += (long double)Kj[(size_t)k * nbf + nu];
    }
  }
}

extern "C" {

int orc_boys(int mmax, double x, double* F) {
  if (mmax < 0 || mmax > 2 * kLmax || !(x >= 0.0)) return -1;
  boys(mmax, x, F);
  return 0;
}

void* orc_create(int natoms, const double* atom_xyz, int nshells, const int32_t* shell_atom, const int32_t* shell_l,
                 const int32_t* shell_nprim, const double* prim_exp, const double* prim_coef) {
  Ctx* c = new Ctx;
  int64_t po = 0;
  int fo = 0;
  for (int s = 0; s < nshells; ++s) {
    Shell sh;
    sh.atom = shell_atom[s]; sh.l = shell_l[s]; sh.nprim = shell_nprim[s]; sh.foff = fo;
    if (sh.l < 0 || sh.l > kLmax || sh.nprim < 1 || sh.atom < 0 || sh.atom >= natoms) { delete c; return nullptr; }
    for (int q = 0; q < 3; ++q) sh.A[q] = atom_xyz[3 * sh.atom + q];
    sh.e.assign(prim_exp + po, prim_exp + po + sh.nprim);
    sh.c.assign(prim_coef + po, prim_coef + po + sh.nprim);
    po += sh.nprim; fo += ncart(sh.l);
    for (int i = 0; i < ncart(sh.l); ++i) c->f2sh.push_back(s);
    c->sh.push_back(std::move(sh));
  }
  c->nbf = fo;
  c->Abound.assign((size_t)nshells * nshells, 0.0);
  for (int a = 0; a < nshells; ++a)
    for (int b = 0; b < nshells; ++b) c->Abound[(size_t)a * nshells + b] = A_bound(c->sh[a], c->sh[b]);
  return c;
}

void orc_destroy(void* h) { delete (Ctx*)h; }
int orc_nbf(void* h) { return ((Ctx*)h)->nbf; }

// A block of shell pair (a,b) at npts points: out[g][ia][ib]
int orc_A_pair(void* h, int a, int b, int64_t npts, const double* pts, double* out) {
  Ctx* c = (Ctx*)h;
  if (a < 0 || b < 0 || a >= (int)c->sh.size() || b >= (int)c->sh.size()) return -1;
  std::vector<PrimPair> pps;
  make_prim_pairs(c->sh[a], c->sh[b], pps);
  const int na = ncart(c->sh[a].l), nb = ncart(c->sh[b].l);
  for (int64_t g = 0; g < npts; ++g) A_block(pps, na, nb, pts + 3 * g, out + (size_t)g * na * nb);
  return 0;
}

// dense collocation Phi[g][mu] for all functions (Eq. 31)
int orc_collocation(void* h, int64_t npts, const double* pts, double* Phi) {
  Ctx* c = (Ctx*)h;
  for (int64_t g = 0; g < npts; ++g)
    for (const Shell& s : c->sh) shell_values(s, pts + 3 * g, Phi + (size_t)g * c->nbf + s.foff);
  return 0;
}

double orc_A_bound(void* h, int a, int b) { Ctx* c = (Ctx*)h; return c->Abound[(size_t)a * c->sh.size() + b]; }
double orc_rcut(void* h, int a, double eps) { return shell_rcut(((Ctx*)h)->sh[a], eps); }

// grid + density-independent plan (R13 batching, R10 B_j, R12 maxima)
int orc_set_grid(void* h, int64_t npts, const double* pts, const double* w, double eps, double h0, int nmax) {
  Ctx* c = (Ctx*)h;
  if (npts < 0 || !(h0 > 0) || nmax < 1 || eps < 0) return -1;
  for (int64_t i = 0; i < npts; ++i) if (!(w[i] >= 0.0)) return -1;
  c->pts.assign(pts, pts + 3 * npts);
  c->w.assign(w, w + npts);
  c->npts = npts; c->eps = eps; c->h0 = h0; c->nmax = nmax;
  do_batching(*c);
  do_basis_screen(*c);
  return 0;
}

int64_t orc_nbatch(void* h) { return (int64_t)((Ctx*)h)->batches.size(); }

// batch_off[nbatch+1], perm[sum |Q_j|] (input indices, batch by batch), bbox[nbatch*6] (lo xyz, hi xyz)
int orc_get_batches(void* h, int64_t* batch_off, int64_t* perm, double* bbox) {
  Ctx* c = (Ctx*)h;
  int64_t o = 0;
  for (size_t j = 0; j < c->batches.size(); ++j) {
    const Batch& b = c->batches[j];
    batch_off[j] = o;
    for (int64_t i : b.pts) perm[o++] = i;
    if (bbox) for (int q = 0; q < 3; ++q) { bbox[6 * j + q] = b.lo[q]; bbox[6 * j + 3 + q] = b.hi[q]; }
  }
  batch_off[c->batches.size()] = o;
  return 0;
}

// CSR of B_j: off[nbatch+1]; ids (may be NULL to query size) ; returns total
int64_t orc_get_B(void* h, int64_t* off, int32_t* ids) {
  Ctx* c = (Ctx*)h;
  int64_t o = 0;
  for (size_t j = 0; j < c->batches.size(); ++j) {
    if (off) off[j] = o;
    for (int a : c->batches[j].B) { if (ids) ids[o] = a; ++o; }
  }
  if (off) off[c->batches.size()] = o;
  return o;
}

// CSR of V_j (valid after orc_build_K / orc_screen): off[nbatch+1]; pairs[2*total] (a<=b); returns total
int64_t orc_get_V(void* h, int64_t* off, int32_t* pairs) {
  Ctx* c = (Ctx*)h;
  int64_t o = 0;
  for (size_t j = 0; j < c->batches.size(); ++j) {
    if (off) off[j] = o;
    for (auto& ab : c->batches[j].V) { if (pairs) { pairs[2 * o] = ab[0]; pairs[2 * o + 1] = ab[1]; } ++o; }
  }
  if (off) off[c->batches.size()] = o;
  return o;
}

int orc_get_maxima(void* h, double* PhiTilde /*[nbatch*nsh]*/, double* phitilde /*[nbatch]*/) {
  Ctx* c = (Ctx*)h;
  const size_t nsh = c->sh.size();
  for (size_t j = 0; j < c->batches.size(); ++j) {
    for (size_t a = 0; a < nsh; ++a) PhiTilde[j * nsh + a] = c->batches[j].PhiTilde[a];
    phitilde[j] = c->batches[j].phitilde;
  }
  return 0;
}

int orc_screen(void* h, const double* P) { do_pair_screen(*(Ctx*)h, P); return 0; }

// K build.  sel_shells: optional list (nsel > 0) of shells S; then only the columns nu in S of
// Kt are computed (G_nu needs only pairs touching S) and K is returned as Kt restricted to those
// columns (other columns 0) -- the caller forms the sampled block K[S,S] = (Kt[S,S]+Kt[S,S]^T)/2.
// With nsel == 0 the full symmetrised K (Eq. 40) is returned.
int orc_build_K(void* h, const double* P, double* K, int nsel, const int32_t* sel_shells) {
  Ctx* c = (Ctx*)h;
  const int nsh = (int)c->sh.size(), nbf = c->nbf;
  for (int i = 0; i < nbf; ++i)
    for (int k = 0; k < i; ++k)
      if (std::fabs(P[(size_t)i * nbf + k] - P[(size_t)k * nbf + i]) > 1e-12 * (1.0 + std::fabs(P[(size_t)i * nbf + k]))) return -2;
  do_pair_screen(*c, P);
  std::vector<char> insel(nsh, nsel > 0 ? 0 : 1);
  for (int i = 0; i < nsel; ++i) insel[sel_shells[i]] = 1;

  int nthreads = 1;
#ifdef _OPENMP
  nthreads = omp_get_max_threads();
#endif
  std::vector<std::vector<long double>> Kacc(nthreads);
  std::vector<double> st_contr(nthreads, 0.0), st_prim(nthreads, 0.0), st_pp(nthreads, 0.0);
  const int64_t nb = (int64_t)c->batches.size();
#ifdef _OPENMP
  const double t0 = omp_get_wtime();
#endif
  if (c->extended) build_batches<long double>(c, P, insel, Kacc, st_contr, st_prim, st_pp);
  else build_batches<double>(c, P, insel, Kacc, st_contr, st_prim, st_pp);
  // reduce the per-thread accumulators in fixed thread order
  std::vector<long double> Kt((size_t)nbf * nbf, 0.0L);
  for (int t = 0; t < nthreads; ++t)
    if (!Kacc[t].empty())
      for (size_t i = 0; i < Kt.size(); ++i) Kt[i] += Kacc[t][i];
  if (nsel > 0) {
    for (size_t i = 0; i < Kt.size(); ++i) K[i] = (double)Kt[i];
  } else {
    for (int i = 0; i < nbf; ++i)       // Eq. 40
      for (int k = 0; k < nbf; ++k) K[(size_t)i * nbf + k] = (double)(0.5L * (Kt[(size_t)i * nbf + k] + Kt[(size_t)k * nbf + i]));
  }
  c->n_int_contr = c->n_int_prim = c->n_pairpoints = 0;
  for (int t = 0; t < nthreads; ++t) { c->n_int_contr += st_contr[t]; c->n_int_prim += st_prim[t]; c->n_pairpoints += st_pp[t]; }
#ifdef _OPENMP
  c->t_build = omp_get_wtime() - t0;
#endif
  return 0;
}

// 1: the sums over sigma, lambda and g of the next orc_build_K run in long double (rounding-order check only); 0: fp64 (default)
int orc_set_extended(void* h, int flag) { ((Ctx*)h)->extended = flag != 0; return 0; }

// stats of the last orc_build_K: contracted integrals, primitive integrals, pair-points, seconds, threads
int orc_get_stats(void* h, double* out5) {
  Ctx* c = (Ctx*)h;
  out5[0] = c->n_int_contr; out5[1] = c->n_int_prim; out5[2] = c->n_pairpoints; out5[3] = c->t_build;
#ifdef _OPENMP
  out5[4] = omp_get_max_threads();
#else
  out5[4] = 1;
#endif
  return 0;
}

}  // extern "C"
