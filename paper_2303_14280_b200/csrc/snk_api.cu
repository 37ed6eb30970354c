// snk_api.cu -- the C ABI of include/snk.h and the host planner behind it.
// Host work here is bookkeeping only (validation, list sizing, super-batch planning, launches);
// every step of the path (rows a0-a7 of DESIGN.md) runs in the kernels of this library.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <limits>
#include <string>
#include <thread>
#include <vector>

#include "snk_internal.h"
#include "snk_kernels.h"
#include "snk_os.cuh"

using namespace snk;

namespace {
thread_local std::string g_create_error;

struct Super { int b0, b1; int64_t slot0, nslots; int t0, t1; int c0, c1, ct0, ct1, max_nrow; };   // batches, tiles, chunks, a4 column tiles

enum Stage { ST_SCREEN = 0, ST_COLLOC, ST_F, ST_G, ST_KT, ST_SYM, ST_COUNT };
}  // namespace

struct snk_ctx {
  int device = -1;              // the CUDA device current at snk_create: every later call must run with it current
  int natoms = 0, nsh = 0, nbf = 0;
  std::vector<double> h_cx, h_cy, h_cz, h_pexp, h_pcoef;
  std::vector<int32_t> h_l, h_foff, h_poff, h_nprim;
  DevBuf<double> d_cx, d_cy, d_cz, d_pexp, d_pcoef, d_rcut2, d_Atil, d_boys;
  DevBuf<int32_t> d_l, d_foff, d_poff, d_nprim, d_lshells;
  PairCand cand{};
  // options
  double eps = 0.0, h0 = 6.0, workspace_gb = 24.0;
  int nmax = 2048;
  int tile_split = 0;           // CTAs per tile in a5; 0 = automatic
  int sm_count = 148;
  // grid state
  bool have_grid = false;
  int64_t npts = 0, npts_kept = 0, nslots = 0, ldj = 0, ld = 0;
  int nbatch = 0, nshw = 0;
  int64_t sum_B = 0, sum_B_fn = 0;
  DevBuf<double> gx, gy, gz, gw, d_PhiTf, d_phit;
  DevBuf<int64_t> slot_src, d_bslot;
  DevBuf<int32_t> d_bn;
  DevBuf<uint32_t> d_bmask;
  DevBuf<unsigned long long> d_phimax, d_Fmax;
  DevBuf<TileRec> d_tiles;
  DevBuf<ChunkRec> d_chunks;    // a4 / a6: chunks of whole batches, their row lists L (functions in the union of B_j)
  DevBuf<int32_t> d_rowlist, d_nrows;
  DevBuf<ColTile> d_ctiles;     // a4: 128-slot column tiles of the chunks
  int64_t lstride = 0;
  double flops_gemm_alg = 0.0;  // 2 |Q_j| nbf(B_j) nbf per contraction, summed over the batches (Eq. 48's operand sizes)
  std::vector<int32_t> h_bn;
  std::vector<int64_t> h_bslot;
  std::vector<TileRec> h_tiles;
  std::vector<Super> supers;
  DevBuf<double> d_Phi, d_F, d_G;
  // build state
  bool have_build = false, have_screen = false, stats_valid = false;
  DevBuf<double> d_absP, d_Ftf, d_FtsT, d_Kt, d_Pin, d_Kout, d_stats, d_cflops;
  DevBuf<int32_t> d_flag, d_np, d_pos, d_ppos;     // per candidate pair: #units, is-pair flag, and their exclusive scans
  DevBuf<unsigned char> d_units;                    // [nunit][kUnitBytes]
  DevBuf<UnitMeta> d_meta;                          // [nunit]
  DevBuf<uint32_t> d_vmask;
  DevBuf<int32_t> d_vlist, d_vcnt;                  // unit-id lists of the current super-batch (k_vlist)
  DevBuf<char> d_tmp;
  int64_t vstride = 0;
  int npair_sig = 0, nunit = 0;
  int64_t nprimpair = 0;
  int cls_beg[kNumClasses + 1] = {0};
  double gemm_flops = 0.0;
  double flops_F = 0.0, flops_Kt = 0.0;     // a4 / a6 flops actually executed per build (blocks with a set activity bit)
  int64_t n_launches = 0;
  // timing
  std::vector<cudaEvent_t> ev_pool;
  struct Span { int stage; int cls; int e0, e1; };
  std::vector<Span> spans;
  int ev_used = 0;
  cudaEvent_t ev_b0 = nullptr, ev_b1 = nullptr, ev_g0 = nullptr, ev_g1 = nullptr;
  cudaStream_t last_stream = nullptr;
  snk_stats stats{};
  std::string err;

  ShellTab tab() const {
    ShellTab t;
    t.cx = d_cx.p; t.cy = d_cy.p; t.cz = d_cz.p; t.l = d_l.p; t.foff = d_foff.p; t.poff = d_poff.p; t.nprim = d_nprim.p;
    t.pexp = d_pexp.p; t.pcoef = d_pcoef.p; t.rcut2 = d_rcut2.p; t.nsh = nsh; t.nbf = nbf;
    return t;
  }
  cudaError_t new_event(int& id) {
    if (ev_used == (int)ev_pool.size()) {
      cudaEvent_t e;
      const cudaError_t rc = cudaEventCreate(&e);
      if (rc != cudaSuccess) return rc;
      ev_pool.push_back(e);
    }
    id = ev_used++;
    return cudaSuccess;
  }
};

#define CK(call)                                                                                        \
  do {                                                                                                  \
    cudaError_t e__ = (call);                                                                           \
    if (e__ != cudaSuccess) {                                                                           \
      char b__[512];                                                                                    \
      snprintf(b__, sizeof b__, "%s:%d: %s -> %s", __FILE__, __LINE__, #call, cudaGetErrorString(e__)); \
      ctx->err = b__;                                                                                   \
      return e__ == cudaErrorMemoryAllocation ? SNK_ENOMEM : SNK_ECUDA;                                 \
    }                                                                                                   \
  } while (0)

#define FAIL(code, msg) do { ctx->err = (msg); return (code); } while (0)

// the context's buffers, events and shared-memory opt-ins belong to one device
#define CHECK_DEVICE()                                                                                              \
  do {                                                                                                              \
    int d__ = -1;                                                                                                   \
    if (cudaGetDevice(&d__) != cudaSuccess || d__ != ctx->device)                                                   \
      FAIL(SNK_ESTATE, "the CUDA device that was current at snk_create must be current for every call on the context"); \
  } while (0)

namespace {

template <class T>
cudaError_t upload(DevBuf<T>& b, const std::vector<T>& v) {
  cudaError_t e = b.reserve(std::max<size_t>(v.size(), 1));
  if (e != cudaSuccess) return e;
  if (!v.empty()) e = cudaMemcpy(b.p, v.data(), v.size() * sizeof(T), cudaMemcpyHostToDevice);
  return e;
}

// Tables for the Taylor path of the device Boys function (R15, layout in snk_os.cuh): for every top order L the scaled
// derivatives F_{L+k}(x_i)/k!, k = 0..7, and e^{-x_i}.  F at the highest order by the all-positive series in long double,
// lower orders by downward recursion.  Own generator of the library (the oracle has its own code).
std::vector<double> make_boys_table() {
  std::vector<double> t((size_t)(kBoysLmax + 1) * kBoysRows * kBoysStride, 0.0);
  const int mtop = kBoysLmax + 7;
  std::vector<long double> F(mtop + 1);
  for (int i = 0; i < kBoysRows; ++i) {
    const long double x = (long double)i * (long double)kBoysDelta;
    const long double ex = expl(-x);
    long double term = 1.0L / (2 * mtop + 1), sum = term;
    for (int k = 1; k < 4000; ++k) {
      term *= 2.0L * x / (2 * mtop + 2 * k + 1);
      sum += term;
      if (term < 1e-22L * sum) break;
    }
    F[mtop] = ex * sum;
    for (int m = mtop; m >= 1; --m) F[m - 1] = (2.0L * x * F[m] + ex) / (2 * m - 1);
    for (int L = 0; L <= kBoysLmax; ++L) {
      double* row = &t[((size_t)L * kBoysRows + i) * kBoysStride];
      long double fact = 1.0L;
      for (int k = 0; k < 8; ++k) { if (k > 0) fact *= k; row[k] = (double)(F[L + k] / fact); }
      row[8] = (double)ex;
    }
  }
  return t;
}

// R11: rigorous bound on |A_{mu nu}(g)| for every shell pair (host, libm: same arithmetic order as documented in DESIGN.md).
void A_bound_rows(const snk_ctx* c, int a0, int a1, double* out) {
  const int nsh = c->nsh;
  auto sg = [&](int s, int k, double& cc, double& zz) {
    const double z = c->h_pexp[c->h_poff[s] + k], co = c->h_pcoef[c->h_poff[s] + k];
    const int l = c->h_l[s];
    if (l == 0) { cc = std::fabs(co); zz = z; }
    else { zz = 0.5 * z; cc = std::fabs(co) * std::pow(l / (std::exp(1.0) * z), 0.5 * l); }
  };
  for (int a = a0; a < a1; ++a)
    for (int b = 0; b < nsh; ++b) {
      const double dx = c->h_cx[a] - c->h_cx[b], dy = c->h_cy[a] - c->h_cy[b], dz = c->h_cz[a] - c->h_cz[b];
      const double AB2 = dx * dx + dy * dy + dz * dz;
      double sum = 0.0;
      for (int k = 0; k < c->h_nprim[a]; ++k)
        for (int l = 0; l < c->h_nprim[b]; ++l) {
          double ca, za, cb, zb;
          sg(a, k, ca, za); sg(b, l, cb, zb);
          const double p = za + zb;
          sum += ca * cb * (2.0 * M_PI / p) * std::exp(-(za * zb / p) * AB2);
        }
      out[(size_t)a * nsh + b] = sum;
    }
}

// R10: cutoff radius on the 0.25-bohr ladder
double shell_rcut(const snk_ctx* c, int s, double eps) {
  if (!(eps > 0.0)) return std::numeric_limits<double>::infinity();
  const int l = c->h_l[s], p0 = c->h_poff[s], np = c->h_nprim[s];
  double zmin = c->h_pexp[p0];
  for (int k = 0; k < np; ++k) zmin = std::min(zmin, c->h_pexp[p0 + k]);
  const double rmin = std::sqrt(l / (2.0 * zmin));
  for (int n = 1; n < 100000; ++n) {
    const double r = 0.25 * n;
    if (r < rmin) continue;
    double env = 0.0;
    for (int k = 0; k < np; ++k) env += std::fabs(c->h_pcoef[p0 + k]) * std::exp(-c->h_pexp[p0 + k] * r * r);
    env *= std::pow(r, l);
    if (env < eps) return r;
  }
  return std::numeric_limits<double>::infinity();
}

// FP64 flop model of the integral kernel: far-field (asymptotic Boys) path, FMA = 2.
// Counted with the same loops as the device templates.
void class_flops(int la, int lb, double& per_prim, double& per_contr) {
  const int L = la + lb;
  double f = 3 + 5 + 1;                     // P - r_g, |.|^2, x = p r^2
  f += 8 + 1 + (L > 0 ? 2 + 2 * L : 0);     // rsqrt, F_0, 1/(2x), upward recursion
  f += (L + 1);                             // seed scaling by pref
  auto nc = [](int l) { return (l + 1) * (l + 2) / 2; };
  for (int l = 0; l < L; ++l)
    for (int n = 0; n < L - l; ++n)
      for (int c = 0; c < nc(l + 1); ++c) {
        // component (i,j,k) of level l+1 in library order
        int ip = 0;
        while ((ip + 1) * (ip + 2) / 2 <= c) ++ip;
        const int i = l + 1 - ip, k = c - ip * (ip + 1) / 2, j = l + 1 - i - k;
        const int aq = i > 0 ? i - 1 : (j > 0 ? j - 1 : k - 1);
        f += 3;                              // mul + fma
        if (aq > 0) f += 3;                  // sub + fma
        if (n == 0 && l + 1 >= la) f += 1;   // contraction accumulate
      }
  if (L == 0 || la == 0) f += 1;
  per_prim = f;
  double h = 0;                              // HRR tree: every shift is one FMA per surviving component
  // nodes at depth s (1..lb) : number of monomials of degree s = nc(s); each holds levels la..L-s
  for (int s = 1; s <= lb; ++s) {
    int comps = 0;
    for (int l = la; l <= L - s; ++l) comps += nc(l);
    h += 2.0 * nc(s) * comps;
  }
  h += 2.0 * 2.0 * nc(la) * nc(lb);          // two contractions, FMA each
  per_contr = h;
}

int set_err(snk_ctx* ctx, int code, const char* msg) { ctx->err = msg; return code; }

// No exception crosses the C ABI (include/snk.h): host allocation failures become SNK_ENOMEM, anything else SNK_ECUDA
// (std::system_error of a worker thread, ...) with the text in snk_last_error.
template <class F>
int guarded(snk_ctx* ctx, F&& body) {
  auto note = [&](const char* what) { try { if (ctx) ctx->err = what; else g_create_error = what; } catch (...) {} };
  try {
    return body();
  } catch (const std::bad_alloc&) {
    note("out of host memory");
    return SNK_ENOMEM;
  } catch (const std::exception& e) {
    note(e.what());
    return SNK_ECUDA;
  } catch (...) {
    note("unknown C++ exception");
    return SNK_ECUDA;
  }
}

}  // namespace

// ---- snk_A_pair_noalloc: the A-block kernel with its primitive-pair scratch in a file-scope device array ------------------
// snk_debug_A_pair cudaMallocs (and frees) a buffer for the primitive-pair records of the shell pair on every call.  Callers
// that must not allocate (CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc) get the same kernel with
// that scratch here: kNoAllocMaxPrims records of 80 bytes = 80 KB, held by every GPU that loads the library until exit.
// In host code `g_noalloc_prims` is only a host-side stand-in for the symbol: its device address comes from
// cudaGetSymbolAddress (noalloc_scratch, once per device, with that device current) and only that pointer goes to kernels.
constexpr int kNoAllocMaxPrims = 1024;
static __device__ __align__(256) unsigned char g_noalloc_prims[kNoAllocMaxPrims * kPrimBytes];
static_assert(sizeof(PrimPair) == kPrimBytes, "PrimPair layout");

namespace {
PrimPair* g_noalloc_ptr[kMaxDevices] = {};

cudaError_t noalloc_scratch(int dev, PrimPair** out) {          // `dev` is the current device
  if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
  if (!g_noalloc_ptr[dev]) {
    void* p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&p, g_noalloc_prims);
    if (e != cudaSuccess) return e;
    g_noalloc_ptr[dev] = static_cast<PrimPair*>(p);
  }
  *out = g_noalloc_ptr[dev];
  return cudaSuccess;
}

// primitive-pair records of shell pair (sa, sb), k-major like the host loop of snk_debug_A_pair (R1: prefactor restored).
// Overwrites entries [0, nprim(sa) nprim(sb)) of the scratch; nothing has to start at zero.
__global__ void k_noalloc_prims(ShellTab sh, int sa, int sb, PrimPair* __restrict__ out) {
  const int npa = sh.nprim[sa], npb = sh.nprim[sb];
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= npa * npb) return;
  const int k = t / npb, l = t - k * npb;
  const double A[3] = {sh.cx[sa], sh.cy[sa], sh.cz[sa]}, B[3] = {sh.cx[sb], sh.cy[sb], sh.cz[sb]};
  const double dx = A[0] - B[0], dy = A[1] - B[1], dz = A[2] - B[2];
  const double AB2 = dx * dx + dy * dy + dz * dz;
  const double za = sh.pexp[sh.poff[sa] + k], zb = sh.pexp[sh.poff[sb] + l];
  const double ps = za + zb;
  PrimPair q;
  q.p2 = 2.0 * ps; q.inv2p = 0.5 / ps;
  q.Px = (za * A[0] + zb * B[0]) / ps; q.Py = (za * A[1] + zb * B[1]) / ps; q.Pz = (za * A[2] + zb * B[2]) / ps;
  q.PAx = q.Px - A[0]; q.PAy = q.Py - A[1]; q.PAz = q.Pz - A[2];
  q.pref = sh.pcoef[sh.poff[sa] + k] * sh.pcoef[sh.poff[sb] + l] * (6.283185307179586 / ps) * exp(-(za * zb / ps) * AB2);
  q.cfar2 = 1.2533141373155002512 * q.pref;
  out[t] = q;
}
}  // namespace

// ====================================================================================================================
extern "C" {

const char* snk_version(void) { return "snk 0.1.0 (sm_100a)"; }

const char* snk_last_error(const snk_ctx* ctx) { return ctx ? ctx->err.c_str() : g_create_error.c_str(); }

int snk_nbf(const snk_ctx* ctx) { return ctx ? ctx->nbf : SNK_EINVAL; }

void snk_destroy(snk_ctx* ctx) {
  if (!ctx) return;
  ctx->d_cx.release(); ctx->d_cy.release(); ctx->d_cz.release(); ctx->d_pexp.release(); ctx->d_pcoef.release();
  ctx->d_rcut2.release(); ctx->d_Atil.release(); ctx->d_boys.release(); ctx->d_l.release(); ctx->d_foff.release();
  ctx->d_poff.release(); ctx->d_nprim.release(); ctx->d_lshells.release();
  ctx->gx.release(); ctx->gy.release(); ctx->gz.release(); ctx->gw.release(); ctx->d_PhiTf.release(); ctx->d_phit.release();
  ctx->slot_src.release(); ctx->d_bslot.release(); ctx->d_bn.release(); ctx->d_bmask.release(); ctx->d_phimax.release();
  ctx->d_Fmax.release(); ctx->d_tiles.release(); ctx->d_chunks.release(); ctx->d_rowlist.release(); ctx->d_nrows.release();
  ctx->d_ctiles.release(); ctx->d_Phi.release(); ctx->d_F.release(); ctx->d_G.release();
  ctx->d_absP.release(); ctx->d_Ftf.release(); ctx->d_FtsT.release(); ctx->d_Kt.release();
  ctx->d_Pin.release(); ctx->d_Kout.release(); ctx->d_stats.release(); ctx->d_cflops.release();
  ctx->d_flag.release(); ctx->d_np.release(); ctx->d_pos.release(); ctx->d_ppos.release(); ctx->d_units.release();
  ctx->d_meta.release(); ctx->d_vmask.release(); ctx->d_vlist.release(); ctx->d_vcnt.release(); ctx->d_tmp.release();
  for (cudaEvent_t e : ctx->ev_pool) cudaEventDestroy(e);
  for (cudaEvent_t e : {ctx->ev_b0, ctx->ev_b1, ctx->ev_g0, ctx->ev_g1}) if (e) cudaEventDestroy(e);
  delete ctx;
}

int snk_create(snk_ctx** out, int32_t natoms, const double* atom_xyz, int32_t nshells, const int32_t* shell_atom,
               const int32_t* shell_l, const int32_t* shell_nprim, const double* prim_exp, const double* prim_coef) {
  snk_ctx* ctx = nullptr;
  const int rc = guarded(nullptr, [&]() -> int {
  if (out) *out = nullptr;
  if (!out || natoms < 1 || nshells < 1 || !atom_xyz || !shell_atom || !shell_l || !shell_nprim || !prim_exp || !prim_coef) {
    g_create_error = "snk_create: NULL argument or empty basis";
    return SNK_EINVAL;
  }
  ctx = new (std::nothrow) snk_ctx;
  if (!ctx) { g_create_error = "snk_create: out of host memory"; return SNK_ENOMEM; }
  auto bail = [&](int code, const std::string& m) { g_create_error = m; snk_destroy(ctx); ctx = nullptr; return code; };
  if (cudaGetDevice(&ctx->device) != cudaSuccess) return bail(SNK_ECUDA, "snk_create: no current CUDA device");
  if (cudaDeviceGetAttribute(&ctx->sm_count, cudaDevAttrMultiProcessorCount, ctx->device) != cudaSuccess || ctx->sm_count < 1) ctx->sm_count = 148;
  ctx->natoms = natoms; ctx->nsh = nshells;
  int64_t po = 0;
  int fo = 0;
  for (int i = 0; i < natoms * 3; ++i) if (!std::isfinite(atom_xyz[i])) return bail(SNK_EINVAL, "snk_create: non-finite atom coordinate");
  for (int s = 0; s < nshells; ++s) {
    const int l = shell_l[s], np = shell_nprim[s], at = shell_atom[s];
    if (l < 0 || l > 3) return bail(SNK_EINVAL, "snk_create: shell_l outside 0..3");
    if (np < 1) return bail(SNK_EINVAL, "snk_create: shell_nprim < 1");
    if (at < 0 || at >= natoms) return bail(SNK_EINVAL, "snk_create: shell_atom out of range");
    ctx->h_cx.push_back(atom_xyz[3 * at]); ctx->h_cy.push_back(atom_xyz[3 * at + 1]); ctx->h_cz.push_back(atom_xyz[3 * at + 2]);
    ctx->h_l.push_back(l); ctx->h_foff.push_back(fo); ctx->h_poff.push_back((int32_t)po); ctx->h_nprim.push_back(np);
    for (int k = 0; k < np; ++k) {
      const double z = prim_exp[po + k], c = prim_coef[po + k];
      if (!(z > 0.0) || !std::isfinite(z)) return bail(SNK_EINVAL, "snk_create: exponent must be finite and > 0");
      if (!std::isfinite(c)) return bail(SNK_EINVAL, "snk_create: non-finite coefficient");
      ctx->h_pexp.push_back(z); ctx->h_pcoef.push_back(c);
    }
    po += np; fo += ncart(l);
  }
  ctx->nbf = fo;
  // candidate-pair enumeration: shells grouped by l
  std::vector<int32_t> lsh;
  int cnt[4] = {0, 0, 0, 0};
  for (int l = 0; l < 4; ++l) {
    ctx->cand.l_off[l] = (int32_t)lsh.size();
    for (int s = 0; s < nshells; ++s) if (ctx->h_l[s] == l) { lsh.push_back(s); ++cnt[l]; }
  }
  ctx->cand.l_off[4] = (int32_t)lsh.size();
  int64_t off = 0;
  for (int la = 0; la < 4; ++la)
    for (int lb = 0; lb <= la; ++lb) {
      const int c = class_id(la, lb);
      ctx->cand.off[c] = off; ctx->cand.cnt_b[c] = cnt[lb]; ctx->cand.la[c] = la; ctx->cand.lb[c] = lb; ctx->cand.same_l[c] = la == lb;
      off += (int64_t)cnt[la] * cnt[lb];
    }
  ctx->cand.off[kNumClasses] = off;
  if (off >= (int64_t)1 << 31) return bail(SNK_EINVAL, "snk_create: too many shells (candidate pairs exceed 2^31)");
  if (nshells > 65535) return bail(SNK_EINVAL, "snk_create: more than 65535 shells (grid.y of the per-shell screening kernels)");

  cudaError_t e = cudaSuccess;
  auto up = [&](auto& buf, const auto& vec) { if (e == cudaSuccess) e = upload(buf, vec); };
  up(ctx->d_cx, ctx->h_cx); up(ctx->d_cy, ctx->h_cy); up(ctx->d_cz, ctx->h_cz); up(ctx->d_pexp, ctx->h_pexp); up(ctx->d_pcoef, ctx->h_pcoef);
  up(ctx->d_l, ctx->h_l); up(ctx->d_foff, ctx->h_foff); up(ctx->d_poff, ctx->h_poff); up(ctx->d_nprim, ctx->h_nprim);
  up(ctx->d_lshells, lsh);
  ctx->cand.shells = ctx->d_lshells.p;
  up(ctx->d_boys, make_boys_table());
  // R11 table
  std::vector<double> At((size_t)nshells * nshells);
  {
    const int nt = (int)std::max(1u, std::min(std::thread::hardware_concurrency(), 16u));
    std::vector<std::thread> th;
    const int chunk = (nshells + nt - 1) / nt;
    for (int t = 0; t < nt; ++t) {
      const int a0 = t * chunk, a1 = std::min(nshells, a0 + chunk);
      if (a0 < a1) th.emplace_back(A_bound_rows, ctx, a0, a1, At.data());
    }
    for (auto& t : th) t.join();
  }
  up(ctx->d_Atil, At);
  if (e == cudaSuccess) e = ctx->d_rcut2.reserve(nshells);
  if (e == cudaSuccess) e = ctx->d_phimax.reserve(1);
  if (e == cudaSuccess) e = ctx->d_Fmax.reserve(nshells);
  if (e == cudaSuccess) e = ctx->d_stats.reserve(32);
  if (e == cudaSuccess) {
    std::vector<double> cf(2 * kNumClasses);
    for (int la = 0; la < 4; ++la)
      for (int lb = 0; lb <= la; ++lb) class_flops(la, lb, cf[class_id(la, lb)], cf[kNumClasses + class_id(la, lb)]);
    e = upload(ctx->d_cflops, cf);
  }
  if (e == cudaSuccess) {
    cudaEventCreate(&ctx->ev_b0); cudaEventCreate(&ctx->ev_b1); cudaEventCreate(&ctx->ev_g0); cudaEventCreate(&ctx->ev_g1);
    e = cudaGetLastError();
  }
  if (e != cudaSuccess)
    return bail(e == cudaErrorMemoryAllocation ? SNK_ENOMEM : SNK_ECUDA, std::string("snk_create: CUDA: ") + cudaGetErrorString(e));
  *out = ctx;
  return SNK_OK;
  });
  if (rc != SNK_OK && ctx) { snk_destroy(ctx); if (out) *out = nullptr; }    // an exception left a half-built context
  return rc;
}

int snk_set_option(snk_ctx* ctx, const char* key, double value) {
  return guarded(ctx, [&]() -> int {
  if (!ctx || !key) return SNK_EINVAL;
  CHECK_DEVICE();
  const std::string k(key);
  if (k == "eps") { if (!(value >= 0.0) || !std::isfinite(value)) FAIL(SNK_EINVAL, "eps must be finite and >= 0"); ctx->eps = value; }
  else if (k == "batch_cell") { if (!(value > 0.0) || !std::isfinite(value)) FAIL(SNK_EINVAL, "batch_cell must be > 0"); ctx->h0 = value; }
  else if (k == "batch_max") { if (!(value >= 32 && value <= 4096) || value != std::floor(value)) FAIL(SNK_EINVAL, "batch_max must be an integer in 32..4096"); ctx->nmax = (int)value; }
  else if (k == "workspace_gb") { if (!(value > 0.0) || !std::isfinite(value)) FAIL(SNK_EINVAL, "workspace_gb must be > 0"); ctx->workspace_gb = value; }
  else if (k == "tile_split") { if (!(value >= 0 && value <= 64) || value != std::floor(value)) FAIL(SNK_EINVAL, "tile_split must be an integer in 0..64 (0 = automatic)"); ctx->tile_split = (int)value; }
  else if (k == "atomics") { if (value != 1.0) FAIL(SNK_EINVAL, "atomics: only 1 is implemented"); }
  else FAIL(SNK_EINVAL, "unknown option key");
  ctx->have_grid = false;      // options take effect at the next snk_set_grid
  ctx->have_build = false;
  return SNK_OK;
  });
}

int snk_set_grid(snk_ctx* ctx, int64_t npts, const double* points, const double* weights, void* stream_) {
  return guarded(ctx, [&]() -> int {
  if (!ctx) return SNK_EINVAL;
  if (npts < 0 || (npts > 0 && (!points || !weights))) FAIL(SNK_EINVAL, "snk_set_grid: bad npts / NULL pointer");
  if (npts >= ((int64_t)1 << 31) - 4096) FAIL(SNK_EINVAL, "snk_set_grid: more than 2^31 points");
  CHECK_DEVICE();
  cudaStream_t s = (cudaStream_t)stream_;
  ctx->last_stream = s;
  ctx->have_grid = false; ctx->have_build = false; ctx->stats_valid = false;
  const int nsh = ctx->nsh;
  CK(cudaEventRecord(ctx->ev_g0, s));
  // R10 cutoffs (host libm), squared
  {
    std::vector<double> rc2(nsh);
    for (int a = 0; a < nsh; ++a) { const double r = shell_rcut(ctx, a, ctx->eps); rc2[a] = r * r; }
    CK(cudaMemcpyAsync(ctx->d_rcut2.p, rc2.data(), nsh * sizeof(double), cudaMemcpyHostToDevice, s));
    CK(cudaStreamSynchronize(s));
  }
  ctx->npts = npts; ctx->nbatch = 0; ctx->npts_kept = 0; ctx->nslots = 0; ctx->sum_B = ctx->sum_B_fn = 0;
  ctx->h_bn.clear(); ctx->h_bslot.clear(); ctx->h_tiles.clear(); ctx->supers.clear();
  ctx->nshw = (nsh + 31) / 32;
  std::vector<int64_t> h_bsrc_begin;
  std::vector<int32_t> h_bcnt;          // |B_j| of the kept batches
  std::vector<int32_t> h_bsrc;
  DevBuf<uint32_t> idx0, idx1, idx2;
  if (npts > 0) {
    // ---- a0: keys, two stable radix passes (path, then root), leaves ----
    DevBuf<unsigned long long> root, path, kin, kout;
    DevBuf<uint8_t> depth;
    DevBuf<int32_t> flag, scan, cnt;
    DevBuf<int64_t> begin;
    DevBuf<double> bbox;
    DevBuf<int> derr;
    auto freeall = [&]() { root.release(); path.release(); kin.release(); kout.release(); depth.release(); flag.release(); scan.release();
                           cnt.release(); begin.release(); bbox.release(); derr.release(); idx0.release(); idx1.release(); idx2.release(); };
    struct Guard { decltype(freeall)& f; ~Guard() { f(); } } guard{freeall};
    CK(root.reserve(npts)); CK(path.reserve(npts)); CK(kin.reserve(npts)); CK(kout.reserve(npts));
    CK(idx0.reserve(npts)); CK(idx1.reserve(npts)); CK(idx2.reserve(npts)); CK(derr.reserve(1));
    CK(cudaMemsetAsync(derr.p, 0, sizeof(int), s));
    CK(run_point_keys(npts, points, weights, ctx->h0, root.p, path.p, idx0.p, derr.p, s));
    int herr = 0;
    CK(cudaMemcpyAsync(&herr, derr.p, sizeof(int), cudaMemcpyDeviceToHost, s));
    CK(cudaStreamSynchronize(s));
    if (herr & 1) FAIL(SNK_EINVAL, "snk_set_grid: negative, NaN or infinite weight");
    if (herr & 2) FAIL(SNK_EINVAL, "snk_set_grid: non-finite or out-of-range point coordinate");
    size_t tb = 0, tb2 = 0;
    CK(run_sort_pairs(nullptr, tb, path.p, kout.p, idx0.p, idx1.p, npts, 60, s));
    CK(run_scan_i32(nullptr, tb2, nullptr, nullptr, npts, true, s));
    CK(ctx->d_tmp.reserve(std::max(tb, tb2) + 256));
    CK(run_sort_pairs(ctx->d_tmp.p, tb, path.p, kout.p, idx0.p, idx1.p, npts, 60, s));
    CK(run_gather_u64(npts, idx1.p, root.p, kin.p, s));
    size_t tb3 = 0;
    CK(run_sort_pairs(nullptr, tb3, kin.p, kout.p, idx1.p, idx2.p, npts, 63, s));
    CK(ctx->d_tmp.reserve(std::max(tb3, tb2) + 256));
    CK(run_sort_pairs(ctx->d_tmp.p, tb3, kin.p, kout.p, idx1.p, idx2.p, npts, 63, s));
    // sorted keys: kout = sorted root; kin <- sorted path
    CK(run_gather_u64(npts, idx2.p, path.p, kin.p, s));
    CK(depth.reserve(npts)); CK(flag.reserve(npts)); CK(scan.reserve(npts));
    CK(run_leaves(npts, kout.p, kin.p, ctx->nmax, depth.p, flag.p, s));
    CK(run_scan_i32(ctx->d_tmp.p, tb2, flag.p, scan.p, npts, true, s));
    int32_t nb_all = 0;
    CK(cudaMemcpyAsync(&nb_all, scan.p + npts - 1, sizeof(int32_t), cudaMemcpyDeviceToHost, s));
    CK(cudaStreamSynchronize(s));
    CK(begin.reserve((size_t)nb_all + 1));
    CK(run_batch_begin(npts, flag.p, scan.p, begin.p, s));
    CK(bbox.reserve((size_t)nb_all * 6));
    CK(run_bbox(nb_all, begin.p, idx2.p, points, bbox.p, s));
    // ---- a1 pass 1: which batches have a non-empty B_j ----
    CK(cnt.reserve(nb_all));
    CK(cudaMemsetAsync(cnt.p, 0, (size_t)nb_all * sizeof(int32_t), s));
    CK(run_basis_screen(ctx->tab(), bbox.p, nullptr, nb_all, ctx->nshw, cnt.p, nullptr, s));
    std::vector<int64_t> h_begin((size_t)nb_all + 1);
    std::vector<int32_t> h_cnt(nb_all);
    CK(cudaMemcpyAsync(h_begin.data(), begin.p, h_begin.size() * sizeof(int64_t), cudaMemcpyDeviceToHost, s));
    CK(cudaMemcpyAsync(h_cnt.data(), cnt.p, h_cnt.size() * sizeof(int32_t), cudaMemcpyDeviceToHost, s));
    CK(cudaStreamSynchronize(s));
    int64_t slot = 0;
    for (int j = 0; j < nb_all; ++j) {
      if (h_cnt[j] == 0) continue;                 // batches with empty B_j are dropped (R10)
      const int n = (int)(h_begin[j + 1] - h_begin[j]);
      h_bsrc.push_back(j); h_bsrc_begin.push_back(h_begin[j]);
      ctx->h_bn.push_back(n); ctx->h_bslot.push_back(slot);
      ctx->sum_B += h_cnt[j];
      h_bcnt.push_back(h_cnt[j]);
      ctx->npts_kept += n;
      slot += (n + kSlotAlign - 1) / kSlotAlign * kSlotAlign;
    }
    ctx->nbatch = (int)ctx->h_bn.size();
    ctx->nslots = slot;
    for (int n : ctx->h_bn)      // k_maxima holds a batch in 16 x 256 registers; only > 4096 coincident points at depth 20 get here
      if (n > 4096) FAIL(SNK_EINVAL, "snk_set_grid: a batch holds more than 4096 points (coincident points beyond octree depth 20)");
    const int nb = ctx->nbatch;
    if (nb > 0) {
      DevBuf<int64_t> d_bsrc_begin;
      DevBuf<int32_t> d_bsrc;
      struct G2 { DevBuf<int64_t>& a; DevBuf<int32_t>& b; ~G2() { a.release(); b.release(); } } g2{d_bsrc_begin, d_bsrc};
      CK(upload(d_bsrc_begin, h_bsrc_begin)); CK(upload(d_bsrc, h_bsrc));
      CK(upload(ctx->d_bn, ctx->h_bn)); CK(upload(ctx->d_bslot, ctx->h_bslot));
      CK(ctx->d_bmask.reserve((size_t)nb * ctx->nshw));
      CK(run_basis_screen(ctx->tab(), bbox.p, d_bsrc.p, nb, ctx->nshw, nullptr, ctx->d_bmask.p, s));
      CK(ctx->gx.reserve(slot)); CK(ctx->gy.reserve(slot)); CK(ctx->gz.reserve(slot)); CK(ctx->gw.reserve(slot)); CK(ctx->slot_src.reserve(slot));
      CK(run_fill_slots(nb, d_bsrc_begin.p, ctx->d_bn.p, ctx->d_bslot.p, idx2.p, points, weights, ctx->gx.p, ctx->gy.p, ctx->gz.p,
                        ctx->gw.p, ctx->slot_src.p, s));
      // ---- Eq. 47 maxima (density independent) ----
      ctx->ldj = (nb + 7) / 8 * 8;
      CK(ctx->d_PhiTf.reserve((size_t)ctx->nbf * ctx->ldj)); CK(ctx->d_phit.reserve(nb));
      CK(cudaMemsetAsync(ctx->d_PhiTf.p, 0, (size_t)ctx->nbf * ctx->ldj * sizeof(double), s));
      CK(cudaMemsetAsync(ctx->d_phimax.p, 0, sizeof(unsigned long long), s));
      CK(run_maxima(ctx->tab(), nb, ctx->d_bn.p, ctx->d_bslot.p, ctx->gx.p, ctx->gy.p, ctx->gz.p, ctx->gw.p, ctx->d_bmask.p, ctx->nshw,
                    ctx->d_PhiTf.p, ctx->ldj, ctx->d_phit.p, ctx->d_phimax.p, s));
      // sum of nbf(B_j) for the stats (host, from the masks)
      std::vector<uint32_t> hm((size_t)nb * ctx->nshw);
      CK(cudaMemcpyAsync(hm.data(), ctx->d_bmask.p, hm.size() * sizeof(uint32_t), cudaMemcpyDeviceToHost, s));
      CK(cudaStreamSynchronize(s));
      ctx->flops_gemm_alg = 0.0;
      for (int j = 0; j < nb; ++j) {
        int64_t nf = 0;
        for (int a = 0; a < nsh; ++a)
          if ((hm[(size_t)j * ctx->nshw + (a >> 5)] >> (a & 31)) & 1u) nf += ncart(ctx->h_l[a]);
        ctx->sum_B_fn += nf;
        ctx->flops_gemm_alg += 2.0 * 2.0 * (double)ctx->h_bn[j] * (double)nf * ctx->nbf;      // a4 and a6
      }
      // ---- tiles and super-batches (Alg. 1 line 8: as many batches as fit the workspace) ----
      for (int j = 0; j < nb; ++j)
        for (int o = 0; o < ctx->h_bn[j]; o += kTile)
          ctx->h_tiles.push_back(TileRec{j, std::min(kTile, ctx->h_bn[j] - o), ctx->h_bslot[j] + o});
      const double budget = ctx->workspace_gb * 1073741824.0;
      int64_t max_slots = (int64_t)(budget / (3.0 * 8.0 * std::max(1, ctx->nbf)));
      max_slots = std::min<int64_t>(max_slots, (int64_t)500000000);           // the kernels address slab rows with a 32-bit byte stride
      max_slots = std::max<int64_t>(max_slots / 128 * 128, 4096 + kSlotAlign);
      int t = 0;
      for (int j = 0; j < nb;) {
        Super sp; sp.b0 = j; sp.slot0 = ctx->h_bslot[j]; sp.t0 = t;
        int64_t n = 0;
        while (j < nb) {
          const int64_t pad = (ctx->h_bn[j] + kSlotAlign - 1) / kSlotAlign * kSlotAlign;
          if (n > 0 && n + pad > max_slots) break;
          n += pad;
          t += (ctx->h_bn[j] + kTile - 1) / kTile;
          ++j;
        }
        sp.b1 = j; sp.nslots = n; sp.t1 = t;
        ctx->supers.push_back(sp);
      }
      // The CTAs of a launch run in tile order and a tile's integral work grows with its points and with the pairs among the
      // shells of B_j: heaviest tiles first inside every super-batch, so that the launch does not end on a few long CTAs.
      for (const Super& sp : ctx->supers)
        std::stable_sort(ctx->h_tiles.begin() + sp.t0, ctx->h_tiles.begin() + sp.t1, [&](const TileRec& x, const TileRec& y) {
          return (double)x.n * h_bcnt[x.batch] * h_bcnt[x.batch] > (double)y.n * h_bcnt[y.batch] * h_bcnt[y.batch];
        });
      CK(upload(ctx->d_tiles, ctx->h_tiles));
      {   // chunks of whole batches (<= kChunkSlots slots, never across super-batches), their row lists, a4 column tiles
        std::vector<ChunkRec> h_chunks;
        std::vector<ColTile> h_ct;
        for (Super& sp : ctx->supers) {
          sp.c0 = (int)h_chunks.size(); sp.ct0 = (int)h_ct.size();
          for (int j = sp.b0; j < sp.b1;) {
            ChunkRec ch; ch.slot0 = ctx->h_bslot[j]; ch.b0 = j; ch.pad = 0;
            int64_t n = 0;
            while (j < sp.b1) {
              const int64_t pad = (ctx->h_bn[j] + kSlotAlign - 1) / kSlotAlign * kSlotAlign;
              if (n > 0 && n + pad > kChunkSlots) break;
              n += pad; ++j;
            }
            ch.b1 = j; ch.nslots = (int32_t)n;
            for (int64_t o = 0; o < n; o += 128) h_ct.push_back(ColTile{ch.slot0 + o, (int32_t)h_chunks.size(), (int32_t)std::min<int64_t>(128, n - o)});
            h_chunks.push_back(ch);
          }
          sp.c1 = (int)h_chunks.size(); sp.ct1 = (int)h_ct.size();
        }
        const int nch = (int)h_chunks.size();
        ctx->lstride = (ctx->nbf + 3) / 4 * 4;
        CK(upload(ctx->d_chunks, h_chunks)); CK(upload(ctx->d_ctiles, h_ct));
        CK(ctx->d_rowlist.reserve((size_t)nch * ctx->lstride)); CK(ctx->d_nrows.reserve(nch));
        CK(run_chunk_rows(ctx->tab(), nch, ctx->d_chunks.p, ctx->d_bmask.p, ctx->nshw, ctx->d_rowlist.p, ctx->lstride, ctx->d_nrows.p, s));
        std::vector<int32_t> h_nrows(nch);
        CK(cudaMemcpyAsync(h_nrows.data(), ctx->d_nrows.p, (size_t)nch * sizeof(int32_t), cudaMemcpyDeviceToHost, s));
        CK(cudaStreamSynchronize(s));
        // executed flops: a4 2 nbf (L padded to the k-tile) columns; a6 2 (L padded to the row tile) slots nbf
        ctx->flops_F = ctx->flops_Kt = 0.0;
        const int tk = f_k_tile(), ta = kt_row_tile();
        for (Super& sp : ctx->supers) {
          sp.max_nrow = 0;
          for (int c = sp.c0; c < sp.c1; ++c) {
            const int nr = h_nrows[c];
            sp.max_nrow = std::max(sp.max_nrow, nr);
            ctx->flops_F += 2.0 * ctx->nbf * (double)((nr + tk - 1) / tk * tk) * h_chunks[c].nslots;
            ctx->flops_Kt += 2.0 * (double)((nr + ta - 1) / ta * ta) * h_chunks[c].nslots * ctx->nbf;
          }
        }
      }
      int64_t ld = 0;
      for (const Super& sp : ctx->supers) ld = std::max(ld, sp.nslots);
      ctx->ld = (ld + 127) / 128 * 128;
      const size_t slab = (size_t)ctx->nbf * ctx->ld;
      CK(ctx->d_Phi.reserve(slab)); CK(ctx->d_F.reserve(slab)); CK(ctx->d_G.reserve(slab));
    }
  }
  CK(ctx->d_Kt.reserve((size_t)ctx->nbf * ctx->nbf));
  CK(cudaEventRecord(ctx->ev_g1, s));
  CK(cudaStreamSynchronize(s));
  float ms = 0;
  cudaEventElapsedTime(&ms, ctx->ev_g0, ctx->ev_g1);
  std::memset(&ctx->stats, 0, sizeof(ctx->stats));
  ctx->stats.ms_set_grid = ms;
  ctx->have_grid = true;
  return SNK_OK;
  });
}

static int build_impl(snk_ctx* ctx, const double* P, double* K, void* stream_, bool screen_only) {
  return guarded(ctx, [&]() -> int {
  if (!ctx) return SNK_EINVAL;
  if (!P || (!K && !screen_only)) FAIL(SNK_EINVAL, "snk_build_K: NULL pointer");
  CHECK_DEVICE();
  if (!ctx->have_grid) FAIL(SNK_ESTATE, "snk_build_K called before snk_set_grid");
  cudaStream_t s = (cudaStream_t)stream_;
  ctx->last_stream = s;
  ctx->stats_valid = false; ctx->have_build = false; ctx->have_screen = false;
  ctx->spans.clear(); ctx->ev_used = 0; ctx->gemm_flops = 0.0; ctx->n_launches = 0;
  const int nbf = ctx->nbf, nsh = ctx->nsh, nb = ctx->nbatch;
  const ShellTab tab = ctx->tab();
  CK(cudaEventRecord(ctx->ev_b0, s));
  if (nb == 0) {
    if (K) CK(cudaMemsetAsync(K, 0, (size_t)nbf * nbf * sizeof(double), s));
    CK(cudaEventRecord(ctx->ev_b1, s));
    ctx->npair_sig = 0; ctx->nunit = 0; ctx->nprimpair = 0; ctx->have_build = true;
    return SNK_OK;
  }
  // SNK_TRACE=1: synchronise after every stage and report it on stderr (debugging aid; perturbs the timings)
  static const bool trace = getenv("SNK_TRACE") != nullptr;
  auto tr = [&](const char* what, int a, int b) {
    if (!trace) return;
    const cudaError_t e = cudaStreamSynchronize(s);
    fprintf(stderr, "[snk] %s %d/%d: %s\n", what, a, b, cudaGetErrorString(e));
  };
  cudaError_t span_rc = cudaSuccess;          // first failure of the timing events (checked with CK after every span)
  auto span_begin = [&](int stage, int cls) {
    snk_ctx::Span sp{stage, cls, -1, -1};
    cudaError_t e = ctx->new_event(sp.e0);
    if (e == cudaSuccess) e = cudaEventRecord(ctx->ev_pool[sp.e0], s);
    if (span_rc == cudaSuccess) span_rc = e;
    return sp;
  };
  auto span_end = [&](snk_ctx::Span sp) {
    cudaError_t e = ctx->new_event(sp.e1);
    if (e == cudaSuccess) e = cudaEventRecord(ctx->ev_pool[sp.e1], s);
    if (span_rc == cudaSuccess) span_rc = e;
    if (sp.e0 >= 0 && sp.e1 >= 0) ctx->spans.push_back(sp);
  };

  // ---- a3: density-dependent screening (Eqs. 43-47) ----
  auto sp = span_begin(ST_SCREEN, -1);
  const int64_t ncand = ctx->cand.off[kNumClasses];
  CK(ctx->d_absP.reserve((size_t)nbf * nbf)); CK(ctx->d_Ftf.reserve((size_t)nbf * ctx->ldj)); CK(ctx->d_FtsT.reserve((size_t)nb * nsh));
  CK(ctx->d_flag.reserve(ncand)); CK(ctx->d_np.reserve(ncand)); CK(ctx->d_pos.reserve(ncand)); CK(ctx->d_ppos.reserve(ncand));
  CK(run_abs((int64_t)nbf * nbf, P, ctx->d_absP.p, s));
  CK(gemm_f64(false, nbf, nb, nbf, ctx->d_absP.p, nbf, ctx->d_PhiTf.p, ctx->ldj, ctx->d_Ftf.p, ctx->ldj, false, nullptr, s));
  ctx->gemm_flops += 2.0 * nbf * (double)nb * nbf;
  CK(cudaMemsetAsync(ctx->d_Fmax.p, 0, (size_t)nsh * sizeof(unsigned long long), s));
  CK(run_shell_max(tab, nb, ctx->d_Ftf.p, ctx->ldj, ctx->d_FtsT.p, nsh, ctx->d_Fmax.p, s));
  CK(run_pair_flags(ctx->cand, tab, ctx->d_Atil.p, (const double*)ctx->d_Fmax.p, (const double*)ctx->d_phimax.p, ctx->eps, ctx->d_flag.p,
                    ctx->d_np.p, s));
  size_t tb = 0;
  CK(run_scan_i32(nullptr, tb, nullptr, nullptr, ncand, false, s));
  CK(ctx->d_tmp.reserve(tb + 256));
  CK(run_scan_i32(ctx->d_tmp.p, tb, ctx->d_flag.p, ctx->d_pos.p, ncand, false, s));
  CK(run_scan_i32(ctx->d_tmp.p, tb, ctx->d_np.p, ctx->d_ppos.p, ncand, false, s));
  // list sizes: the one synchronisation of the build
  int32_t h_last[4] = {0, 0, 0, 0};
  int32_t h_cls[kNumClasses] = {0};
  CK(cudaMemcpyAsync(&h_last[0], ctx->d_pos.p + ncand - 1, 4, cudaMemcpyDeviceToHost, s));
  CK(cudaMemcpyAsync(&h_last[1], ctx->d_flag.p + ncand - 1, 4, cudaMemcpyDeviceToHost, s));
  CK(cudaMemcpyAsync(&h_last[2], ctx->d_ppos.p + ncand - 1, 4, cudaMemcpyDeviceToHost, s));
  CK(cudaMemcpyAsync(&h_last[3], ctx->d_np.p + ncand - 1, 4, cudaMemcpyDeviceToHost, s));
  for (int c = 0; c < kNumClasses; ++c)
    if (ctx->cand.off[c] < ncand) CK(cudaMemcpyAsync(&h_cls[c], ctx->d_pos.p + ctx->cand.off[c], 4, cudaMemcpyDeviceToHost, s));
  CK(cudaStreamSynchronize(s));
  const int nunit = h_last[0] + h_last[1];
  const int npair = h_last[2] + h_last[3];
  for (int c = 0; c < kNumClasses; ++c) ctx->cls_beg[c] = ctx->cand.off[c] < ncand ? h_cls[c] : nunit;
  ctx->cls_beg[kNumClasses] = nunit;
  ctx->npair_sig = npair; ctx->nunit = nunit;
  ctx->vstride = (nunit + 31) / 32 + 1;
  CK(ctx->d_units.reserve((size_t)std::max(nunit, 1) * kUnitBytes)); CK(ctx->d_meta.reserve(std::max(nunit, 1)));
  CK(ctx->d_vmask.reserve((size_t)nb * ctx->vstride));
  {   // unit-id lists: one row of nunit ints per batch of the largest super-batch (a class's slot is as long as the class)
    int max_nb = 1;
    for (const Super& su : ctx->supers) max_nb = std::max(max_nb, su.b1 - su.b0);
    CK(ctx->d_vlist.reserve((size_t)max_nb * std::max(nunit, 1))); CK(ctx->d_vcnt.reserve((size_t)max_nb * kNumClasses));
  }
  CK(run_unit_fill(ctx->cand, tab, ctx->d_flag.p, ctx->d_pos.p, ctx->d_Atil.p, 1e-4 * ctx->eps, (const double*)ctx->d_Fmax.p,
                   (const double*)ctx->d_phimax.p, ctx->ld, ctx->d_units.p, ctx->d_meta.p, s));
  CK(cudaMemsetAsync(ctx->d_vmask.p, 0, (size_t)nb * ctx->vstride * sizeof(uint32_t), s));
  CK(run_vmask(nb, nunit, ctx->d_meta.p, ctx->d_FtsT.p, nsh, ctx->d_phit.p, ctx->eps, ctx->d_vmask.p, ctx->vstride, s));
  ctx->n_launches += 6;
  span_end(sp);
  tr("screen", nunit, npair);
  ctx->have_screen = true;
  if (screen_only) {
    CK(span_rc);
    CK(cudaEventRecord(ctx->ev_b1, s));
    return SNK_OK;
  }

  CK(cudaMemsetAsync(ctx->d_Kt.p, 0, (size_t)nbf * nbf * sizeof(double), s));
  for (const Super& su : ctx->supers) {
    const int ntiles = su.t1 - su.t0;
    // ---- a2: collocation ----
    sp = span_begin(ST_COLLOC, -1);
    CK(run_colloc(tab, ctx->d_tiles.p + su.t0, ntiles, ctx->gx.p, ctx->gy.p, ctx->gz.p, ctx->d_bmask.p, ctx->nshw, ctx->d_Phi.p, ctx->ld,
                  su.slot0, s));
    span_end(sp);
    // ---- a4: F = P * Phi ----
    sp = span_begin(ST_F, -1);
    tr("colloc", (int)(&su - ctx->supers.data()), (int)ctx->supers.size());
    CK(gemm_f(nbf, su.slot0, su.ct1 - su.ct0, ctx->d_ctiles.p + su.ct0, su.c0, ctx->d_nrows.p + su.c0,
              ctx->d_rowlist.p + (int64_t)su.c0 * ctx->lstride, ctx->lstride, P, ctx->d_Phi.p, ctx->d_F.p, ctx->ld, s));
    span_end(sp);
    tr("F", (int)(&su - ctx->supers.data()), (int)ctx->supers.size());
    // ---- a5: G ----
    sp = span_begin(ST_G, -1);
    CK(cudaMemsetAsync(ctx->d_G.p, 0, (size_t)nbf * ctx->ld * sizeof(double), s));
    IntParams ip;
    ip.gx = ctx->gx.p; ip.gy = ctx->gy.p; ip.gz = ctx->gz.p; ip.F = ctx->d_F.p; ip.G = ctx->d_G.p; ip.ld = ctx->ld; ip.slot0 = su.slot0;
    ip.tiles = ctx->d_tiles.p + su.t0; ip.ntiles = ntiles;
    CK(run_vlist(su.b0, su.b1 - su.b0, ctx->cls_beg, ctx->d_vmask.p, ctx->vstride, ctx->d_vlist.p, nunit, ctx->d_vcnt.p, s));
    ctx->n_launches += 1;
    ip.vlist = ctx->d_vlist.p; ip.vlstride = nunit; ip.vcnt = ctx->d_vcnt.p; ip.b0 = su.b0;
    ip.units = ctx->d_units.p; ip.meta = ctx->d_meta.p; ip.boys = ctx->d_boys.p;
    // CTAs per tile (each takes a contiguous share of the tile's unit list), chosen per class:
    //  * L2: the CTAs of a launch that are resident at one time (about 3 per SM) re-read the F rows of their tiles once per
    //    partner shell; with one tile per CTA those F blocks (nbf x 1 KB each) are hundreds of MB and the re-reads go to HBM.
    //    Sharing a tile among n CTAs divides the resident blocks by n: n is set so that they fit about 48 MB of the 126 MB L2
    //    (measured: config 3 build 1316 -> 1262 ms at n = 4..8, reduced-grid config 4 18.7 -> 16.8 s from n = 4 to 32);
    //  * tail: a launch with few tiles (large basis, small super-batch) would leave its last wave mostly empty;
    //  * but a CTA should keep about a thousand units of the class, else the per-CTA set-up shows (d-d: 60 % slower at n = 16).
    auto split_for = [&](int c) {
      if (ctx->tile_split > 0) return ctx->tile_split;
      const int by_units = std::max(1, (ctx->cls_beg[c + 1] - ctx->cls_beg[c]) / 1024);
      const int by_l2 = (int)std::ceil(3.0 * ctx->sm_count * (double)nbf * 1024.0 / 48e6);
      const int by_tail = 4000 / std::max(1, ntiles);
      return std::max(1, std::min(std::min(32, by_units), std::max(by_l2, by_tail)));
    };
    for (int c = 0; c < kNumClasses; ++c) {
      ip.pbeg = ctx->cls_beg[c]; ip.pend = ctx->cls_beg[c + 1]; ip.cls = c; ip.nsplit = split_for(c);
      if (ip.pend <= ip.pbeg) continue;
      auto spc = span_begin(ST_COUNT, c);
      CK(launch_integrals(c, ip, s));
      ctx->n_launches += 1;
      span_end(spc);
      tr("G class", c, kNumClasses);
    }
    span_end(sp);
    // ---- a6: Kt += Phi diag(w) G^T ----
    sp = span_begin(ST_KT, -1);
    CK(gemm_kt(nbf, su.slot0, su.c1 - su.c0, su.max_nrow, ctx->d_chunks.p + su.c0, ctx->d_nrows.p + su.c0,
               ctx->d_rowlist.p + (int64_t)su.c0 * ctx->lstride, ctx->lstride, ctx->d_Phi.p, ctx->d_G.p, ctx->ld, ctx->gw.p, ctx->d_Kt.p, s));
    ctx->n_launches += 3;   // collocation, F GEMM, Kt GEMM
    span_end(sp);
    tr("Kt", (int)(&su - ctx->supers.data()), (int)ctx->supers.size());
  }
  ctx->gemm_flops += ctx->flops_F + ctx->flops_Kt;
  // ---- a7 ----
  sp = span_begin(ST_SYM, -1);
  CK(run_symmetrise(nbf, ctx->d_Kt.p, K, s));
  ctx->n_launches += 1;
  span_end(sp);
  CK(span_rc);
  CK(cudaEventRecord(ctx->ev_b1, s));
  ctx->have_build = true;
  return SNK_OK;
  });
}

int snk_build_K(snk_ctx* ctx, const double* P, double* K, void* stream_) { return build_impl(ctx, P, K, stream_, false); }

int snk_screen(snk_ctx* ctx, const double* P, void* stream_) { return build_impl(ctx, P, nullptr, stream_, true); }

int snk_batch_costs(snk_ctx* ctx, double* cost) {
  return guarded(ctx, [&]() -> int {
  if (!ctx) return SNK_EINVAL;
  if (!cost) FAIL(SNK_EINVAL, "snk_batch_costs: NULL pointer");
  CHECK_DEVICE();
  if (!ctx->have_grid || !ctx->have_screen) FAIL(SNK_ESTATE, "snk_batch_costs needs snk_set_grid and snk_screen / snk_build_K first");
  cudaStream_t s = ctx->last_stream;
  const int nb = ctx->nbatch;
  if (nb == 0) return SNK_OK;
  DevBuf<double> d;
  CK(d.reserve(nb));
  CK(run_batch_costs(nb, ctx->nunit, ctx->d_meta.p, ctx->d_bn.p, ctx->d_vmask.p, ctx->vstride, d.p, s));
  CK(cudaMemcpyAsync(cost, d.p, (size_t)nb * sizeof(double), cudaMemcpyDeviceToHost, s));
  CK(cudaStreamSynchronize(s));
  return SNK_OK;
  });
}

int snk_build_K_host(snk_ctx* ctx, const double* P_host, double* K_host, void* stream_) {
  return guarded(ctx, [&]() -> int {
  if (!ctx) return SNK_EINVAL;
  if (!P_host || !K_host) FAIL(SNK_EINVAL, "snk_build_K_host: NULL pointer");
  CHECK_DEVICE();
  cudaStream_t s = (cudaStream_t)stream_;
  const size_t n = (size_t)ctx->nbf * ctx->nbf;
  CK(ctx->d_Pin.reserve(n)); CK(ctx->d_Kout.reserve(n));
  CK(cudaMemcpyAsync(ctx->d_Pin.p, P_host, n * sizeof(double), cudaMemcpyHostToDevice, s));
  const int rc = snk_build_K(ctx, ctx->d_Pin.p, ctx->d_Kout.p, stream_);
  if (rc != SNK_OK) return rc;
  CK(cudaMemcpyAsync(K_host, ctx->d_Kout.p, n * sizeof(double), cudaMemcpyDeviceToHost, s));
  CK(cudaStreamSynchronize(s));
  return SNK_OK;
  });
}

int snk_get_stats(snk_ctx* ctx, snk_stats* out) {
  return guarded(ctx, [&]() -> int {
  if (!ctx || !out) return SNK_EINVAL;
  CHECK_DEVICE();
  cudaStream_t s = ctx->last_stream;
  CK(cudaStreamSynchronize(s));
  snk_stats& st = ctx->stats;
  st.npts = ctx->npts; st.npts_kept = ctx->npts_kept; st.nbatch = ctx->nbatch; st.sum_B = ctx->sum_B; st.sum_B_fn = ctx->sum_B_fn;
  st.nsuper = (int64_t)ctx->supers.size();
  if (ctx->have_build && !ctx->stats_valid) {
    if (ctx->nunit > 0) {      // primitive pairs kept (R14): from the unit metadata, off the timed path
      std::vector<UnitMeta> hm(ctx->nunit);
      CK(cudaMemcpyAsync(hm.data(), ctx->d_meta.p, hm.size() * sizeof(UnitMeta), cudaMemcpyDeviceToHost, s));
      CK(cudaStreamSynchronize(s));
      ctx->nprimpair = 0;
      for (const UnitMeta& m : hm) ctx->nprimpair += m.nprim_first & 0xff;
    }
    st.npair_sig = ctx->npair_sig; st.nprimpair = ctx->nprimpair; st.flops_gemm = ctx->gemm_flops;
    double h[32] = {0};
    if (ctx->nbatch > 0 && ctx->nunit > 0) {
      CK(cudaMemsetAsync(ctx->d_stats.p, 0, 32 * sizeof(double), s));
      CK(run_vstats(ctx->nbatch, ctx->nunit, ctx->d_meta.p, ctx->tab(), ctx->d_bn.p, ctx->d_vmask.p, ctx->vstride, ctx->d_cflops.p,
                    ctx->d_cflops.p + kNumClasses, ctx->d_stats.p, s));
      CK(cudaMemcpyAsync(h, ctx->d_stats.p, 32 * sizeof(double), cudaMemcpyDeviceToHost, s));
      CK(cudaStreamSynchronize(s));
    }
    st.sum_V = (int64_t)h[0]; st.n_pairpoints = h[1]; st.n_int_contracted = h[2]; st.n_int_primitive = h[3];
    for (int c = 0; c < kNumClasses; ++c) { st.n_int_class[c] = h[4 + c]; st.flops_class[c] = h[16 + c]; }
    st.n_launches = ctx->n_launches;
    st.flops_gemm_alg = ctx->flops_gemm_alg;
    st.flops_integral = h[14];
    double acc[ST_COUNT] = {0};
    for (int c = 0; c < kNumClasses; ++c) st.ms_G_class[c] = 0.0;
    for (const auto& sp : ctx->spans) {
      float ms = 0;
      cudaEventElapsedTime(&ms, ctx->ev_pool[sp.e0], ctx->ev_pool[sp.e1]);
      if (sp.stage == ST_COUNT) st.ms_G_class[sp.cls] += ms; else acc[sp.stage] += ms;
    }
    st.ms_screen = acc[ST_SCREEN]; st.ms_colloc = acc[ST_COLLOC]; st.ms_F = acc[ST_F]; st.ms_G = acc[ST_G]; st.ms_Kt = acc[ST_KT];
    st.ms_sym = acc[ST_SYM];
    float ms = 0;
    cudaEventElapsedTime(&ms, ctx->ev_b0, ctx->ev_b1);
    st.ms_build = ms;
    ctx->stats_valid = true;
  }
  *out = st;
  return SNK_OK;
  });
}

int snk_export_lists(snk_ctx* ctx, int64_t* sizes, int64_t* batch_off, int64_t* perm, int64_t* B_off, int32_t* B_ids, int64_t* V_off,
                     int32_t* V_pairs) {
  return guarded(ctx, [&]() -> int {
  if (!ctx || !sizes) return SNK_EINVAL;
  CHECK_DEVICE();
  if (!ctx->have_grid) FAIL(SNK_ESTATE, "snk_export_lists before snk_set_grid");
  cudaStream_t s = ctx->last_stream;
  CK(cudaStreamSynchronize(s));
  const int nb = ctx->nbatch, nsh = ctx->nsh;
  snk_stats st;
  const int rc = snk_get_stats(ctx, &st);
  if (rc != SNK_OK) return rc;
  sizes[0] = nb; sizes[1] = ctx->npts_kept; sizes[2] = ctx->sum_B; sizes[3] = ctx->have_build ? st.sum_V : 0;
  if (batch_off) {
    int64_t o = 0;
    for (int j = 0; j < nb; ++j) { batch_off[j] = o; o += ctx->h_bn[j]; }
    batch_off[nb] = o;
  }
  if (perm && nb > 0) {
    std::vector<int64_t> src(ctx->nslots);
    CK(cudaMemcpy(src.data(), ctx->slot_src.p, src.size() * sizeof(int64_t), cudaMemcpyDeviceToHost));
    int64_t o = 0;
    for (int j = 0; j < nb; ++j)
      for (int i = 0; i < ctx->h_bn[j]; ++i) perm[o++] = src[ctx->h_bslot[j] + i];
  }
  if ((B_off || B_ids) && nb > 0) {
    std::vector<uint32_t> hm((size_t)nb * ctx->nshw);
    CK(cudaMemcpy(hm.data(), ctx->d_bmask.p, hm.size() * sizeof(uint32_t), cudaMemcpyDeviceToHost));
    int64_t o = 0;
    for (int j = 0; j < nb; ++j) {
      if (B_off) B_off[j] = o;
      for (int a = 0; a < nsh; ++a)
        if ((hm[(size_t)j * ctx->nshw + (a >> 5)] >> (a & 31)) & 1u) { if (B_ids) B_ids[o] = a; ++o; }
    }
    if (B_off) B_off[nb] = o;
  } else if (B_off) B_off[0] = 0;
  if ((V_off || V_pairs) && nb > 0) {
    if (!ctx->have_build) FAIL(SNK_ESTATE, "snk_export_lists: V_j need a prior snk_build_K");
    const int np = ctx->nunit;
    std::vector<UnitMeta> hp(std::max(np, 1));
    std::vector<uint32_t> hv((size_t)nb * ctx->vstride);
    if (np > 0) CK(cudaMemcpy(hp.data(), ctx->d_meta.p, (size_t)np * sizeof(UnitMeta), cudaMemcpyDeviceToHost));
    CK(cudaMemcpy(hv.data(), ctx->d_vmask.p, hv.size() * sizeof(uint32_t), cudaMemcpyDeviceToHost));
    int64_t o = 0;
    std::vector<std::pair<int32_t, int32_t>> tmp;
    for (int j = 0; j < nb; ++j) {
      if (V_off) V_off[j] = o;
      tmp.clear();
      for (int i = 0; i < np; ++i)
        if (((hv[(size_t)j * ctx->vstride + (i >> 5)] >> (i & 31)) & 1u) && ((hp[i].nprim_first >> 8) & 1))
          tmp.emplace_back(std::min(hp[i].sa, hp[i].sb), std::max(hp[i].sa, hp[i].sb));
      std::sort(tmp.begin(), tmp.end());
      for (auto& ab : tmp) { if (V_pairs) { V_pairs[2 * o] = ab.first; V_pairs[2 * o + 1] = ab.second; } ++o; }
    }
    if (V_off) V_off[nb] = o;
  } else if (V_off) V_off[0] = 0;
  return SNK_OK;
  });
}

int snk_debug_boys(int32_t mmax, int64_t n, const double* x, double* out, void* stream_) {
  return guarded((snk_ctx*)nullptr, [&]() -> int {
  if (mmax < 0 || mmax > 6 || n < 0 || (n > 0 && (!x || !out))) return SNK_EINVAL;
  static DevBuf<double> tabs[kMaxDevices];      // process-lifetime table of the hook, one per device
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) return SNK_ECUDA;
  DevBuf<double>& tab = tabs[dev];
  if (!tab.p) {
    if (upload(tab, make_boys_table()) != cudaSuccess) return SNK_ECUDA;
  }
  return launch_debug_boys(mmax, n, x, tab.p, out, (cudaStream_t)stream_) == cudaSuccess ? SNK_OK : SNK_ECUDA;
  });
}

int snk_debug_A_pair(snk_ctx* ctx, int32_t a, int32_t b, int64_t n, const double* pts, double* out, void* stream_) {
  return guarded(ctx, [&]() -> int {
  if (!ctx) return SNK_EINVAL;
  if (a < 0 || b < 0 || a >= ctx->nsh || b >= ctx->nsh || n < 0 || (n > 0 && (!pts || !out))) FAIL(SNK_EINVAL, "snk_debug_A_pair: bad argument");
  CHECK_DEVICE();
  cudaStream_t s = (cudaStream_t)stream_;
  const bool tr = ctx->h_l[a] < ctx->h_l[b];
  const int sa = tr ? b : a, sb = tr ? a : b;
  const double A[3] = {ctx->h_cx[sa], ctx->h_cy[sa], ctx->h_cz[sa]}, B[3] = {ctx->h_cx[sb], ctx->h_cy[sb], ctx->h_cz[sb]};
  const double AB[3] = {A[0] - B[0], A[1] - B[1], A[2] - B[2]};
  const double AB2 = AB[0] * AB[0] + AB[1] * AB[1] + AB[2] * AB[2];
  std::vector<PrimPair> pp;
  for (int k = 0; k < ctx->h_nprim[sa]; ++k)
    for (int l = 0; l < ctx->h_nprim[sb]; ++l) {
      const double za = ctx->h_pexp[ctx->h_poff[sa] + k], zb = ctx->h_pexp[ctx->h_poff[sb] + l];
      PrimPair q;
      const double ps = za + zb;
      q.p2 = 2.0 * ps; q.inv2p = 0.5 / ps;
      q.Px = (za * A[0] + zb * B[0]) / ps; q.Py = (za * A[1] + zb * B[1]) / ps; q.Pz = (za * A[2] + zb * B[2]) / ps;
      q.PAx = q.Px - A[0]; q.PAy = q.Py - A[1]; q.PAz = q.Pz - A[2];
      q.pref = ctx->h_pcoef[ctx->h_poff[sa] + k] * ctx->h_pcoef[ctx->h_poff[sb] + l] * (2.0 * M_PI / ps) * std::exp(-(za * zb / ps) * AB2);
      q.cfar2 = 1.2533141373155002512 * q.pref;
      pp.push_back(q);
    }
  DevBuf<PrimPair> d;
  CK(d.reserve(pp.size()));
  CK(cudaMemcpyAsync(d.p, pp.data(), pp.size() * sizeof(PrimPair), cudaMemcpyHostToDevice, s));
  cudaError_t e = launch_debug_A(ctx->h_l[sa], ctx->h_l[sb], tr, d.p, (int)pp.size(), AB[0], AB[1], AB[2], pts, n, ctx->d_boys.p, out, s);
  cudaError_t e2 = cudaStreamSynchronize(s);
  d.release();
  CK(e); CK(e2);
  return SNK_OK;
  });
}

int snk_A_pair_noalloc(snk_ctx* ctx, int32_t a, int32_t b, int64_t n, const double* pts, double* out, void* stream_) {
  return guarded(ctx, [&]() -> int {
  if (!ctx) return SNK_EINVAL;
  if (a < 0 || b < 0 || a >= ctx->nsh || b >= ctx->nsh || n < 0 || (n > 0 && (!pts || !out))) FAIL(SNK_EINVAL, "snk_A_pair_noalloc: bad argument");
  CHECK_DEVICE();
  cudaStream_t s = (cudaStream_t)stream_;
  const bool tr = ctx->h_l[a] < ctx->h_l[b];
  const int sa = tr ? b : a, sb = tr ? a : b;
  const int np = ctx->h_nprim[sa] * ctx->h_nprim[sb];
  if (np > kNoAllocMaxPrims)
    FAIL(SNK_EINVAL, "snk_A_pair_noalloc: the shell pair has more than 1024 primitive pairs (the fixed scratch); use snk_debug_A_pair");
  PrimPair* scratch = nullptr;
  CK(noalloc_scratch(ctx->device, &scratch));
  if (n == 0) return SNK_OK;
  k_noalloc_prims<<<(np + 127) / 128, 128, 0, s>>>(ctx->tab(), sa, sb, scratch);
  CK(cudaGetLastError());
  const double AB[3] = {ctx->h_cx[sa] - ctx->h_cx[sb], ctx->h_cy[sa] - ctx->h_cy[sb], ctx->h_cz[sa] - ctx->h_cz[sb]};
  CK(launch_debug_A(ctx->h_l[sa], ctx->h_l[sb], tr, scratch, np, AB[0], AB[1], AB[2], pts, n, ctx->d_boys.p, out, s));
  return SNK_OK;
  });
}

int snk_measure_fp64_peak(double* dfma_tflops, double* dmma_tflops, int32_t reps) {
  return guarded((snk_ctx*)nullptr, [&]() -> int {
  if (!dfma_tflops || !dmma_tflops || reps < 1) return SNK_EINVAL;
  return run_fp64_peak(dfma_tflops, dmma_tflops, reps) == cudaSuccess ? SNK_OK : SNK_ECUDA;
  });
}

}  // extern "C"
