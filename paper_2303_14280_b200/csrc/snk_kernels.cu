// snk_kernels.cu -- everything on the path except the integral kernel and the GEMM:
//   a0 batching keys / leaves / bboxes (R13)       a1 B_j sphere-box tests (Eq. 41)
//   Eq. 47 maxima   a3 pair screening (Eqs. 43-46)  a2 collocation (Eq. 31)   a7 symmetrise (Eq. 40)
#include <cub/cub.cuh>

#include "snk_internal.h"
#include "snk_kernels.h"
#include "snk_os.cuh"

namespace snk {

// ------------------------------------------------------------------------------------------------------------
// a0: keys.  root cell = floor(x/h0) per axis (21 bits each, biased); path = 3 bits per octree level, 20 levels,
// child bit = (coordinate >= geometric midpoint) -> points on a split plane go to the upper child (R13).
// ------------------------------------------------------------------------------------------------------------
__global__ void k_point_keys(int64_t n, const double* __restrict__ pts, const double* __restrict__ w, double h0,
                             unsigned long long* __restrict__ root, unsigned long long* __restrict__ path, uint32_t* __restrict__ idx,
                             int* __restrict__ err) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const double c[3] = {pts[3 * i], pts[3 * i + 1], pts[3 * i + 2]};
  const double wi = w[i];
  if (!(wi >= 0.0) || isinf(wi)) atomicOr(err, 1);
  unsigned long long r = 0, p = 0;
  double lo[3], hi[3];
  bool bad = false;
#pragma unroll
  for (int q = 0; q < 3; ++q) {
    if (!isfinite(c[q])) { bad = true; lo[q] = hi[q] = 0; continue; }
    const double f = floor(c[q] / h0);
    if (fabs(f) >= 1048575.0) { bad = true; lo[q] = hi[q] = 0; continue; }
    const long long ic = (long long)f;
    r = (r << 21) | (unsigned long long)(ic + 1048576);
    lo[q] = (double)ic * h0;
    hi[q] = (double)(ic + 1) * h0;
  }
  if (bad) { atomicOr(err, 2); r = 0; }
  for (int d = 0; d < kMaxDepth; ++d) {
    unsigned b = 0;
#pragma unroll
    for (int q = 0; q < 3; ++q) {
      const double mid = 0.5 * (lo[q] + hi[q]);
      const bool up = c[q] >= mid;
      b = (b << 1) | (up ? 1u : 0u);
      if (up) lo[q] = mid; else hi[q] = mid;
    }
    p = (p << 3) | b;
  }
  root[i] = r; path[i] = p; idx[i] = (uint32_t)i;
}

template <class T>
__global__ void k_gather(int64_t n, const uint32_t* __restrict__ idx, const T* __restrict__ src, T* __restrict__ dst) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) dst[i] = src[idx[i]];
}

// number of points sharing (root, first d levels of path) with sorted position i
__device__ __forceinline__ int64_t node_count(const unsigned long long* __restrict__ root, const unsigned long long* __restrict__ path,
                                              int64_t n, int64_t i, int d) {
  const int sh = 3 * (kMaxDepth - d);
  const unsigned long long r = root[i], pf = sh >= 60 ? 0ull : (path[i] >> sh);
  auto less = [&](int64_t k) {      // key(k) < key(i)
    const unsigned long long rk = root[k];
    if (rk != r) return rk < r;
    const unsigned long long pk = sh >= 60 ? 0ull : (path[k] >> sh);
    return pk < pf;
  };
  auto leq = [&](int64_t k) {       // key(k) <= key(i)
    const unsigned long long rk = root[k];
    if (rk != r) return rk < r;
    const unsigned long long pk = sh >= 60 ? 0ull : (path[k] >> sh);
    return pk <= pf;
  };
  int64_t a = 0, b = i;             // first k with !less(k) in [0, i]
  while (a < b) { const int64_t m = (a + b) >> 1; if (less(m)) a = m + 1; else b = m; }
  const int64_t first = a;
  a = i; b = n;                     // first k with !leq(k) in [i, n]
  while (a < b) { const int64_t m = (a + b) >> 1; if (leq(m)) a = m + 1; else b = m; }
  return a - first;
}

// leaf depth of every sorted point: smallest d whose node holds <= nmax points (else kMaxDepth); start flags
__global__ void k_leaf_depth(int64_t n, const unsigned long long* __restrict__ root, const unsigned long long* __restrict__ path, int nmax,
                             uint8_t* __restrict__ depth) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  int lo = 0, hi = kMaxDepth;       // count is non-increasing in d: find the first d with count <= nmax
  while (lo < hi) {
    const int m = (lo + hi) >> 1;
    if (node_count(root, path, n, i, m) <= nmax) hi = m; else lo = m + 1;
  }
  depth[i] = (uint8_t)lo;
}

__global__ void k_start_flags(int64_t n, const unsigned long long* __restrict__ root, const unsigned long long* __restrict__ path,
                              const uint8_t* __restrict__ depth, int32_t* __restrict__ flag) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  int f = 1;
  if (i > 0 && root[i] == root[i - 1]) {
    const int sh = 3 * (kMaxDepth - depth[i]);
    const unsigned long long a = sh >= 60 ? 0ull : path[i] >> sh, b = sh >= 60 ? 0ull : path[i - 1] >> sh;
    f = a != b;
  }
  flag[i] = f;
}

// batch_begin[bid] = first sorted position of batch bid (scan = inclusive scan of flags)
__global__ void k_batch_begin(int64_t n, const int32_t* __restrict__ flag, const int32_t* __restrict__ scan, int64_t* __restrict__ begin) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  if (flag[i]) begin[scan[i] - 1] = i;
  if (i == n - 1) begin[scan[i]] = n;
}

// tight bbox of each batch (exact min/max of its points): one CTA per batch
__global__ void k_bbox(const int64_t* __restrict__ begin, const uint32_t* __restrict__ idx, const double* __restrict__ pts,
                       double* __restrict__ bbox) {
  const int64_t j = blockIdx.x;
  const int64_t b0 = begin[j], b1 = begin[j + 1];
  double lo[3] = {INFINITY, INFINITY, INFINITY}, hi[3] = {-INFINITY, -INFINITY, -INFINITY};
  for (int64_t i = b0 + threadIdx.x; i < b1; i += blockDim.x) {
    const int64_t s = idx[i];
#pragma unroll
    for (int q = 0; q < 3; ++q) { const double v = pts[3 * s + q]; lo[q] = fmin(lo[q], v); hi[q] = fmax(hi[q], v); }
  }
  __shared__ double slo[3][32], shi[3][32];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
#pragma unroll
  for (int q = 0; q < 3; ++q) {
    for (int o = 16; o; o >>= 1) { lo[q] = fmin(lo[q], __shfl_xor_sync(~0u, lo[q], o)); hi[q] = fmax(hi[q], __shfl_xor_sync(~0u, hi[q], o)); }
    if (lane == 0) { slo[q][wid] = lo[q]; shi[q][wid] = hi[q]; }
  }
  __syncthreads();
  if (threadIdx.x < 3) {
    const int q = threadIdx.x;
    double a = slo[q][0], b = shi[q][0];
    for (int k = 1; k < nw; ++k) { a = fmin(a, slo[q][k]); b = fmax(b, shi[q][k]); }
    bbox[6 * j + q] = a; bbox[6 * j + 3 + q] = b;
  }
}

// a1: shell a in B_j iff dist^2(A, bbox_j) <= rcut_a^2 (R10).  mode 0: count shells per batch; mode 1: bit masks.
__global__ void k_basis_screen(ShellTab sh, const double* __restrict__ bbox, const int32_t* __restrict__ batch_src, int nbatch, int nshw,
                               int32_t* __restrict__ count, uint32_t* __restrict__ mask) {
  const int j = blockIdx.x;                      // batches on grid.x: more than 65535 of them at the paper's scale
  const int a = blockIdx.y * blockDim.x + threadIdx.x;
  const double* bb = bbox + 6 * (int64_t)(batch_src ? batch_src[j] : j);
  bool in = false;
  if (a < sh.nsh) {
    const double c[3] = {sh.cx[a], sh.cy[a], sh.cz[a]};
    double d2 = 0.0;
#pragma unroll
    for (int q = 0; q < 3; ++q) {
      const double d = fmax(0.0, fmax(bb[q] - c[q], c[q] - bb[3 + q]));
      d2 += d * d;
    }
    in = d2 <= sh.rcut2[a];
  }
  const unsigned bal = __ballot_sync(~0u, in);
  if ((threadIdx.x & 31) == 0) {
    if (mask) { if ((a >> 5) < nshw) mask[(int64_t)j * nshw + (a >> 5)] = bal; }
    else if (bal) atomicAdd(count + j, __popc(bal));
  }
}

// slots: batch j occupies [slot, slot + n) (+ padding to kSlotAlign with w = 0 and the batch's first point)
__global__ void k_fill_slots(const int64_t* __restrict__ bsrc_begin, const int32_t* __restrict__ bn, const int64_t* __restrict__ bslot,
                             const uint32_t* __restrict__ idx, const double* __restrict__ pts, const double* __restrict__ w,
                             double* __restrict__ gx, double* __restrict__ gy, double* __restrict__ gz, double* __restrict__ gw,
                             int64_t* __restrict__ slot_src) {
  const int j = blockIdx.x;
  const int64_t b0 = bsrc_begin[j], s0 = bslot[j];
  const int n = bn[j], npad = (n + kSlotAlign - 1) / kSlotAlign * kSlotAlign;
  for (int i = threadIdx.x; i < npad; i += blockDim.x) {
    const int64_t src = idx[b0 + (i < n ? i : 0)];
    gx[s0 + i] = pts[3 * src]; gy[s0 + i] = pts[3 * src + 1]; gz[s0 + i] = pts[3 * src + 2];
    gw[s0 + i] = i < n ? w[src] : 0.0;
    slot_src[s0 + i] = i < n ? src : -1;
  }
}

// radial part + components of one shell at displacement (x,y,z); out[ncart(l)]
__device__ __forceinline__ void shell_eval(const ShellTab& sh, int a, double x, double y, double z, double (&out)[10]) {
  const double r2 = x * x + y * y + z * z;
  const int p0 = sh.poff[a], np = sh.nprim[a];
  double rad = 0.0;
  for (int k = 0; k < np; ++k) rad = fma(sh.pcoef[p0 + k], exp(-sh.pexp[p0 + k] * r2), rad);
  switch (sh.l[a]) {
    case 0: out[0] = rad; break;
    case 1: out[0] = x * rad; out[1] = y * rad; out[2] = z * rad; break;
    case 2: {
      const double xr = x * rad, yr = y * rad;
      out[0] = x * xr; out[1] = y * xr; out[2] = z * xr; out[3] = y * yr; out[4] = z * yr; out[5] = z * z * rad; break;
    }
    default: {
      const double xx = x * x * rad, yy = y * y * rad, zz = z * z * rad;
      out[0] = x * xx; out[1] = y * xx; out[2] = z * xx; out[3] = x * yy; out[4] = x * y * z * rad; out[5] = x * zz;
      out[6] = y * yy; out[7] = z * yy; out[8] = y * zz; out[9] = z * zz; break;
    }
  }
}

// Eq. 47 (R12): PhiTilde_a(j) = max_g max_{mu in a} sqrt(w_g)|Phi[g,mu]| (written per FUNCTION of a),
//               phitilde(j)  = max_g sqrt(w_g) sum_{mu in B_j} |Phi[g,mu]|.   One CTA per batch.
constexpr int kMaxPerThread = 16;   // batch_max <= 4096, 256 threads
__global__ void __launch_bounds__(256) k_maxima(ShellTab sh, const int32_t* __restrict__ bn, const int64_t* __restrict__ bslot,
                                                const double* __restrict__ gx, const double* __restrict__ gy, const double* __restrict__ gz,
                                                const double* __restrict__ gw, const uint32_t* __restrict__ bmask, int nshw,
                                                double* __restrict__ PhiTf, int64_t ldj, double* __restrict__ phit,
                                                unsigned long long* __restrict__ phimax_bits) {
  extern __shared__ unsigned long long smax[];     // [nsh] bit patterns of non-negative doubles
  const int j = blockIdx.x, n = bn[j];
  const int64_t s0 = bslot[j];
  for (int a = threadIdx.x; a < sh.nsh; a += blockDim.x) smax[a] = 0ull;
  __syncthreads();
  double px[kMaxPerThread], py[kMaxPerThread], pz[kMaxPerThread], sw[kMaxPerThread], sum[kMaxPerThread];
#pragma unroll
  for (int q = 0; q < kMaxPerThread; ++q) {
    const int i = threadIdx.x + q * 256;
    const bool ok = i < n;
    px[q] = ok ? gx[s0 + i] : 0.0; py[q] = ok ? gy[s0 + i] : 0.0; pz[q] = ok ? gz[s0 + i] : 0.0;
    sw[q] = ok ? sqrt(gw[s0 + i]) : -1.0;
    sum[q] = 0.0;
  }
  const uint32_t* m = bmask + (int64_t)j * nshw;
  for (int wd = 0; wd < nshw; ++wd) {
    uint32_t bits = m[wd];
    while (bits) {
      const int a = (wd << 5) + __ffs(bits) - 1;
      bits &= bits - 1;
      const double cx = sh.cx[a], cy = sh.cy[a], cz = sh.cz[a];
      const int nc = ncart(sh.l[a]);
      double mx = 0.0;
#pragma unroll
      for (int q = 0; q < kMaxPerThread; ++q) {
        if (sw[q] < 0.0) continue;
        double v[10];
        shell_eval(sh, a, px[q] - cx, py[q] - cy, pz[q] - cz, v);
        double s = 0.0, vm = 0.0;
        for (int c = 0; c < nc; ++c) { const double av = fabs(v[c]); s += av; vm = fmax(vm, av); }
        sum[q] += s;
        mx = fmax(mx, sw[q] * vm);
      }
      for (int o = 16; o; o >>= 1) mx = fmax(mx, __shfl_xor_sync(~0u, mx, o));
      if ((threadIdx.x & 31) == 0 && mx > 0.0) atomicMax(&smax[a], (unsigned long long)__double_as_longlong(mx));
    }
  }
  double pm = 0.0;
#pragma unroll
  for (int q = 0; q < kMaxPerThread; ++q) if (sw[q] >= 0.0) pm = fmax(pm, sw[q] * sum[q]);
  for (int o = 16; o; o >>= 1) pm = fmax(pm, __shfl_xor_sync(~0u, pm, o));
  __shared__ unsigned long long spm;
  if (threadIdx.x == 0) spm = 0ull;
  __syncthreads();
  if ((threadIdx.x & 31) == 0) atomicMax(&spm, (unsigned long long)__double_as_longlong(pm));
  __syncthreads();
  if (threadIdx.x == 0) { phit[j] = __longlong_as_double((long long)spm); atomicMax(phimax_bits, spm); }
  for (int a = threadIdx.x; a < sh.nsh; a += blockDim.x) {
    const double v = __longlong_as_double((long long)smax[a]);
    const int f0 = sh.foff[a], nc = ncart(sh.l[a]);
    for (int c = 0; c < nc; ++c) PhiTf[(int64_t)(f0 + c) * ldj + j] = v;
  }
}

// ------------------------------------------------------------------------------------------------------------
// a3: density-dependent screening
// ------------------------------------------------------------------------------------------------------------
__global__ void k_abs(int64_t n, const double* __restrict__ in, double* __restrict__ out) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) out[i] = fabs(in[i]);
}

// Ftilde_a(j) = max_{mu in a} Ftf[mu][j]  ->  FtsT[j][a];  Fmax[a] = max_j
__global__ void k_shell_max(ShellTab sh, int nbatch, const double* __restrict__ Ftf, int64_t ldj, double* __restrict__ FtsT, int nshld,
                            unsigned long long* __restrict__ Fmax_bits) {
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  const int a = blockIdx.y;
  double v = 0.0;
  if (j < nbatch) {
    const int f0 = sh.foff[a], nc = ncart(sh.l[a]);
    for (int c = 0; c < nc; ++c) v = fmax(v, Ftf[(int64_t)(f0 + c) * ldj + j]);
    FtsT[(int64_t)j * nshld + a] = v;
  }
  for (int o = 16; o; o >>= 1) v = fmax(v, __shfl_xor_sync(~0u, v, o));
  if ((threadIdx.x & 31) == 0 && v > 0.0) atomicMax(Fmax_bits + a, (unsigned long long)__double_as_longlong(v));
}

__device__ __forceinline__ bool cand_decode(const PairCand& pc, int64_t i, int& a, int& b) {
  int c = 0;
#pragma unroll
  for (int k = 1; k < kNumClasses; ++k) if (i >= pc.off[k]) c = k;
  const int64_t r = i - pc.off[c];
  const int nb = pc.cnt_b[c];
  const int ia = (int)(r / nb), ib = (int)(r % nb);
  if (pc.same_l[c] && ia > ib) return false;
  a = pc.shells[pc.l_off[pc.la[c]] + ia];
  b = pc.shells[pc.l_off[pc.lb[c]] + ib];
  return true;
}

// candidate pair i is globally significant iff its Eq. 44/45 estimate with the per-shell maxima over batches reaches eps.
// nunit[i] = number of pair units it will occupy (ceil(K_a K_b / kUnitPrims)), ispair[i] = 0/1.
__global__ void k_pair_flags(PairCand pc, ShellTab sh, const double* __restrict__ Atil, const double* __restrict__ Fmax,
                             const double* __restrict__ phimax, double eps, int32_t* __restrict__ nunit, int32_t* __restrict__ ispair) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= pc.off[kNumClasses]) return;
  int a, b, f = 0, nu = 0;
  if (cand_decode(pc, i, a, b)) {
    const double At = Atil[(int64_t)a * sh.nsh + b];
    const double fa = Fmax[a], fb = Fmax[b];
    const double eE = fa * fb * At, eK = fmax(fa, fb) * (*phimax) * At;
    f = (eE >= eps || eK >= eps) ? 1 : 0;
    nu = f ? (sh.nprim[a] * sh.nprim[b] + kUnitPrims - 1) / kUnitPrims : 0;
  }
  nunit[i] = nu; ispair[i] = f;
}

// Pair units of every significant pair: header, primitive-pair table (R1 prefactor) and the screening metadata.
// R14: a primitive pair whose rigorous s-type bound (same construction as R11) times the largest density factor of
// Eqs. 44/45 is below prim_thresh / (K_a K_b) is dropped (never when eps = 0).  Kept primitive pairs are packed into the
// pair's units in order; trailing units may stay empty (nprim = 0) and are then never part of V_j.
__global__ void k_unit_fill(PairCand pc, ShellTab sh, const int32_t* __restrict__ nunit, const int32_t* __restrict__ pos,
                            const double* __restrict__ Atil, double prim_thresh, const double* __restrict__ Fmax,
                            const double* __restrict__ phimax, int64_t ld, unsigned char* __restrict__ units,
                            UnitMeta* __restrict__ meta) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= pc.off[kNumClasses] || nunit[i] == 0) return;
  int a, b;
  cand_decode(pc, i, a, b);
  const int la = sh.l[a], lb = sh.l[b];
  const int pa = sh.poff[a], pb = sh.poff[b], ka = sh.nprim[a], kb = sh.nprim[b];
  const double A[3] = {sh.cx[a], sh.cy[a], sh.cz[a]}, B[3] = {sh.cx[b], sh.cy[b], sh.cz[b]};
  const double ABx = A[0] - B[0], ABy = A[1] - B[1], ABz = A[2] - B[2];
  const double AB2 = ABx * ABx + ABy * ABy + ABz * ABz;
  const double At = Atil[(int64_t)a * sh.nsh + b];
  const double dens = fmax(Fmax[a] * Fmax[b], fmax(Fmax[a], Fmax[b]) * (*phimax));
  const double thr = prim_thresh / (double)(ka * kb);
  const int u0 = pos[i], nu = nunit[i];
  int n = 0;                                   // primitive pairs kept so far
  for (int k = 0; k < ka; ++k)
    for (int l = 0; l < kb; ++l) {
      const double za = sh.pexp[pa + k], zb = sh.pexp[pb + l], ca = sh.pcoef[pa + k], cb = sh.pcoef[pb + l];
      if (prim_thresh > 0.0) {
        const double zza = la ? 0.5 * za : za, zzb = lb ? 0.5 * zb : zb;
        const double cca = la ? fabs(ca) * pow((double)la / (2.718281828459045 * za), 0.5 * la) : fabs(ca);
        const double ccb = lb ? fabs(cb) * pow((double)lb / (2.718281828459045 * zb), 0.5 * lb) : fabs(cb);
        const double pp = zza + zzb;
        if (cca * ccb * (6.283185307179586 / pp) * exp(-(zza * zzb / pp) * AB2) * dens < thr) continue;
      }
      PrimPair q;
      const double pp = za + zb;
      q.p2 = 2.0 * pp;
      q.inv2p = 0.5 / pp;
      q.Px = (za * A[0] + zb * B[0]) / pp; q.Py = (za * A[1] + zb * B[1]) / pp; q.Pz = (za * A[2] + zb * B[2]) / pp;
      q.PAx = q.Px - A[0]; q.PAy = q.Py - A[1]; q.PAz = q.Pz - A[2];
      q.pref = ca * cb * (6.283185307179586 / pp) * exp(-(za * zb / pp) * AB2);
      q.cfar2 = 1.2533141373155002512 * q.pref;   // pref sqrt(pi/2): far-field seed constant (snk_os.cuh)
      *reinterpret_cast<PrimPair*>(units + (size_t)(u0 + n / kUnitPrims) * kUnitBytes + 64 + (n % kUnitPrims) * kPrimBytes) = q;
      ++n;
    }
  for (int u = 0; u < nu; ++u) {
    const int np = max(0, min(kUnitPrims, n - u * kUnitPrims));
    UnitHdr h;
    h.fa = sh.foff[a]; h.fb = sh.foff[b]; h.nprim = np; h.first = u == 0;
    h.ABx = ABx; h.ABy = ABy; h.ABz = ABz; h.sa = a; h.sb = b; h.offa = (int64_t)h.fa * ld; h.offb = (int64_t)h.fb * ld;
    *reinterpret_cast<UnitHdr*>(units + (size_t)(u0 + u) * kUnitBytes) = h;
    UnitMeta m;
    m.sa = a; m.sb = b; m.fb = h.fb; m.nprim_first = np | ((u == 0) << 8); m.At = At;
    meta[u0 + u] = m;
  }
}

// V_j bit masks (Eq. 43): one thread per (batch, unit); every unit of a pair takes the pair's decision
__global__ void k_vmask(int nunit, const UnitMeta* __restrict__ meta, const double* __restrict__ FtsT, int nshld,
                        const double* __restrict__ phit, double eps, uint32_t* __restrict__ vmask, int64_t vstride) {
  const int nblk_u = (nunit + 255) / 256;            // flattened grid: the batch index may exceed grid.y's 65535
  const int j = blockIdx.x / nblk_u;
  const int i = (blockIdx.x % nblk_u) * blockDim.x + threadIdx.x;
  bool keep = false;
  if (i < nunit) {
    const UnitMeta m = meta[i];
    const double* F = FtsT + (int64_t)j * nshld;
    const double fa = F[m.sa], fb = F[m.sb];
    const double eE = fa * fb * m.At, eK = fmax(fa, fb) * phit[j] * m.At;
    keep = (eE >= eps || eK >= eps) && (m.nprim_first & 0xff) > 0;
  }
  const unsigned bal = __ballot_sync(~0u, keep);
  if ((threadIdx.x & 31) == 0 && (i >> 5) < vstride) vmask[(int64_t)j * vstride + (i >> 5)] = bal;
}

// Unit lists of the batches [b0, b0 + nb) for the integral kernel: the set bits of V_j, class by class, as unit ids.
// list[(j - b0) * stride + cls_beg[c] + q] = q-th kept unit of class c in batch j (ascending: the (a, b) order of the unit table),
// cnt[(j - b0) * kNumClasses + c] = their number.  The slot of a class inside a batch's row is as long as the class itself, so no
// offsets have to be scanned and nothing has to be sized on the host.  One CTA per batch.
struct ClassBeg { int v[kNumClasses + 1]; };
__global__ void __launch_bounds__(256) k_vlist(int b0, ClassBeg cb, const uint32_t* __restrict__ vmask, int64_t vstride,
                                               int32_t* __restrict__ list, int64_t stride, int32_t* __restrict__ cnt) {
  __shared__ int wsum[8];
  const int jj = blockIdx.x, t = threadIdx.x, lane = t & 31, warp = t >> 5;
  const uint32_t* __restrict__ mrow = vmask + (int64_t)(b0 + jj) * vstride;
  int32_t* __restrict__ out_b = list + (int64_t)jj * stride;
  for (int c = 0; c < kNumClasses; ++c) {
    const int pbeg = cb.v[c], pend = cb.v[c + 1];
    int running = 0;
    if (pend > pbeg) {
      const int w0 = pbeg >> 5, w1 = (pend + 31) >> 5;
      int32_t* __restrict__ out = out_b + pbeg;
      for (int wb = w0; wb < w1; wb += 256) {
        const int w = wb + t;
        uint32_t word = 0u;
        if (w < w1) {
          word = mrow[w];
          if (w == w0) word &= 0xffffffffu << (pbeg & 31);
          if (w == w1 - 1 && (pend & 31)) word &= 0xffffffffu >> (32 - (pend & 31));
        }
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
        const int id0 = w << 5;
        while (word) { const int b = __ffs(word) - 1; word &= word - 1; out[o++] = id0 + b; }
        running += total;
        __syncthreads();
      }
    }
    if (t == 0) cnt[jj * kNumClasses + c] = running;
  }
}

// counters for snk_stats: out[0]=sum|V_j|, [1]=pair-points, [2]=contracted integrals, [3]=primitive integrals,
// [4..13] contracted integrals per class, [14] flop model, [16..25] flop model per class.  Pair-level quantities are
// counted on the first unit of a pair only.
// One CTA per batch walks the batch's V_j mask; sums are kept in registers, reduced over the CTA and leave with 23 atomics
// per batch (one atomic per kept unit and counter would serialise 10^11 same-address updates at the paper's scale).
__global__ void __launch_bounds__(256) k_vstats(int nunit, const UnitMeta* __restrict__ meta, ShellTab sh, const int32_t* __restrict__ bn,
                                                const uint32_t* __restrict__ vmask, int64_t vstride,
                                                const double* __restrict__ class_flops_prim, const double* __restrict__ class_flops_contr,
                                                double* __restrict__ out) {
  constexpr int NV = 3 + 2 * kNumClasses;
  __shared__ double red[8][NV];
  const int j = blockIdx.x;
  const double nq = bn[j];
  double v[NV];                                  // [0] kept pairs, [1] pair-points, [2] primitive integrals, then per class
#pragma unroll
  for (int k = 0; k < NV; ++k) v[k] = 0.0;
  const uint32_t* __restrict__ mrow = vmask + (int64_t)j * vstride;
  for (int i = threadIdx.x; i < nunit; i += 256) {
    if (!((mrow[i >> 5] >> (i & 31)) & 1u)) continue;
    const UnitMeta m = meta[i];
    const int la = sh.l[m.sa], lb = sh.l[m.sb];
    const int np = m.nprim_first & 0xff;
    const double first = (double)((m.nprim_first >> 8) & 1);
    const double nc = (double)(ncart(la) * ncart(lb));
    const int cls = la * (la + 1) / 2 + lb;
    v[0] += first; v[1] += first * nq; v[2] += nq * nc * np;
    const double vi = first * nq * nc, vf = nq * (class_flops_prim[cls] * np + class_flops_contr[cls] * first);
#pragma unroll
    for (int c = 0; c < kNumClasses; ++c)
      if (c == cls) { v[3 + c] += vi; v[3 + kNumClasses + c] += vf; }
  }
#pragma unroll
  for (int k = 0; k < NV; ++k) {
    double x = v[k];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5][k] = x;
  }
  __syncthreads();
  if (threadIdx.x < NV) {
    const int k = threadIdx.x;
    double x = 0.0;
#pragma unroll
    for (int w = 0; w < 8; ++w) x += red[w][k];
    if (x != 0.0) {
      if (k == 0) atomicAdd(out + 0, x);
      else if (k == 1) atomicAdd(out + 1, x);
      else if (k == 2) atomicAdd(out + 3, x);
      else if (k < 3 + kNumClasses) { atomicAdd(out + 4 + (k - 3), x); atomicAdd(out + 2, x); }
      else { atomicAdd(out + 16 + (k - 3 - kNumClasses), x); atomicAdd(out + 14, x); }
    }
  }
}

// ------------------------------------------------------------------------------------------------------------
// a2: collocation Phi[mu][slot] (Eq. 31), zero for shells outside B_j.  One thread per grid point, one CTA per
// (tile, chunk of 64 shells); stores are coalesced along the slot index.
// ------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kTile) k_colloc(ShellTab sh, const TileRec* __restrict__ tiles, const double* __restrict__ gx,
                                                  const double* __restrict__ gy, const double* __restrict__ gz,
                                                  const uint32_t* __restrict__ bmask, int nshw, double* __restrict__ Phi, int64_t ld,
                                                  int64_t slot0) {
  const TileRec tile = tiles[blockIdx.x];
  const int t = threadIdx.x;
  const int npad = (tile.n + kSlotAlign - 1) / kSlotAlign * kSlotAlign;
  if (t >= npad) return;
  const int64_t slot = tile.slot + t;
  const double x = gx[slot], y = gy[slot], z = gz[slot];
  double* __restrict__ out = Phi + (slot - slot0);
  const uint32_t* m = bmask + (int64_t)tile.batch * nshw;
  const int a0 = blockIdx.y * 64, a1 = min(a0 + 64, sh.nsh);
  for (int a = a0; a < a1; ++a) {
    const int f0 = sh.foff[a], nc = ncart(sh.l[a]);
    if ((m[a >> 5] >> (a & 31)) & 1u) {
      double v[10];
      shell_eval(sh, a, x - sh.cx[a], y - sh.cy[a], z - sh.cz[a], v);
      for (int c = 0; c < nc; ++c) out[(int64_t)(f0 + c) * ld] = v[c];
    } else {
      for (int c = 0; c < nc; ++c) out[(int64_t)(f0 + c) * ld] = 0.0;
    }
  }
}

// a7: K = (Kt + Kt^T)/2 (Eq. 40)
__global__ void k_symmetrise(int n, const double* __restrict__ Kt, double* __restrict__ K) {
  __shared__ double tile[32][33];
  const int bx = blockIdx.x * 32, by = blockIdx.y * 32;
  const int tx = threadIdx.x, ty = threadIdx.y;
  for (int r = ty; r < 32; r += 8) {
    const int i = bx + r, jj = by + tx;            // read Kt[bx-block rows][by-block cols] transposed source
    tile[r][tx] = (i < n && jj < n) ? Kt[(int64_t)i * n + jj] : 0.0;
  }
  __syncthreads();
  for (int r = ty; r < 32; r += 8) {
    const int i = by + r, jj = bx + tx;            // K[i][jj] = (Kt[i][jj] + Kt[jj][i])/2 ; Kt[jj][i] = tile[tx][r]
    if (i < n && jj < n) K[(int64_t)i * n + jj] = 0.5 * (Kt[(int64_t)i * n + jj] + tile[tx][r]);
  }
}

__global__ void k_zero_pad_cols(double* __restrict__ A, int64_t rows, int64_t ld, int64_t c0, int64_t c1) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t w = c1 - c0;
  if (i < rows * w) A[(i / w) * ld + c0 + (i % w)] = 0.0;
}

// ------------------------------------------------------------------------------------------------------------
// host-side launch wrappers
// ------------------------------------------------------------------------------------------------------------
static inline unsigned nblk(int64_t n, int b) { return (unsigned)((n + b - 1) / b); }

cudaError_t run_point_keys(int64_t n, const double* pts, const double* w, double h0, unsigned long long* root, unsigned long long* path,
                           uint32_t* idx, int* err, cudaStream_t s) {
  if (n > 0) k_point_keys<<<nblk(n, 256), 256, 0, s>>>(n, pts, w, h0, root, path, idx, err);
  return cudaGetLastError();
}

cudaError_t run_sort_pairs(void* tmp, size_t& tmp_bytes, const unsigned long long* kin, unsigned long long* kout, const uint32_t* vin,
                           uint32_t* vout, int64_t n, int end_bit, cudaStream_t s) {
  return cub::DeviceRadixSort::SortPairs(tmp, tmp_bytes, kin, kout, vin, vout, (int)n, 0, end_bit, s);
}

cudaError_t run_gather_u64(int64_t n, const uint32_t* idx, const unsigned long long* src, unsigned long long* dst, cudaStream_t s) {
  if (n > 0) k_gather<unsigned long long><<<nblk(n, 256), 256, 0, s>>>(n, idx, src, dst);
  return cudaGetLastError();
}

cudaError_t run_leaves(int64_t n, const unsigned long long* root, const unsigned long long* path, int nmax, uint8_t* depth, int32_t* flag,
                       cudaStream_t s) {
  if (n > 0) {
    k_leaf_depth<<<nblk(n, 256), 256, 0, s>>>(n, root, path, nmax, depth);
    k_start_flags<<<nblk(n, 256), 256, 0, s>>>(n, root, path, depth, flag);
  }
  return cudaGetLastError();
}

cudaError_t run_scan_i32(void* tmp, size_t& tmp_bytes, const int32_t* in, int32_t* out, int64_t n, bool inclusive, cudaStream_t s) {
  if (inclusive) return cub::DeviceScan::InclusiveSum(tmp, tmp_bytes, in, out, (int)n, s);
  return cub::DeviceScan::ExclusiveSum(tmp, tmp_bytes, in, out, (int)n, s);
}

cudaError_t run_batch_begin(int64_t n, const int32_t* flag, const int32_t* scan, int64_t* begin, cudaStream_t s) {
  if (n > 0) k_batch_begin<<<nblk(n, 256), 256, 0, s>>>(n, flag, scan, begin);
  return cudaGetLastError();
}

cudaError_t run_bbox(int nbatch, const int64_t* begin, const uint32_t* idx, const double* pts, double* bbox, cudaStream_t s) {
  if (nbatch > 0) k_bbox<<<nbatch, 256, 0, s>>>(begin, idx, pts, bbox);
  return cudaGetLastError();
}

cudaError_t run_basis_screen(const ShellTab& sh, const double* bbox, const int32_t* batch_src, int nbatch, int nshw, int32_t* count,
                             uint32_t* mask, cudaStream_t s) {
  if (nbatch > 0) {
    dim3 g((unsigned)nbatch, (unsigned)(nshw * 32 + 127) / 128);
    k_basis_screen<<<g, 128, 0, s>>>(sh, bbox, batch_src, nbatch, nshw, count, mask);
  }
  return cudaGetLastError();
}

cudaError_t run_fill_slots(int nbatch, const int64_t* bsrc_begin, const int32_t* bn, const int64_t* bslot, const uint32_t* idx,
                           const double* pts, const double* w, double* gx, double* gy, double* gz, double* gw, int64_t* slot_src,
                           cudaStream_t s) {
  if (nbatch > 0) k_fill_slots<<<nbatch, 256, 0, s>>>(bsrc_begin, bn, bslot, idx, pts, w, gx, gy, gz, gw, slot_src);
  return cudaGetLastError();
}

cudaError_t run_maxima(const ShellTab& sh, int nbatch, const int32_t* bn, const int64_t* bslot, const double* gx, const double* gy,
                       const double* gz, const double* gw, const uint32_t* bmask, int nshw, double* PhiTf, int64_t ldj, double* phit,
                       unsigned long long* phimax_bits, cudaStream_t s) {
  if (nbatch > 0) {
    const size_t sm = (size_t)sh.nsh * sizeof(unsigned long long);
    if (sm > 48 * 1024) cudaFuncSetAttribute(k_maxima, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
    k_maxima<<<nbatch, 256, sm, s>>>(sh, bn, bslot, gx, gy, gz, gw, bmask, nshw, PhiTf, ldj, phit, phimax_bits);
  }
  return cudaGetLastError();
}

cudaError_t run_abs(int64_t n, const double* in, double* out, cudaStream_t s) {
  if (n > 0) k_abs<<<nblk(n, 256), 256, 0, s>>>(n, in, out);
  return cudaGetLastError();
}

cudaError_t run_shell_max(const ShellTab& sh, int nbatch, const double* Ftf, int64_t ldj, double* FtsT, int nshld,
                          unsigned long long* Fmax_bits, cudaStream_t s) {
  if (nbatch > 0) {
    dim3 g(nblk(nbatch, 128), (unsigned)sh.nsh);
    k_shell_max<<<g, 128, 0, s>>>(sh, nbatch, Ftf, ldj, FtsT, nshld, Fmax_bits);
  }
  return cudaGetLastError();
}

cudaError_t run_pair_flags(const PairCand& pc, const ShellTab& sh, const double* Atil, const double* Fmax, const double* phimax, double eps,
                           int32_t* nunit, int32_t* ispair, cudaStream_t s) {
  const int64_t n = pc.off[kNumClasses];
  if (n > 0) k_pair_flags<<<nblk(n, 256), 256, 0, s>>>(pc, sh, Atil, Fmax, phimax, eps, nunit, ispair);
  return cudaGetLastError();
}

cudaError_t run_unit_fill(const PairCand& pc, const ShellTab& sh, const int32_t* nunit, const int32_t* pos, const double* Atil,
                          double prim_thresh, const double* Fmax, const double* phimax, int64_t ld, unsigned char* units,
                          UnitMeta* meta, cudaStream_t s) {
  const int64_t n = pc.off[kNumClasses];
  if (n > 0) k_unit_fill<<<nblk(n, 128), 128, 0, s>>>(pc, sh, nunit, pos, Atil, prim_thresh, Fmax, phimax, ld, units, meta);
  return cudaGetLastError();
}

cudaError_t run_vmask(int nbatch, int nunit, const UnitMeta* meta, const double* FtsT, int nshld, const double* phit, double eps,
                      uint32_t* vmask, int64_t vstride, cudaStream_t s) {
  if (nbatch > 0 && nunit > 0) {
    const int64_t nb = (int64_t)nbatch * nblk(nunit, 256);
    if (nb > 0x7fffffff) return cudaErrorInvalidConfiguration;
    k_vmask<<<(unsigned)nb, 256, 0, s>>>(nunit, meta, FtsT, nshld, phit, eps, vmask, vstride);
  }
  return cudaGetLastError();
}

// work estimate of a batch for Alg. 2: primitive pair-points = |Q_j| * sum of the primitive pairs of the
// units kept in V_j (what the integral kernel's time is proportional to).  One CTA per batch.
__global__ void __launch_bounds__(256) k_batch_costs(int nunit, const UnitMeta* __restrict__ meta, const int32_t* __restrict__ bn,
                                                     const uint32_t* __restrict__ vmask, int64_t vstride, double* __restrict__ cost) {
  __shared__ double red[8];
  const int j = blockIdx.x;
  const uint32_t* __restrict__ mrow = vmask + (int64_t)j * vstride;
  double v = 0.0;
  for (int i = threadIdx.x; i < nunit; i += 256)
    if ((mrow[i >> 5] >> (i & 31)) & 1u) v += (double)(meta[i].nprim_first & 0xff);
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(~0u, v, d);
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
  __syncthreads();
  if (threadIdx.x == 0) {
    double t = 0.0;
    for (int k = 0; k < 8; ++k) t += red[k];
    cost[j] = t * (double)bn[j];
  }
}

cudaError_t run_batch_costs(int nbatch, int nunit, const UnitMeta* meta, const int32_t* bn, const uint32_t* vmask, int64_t vstride,
                            double* cost, cudaStream_t s) {
  if (nbatch > 0) k_batch_costs<<<(unsigned)nbatch, 256, 0, s>>>(nunit, meta, bn, vmask, vstride, cost);
  return cudaGetLastError();
}

cudaError_t run_vlist(int b0, int nb, const int* cls_beg, const uint32_t* vmask, int64_t vstride, int32_t* list, int64_t stride,
                      int32_t* cnt, cudaStream_t s) {
  if (nb > 0) {
    ClassBeg cb;
    for (int c = 0; c <= kNumClasses; ++c) cb.v[c] = cls_beg[c];
    k_vlist<<<(unsigned)nb, 256, 0, s>>>(b0, cb, vmask, vstride, list, stride, cnt);
  }
  return cudaGetLastError();
}

cudaError_t run_vstats(int nbatch, int nunit, const UnitMeta* meta, const ShellTab& sh, const int32_t* bn, const uint32_t* vmask,
                       int64_t vstride, const double* cfp, const double* cfc, double* out, cudaStream_t s) {
  if (nbatch > 0 && nunit > 0) {
    k_vstats<<<(unsigned)nbatch, 256, 0, s>>>(nunit, meta, sh, bn, vmask, vstride, cfp, cfc, out);
  }
  return cudaGetLastError();
}

cudaError_t run_colloc(const ShellTab& sh, const TileRec* tiles, int ntiles, const double* gx, const double* gy, const double* gz,
                       const uint32_t* bmask, int nshw, double* Phi, int64_t ld, int64_t slot0, cudaStream_t s) {
  if (ntiles > 0) {
    dim3 g((unsigned)ntiles, (unsigned)((sh.nsh + 63) / 64));
    k_colloc<<<g, kTile, 0, s>>>(sh, tiles, gx, gy, gz, bmask, nshw, Phi, ld, slot0);
  }
  return cudaGetLastError();
}

cudaError_t run_symmetrise(int n, const double* Kt, double* K, cudaStream_t s) {
  if (n > 0) {
    dim3 g((unsigned)((n + 31) / 32), (unsigned)((n + 31) / 32)), b(32, 8);
    k_symmetrise<<<g, b, 0, s>>>(n, Kt, K);
  }
  return cudaGetLastError();
}

cudaError_t run_zero_pad_cols(double* A, int64_t rows, int64_t ld, int64_t c0, int64_t c1, cudaStream_t s) {
  if (rows > 0 && c1 > c0) k_zero_pad_cols<<<nblk(rows * (c1 - c0), 256), 256, 0, s>>>(A, rows, ld, c0, c1);
  return cudaGetLastError();
}

}  // namespace snk
