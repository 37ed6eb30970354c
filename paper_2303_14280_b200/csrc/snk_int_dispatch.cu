// class dispatch of the integral-contraction kernels + Boys test hook
#include "snk_int_kernel.cuh"
namespace snk {
SNK_DECLARE_CLASS(0, 0) SNK_DECLARE_CLASS(1, 0) SNK_DECLARE_CLASS(1, 1) SNK_DECLARE_CLASS(2, 0) SNK_DECLARE_CLASS(2, 1)
SNK_DECLARE_CLASS(2, 2) SNK_DECLARE_CLASS(3, 0) SNK_DECLARE_CLASS(3, 1) SNK_DECLARE_CLASS(3, 2) SNK_DECLARE_CLASS(3, 3)

cudaError_t launch_integrals(int cls, const IntParams& p, cudaStream_t s) {
  switch (cls) {
    case 0: return launch_class_00(p, s);
    case 1: return launch_class_10(p, s);
    case 2: return launch_class_11(p, s);
    case 3: return launch_class_20(p, s);
    case 4: return launch_class_21(p, s);
    case 5: return launch_class_22(p, s);
    case 6: return launch_class_30(p, s);
    case 7: return launch_class_31(p, s);
    case 8: return launch_class_32(p, s);
    case 9: return launch_class_33(p, s);
  }
  return cudaErrorInvalidValue;
}

cudaError_t launch_debug_A(int la, int lb, bool tr, const PrimPair* prims, int nprim, double ABx, double ABy, double ABz,
                           const double* pts, int64_t n, const double* boys, double* out, cudaStream_t s) {
  switch (class_id(la, lb)) {
    case 0: return launch_dbgA_00(tr, prims, nprim, ABx, ABy, ABz, pts, n, boys, out, s);
    case 1: return launch_dbgA_10(tr, prims, nprim, ABx, ABy, ABz, pts, n, boys, out, s);
    case 2: return launch_dbgA_11(tr, prims, nprim, ABx, ABy, ABz, pts, n, boys, out, s);
    case 3: return launch_dbgA_20(tr, prims, nprim, ABx, ABy, ABz, pts, n, boys, out, s);
    case 4: return launch_dbgA_21(tr, prims, nprim, ABx, ABy, ABz, pts, n, boys, out, s);
    case 5: return launch_dbgA_22(tr, prims, nprim, ABx, ABy, ABz, pts, n, boys, out, s);
    case 6: return launch_dbgA_30(tr, prims, nprim, ABx, ABy, ABz, pts, n, boys, out, s);
    case 7: return launch_dbgA_31(tr, prims, nprim, ABx, ABy, ABz, pts, n, boys, out, s);
    case 8: return launch_dbgA_32(tr, prims, nprim, ABx, ABy, ABz, pts, n, boys, out, s);
    case 9: return launch_dbgA_33(tr, prims, nprim, ABx, ABy, ABz, pts, n, boys, out, s);
  }
  return cudaErrorInvalidValue;
}

template <int M>
__global__ void k_debug_boys(int64_t n, const double* x, const double* tab, double* out) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  double F[M + 1];
  boys<M>(x[i], tab, F);
#pragma unroll
  for (int m = 0; m <= M; ++m) out[i * (M + 1) + m] = F[m];
}

cudaError_t launch_debug_boys(int mmax, int64_t n, const double* x, const double* tab, double* out, cudaStream_t s) {
  if (n <= 0) return cudaSuccess;
  const unsigned g = (unsigned)((n + 127) / 128);
  switch (mmax) {
    case 0: k_debug_boys<0><<<g, 128, 0, s>>>(n, x, tab, out); break;
    case 1: k_debug_boys<1><<<g, 128, 0, s>>>(n, x, tab, out); break;
    case 2: k_debug_boys<2><<<g, 128, 0, s>>>(n, x, tab, out); break;
    case 3: k_debug_boys<3><<<g, 128, 0, s>>>(n, x, tab, out); break;
    case 4: k_debug_boys<4><<<g, 128, 0, s>>>(n, x, tab, out); break;
    case 5: k_debug_boys<5><<<g, 128, 0, s>>>(n, x, tab, out); break;
    case 6: k_debug_boys<6><<<g, 128, 0, s>>>(n, x, tab, out); break;
    default: return cudaErrorInvalidValue;
  }
  return cudaGetLastError();
}
}  // namespace snk
