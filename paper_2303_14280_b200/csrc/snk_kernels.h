// snk_kernels.h -- launch wrappers of snk_kernels.cu (internal)
#pragma once
#include "snk_internal.h"

namespace snk {

// enumeration of all candidate shell pairs, class by class (class = (la,lb), la >= lb), inside a class row-major
// over (shells of la) x (shells of lb); for la == lb only ia <= ib is a candidate.  Order = sort key (class, a, b).
struct PairCand {
  int64_t off[kNumClasses + 1];
  int32_t cnt_b[kNumClasses];
  int32_t la[kNumClasses], lb[kNumClasses], same_l[kNumClasses];
  int32_t l_off[5];
  const int32_t* shells;   // DEVICE: shell ids grouped by l, ascending inside a group
};

cudaError_t run_point_keys(int64_t n, const double* pts, const double* w, double h0, unsigned long long* root, unsigned long long* path,
                           uint32_t* idx, int* err, cudaStream_t s);
cudaError_t run_sort_pairs(void* tmp, size_t& tmp_bytes, const unsigned long long* kin, unsigned long long* kout, const uint32_t* vin,
                           uint32_t* vout, int64_t n, int end_bit, cudaStream_t s);
cudaError_t run_gather_u64(int64_t n, const uint32_t* idx, const unsigned long long* src, unsigned long long* dst, cudaStream_t s);
cudaError_t run_leaves(int64_t n, const unsigned long long* root, const unsigned long long* path, int nmax, uint8_t* depth, int32_t* flag,
                       cudaStream_t s);
cudaError_t run_scan_i32(void* tmp, size_t& tmp_bytes, const int32_t* in, int32_t* out, int64_t n, bool inclusive, cudaStream_t s);
cudaError_t run_batch_begin(int64_t n, const int32_t* flag, const int32_t* scan, int64_t* begin, cudaStream_t s);
cudaError_t run_bbox(int nbatch, const int64_t* begin, const uint32_t* idx, const double* pts, double* bbox, cudaStream_t s);
cudaError_t run_basis_screen(const ShellTab& sh, const double* bbox, const int32_t* batch_src, int nbatch, int nshw, int32_t* count,
                             uint32_t* mask, cudaStream_t s);
cudaError_t run_fill_slots(int nbatch, const int64_t* bsrc_begin, const int32_t* bn, const int64_t* bslot, const uint32_t* idx,
                           const double* pts, const double* w, double* gx, double* gy, double* gz, double* gw, int64_t* slot_src,
                           cudaStream_t s);
cudaError_t run_maxima(const ShellTab& sh, int nbatch, const int32_t* bn, const int64_t* bslot, const double* gx, const double* gy,
                       const double* gz, const double* gw, const uint32_t* bmask, int nshw, double* PhiTf, int64_t ldj, double* phit,
                       unsigned long long* phimax_bits, cudaStream_t s);
cudaError_t run_abs(int64_t n, const double* in, double* out, cudaStream_t s);
cudaError_t run_shell_max(const ShellTab& sh, int nbatch, const double* Ftf, int64_t ldj, double* FtsT, int nshld,
                          unsigned long long* Fmax_bits, cudaStream_t s);
cudaError_t run_pair_flags(const PairCand& pc, const ShellTab& sh, const double* Atil, const double* Fmax, const double* phimax, double eps,
                           int32_t* nunit, int32_t* ispair, cudaStream_t s);
cudaError_t run_unit_fill(const PairCand& pc, const ShellTab& sh, const int32_t* nunit, const int32_t* pos, const double* Atil,
                          double prim_thresh, const double* Fmax, const double* phimax, int64_t ld, unsigned char* units,
                          UnitMeta* meta, cudaStream_t s);
cudaError_t run_vmask(int nbatch, int nunit, const UnitMeta* meta, const double* FtsT, int nshld, const double* phit, double eps,
                      uint32_t* vmask, int64_t vstride, cudaStream_t s);
cudaError_t run_batch_costs(int nbatch, int nunit, const UnitMeta* meta, const int32_t* bn, const uint32_t* vmask, int64_t vstride,
                            double* cost, cudaStream_t s);
cudaError_t run_vlist(int b0, int nb, const int* cls_beg, const uint32_t* vmask, int64_t vstride, int32_t* list, int64_t stride,
                      int32_t* cnt, cudaStream_t s);
cudaError_t run_vstats(int nbatch, int nunit, const UnitMeta* meta, const ShellTab& sh, const int32_t* bn, const uint32_t* vmask,
                       int64_t vstride, const double* cfp, const double* cfc, double* out, cudaStream_t s);
cudaError_t run_colloc(const ShellTab& sh, const TileRec* tiles, int ntiles, const double* gx, const double* gy, const double* gz,
                       const uint32_t* bmask, int nshw, double* Phi, int64_t ld, int64_t slot0, cudaStream_t s);
cudaError_t run_symmetrise(int n, const double* Kt, double* K, cudaStream_t s);
// a4 / a6 (snk_gemm_kt.cu): row lists of the chunks, F = P Phi and Kt += Phi diag(w) G^T packed to them
cudaError_t run_chunk_rows(const ShellTab& sh, int nchunks, const ChunkRec* chunks, const uint32_t* bmask, int nshw, int32_t* rowlist,
                           int64_t lstride, int32_t* nrows, cudaStream_t s);
cudaError_t gemm_f(int64_t nbf, int64_t slot0, int ntiles, const ColTile* tiles, int chunk0, const int32_t* nrows, const int32_t* rowlist,
                   int64_t lstride, const double* P, const double* Phi, double* F, int64_t ld, cudaStream_t s);
int kt_row_tile();   // packed Phi rows per CTA tile of k_gemm_kt
int f_k_tile();      // packed k entries per step of k_gemm_f
cudaError_t gemm_kt(int64_t nbf, int64_t slot0, int nchunks, int max_nrow, const ChunkRec* chunks, const int32_t* nrows,
                    const int32_t* rowlist, int64_t lstride, const double* Phi, const double* G, int64_t ld, const double* wts, double* Kt,
                    cudaStream_t s);
cudaError_t run_zero_pad_cols(double* A, int64_t rows, int64_t ld, int64_t c0, int64_t c1, cudaStream_t s);
cudaError_t run_fp64_peak(double* dfma_tflops, double* dmma_tflops, int reps);

}  // namespace snk
