// common.cuh -- internal declarations shared by the translation units of libhdc.so (sm_100a only).
// Nothing here is part of the public ABI (include/hdc.h is).  No code is shared with oracle/.
#pragma once
#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "hdc.h"

namespace hdc {

// ---- operand kinds of the contraction loaders (device-side view of a matrix element) ----------
enum OperandKind : int {
  OPK_F32 = 0,        // float
  OPK_BF16 = 1,       // __nv_bfloat16, widened exactly
  OPK_F32_RBF16 = 2,  // float rounded to nearest-even bf16 on load (precision BF16 / hv_bits 16)
  OPK_BITS = 3,       // packed hypervector bits: element k -> bit k&31 of word k>>5, value 1-2*bit
  OPK_I8 = 4,         // int8
  OPK_F32_RF16 = 5,   // float rounded to nearest-even IEEE half on load (hv code HDC_HV_F16, precision HDC_F16)
  OPK_BF16_RF16 = 6,  // __nv_bfloat16 widened, then rounded to IEEE half (precision HDC_F16 on bf16 inputs)
  OPK_F16 = 7,        // __half (staged operands of the tcgen05 path)
  OPK_I16 = 8         // int16 (class codes of hv code HDC_HV_I16)
};

struct Operand {
  const void* p;
  int64_t ld;  // in elements (words for OPK_BITS)
  int kind;
};

// Reduction perforation of the similarity (include/hdc.h knobs perf_begin /
// perf_stride): the visited dimensions are d = begin + j*stride < D_eff.
struct Perf {
  int begin;
  int stride;
};
__host__ __device__ __forceinline__ bool perf_visits(const Perf& pf, int d) {
  return d >= pf.begin && (pf.stride <= 1 || (d - pf.begin) % pf.stride == 0);
}
static inline int perf_count(const Perf& pf, int D_eff) {
  const int st = pf.stride <= 1 ? 1 : pf.stride;
  return D_eff > pf.begin ? (D_eff - pf.begin + st - 1) / st : 0;
}
static inline bool perf_on(const Perf& pf) { return pf.begin > 0 || pf.stride > 1; }

enum EpilogueKind : int { EPI_SIGN = 0, EPI_SCORE = 1, EPI_ARGMAX = 2, EPI_INFER = 3 };

// Epilogue of C[m,n] = sum_k A[m,k] * B[n,k]
struct Epilogue {
  int kind;
  // EPI_SIGN: bit[m,n] = [acc < 0] packed into bits[m][n>>5]; optional raw accumulators
  uint32_t* bits;
  int64_t ldbits;
  void* raw;  // float* (float accumulate) or int32_t* (integer accumulate), nullable
  int64_t ldraw;
  // EPI_SCORE: S[m,n] = acc * colscale[n] (colscale nullable => 1); s_i32 = 1 => store as int32 (2: int64, widedot.cu only)
  void* S;
  int64_t lds;
  int s_i32;
  const double* colscale;
  const float* colscale_f;  // the same scales rounded to fp32 (sim_tc_kernel compares in fp32: FP64 is slow here)
  // EPI_ARGMAX: label = argmax_n acc*colscale[n], ties to lowest n; best/second nullable.
  // ham_D > 0: report best/second as Hamming distances (ham_D - dot)/2 (bits x bits).
  int32_t* labels;
  float* best;
  float* second;
  int ham_D;
  // EPI_INFER (gemm_tc.cu only): sign of the accumulators (packed into `bits` when it is not NULL) followed by
  // the similarity search of the signed row against K <= 32 class hypervectors and the arg-max, all in the
  // epilogue: score[m,k] = sum_n sgn(acc[m,n]) * cls[k][n].  cls: fp32 [KC][ldcls] class operand prepared by
  // launch_class_operand_f32 (KC = 8, 16 or 32 rows, ldcls a multiple of 256, zeros beyond K / D_eff);
  // labels / best / second / colscale / ham_D as for EPI_ARGMAX.
  const float* cls;
  int64_t ldcls;
  int K;
};

// ---- launchers (each returns the CUDA error of its launches and adds to *nlaunch) -------------
cudaError_t launch_gemm_simt(const Operand& A, const Operand& B, int64_t M, int Nc, int Kr,
                             bool int_acc, const Epilogue& e, cudaStream_t st, int64_t* nlaunch);

// tcgen05 path (gemm_tc.cu): both operands K-contiguous bf16 or int8, 16-byte aligned bases and row
// strides.  The reduction axis is a list of `nseg` segments of Kr elements: segment s reads A
// columns [a_seg(s)*seg_stride, +Kr) and B columns [b_seg(s)*seg_stride, +Kr), a_seg(s) = 4-bit
// field s of a_segs (nseg = 1, a_segs = b_segs = 0: a plain GEMM).  Columns >= cols_a / cols_b read
// as zero (TMA out-of-bounds fill), so Kr need not be a multiple of the k-block.
// Returns cudaErrorNotSupported when the operands do not meet the alignment rules.
struct TcContext;  // opaque: holds the cuTensorMapEncodeTiled entry point
TcContext* tc_context_create();
void tc_context_destroy(TcContext*);
struct TcOperands {
  const void* A;
  const void* B;
  int elem_kind;  // OPK_BF16 | OPK_F16 | OPK_I8
  int64_t lda, ldb;
  int64_t cols_a, cols_b;
  int Kr;
  int nseg;
  uint32_t a_segs, b_segs;
  int seg_stride;
  int Kvalid;  // 0 = Kr; else: columns >= Kvalid of every segment are known to be zero (staged padding), so the MMAs
               // of the last k-block that would only read them are not issued
};
// cta_group: 1 / 2 force the 1-CTA / CTA-pair kernel, anything else chooses by problem size
cudaError_t launch_gemm_tc(TcContext* tc, const TcOperands& o, int64_t M, int Nc, const Epilogue& e,
                           int sm_count, int cta_group, cudaStream_t st, int64_t* nlaunch);

// similarity on the tensor cores from packed queries (simtc.cu).  cop: workspace of
// sim_tc_operand_bytes() for the staged class operand; amax_scratch: one float (hv_bits 8).
// e.kind is EPI_SCORE or EPI_ARGMAX; e.ham_D > 0 reports Hamming distances (hv_bits 1).
size_t sim_tc_operand_bytes(int K, int hv_bits, int D_eff);
cudaError_t launch_sim_tc(TcContext* tc, const uint32_t* Hbits, int64_t N, int64_t ldh, const float* C_acc,
                          int K, int64_t ldc, int D_eff, int hv_bits, void* cop, float* amax_scratch,
                          const Epilogue& e, Perf pf, double* partial, bool cop_ready, bool prep_only, int sm_count,
                          int force_cg, cudaStream_t st, int64_t* nlaunch, int piece = 0, int width = 0,
                          int* live = nullptr);
// piece > 0 (with hv_bits = HDC_HV_I16): the staged operand is the balanced base-65536 piece `piece - 1` of the
// `width`-bit integer code rint(C_acc) (HDC_HV_I32 / HDC_HV_I64, reading A22) instead of the scaled int16 code
// live (piece mode, nullable): one int, set to 1 by the preparation when the piece holds a nonzero code (the caller
// zeroes it first: launch_wide_prepare); the contraction returns at once while it is 0
// force_cg: 1 / 2 = one-CTA / CTA-pair kernel (knobs HDC_FLAG_TC_1CTA / _2CTA), else by problem size
// cop_ready: cop already holds the staged class operand of the same (C_acc, knobs) -- skip its preparation
// prep_only: stage the class operand into cop (and amax) and return without contracting
// partial: workspace of sim_tc_partial_bytes() (0 bytes / NULL: no split of the reduction axis)
size_t sim_tc_partial_bytes(int64_t N, int K, int hv_bits, int D_eff, int sm_count);
// amax = max |C[k][d]| over k < K and the visited d < D_eff (amax zeroed here)
cudaError_t launch_tensor_amax(const float* C, int K, int D_eff, int64_t ldc, Perf pf, float* amax,
                               cudaStream_t st, int64_t* nlaunch);
// mask[w] = bits of word w whose dimension is visited and < D_eff (W words)
// ADC-quantised chunked dot (adc.cu): transfer function tabulated by the number of
// differing bits in a chunk -- full[i] for 128-dimension chunks, tail[i] for the ragged last chunk.
struct AdcTables {
  int full[129];
  int tail[129];
};
size_t adc_class_bytes(int K, int D_eff);
cudaError_t launch_adc_similarity(const uint32_t* H, int64_t N, int64_t ldh, const float* C_acc, int K,
                                  int64_t ldc, int D_eff, const AdcTables& tab, uint32_t* class_ws, int32_t* S,
                                  int64_t lds, int32_t* labels, int sm_count, int smem_optin, cudaStream_t st,
                                  int64_t* nlaunch);

// Perforated encode contraction: compacted copy of the visited columns (esize = element bytes 1/2/4)
// and the compensation scale applied to the optional raw accumulators.
cudaError_t launch_gather_cols(const void* src, int esize, int64_t rows, int64_t ld_src, Perf pf, int n_vis,
                               void* dst, int64_t ld_dst, cudaStream_t st, int64_t* nlaunch);
cudaError_t launch_scale_raw(void* raw, int64_t rows, int cols, int64_t ld, float scale, int from_i32,
                             cudaStream_t st, int64_t* nlaunch);
cudaError_t launch_perf_mask(uint32_t* mask, int W, int D_eff, Perf pf, cudaStream_t st, int64_t* nlaunch);

// fp32/bf16 -> bf16 staging with zero padding of the reduction axis: dst [rows][ld_dst]
// HDC_FLAG_F32_FAST staging: per-row power-of-two scale + 2-way half split ([h1 | h2], seg columns each);
// expo[row] = the exponent applied; launch_unscale_raw undoes both operands' scales on raw accumulators.
cudaError_t launch_split2_f16(const void* src, int src_kind, int64_t rows, int cols, int64_t ld_src, __half* dst,
                              int seg, int* expo, cudaStream_t st, int64_t* nlaunch);
cudaError_t launch_unscale_raw(float* raw, int64_t rows, int cols, int64_t ld, const int* ex, const int* ep,
                               cudaStream_t st, int64_t* nlaunch);
cudaError_t launch_convert_f16(const void* src, int src_kind, int64_t rows, int cols, int64_t ld_src,
                               __half* dst, int64_t ld_dst, cudaStream_t st, int64_t* nlaunch);
cudaError_t launch_convert_bf16(const void* src, int src_kind, int64_t rows, int cols, int64_t ld_src,
                                __nv_bfloat16* dst, int64_t ld_dst, cudaStream_t st, int64_t* nlaunch);
// fp32/bf16 -> three bf16 segments [x1 | x2 | x3] with x1 = bf16(x), x2 = bf16(x - x1),
// x3 = bf16(x - x1 - x2) (each subtraction exact in fp32): dst [rows][3*seg] , zero padded
cudaError_t launch_split3_bf16(const void* src, int src_kind, int64_t rows, int cols, int64_t ld_src,
                               __nv_bfloat16* dst, int seg, cudaStream_t st, int64_t* nlaunch);
// per-row symmetric int8 quantisation (S1/A7): dst [rows][ld_dst] int8, zero padded
cudaError_t launch_quantize_rows_i8(const void* src, int src_kind, int64_t rows, int cols, int64_t ld_src,
                                    int8_t* dst, int64_t ld_dst, cudaStream_t st, int64_t* nlaunch);
// per-tensor symmetric int8 of C_acc[k<K][d<D_eff] (S5): amax_scratch is one float in ws
cudaError_t launch_quantize_tensor_i8(const float* C, int K, int D_eff, int64_t ldc, Perf pf, int8_t* dst,
                                      int64_t ld_dst, float* amax_scratch, cudaStream_t st,
                                      int64_t* nlaunch);
// per-tensor symmetric int16 of C_acc[k<K][d<D_eff] (S5 at HDC_HV_I16, A21): scale 32767 / amax
cudaError_t launch_quantize_tensor_i16(const float* C, int K, int D_eff, int64_t ldc, Perf pf, int16_t* dst,
                                       int64_t ld_dst, float* amax_scratch, cudaStream_t st,
                                       int64_t* nlaunch);
// class operand of the fused inference epilogue (EPI_INFER): dst [KC][ld_dst] fp32, row k < K = the class
// operand at hv_bits (32: C_acc; 16 / HDC_HV_F16: RNE to bf16 / half; 8: per-tensor int8 code, scale 127 / *amax;
// 1: +-1 from the sign), zero for d >= D_eff, unvisited d and rows >= K
cudaError_t launch_class_operand_f32(const float* C, int K, int D_eff, int64_t ldc, int hv_bits, Perf pf,
                                     const float* amax, float* dst, int KC, int64_t ld_dst, cudaStream_t st,
                                     int64_t* nlaunch);
// sign bits of C_acc: cbits [K][W] (tail bits zero)
cudaError_t launch_sign_bits(const float* C, int K, int D_eff, int64_t ldc, uint32_t* cbits, int W,
                             cudaStream_t st, int64_t* nlaunch);
// colscale[k] = cos ? (nrm_k > 0 ? 1/(sqrt(n_visited)*nrm_k) : 0) : 1, nrm over the visited
// dimensions of the operand as loaded
// colscale_f (nullable): receives (float)colscale[k]
cudaError_t launch_col_scale(const Operand& C, int K, int D_eff, int cos, Perf pf, double* colscale,
                             cudaStream_t st, int64_t* nlaunch, float* colscale_f = nullptr);

// 32- / 64-bit integer class operands (widedot.cu; hv codes HDC_HV_I32 / HDC_HV_I64, reading A22): the codes
// rint(C_acc) staged as byte planes (wide_operand_bytes; 0 for any other hv_bits) with the cosine scales, and
// the dp4a contraction of packed queries against them (e.kind EPI_ARGMAX, or EPI_SCORE with e.s_i32 = 0 for
// fp32 scores, 2 for int64 scores)
size_t wide_operand_bytes(int K, int hv_bits, int D_eff);
// tensor-core route: the 16-bit pieces of the codes are contracted one by one by sim_tc_kernel (int32 scores
// S_j [rows][K], j < pieces, piece j at Sp + j * rows * K) and recombined here as sum_j S_j << 16j in 64 bits
// before the same epilogue (arg-max / fp32 / int64 scores); e's row pointers are those of the first row
cudaError_t launch_wide_combine(const int32_t* Sp, int pieces, int64_t rows, int K, int cos, const double* colscale,
                                const int* live, const Epilogue& e, cudaStream_t st, int64_t* nlaunch);
// live: `pieces` ints, piece j is read only where live[j] != 0 (its scores were not written otherwise)
cudaError_t launch_wide_prepare(const float* C_acc, int K, int64_t ldc, int D_eff, int hv_bits, Perf pf, int cos,
                                uint32_t* planes, double* colscale, cudaStream_t st, int64_t* nlaunch,
                                int* live = nullptr);   // live (nullable): four ints, zeroed here
cudaError_t launch_wide_dot(const uint32_t* Hbits, int64_t N, int64_t ldh, int K, int D_eff, int hv_bits, int cos,
                            const uint32_t* planes, const double* colscale, const Epilogue& e, cudaStream_t st,
                            int64_t* nlaunch);

// packed XOR+popcount similarity with class bits in shared memory (hamming.cu)
// mask (nullable): W words; distances count only the bits set in it (reduction perforation)
cudaError_t launch_hamming(const uint32_t* Hbits, int64_t N, int64_t ldh, const uint32_t* Cbits, int K,
                           int W, int D_eff, const uint32_t* mask, int32_t* dist, int64_t lds, int32_t* labels,
                           float* best, float* second, int sm_count, int smem_optin, cudaStream_t st,
                           int64_t* nlaunch);

// level-ID encode (levelid.cu)
// levels: uint8_t indices, or uint16_t when lvl16 != 0 (general kernel only)
cudaError_t launch_levelid(const void* levels, int lvl16, int64_t N, int F, int64_t ldl, const uint32_t* ID,
                           int64_t ldid, const uint32_t* LV, int Q, int64_t ldlv, int D_eff,
                           uint32_t* Hbits, int64_t ldh, int sm_count, int smem_optin, cudaStream_t st,
                           int64_t* nlaunch);

// class update (train.cu): delta int32 [K][W*32] workspace
cudaError_t launch_class_update(const uint32_t* Hbits, int64_t n0, int64_t nb, int64_t ldh,
                                const int32_t* y, const int32_t* pred /*null => bundle*/, float* C_acc,
                                int K, int64_t ldc, int D_eff, float lr, int32_t* delta,
                                unsigned long long* n_wrong, int sm_count, cudaStream_t st,
                                int64_t* nlaunch);

// the two halves of launch_class_update (multi-GPU training exchanges delta between them)
cudaError_t launch_class_delta(const uint32_t* Hbits, int64_t n0, int64_t nb, int64_t ldh, const int32_t* y,
                               const int32_t* pred, int K, int D_eff, int32_t* delta,
                               unsigned long long* n_wrong, int sm_count, cudaStream_t st, int64_t* nlaunch);
cudaError_t launch_apply_update(float* C_acc, int K, int64_t ldc, int D_eff, const int32_t* delta, float lr,
                                int sm_count, cudaStream_t st, int64_t* nlaunch);

// HD-Clustering re-bundle step (train.cu): counts members per cluster (members: int32 [K] workspace),
// adds the number of samples with assign != prev to *n_changed (both nullable) and zeroes the
// accumulator rows of the clusters that have members
cudaError_t launch_kmeans_reset(const int32_t* assign, const int32_t* prev, int64_t N, float* C_acc, int K,
                                int64_t ldc, int D_eff, int32_t* members, unsigned long long* n_changed,
                                int sm_count, cudaStream_t st, int64_t* nlaunch);

static inline int64_t round_up(int64_t x, int64_t m) { return (x + m - 1) / m * m; }
static inline int words_of(int D_eff) { return (D_eff + 31) >> 5; }

}  // namespace hdc
