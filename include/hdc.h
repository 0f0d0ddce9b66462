/* hdc.h -- C ABI of libhdc.so: the data-parallel HDC hot path of arxiv/paper_2606_26547
 * (ApproxHDC) as hand-written CUDA for NVIDIA B200 (sm_100a).
 *
 * The path (section 2.1, Listing 1 L63-L81): (1) encode feature vectors into D-dimensional
 * hypervectors, (2) similarity search against K class hypervectors, (3) arg-extremum and the
 * perceptron-style class update.  The paper's approximation knobs (section 4.2: reduction perforation
 * L155, binarization L161, encoding dimensionality L163, element type L165, algorithmic choice
 * L167, retraining epochs L181) are RUNTIME arguments (`hdc_knobs_t`, the `epochs` loop is the
 * caller's).
 *
 * General contract
 *  - Every data pointer is a DEVICE pointer owned by the caller, unless the parameter name ends in
 *    `_host` (then it is a host pointer, pinned for full speed).  A call may be made with any device current:
 *    its work goes to the handle's device.  Nothing is allocated or freed
 *    inside a compute call; scratch comes from the caller's workspace `ws` (size from
 *    hdc_workspace_bytes()).  `stream` is a cudaStream_t (NULL = legacy default stream).  Calls
 *    enqueue work and return; they do not synchronise (the `_host` entry point does, it says so).
 *  - Return value: HDC_OK (0) or a negative hdc_status.  Argument errors are detected on the host
 *    BEFORE anything is enqueued.  A failed launch maps to HDC_ERR_CUDA; hdc_last_error() gives
 *    the text.  Device faults are sticky CUDA errors seen at the caller's next synchronisation.
 *  - Layouts are row-major with the reduction axis contiguous: X[N][ldx], P[D][ldp] (row d =
 *    projection d, Listing 1 `hypermatrix<2048,617>` L65), C[K][ldc] (`hypermatrix<26,2048>`
 *    L66).  `ld*` are in ELEMENTS (uint32 words for bit matrices).  Base pointers must be 16-byte
 *    aligned and fp32/bf16 leading dimensions a multiple of 4 / 8 elements where stated.
 *  - Packed hypervectors: bipolar value v in {+1,-1} is stored as bit b = [v == -1]; element d is
 *    bit (d & 31) of uint32 word (d >> 5), LSB first.  Exactly W = ceil(D_eff/32) words are
 *    written per row; bits >= D_eff of the last word are written as 0.  sgn(0) = +1 (bit 0).
 *  - D_eff (1 <= D_eff <= D): every reduction over d and every output row is restricted to
 *    d < D_eff and nothing is rescaled (L61 "only the first 1024 elements", L155 "used as-is").
 *    Results equal those obtained by slicing every [.][D] array to its first D_eff columns.
 *  - arg-max / arg-min ties go to the lowest class index.  Inputs must be finite.
 *  - Empty inputs: a call with N == 0 validates its other arguments, enqueues nothing and returns
 *    HDC_OK; the per-sample pointers (X, levels, Hbits, S, labels, y, pred) may then be NULL.
 *  - Outputs must not alias inputs (except C_acc, which is in/out).  A handle is not thread-safe;
 *    distinct handles are independent.  There is no CPU fallback and no other architecture:
 *    hdc_create() fails with HDC_ERR_ARCH unless the device is compute capability 10.0 (the library
 *    holds sm_100a code only).
 */
#ifndef HDC_H_
#define HDC_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct hdc_ctx* hdc_handle_t;

typedef enum {
  HDC_OK = 0,
  HDC_ERR_INVALID_ARG = -1, /* null pointer, size <= 0, D_eff out of range, bad enum        */
  HDC_ERR_UNSUPPORTED = -2, /* a valid combination this build does not implement             */
  HDC_ERR_ALIGNMENT = -3,   /* base pointer / leading dimension alignment                    */
  HDC_ERR_WORKSPACE = -4,   /* ws == NULL or ws_bytes < hdc_workspace_bytes(...)             */
  HDC_ERR_CUDA = -5,        /* CUDA runtime / launch error (text in hdc_last_error)          */
  HDC_ERR_ARCH = -6         /* device is not sm_100                                          */
} hdc_status;

/* element types of buffers */
enum { HDC_F32 = 0, HDC_BF16 = 1, HDC_I8 = 2, HDC_B1 = 3, HDC_U8 = 4, HDC_I32 = 5, HDC_F16 = 6, HDC_I64 = 7 };
/* similarity kinds (L167 algorithmic choice) */
enum { HDC_SIM_DOT = 0, HDC_SIM_COS = 1, HDC_SIM_HAMMING = 2 };
/* knobs.hv_bits codes (not widths): 16-bit IEEE half class operand (L165 "FP16"); 16-, 32- and 64-bit
 * integer class operands (L165 "integer data types (8, 16, 32, or 64-bit)") */
enum { HDC_HV_F16 = 17, HDC_HV_I16 = 18, HDC_HV_I32 = 19, HDC_HV_I64 = 20 };
/* hdc_train_epoch modes */
enum { HDC_TRAIN_BUNDLE = 0, HDC_TRAIN_PERCEPTRON = 1, HDC_TRAIN_KMEANS = 2 };
/* hdc_encode_rp outputs (bit-or) */
enum { HDC_OUT_BITS = 1, HDC_OUT_RAW = 4 };
/* hdc_workspace_bytes ops */
enum { HDC_OP_ENCODE_RP = 0, HDC_OP_ENCODE_LEVELID = 1, HDC_OP_SIMILARITY = 2, HDC_OP_CLASSIFY = 3,
       HDC_OP_TRAIN_EPOCH = 4, HDC_OP_INFER_RP_HOST = 5, HDC_OP_INFER_RP = 6 };
/* knobs.flags */
enum {
  HDC_FLAG_NONE = 0,
  HDC_FLAG_SIMT = 1, /* force the CUDA-core (FFMA / popcount) kernels where a tensor-core kernel
                        exists for the same operation (debugging, A/B measurement)              */
  HDC_FLAG_TC_1CTA = 2, /* encode and similarity contractions: force the one-CTA-per-tile tcgen05 kernels */
  HDC_FLAG_TC_2CTA = 4, /* ... force the CTA-pair (cta_group::2) tcgen05 kernels; without either flag the
                           library chooses by problem size                                      */
  HDC_FLAG_F32_FAST = 8, /* precision HDC_F32 only, OFF by default: contract 2-way IEEE-half splits of
                           the row-scaled operands (22 of the 24 mantissa bits, three tensor-core
                           products instead of six; |error| <= 3 * 2^-22 * sum|x p|).  An extra point
                           of the element-precision knob (L165) between bf16 and fp32, not fp32.  */
  HDC_FLAG_FUSED_INFER = 16 /* hdc_infer_rp / hdc_infer_rp_host only, OFF by default: for K <= 32 and
                           N >= 12288 run encode + similarity + arg-max as ONE kernel (the epilogue warps of the
                           contraction search each signed row against the class hypervectors on the CUDA
                           cores; the hypervectors need not reach HBM).  Same results as the two kernels;
                           measured SLOWER than them on B200 (the class values reach the FFMAs through shared
                           memory, whose bandwidth the tensor-core operand traffic already uses up:
                           DESIGN.md section 6), kept as a tested A/B switch.                              */
};

/* Approximation knobs (section 4.2).
 *  D_eff      effective dimensionality, 1..D (L61, L155, L163).
 *  precision  operand type of the encode contraction (L165): HDC_F32 | HDC_BF16 | HDC_F16 | HDC_I8 |
 *             HDC_B1.  HDC_F16: operands rounded to nearest-even IEEE half, fp32 accumulate.
 *             HDC_BF16: operands rounded to nearest-even bf16, fp32 accumulate.  HDC_I8: per-row
 *             symmetric int8 of X and of P (a = max|row|, s = 127/a, q = clamp(rint(x*s),+-127)),
 *             int32 accumulate.  HDC_B1: packed hypervectors with the real-valued contraction in
 *             bf16 (same contraction as HDC_BF16).
 *  hv_bits    element width of the CLASS hypervectors in similarity / classify / train (L165):
 *             32 fp32 | 16 bf16 (RNE of C_acc) | HDC_HV_F16 IEEE half (RNE of C_acc; |c| > 65504
 *             overflows, outside the contract) | 8 int8 (per-tensor symmetric over k<K, d<D_eff)
 *             | HDC_HV_I16 int16 (per-tensor symmetric over k<K, d<D_eff: s = 32767/max|c|,
 *             q = clamp(rint(c*s), +-32767); int32 accumulate, exact: D_eff*32767 < 2^31)
 *             | HDC_HV_I32 / HDC_HV_I64 32- / 64-bit integers: the accumulators themselves,
 *             q = rint(c) (half to even), NO scale, saturating at +-(2^31 - 1) / +-(2^63 - 1); scores
 *             are exact integers accumulated in 64 bits (contract: sum_d |q[k,d]| < 2^63, beyond it the
 *             sums wrap), DOT / COS only; contracted on the tensor cores as balanced 16-bit pieces of the
 *             codes (each an int16-style operand, exact int32 scores, recombined in 64 bits), or with
 *             HDC_FLAG_SIMT by dp4a over the byte planes of the codes
 *             | 1 sign bit [C_acc < 0].  Query hypervectors are always bipolar (packed bits).
 *  sim        HDC_SIM_*; HDC_SIM_HAMMING requires hv_bits == 1.
 *  flags      HDC_FLAG_*.
 *  perf_begin, perf_stride   reduction perforation of the SIMILARITY (L155 "skip iterations at
 *             regular intervals, defined by a specified stride"; parameters starting offset, ending
 *             offset, stride: L76-L77, L130): the reductions over d in hdc_similarity / hdc_classify
 *             and in the prediction step of hdc_train_epoch visit d = perf_begin + j*perf_stride
 *             < D_eff only (D_eff is the ending offset).  Results equal those obtained by gathering
 *             the visited dimensions of both operands; nothing is rescaled (L155); the int8 class
 *             scale and the cosine norms are taken over the visited dimensions.  0 <= perf_begin
 *             < D_eff; perf_stride 0 or 1 = every dimension.  Encoders and class updates are not
 *             perforated by these two (L157, L187).  Not available with HDC_FLAG_SIMT for DOT /
 *             COS (HDC_ERR_UNSUPPORTED).
 *  enc_perf_begin, enc_perf_stride   reduction perforation of the ENCODE contraction, read by
 *             hdc_encode_rp and hdc_infer_rp_host only (L155: "for operations such as matrix-vector
 *             dot products, the results are scaled appropriately to compensate for the skipped
 *             iterations"): the F reduction visits f = enc_perf_begin + j*enc_perf_stride < F, the
 *             operands at `precision` are those of the gathered columns (per-row int8 scales over
 *             the visited features) and the accumulators are multiplied by F / F_visited.  Off
 *             (0, 0) by default: the paper keeps perforation out of the encoders because it "often
 *             degrades the quality-of-service" (L157, L187).  0 <= enc_perf_begin < F;
 *             enc_perf_stride 0 or 1 = every feature.                                            */
typedef struct {
  int32_t D_eff;
  int32_t precision;
  int32_t hv_bits;
  int32_t sim;
  int32_t flags;
  int32_t perf_begin;
  int32_t perf_stride;
  int32_t enc_perf_begin;
  int32_t enc_perf_stride;
} hdc_knobs_t;

/* ---- handle ------------------------------------------------------------------------------ */
/* Creates a context on CUDA device `device` (sets nothing globally except cudaSetDevice during
 * the call).  HDC_ERR_ARCH unless compute capability 10.0; HDC_ERR_CUDA if no device. */
int32_t hdc_create(hdc_handle_t* out, int32_t device);
int32_t hdc_destroy(hdc_handle_t h);
/* Host string describing the last error on this handle; valid until the next call on it. */
const char* hdc_last_error(hdc_handle_t h);
/* ABI version of this header (major*100 + minor). */
int32_t hdc_version(void);
/* Number of kernel launches this handle has enqueued since creation (bench `gpu_launches`). */
int64_t hdc_launch_count(hdc_handle_t h);

/* Which kernels the handle has chosen since creation (a tensor-core request that silently ran on the CUDA
 * cores, or a fused inference that ran as two kernels, costs a multiple of the time with HDC_OK: this makes it
 * visible).  HDC_STAT_TC_LAUNCHES: encode contractions on the tcgen05 kernels; HDC_STAT_SIMT_FALLBACKS: encode
 * contractions for which the tensor path was asked (no HDC_FLAG_SIMT) but refused the operands, so the
 * CUDA-core kernel ran (hdc_last_error then says so); HDC_STAT_INFER_FUSED / _UNFUSED: hdc_infer_rp /
 * hdc_infer_rp_host passes (per chunk) through the fused kernel / through encode + classify.  -1: bad id. */
enum { HDC_STAT_TC_LAUNCHES = 0, HDC_STAT_SIMT_FALLBACKS = 1, HDC_STAT_INFER_FUSED = 2, HDC_STAT_INFER_UNFUSED = 3,
       HDC_STAT_COUNT = 4 };
int64_t hdc_stat(hdc_handle_t h, int32_t stat_id);

/* Per-kernel device timing (for roofline reporting).  While enabled, the dominant kernel of each
 * entry point is bracketed by CUDA events on the caller's stream: HDC_K_ENCODE_GEMM (contraction of
 * hdc_encode_rp, staging excluded), HDC_K_SIM (similarity / classify kernel, operand staging
 * excluded), HDC_K_LEVELID, HDC_K_CLASS_UPDATE.  hdc_kernel_time() synchronises the recorded events,
 * returns the summed milliseconds and the number of launches of that kernel since the last call (or
 * since enabling) and resets them.  At most 1024 launches per kernel id are kept between reads. */
enum { HDC_K_ENCODE_GEMM = 0, HDC_K_SIM = 1, HDC_K_LEVELID = 2, HDC_K_CLASS_UPDATE = 3, HDC_K_COUNT = 4 };
int32_t hdc_kernel_timing(hdc_handle_t h, int32_t enable);
int32_t hdc_kernel_time(hdc_handle_t h, int32_t kernel_id, float* ms_total, int64_t* launches);

/* Bytes of device workspace the given op needs for these sizes and knobs (0 is possible).
 * F_or_Q: F for encode_rp / infer_rp / infer_rp_host, Q for encode_levelid, ignored otherwise.
 * For HDC_OP_TRAIN_EPOCH, N is the mini-batch size actually used (batch, or N when batch = 0); for
 * HDC_TRAIN_KMEANS and hdc_train_delta it is the number of samples of the call. */
size_t hdc_workspace_bytes(hdc_handle_t h, int32_t op, int64_t N, int32_t F_or_Q, int32_t D,
                           int32_t K, const hdc_knobs_t* knobs);

/* ---- (1a) random-projection encode + sign + pack ------------------------------------------
 * PAPER.md Listing 1 L68-L70 `__hetero_hdc_matmul`, L155, L161 (automatic binarization).
 *   acc[n,d] = sum_{f<F} x~[n,f] * p~[d,f],   bit[n,d] = [acc[n,d] < 0],   d < D_eff
 * (x~, p~ = operands at knobs->precision).  The F reduction is perforated only when
 * knobs->enc_perf_* ask for it (see hdc_knobs_t); the bits do not depend on the compensation scale.
 * X [N][ldx] of x_dtype (HDC_F32 or HDC_BF16); P [D][ldp] of p_dtype (HDC_F32 or HDC_BF16).
 * A bf16 input under precision HDC_F32 is widened exactly.  out_kinds: HDC_OUT_BITS writes
 * Hbits [N][ldh_words]; HDC_OUT_RAW additionally writes the accumulators to Hraw [N][ldraw]
 * (float for F32/BF16/B1, int32 for I8; with a perforated reduction always float:
 * fl32(fl32(acc) * fl32(F / F_visited))).  Unused outputs may be NULL. */
int32_t hdc_encode_rp(hdc_handle_t h, const void* X, int32_t x_dtype, int64_t N, int32_t F,
                      int64_t ldx, const void* P, int32_t p_dtype, int32_t D, int64_t ldp,
                      const hdc_knobs_t* knobs, int32_t out_kinds, uint32_t* Hbits,
                      int64_t ldh_words, void* Hraw, int64_t ldraw, void* ws, size_t ws_bytes,
                      void* stream);

/* ---- (1b) level-ID record encode ----------------------------------------------------------
 * PAPER.md L167 ("ID-based encoding"), L183 (N_LEVELS), L239 (Level-ID); bind = XOR, bundle =
 * majority (BASELINE.json north_star).
 *   cnt[n,d] = sum_{f<F} ( ID[f,d] XOR LV[levels[n,f], d] ),   bit[n,d] = [2*cnt > F]
 * levels [N][ldl] uint8 level indices, each < Q <= 256 (unchecked on device); F above what one CTA can stage
 * in shared memory (about 7000 features; 3500 for the 16-bit variant) returns HDC_ERR_UNSUPPORTED;
 * IDbits [F][ldid_words], LVbits [Q][ldlv_words] packed tables covering D bits. */
int32_t hdc_encode_levelid(hdc_handle_t h, const uint8_t* levels, int64_t N, int32_t F, int64_t ldl,
                           const uint32_t* IDbits, int64_t ldid_words, const uint32_t* LVbits,
                           int32_t Q, int64_t ldlv_words, int32_t D, const hdc_knobs_t* knobs,
                           uint32_t* Hbits, int64_t ldh_words, void* ws, size_t ws_bytes,
                           void* stream);
/* Same with 16-bit level indices, 1 <= Q <= 65535 (PAPER.md L183 N_LEVELS "quantization granularity",
 * L255: the Micro-HD comparison tunes the number of levels up to 814).  levels [N][ldl] uint16. */
int32_t hdc_encode_levelid_u16(hdc_handle_t h, const uint16_t* levels, int64_t N, int32_t F, int64_t ldl,
                               const uint32_t* IDbits, int64_t ldid_words, const uint32_t* LVbits, int32_t Q,
                               int64_t ldlv_words, int32_t D, const hdc_knobs_t* knobs, uint32_t* Hbits,
                               int64_t ldh_words, void* ws, size_t ws_bytes, void* stream);

/* ---- (2) similarity -----------------------------------------------------------------------
 * PAPER.md L72-L74 `__hetero_hdc_hamming_distance`, L110 `__hetero_hdc_cos_sim`, L197 dot.
 * Hbits [N][ldh_words] packed queries; C_acc [K][ldc] fp32 class accumulators, from which the
 * class operand is derived at knobs->hv_bits.  Over d < D_eff:
 *   HAMMING  dist[n,k] = popcount(h[n] xor cbit[k])                       -> S int32 [N][lds]
 *   DOT      s[n,k]   = sum_d v[n,d]*c[k,d]                               -> S fp32 (int32 if hv_bits 8, HDC_HV_I16 or 1)
 *   COS      s[n,k]   = DOT / (sqrt(D_eff) * sqrt(sum_d c[k,d]^2)), 0 if the norm is 0   -> S fp32
 * s_dtype must be HDC_I32 for HAMMING, HDC_F32 for COS, HDC_F32 or HDC_I32 for DOT (HDC_I32 only
 * for hv_bits 8, HDC_HV_I16 or 1; fp32 scores of an int16 operand are the exact int32 sum rounded once).
 * hv_bits HDC_HV_I32 / HDC_HV_I64: DOT writes HDC_F32 (the exact 64-bit sum rounded once) or HDC_I64
 * (S int64 [N][lds], 8-byte aligned), COS writes HDC_F32. */
int32_t hdc_similarity(hdc_handle_t h, const uint32_t* Hbits, int64_t N, int64_t ldh_words,
                       const float* C_acc, int32_t K, int64_t ldc, int32_t D,
                       const hdc_knobs_t* knobs, void* S, int32_t s_dtype, int64_t lds, void* ws,
                       size_t ws_bytes, void* stream);

/* ---- (2') chunked, ADC-quantised dot similarity (SpecPCM simulator) --------------------------
 * "The SpecPCM simulator computes dot-product similarity over 128-element array
 * chunks, with each partial dot product quantized by the ADC before accumulation"; hardware knobs
 * ADC_RES, ADC_STEP, ADC_FLOOR, ADC_CEIL; MLC = 1: +-1 hypervectors (class operand = sign of C_acc).
 *   s[n,k] = sum_j adc( sum_{d in [128 j, 128 j + 128), d < D_eff} v[n,d] * c[k,d] )
 *   adc(p) = floor + step * min( (clamp(p, floor, ceil) - floor + step/2) / step , 2^res - 1 )
 * (integer arithmetic, step/2 and the division rounded down: nearest code, halves up; the paper
 * prints no formula: DESIGN.md reading A19.  floor -127, ceil 128, res 8, step 1 -- the paper's
 * baseline window -- is transparent on [-127, 128]).  1 <= res <= 16, 1 <= step <= 65536, floor <= ceil,
 * |floor|, |ceil| <= 32768; only knobs->D_eff is read.  S (int32 [N][lds], nullable) receives the
 * scores, labels (int32 [N], nullable) the arg-max with ties to the lowest k; at least one of them.
 * Workspace: hdc_workspace_bytes(HDC_OP_SIMILARITY, ...) suffices. */
typedef struct {
  int32_t res;   /* ADC_RES: number of output bits */
  int32_t step;  /* ADC_STEP: input units per code */
  int32_t floor; /* ADC_FLOOR: lowest input / level */
  int32_t ceil;  /* ADC_CEIL: highest input */
} hdc_adc_t;
int32_t hdc_similarity_adc(hdc_handle_t h, const uint32_t* Hbits, int64_t N, int64_t ldh_words,
                           const float* C_acc, int32_t K, int64_t ldc, int32_t D,
                           const hdc_knobs_t* knobs, const hdc_adc_t* adc, int32_t* S, int64_t lds,
                           int32_t* labels, void* ws, size_t ws_bytes, void* stream);

/* ---- (2+3a) classify = similarity + arg-extremum, fused (no S matrix) ----------------------
 * PAPER.md Listing 1 L72-L80.  labels[n] = arg-max (DOT, COS) or arg-min (HAMMING) over k, ties
 * to the lowest k.  best / second (nullable, fp32 [N]) receive the winning and runner-up score
 * (distances as floats for HAMMING; second = best when K == 1 or on a tie). */
int32_t hdc_classify(hdc_handle_t h, const uint32_t* Hbits, int64_t N, int64_t ldh_words,
                     const float* C_acc, int32_t K, int64_t ldc, int32_t D,
                     const hdc_knobs_t* knobs, int32_t* labels, float* best, float* second,
                     void* ws, size_t ws_bytes, void* stream);

/* ---- (3b,3c) one-pass bundling and one retraining epoch ------------------------------------
 * PAPER.md L53 (class hypervectors by vector addition), L181 (TRAIN_ITERATIONS); the update
 * rule is the perceptron-style reading S9 of DESIGN.md.
 *  mode HDC_TRAIN_BUNDLE:      C_acc[k,d] += sum_{n: y_n = k} v[n,d]             (knobs: D_eff only)
 *  mode HDC_TRAIN_PERCEPTRON:  samples in index order; per mini-batch of `batch` samples
 *      (0 => N): yhat = classify(h) with the current C_acc at knobs->{hv_bits,sim};
 *      Delta[k,d] = sum_{yhat_n != y_n} ([k = y_n] - [k = yhat_n]) * v[n,d]   (integer);
 *      C_acc[k,d] = fl32(C_acc[k,d] + fl32(lr * (float)Delta[k,d])).
 *  mode HDC_TRAIN_KMEANS (HD-Clustering; reading A16): one Lloyd
 *      iteration over all N samples: a = classify(h) with the current C_acc at knobs->{hv_bits,sim};
 *      every cluster with at least one member is re-bundled, C_acc[k,d] = sum_{n: a_n = k} v[n,d];
 *      a cluster without members keeps its accumulator.  y is the PREVIOUS assignment (nullable),
 *      pred receives a, n_wrong is incremented by #{n : a_n != y_n} (0 moved = converged);
 *      lr and batch are ignored.
 * y [N] int32 labels in [0,K) (unchecked on device).  pred (nullable, int32 [N]) receives yhat;
 * n_wrong (nullable, device uint64) is INCREMENTED by the number of mispredictions.
 * Deterministic: integer Delta, no floating-point atomics. */
int32_t hdc_train_epoch(hdc_handle_t h, int32_t mode, const uint32_t* Hbits, int64_t N,
                        int64_t ldh_words, const int32_t* y, float* C_acc, int32_t K, int64_t ldc,
                        int32_t D, const hdc_knobs_t* knobs, float lr, int64_t batch, int32_t* pred,
                        unsigned long long* n_wrong, void* ws, size_t ws_bytes, void* stream);

/* ---- (3c) the two halves of a retraining mini-batch, for data-parallel training ------------------
 * hdc_train_epoch(PERCEPTRON) is, per mini-batch, hdc_train_delta followed by hdc_train_apply.
 * With the mini-batch split over several GPUs every rank calls hdc_train_delta
 * on its shard, the int32 deltas are summed across ranks (one all-reduce of K*W*32 integers: integer
 * addition, so the result does not depend on the order), and every rank calls hdc_train_apply with
 * the summed delta: the replicas of C_acc stay bit-identical.
 *  hdc_train_delta: yhat = classify(h) with C_acc at knobs->{hv_bits, sim, perforation};
 *      delta[k][d] = sum_{n < N, yhat_n != y_n} ([k = y_n] - [k = yhat_n]) * v[n,d], written (not
 *      accumulated) as int32 [K][W*32], W = ceil(D_eff/32); pred (nullable) receives yhat; n_wrong
 *      (nullable) is incremented.  N == 0 writes zeros.  Workspace: HDC_OP_TRAIN_EPOCH for N.
 *  hdc_train_apply: C_acc[k,d] = fl32(C_acc[k,d] + fl32(lr * (float)delta[k][d])) for d < D_eff. */
int32_t hdc_train_delta(hdc_handle_t h, const uint32_t* Hbits, int64_t N, int64_t ldh_words,
                        const int32_t* y, const float* C_acc, int32_t K, int64_t ldc, int32_t D,
                        const hdc_knobs_t* knobs, int32_t* delta, int32_t* pred,
                        unsigned long long* n_wrong, void* ws, size_t ws_bytes, void* stream);
int32_t hdc_train_apply(hdc_handle_t h, float* C_acc, int32_t K, int64_t ldc, int32_t D,
                        const hdc_knobs_t* knobs, const int32_t* delta, float lr, void* stream);

/* ---- (1a)+(2)+(3a) inference in one call ----------------------------------------------------
 * PAPER.md Listing 1 L63-L81 (`inference`: matmul -> hamming_distance / cos_sim -> arg_min as one task),
 * L161 (binarization between them).  labels[n] = hdc_classify(hdc_encode_rp(X))[n] with the same knobs:
 * operand precisions, D_eff, similarity, class width and perforation exactly as in those two calls (integer
 * class operands -- hv_bits 8 and 1 -- give the same labels bit for bit; float class operands the same
 * scores up to fp32 summation order, i.e. within the 1e-3 tolerance of the float paths).  best / second
 * (nullable) as in hdc_classify.  Hbits (NULLABLE, [N][ldh_words]) additionally receives the hypervectors.
 * The call runs the encode and the classify kernels one after the other on `stream` (the hypervectors
 * stay in the workspace when Hbits is NULL).  With HDC_FLAG_FUSED_INFER, K <= 32 and N >= 12288 the three
 * steps run as ONE kernel instead (see the flag; hdc_stat says which path ran).
 * Workspace: hdc_workspace_bytes(HDC_OP_INFER_RP, N, F, D, K, knobs). */
int32_t hdc_infer_rp(hdc_handle_t h, const void* X, int32_t x_dtype, int64_t N, int32_t F, int64_t ldx,
                     const void* P, int32_t p_dtype, int32_t D, int64_t ldp, const float* C_acc, int32_t K,
                     int64_t ldc, const hdc_knobs_t* knobs, int32_t* labels, float* best, float* second,
                     uint32_t* Hbits, int64_t ldh_words, void* ws, size_t ws_bytes, void* stream);

/* ---- prepared model: the query-independent operands, converted once ------------------------
 * Every plain entry point derives the operands of its contraction from the caller's P and C_acc inside
 * the call (staged projection at knobs->precision; class operand at knobs->hv_bits with its int8 scale,
 * cosine scales, perforation mask) -- right for training, where C_acc changes every mini-batch, wasteful
 * for a server that classifies small batches against a fixed model.  hdc_model_prepare runs exactly those
 * preparation kernels once, into `blob` (DEVICE memory of the caller, >= hdc_model_bytes(), 256-byte
 * aligned), and fills the host descriptor *out; the *_m entry points take the descriptor instead of
 * (P, C_acc, knobs) and launch only the per-query kernels.  Results are identical, bit for bit, to the
 * plain entry points with the same arguments.  P or C_acc may be NULL (a model with one half only; F / K
 * are then ignored).  The descriptor is plain data (copy it freely); P, C_acc and blob must stay alive and
 * unchanged while it is in use (the CUDA-core kernels of HDC_FLAG_SIMT read P and C_acc in place).  The
 * knobs are fixed at preparation (the staged layouts depend on them) and stored in the descriptor.
 * Workspace of the *_m calls: as for hdc_encode_rp / hdc_classify / hdc_infer_rp. */
typedef struct {
  uint32_t magic;
  int32_t F, D, K, p_dtype;
  int64_t ldp, ldc;
  const void* P;
  const float* C_acc;
  void* blob;
  size_t blob_bytes;
  hdc_knobs_t knobs;
} hdc_model_t;
size_t hdc_model_bytes(hdc_handle_t h, int32_t F, int32_t D, int32_t K, const hdc_knobs_t* knobs);
int32_t hdc_model_prepare(hdc_handle_t h, const void* P, int32_t p_dtype, int32_t F, int32_t D, int64_t ldp,
                          const float* C_acc, int32_t K, int64_t ldc, const hdc_knobs_t* knobs, void* blob,
                          size_t blob_bytes, hdc_model_t* out, void* stream);
/* = hdc_encode_rp (HDC_OUT_BITS) / hdc_classify / hdc_infer_rp with the model's P, C_acc and knobs */
int32_t hdc_encode_rp_m(hdc_handle_t h, const void* X, int32_t x_dtype, int64_t N, int64_t ldx,
                        const hdc_model_t* m, uint32_t* Hbits, int64_t ldh_words, void* ws, size_t ws_bytes,
                        void* stream);
int32_t hdc_classify_m(hdc_handle_t h, const uint32_t* Hbits, int64_t N, int64_t ldh_words, const hdc_model_t* m,
                       int32_t* labels, float* best, float* second, void* ws, size_t ws_bytes, void* stream);
int32_t hdc_infer_rp_m(hdc_handle_t h, const void* X, int32_t x_dtype, int64_t N, int64_t ldx,
                       const hdc_model_t* m, int32_t* labels, float* best, float* second, uint32_t* Hbits,
                       int64_t ldh_words, void* ws, size_t ws_bytes, void* stream);

/* ---- classify without any allocation or caller workspace ----------------------------------------
 * = hdc_classify for knobs->sim == HDC_SIM_HAMMING, knobs->hv_bits == 1 (Hamming distance,
 * arg-min, ties to the lowest k; perforation knobs honoured), same labels / best / second bit for bit, for callers
 * that can neither allocate device memory nor hand over a workspace (under CUDA graph capture, tight serving
 * loops).  The scratch the call needs -- the packed sign bits of the class accumulators, K * W words, and the
 * perforation mask, W words, W = ceil(D_eff / 32) -- lives in a fixed array inside the library
 * (HDC_STATIC_SCRATCH_BYTES of device memory on every GPU that loads the library, held until the process exits).
 * Limits: (K + 1) * W * 4 <= HDC_STATIC_SCRATCH_BYTES and K <= 64; beyond them the call returns
 * HDC_ERR_UNSUPPORTED (message in hdc_last_error) and launches nothing.  The call performs no cudaMalloc /
 * cudaFree and calls no allocating library routine.
 * The array is SHARED by every call on that GPU (all handles, all streams) and keeps the previous call's contents
 * (each call rewrites every word it reads): two calls that may overlap on the GPU -- different streams without an
 * event between them, or two host threads -- race on it; serialise them.  Other argument rules as hdc_classify. */
#define HDC_STATIC_SCRATCH_BYTES (1u << 20)
int32_t hdc_classify_hamming_static(hdc_handle_t h, const uint32_t* Hbits, int64_t N, int64_t ldh_words,
                                    const float* C_acc, int32_t K, int64_t ldc, int32_t D,
                                    const hdc_knobs_t* knobs, int32_t* labels, float* best, float* second,
                                    void* stream);

/* ---- end-to-end inference from host buffers ------------------------------------------------
 * encode_rp + classify for N queries whose features live in HOST memory (pinned for full speed):
 * copies X_host in chunks to the device (inside the call), runs hdc_infer_rp per chunk and copies the
 * labels back to labels_host; synchronises `stream` before returning.  P and C_acc are device
 * pointers as above.  Used for the end-to-end (`e2e`) measurement. */
int32_t hdc_infer_rp_host(hdc_handle_t h, const void* X_host, int32_t x_dtype, int64_t N, int32_t F,
                          int64_t ldx, const void* P, int32_t p_dtype, int32_t D, int64_t ldp,
                          const float* C_acc, int32_t K, int64_t ldc, const hdc_knobs_t* knobs,
                          int32_t* labels_host, void* ws, size_t ws_bytes, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* HDC_H_ */
