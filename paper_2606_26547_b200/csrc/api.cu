// api.cu -- the C ABI of libhdc.so (include/hdc.h): argument validation on the host before anything
// is enqueued, workspace carving, and the sequencing of the kernels of each entry point.  No
// arithmetic of the method lives here.
#include <stdio.h>

#include <string>
#include <utility>
#include <vector>

#include "common.cuh"

struct hdc_ctx {
  int device = 0;
  int sm_count = 0;
  int smem_optin = 0;
  int64_t launches = 0;
  std::string err;
  hdc::TcContext* tc = nullptr;
  cudaStream_t copy_stream = nullptr;
  cudaEvent_t ev_copied[2] = {nullptr, nullptr};
  cudaEvent_t ev_done[2] = {nullptr, nullptr};
  cudaEvent_t ev_entry = nullptr;
  bool timing = false;
  // Where the per-call-invariant operands live (staged projection, class operand, scales) and whether this
  // pass prepares them, uses them, or both.  model == nullptr: they are carved from the call's workspace and
  // prepared in the call (the plain entry points).  hdc_model_prepare: PREP_ONLY into the caller's blob; the
  // *_m entry points and the chunks of hdc_infer_rp_host after the first: RUN_ONLY.
  void* model = nullptr;  // hdc::Bump*
  size_t model_cap = 0;
  int prep_mode = 0;  // PREP_AND_RUN
  std::vector<std::pair<cudaEvent_t, cudaEvent_t>> tev[HDC_K_COUNT];  // event pool per kernel id
  size_t tused[HDC_K_COUNT] = {0, 0, 0, 0};
  int64_t stats[HDC_STAT_COUNT] = {0, 0, 0, 0};
  uint32_t* static_scratch = nullptr;  // device address of g_static_scratch on this handle's device (resolved once)
};

namespace hdc {
namespace {

// Bump allocator over the caller's workspace; with base == nullptr it only measures.
struct Bump {
  char* base;
  size_t off = 0;
  explicit Bump(void* b) : base((char*)b) {}
  template <typename T>
  T* take(size_t count) {
    off = (size_t)round_up((int64_t)off, 256);
    T* p = base ? reinterpret_cast<T*>(base + off) : nullptr;
    off += count * sizeof(T);
    return p;
  }
};

enum PrepMode : int { PREP_AND_RUN = 0, PREP_ONLY = 1, RUN_ONLY = 2 };
// the allocator of the persistent operands of this pass
Bump& persistent(hdc_ctx* h, Bump& b) { return h->model ? *static_cast<Bump*>(h->model) : b; }
bool persistent_fits(const hdc_ctx* h, Bump& b, size_t ws_bytes) {
  if (b.off > ws_bytes) return false;
  return !h->model || static_cast<Bump*>(h->model)->off <= h->model_cap;
}
bool do_prep(const hdc_ctx* h) { return h->prep_mode != RUN_ONLY; }
bool prep_only(const hdc_ctx* h) { return h->prep_mode == PREP_ONLY; }

int fail(hdc_ctx* h, int code, const char* msg) {
  if (h) h->err = msg;
  return code;
}
int cuda_fail(hdc_ctx* h, cudaError_t e, const char* where) {
  if (h) h->err = std::string(where) + ": " + cudaGetErrorString(e);
  return HDC_ERR_CUDA;
}
// Brackets one kernel launch with CUDA events on `st` while hdc_kernel_timing is enabled.
struct Timed {
  hdc_ctx* h;
  cudaStream_t st;
  cudaEvent_t stop = nullptr;
  Timed(hdc_ctx* h_, int id, cudaStream_t st_) : h(h_), st(st_) {
    if (!h->timing || h->tused[id] >= 1024) return;
    if (h->tused[id] == h->tev[id].size()) {
      cudaEvent_t a, b;
      if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) return;
      h->tev[id].push_back({a, b});
    }
    auto& pr = h->tev[id][h->tused[id]++];
    cudaEventRecord(pr.first, st);
    stop = pr.second;
  }
  ~Timed() {
    if (stop) cudaEventRecord(stop, st);
  }
};

// Work of a handle goes to the handle's device whatever device the caller left current (restored on return).
struct DeviceGuard {
  int prev = -1;
  bool switched = false;
  explicit DeviceGuard(int device) {
    if (cudaGetDevice(&prev) == cudaSuccess && prev != device) switched = cudaSetDevice(device) == cudaSuccess;
  }
  ~DeviceGuard() {
    if (switched) cudaSetDevice(prev);
  }
};

bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15) == 0; }

int check_knobs(hdc_ctx* h, const hdc_knobs_t* k, int D) {
  if (!k) return fail(h, HDC_ERR_INVALID_ARG, "knobs is NULL");
  if (k->D_eff < 1 || k->D_eff > D) return fail(h, HDC_ERR_INVALID_ARG, "D_eff outside 1..D");
  return HDC_OK;
}
int check_sim_knobs(hdc_ctx* h, const hdc_knobs_t* k) {
  if (k->hv_bits != 32 && k->hv_bits != 16 && k->hv_bits != HDC_HV_F16 && k->hv_bits != HDC_HV_I16 &&
      k->hv_bits != HDC_HV_I32 && k->hv_bits != HDC_HV_I64 && k->hv_bits != 8 && k->hv_bits != 1)
    return fail(h, HDC_ERR_INVALID_ARG, "hv_bits must be 32, 16, HDC_HV_F16, HDC_HV_I16, HDC_HV_I32, HDC_HV_I64, 8 or 1");
  if (k->sim != HDC_SIM_DOT && k->sim != HDC_SIM_COS && k->sim != HDC_SIM_HAMMING)
    return fail(h, HDC_ERR_INVALID_ARG, "bad sim");
  if (k->sim == HDC_SIM_HAMMING && k->hv_bits != 1)
    return fail(h, HDC_ERR_INVALID_ARG, "HDC_SIM_HAMMING requires hv_bits == 1");
  if (k->perf_stride < 0 || k->perf_begin < 0 || k->perf_begin >= k->D_eff)
    return fail(h, HDC_ERR_INVALID_ARG, "perforation: need perf_stride >= 0 and 0 <= perf_begin < D_eff");
  return HDC_OK;
}
bool wide_int(const hdc_knobs_t* k) { return k->hv_bits == HDC_HV_I32 || k->hv_bits == HDC_HV_I64; }
// Rows per pass of the tensor-core route of the 32- / 64-bit integer class operands: the int32 scores of one 16-bit
// piece of a pass ([rows][K]) stay around 32 MB (L2-resident between sim_tc_kernel and the combine kernel), but a
// pass is never smaller than one wave of 128-row tiles on 148 SMs
int64_t wide_chunk_rows(int64_t N, int K) {
  int64_t rows = ((int64_t)8 << 20) / (K > 0 ? K : 1);
  rows -= rows % 256;
  if (rows < 18944) rows = 18944;
  return N < rows ? (N > 0 ? N : 1) : rows;
}
// workspace of that route: persistent class pieces (pm) and per-pass piece scores (b)
void wide_tc_ws(int64_t N, int K, const hdc_knobs_t* k, Bump* pm, Bump* b) {
  if (!wide_int(k)) return;
  const int pieces = k->hv_bits == HDC_HV_I32 ? 2 : 4;
  if (pm) {
    for (int j = 0; j < pieces; ++j) pm->take<uint8_t>(sim_tc_operand_bytes(K, HDC_HV_I16, k->D_eff));
    pm->take<int>(4);   // live flags of the pieces
  }
  if (b) b->take<int32_t>((size_t)pieces * (size_t)wide_chunk_rows(N, K) * (size_t)K);
}
Perf perf_of(const hdc_knobs_t* k) { return Perf{k->perf_begin, k->perf_stride <= 1 ? 1 : k->perf_stride}; }
Perf enc_perf_of(const hdc_knobs_t* k) {
  return Perf{k->enc_perf_begin, k->enc_perf_stride <= 1 ? 1 : k->enc_perf_stride};
}

// ------------------------------------------------------------------------------------- encode
// Reduction-segment schedule of the fp32-precision contraction over 3-way bf16 splits: segment s
// multiplies A part a(s) with B part b(s); smallest terms first (x3p1, x2p2, x1p3, x2p1, x1p2, x1p1).
constexpr uint32_t SPLIT_A_SEGS = 0x001012u;  // nibble s = a(s): 2,1,0,1,0,0
constexpr uint32_t SPLIT_B_SEGS = 0x010210u;  // nibble s = b(s): 0,1,2,0,1,0
// HDC_FLAG_F32_FAST: 2-way half splits, three products (h2 p1, h1 p2, h1 p1)
constexpr uint32_t SPLIT2_A_SEGS = 0x001u;  // a(s): 1,0,0
constexpr uint32_t SPLIT2_B_SEGS = 0x010u;  // b(s): 0,1,0

struct EncodePlan {
  bool tc = false;         // tensor-core kernel
  void* Xs = nullptr;      // staged X (bf16, 3 x bf16 or int8), null = use input in place
  void* Ps = nullptr;      // staged P
  int64_t ldxs = 0, ldps = 0;
  int Fp = 0;
  int* ex = nullptr;       // HDC_FLAG_F32_FAST: per-row scale exponents of X and of P
  int* ep = nullptr;
};

// 1 / 2 when the knobs force the 1-CTA / CTA-pair contraction kernel, 0 = by problem size
int tc_cta_group(const hdc_knobs_t* k) {
  return (k->flags & HDC_FLAG_TC_1CTA) ? 1 : (k->flags & HDC_FLAG_TC_2CTA) ? 2 : 0;
}

bool use_tc(const hdc_ctx* h, const hdc_knobs_t* k) {
  return h->tc != nullptr && !(k->flags & HDC_FLAG_SIMT);
}

// Carves the staging buffers of hdc_encode_rp.  x_inplace / p_inplace: operand usable as given.
// X staging comes from b (scratch), P staging from pm (persistent: may be the same allocator).
void plan_encode(const hdc_ctx* h, int64_t N, int F, int D_eff, const hdc_knobs_t* k, bool x_inplace,
                 bool p_inplace, Bump& b, Bump& pm, EncodePlan& pl) {
  const int prec = k->precision;
  pl.tc = use_tc(h, k);
  pl.Fp = (int)round_up(F, 64);
  if (prec == HDC_F32) {
    if (!pl.tc) return;  // FFMA kernel reads the operands in place
    if (k->flags & HDC_FLAG_F32_FAST) {
      pl.ldxs = pl.ldps = 2 * (int64_t)pl.Fp;
      pl.Xs = b.take<__half>((size_t)N * pl.ldxs);
      pl.Ps = pm.take<__half>((size_t)D_eff * pl.ldps);
      pl.ex = b.take<int>((size_t)N);
      pl.ep = pm.take<int>((size_t)D_eff);
      return;
    }
    pl.ldxs = pl.ldps = 3 * (int64_t)pl.Fp;
    pl.Xs = b.take<__nv_bfloat16>((size_t)N * pl.ldxs);
    pl.Ps = pm.take<__nv_bfloat16>((size_t)D_eff * pl.ldps);
    return;
  }
  if (prec == HDC_I8) {
    pl.ldxs = pl.ldps = pl.Fp;
    if (!x_inplace) pl.Xs = b.take<int8_t>((size_t)N * pl.Fp);
    if (!p_inplace) pl.Ps = pm.take<int8_t>((size_t)D_eff * pl.Fp);
    return;
  }
  // BF16 / B1 / F16 (half operands are always staged: the inputs are fp32 or bf16)
  if (!pl.tc) return;  // CUDA-core kernel rounds on load, no staging
  if (prec == HDC_F16) x_inplace = p_inplace = false;
  pl.ldxs = pl.ldps = pl.Fp;
  if (!x_inplace) pl.Xs = b.take<__nv_bfloat16>((size_t)N * pl.Fp);
  if (!p_inplace) pl.Ps = pm.take<__nv_bfloat16>((size_t)D_eff * pl.Fp);
}

// infer (nullable): the epilogue of the fused inference kernel (EPI_INFER: labels, class operand, scales); the
// contraction then signs, optionally packs (Hbits may be NULL) and classifies in one kernel.  Only the
// tensor-core path has it: the caller checks infer_fusable() first.
// Order in every branch: stage P (persistent; skipped when a prepared model is used), return if only
// preparing, stage X, contract.
int encode_rp_core(hdc_ctx* h, const void* X, int x_dtype, int64_t N, int F, int64_t ldx, const void* P,
                   int p_dtype, int64_t ldp, const hdc_knobs_t* k, int out_kinds, uint32_t* Hbits,
                   int64_t ldh, void* Hraw, int64_t ldraw, Bump& b, size_t ws_bytes, cudaStream_t st,
                   const Epilogue* infer = nullptr) {
  const int D_eff = k->D_eff;
  const int prec = k->precision;
  const bool want_raw = (out_kinds & HDC_OUT_RAW) != 0;
  Epilogue e{};
  if (infer) e = *infer;
  e.kind = infer ? EPI_INFER : EPI_SIGN;
  e.bits = Hbits;
  e.ldbits = ldh;
  e.raw = want_raw ? Hraw : nullptr;
  e.ldraw = ldraw;
  // a tensor-core launch that cannot take these operands: the CUDA-core kernel runs instead (counted, so that
  // a silent 3x slow-down is visible through hdc_stat); the fused inference epilogue has no such fallback
  auto tc_refused = [&](const char* what) -> int {
    if (infer) return fail(h, HDC_ERR_UNSUPPORTED, "infer_rp: operands not usable by the fused tensor-core kernel");
    ++h->stats[HDC_STAT_SIMT_FALLBACKS];
    h->err = std::string(what) + ": tensor-core kernel refused the operands, CUDA-core kernel used";
    return HDC_OK;
  };
  // runs the tensor-core contraction; HDC_OK, an error, or 1 = refused (fall through to the CUDA cores)
  auto contract_tc = [&](const TcOperands& o, const char* what) -> int {
    cudaError_t ce;
    {
      Timed tm(h, HDC_K_ENCODE_GEMM, st);
      ce = launch_gemm_tc(h->tc, o, N, D_eff, e, h->sm_count, tc_cta_group(k), st, &h->launches);
    }
    if (ce == cudaSuccess) {
      ++h->stats[HDC_STAT_TC_LAUNCHES];
      return HDC_OK;
    }
    if (ce != cudaErrorNotSupported) return cuda_fail(h, ce, what);
    if (int rc = tc_refused(what)) return rc;
    return 1;
  };
  const int xk = x_dtype == HDC_BF16 ? OPK_BF16 : OPK_F32;
  const int pk = p_dtype == HDC_BF16 ? OPK_BF16 : (p_dtype == HDC_I8 ? OPK_I8 : OPK_F32);
  const bool modelled = h->model != nullptr;   // P must then be staged into the model, never used in place
  cudaError_t ce;
  EncodePlan pl;
  Bump& pm = persistent(h, b);

  if (prec == HDC_F32) {
    plan_encode(h, N, F, D_eff, k, false, false, b, pm, pl);
    if (!persistent_fits(h, b, ws_bytes)) return fail(h, HDC_ERR_WORKSPACE, "encode_rp: workspace too small");
    if (pl.tc && (k->flags & HDC_FLAG_F32_FAST)) {
      if (do_prep(h)) {
        ce = launch_split2_f16(P, pk, D_eff, F, ldp, (__half*)pl.Ps, pl.Fp, pl.ep, st, &h->launches);
        if (ce != cudaSuccess) return cuda_fail(h, ce, "split P");
      }
      if (prep_only(h)) return HDC_OK;
      ce = launch_split2_f16(X, xk, N, F, ldx, (__half*)pl.Xs, pl.Fp, pl.ex, st, &h->launches);
      if (ce != cudaSuccess) return cuda_fail(h, ce, "split X");
      TcOperands o{pl.Xs, pl.Ps, OPK_F16, pl.ldxs, pl.ldps, pl.ldxs, pl.ldps, pl.Fp, 3,
                   SPLIT2_A_SEGS, SPLIT2_B_SEGS, pl.Fp, F};
      int rc = contract_tc(o, "encode_rp fp32 (2 x fp16) tcgen05");
      if (rc == HDC_OK && want_raw) {
        ce = launch_unscale_raw((float*)Hraw, N, D_eff, ldraw, pl.ex, pl.ep, st, &h->launches);
        if (ce != cudaSuccess) return cuda_fail(h, ce, "unscale raw");
      }
      if (rc <= 0) return rc;
      pl.tc = false;  // the workspace was planned for the 2-way split: go straight to the CUDA-core kernel
    }
    if (pl.tc) {
      if (do_prep(h)) {
        ce = launch_split3_bf16(P, pk, D_eff, F, ldp, (__nv_bfloat16*)pl.Ps, pl.Fp, st, &h->launches);
        if (ce != cudaSuccess) return cuda_fail(h, ce, "split P");
      }
      if (prep_only(h)) return HDC_OK;
      ce = launch_split3_bf16(X, xk, N, F, ldx, (__nv_bfloat16*)pl.Xs, pl.Fp, st, &h->launches);
      if (ce != cudaSuccess) return cuda_fail(h, ce, "split X");
      TcOperands o{pl.Xs, pl.Ps, OPK_BF16, pl.ldxs, pl.ldps, pl.ldxs, pl.ldps, pl.Fp, 6,
                   SPLIT_A_SEGS, SPLIT_B_SEGS, pl.Fp, F};
      int rc = contract_tc(o, "encode_rp fp32 tcgen05");
      if (rc <= 0) return rc;
    }
    if (prep_only(h)) return HDC_OK;  // the CUDA-core kernel reads P in place
    {
      Timed tm(h, HDC_K_ENCODE_GEMM, st);
      ce = launch_gemm_simt(Operand{X, ldx, xk}, Operand{P, ldp, pk}, N, D_eff, F, false, e, st, &h->launches);
    }
    return ce == cudaSuccess ? HDC_OK : cuda_fail(h, ce, "encode_rp fp32");
  }

  const bool tc_ok_x = x_dtype == HDC_BF16 && (ldx % 8) == 0 && aligned16(X);
  const bool tc_ok_p = !modelled && p_dtype == HDC_BF16 && (ldp % 8) == 0 && aligned16(P);
  if (prec == HDC_I8) {
    const bool p_in = !modelled && p_dtype == HDC_I8 && (ldp % 16) == 0 && aligned16(P);
    plan_encode(h, N, F, D_eff, k, false, p_in, b, pm, pl);
    if (!persistent_fits(h, b, ws_bytes)) return fail(h, HDC_ERR_WORKSPACE, "encode_rp: workspace too small");
    const void* Pq = P;
    int64_t ldpq = ldp;
    if (!p_in) {
      if (do_prep(h)) {
        ce = launch_quantize_rows_i8(P, pk, D_eff, F, ldp, (int8_t*)pl.Ps, pl.ldps, st, &h->launches);
        if (ce != cudaSuccess) return cuda_fail(h, ce, "quantize P");
      }
      Pq = pl.Ps;
      ldpq = pl.ldps;
    }
    if (prep_only(h)) return HDC_OK;
    ce = launch_quantize_rows_i8(X, xk, N, F, ldx, (int8_t*)pl.Xs, pl.ldxs, st, &h->launches);
    if (ce != cudaSuccess) return cuda_fail(h, ce, "quantize X");
    if (pl.tc) {
      TcOperands o{pl.Xs, Pq, OPK_I8, pl.ldxs, ldpq, F, F, F, 1, 0u, 0u, 0};
      int rc = contract_tc(o, "encode_rp int8 tcgen05");
      if (rc <= 0) return rc;
    }
    ce = launch_gemm_simt(Operand{pl.Xs, pl.ldxs, OPK_I8}, Operand{Pq, ldpq, OPK_I8}, N, D_eff, F, true, e,
                          st, &h->launches);
    return ce == cudaSuccess ? HDC_OK : cuda_fail(h, ce, "encode_rp int8");
  }

  if (prec == HDC_F16) {
    plan_encode(h, N, F, D_eff, k, false, false, b, pm, pl);
    if (!persistent_fits(h, b, ws_bytes)) return fail(h, HDC_ERR_WORKSPACE, "encode_rp: workspace too small");
    if (pl.tc) {
      if (do_prep(h)) {
        ce = launch_convert_f16(P, pk, D_eff, F, ldp, (__half*)pl.Ps, pl.ldps, st, &h->launches);
        if (ce != cudaSuccess) return cuda_fail(h, ce, "convert P");
      }
      if (prep_only(h)) return HDC_OK;
      ce = launch_convert_f16(X, xk, N, F, ldx, (__half*)pl.Xs, pl.ldxs, st, &h->launches);
      if (ce != cudaSuccess) return cuda_fail(h, ce, "convert X");
      TcOperands o{pl.Xs, pl.Ps, OPK_F16, pl.ldxs, pl.ldps, F, F, F, 1, 0u, 0u, 0};
      int rc = contract_tc(o, "encode_rp fp16 tcgen05");
      if (rc <= 0) return rc;
    }
    if (prep_only(h)) return HDC_OK;
    const int xr = x_dtype == HDC_BF16 ? OPK_BF16_RF16 : OPK_F32_RF16;
    const int pr = p_dtype == HDC_BF16 ? OPK_BF16_RF16 : OPK_F32_RF16;
    ce = launch_gemm_simt(Operand{X, ldx, xr}, Operand{P, ldp, pr}, N, D_eff, F, false, e, st, &h->launches);
    return ce == cudaSuccess ? HDC_OK : cuda_fail(h, ce, "encode_rp fp16");
  }

  // BF16 / B1
  plan_encode(h, N, F, D_eff, k, tc_ok_x, tc_ok_p, b, pm, pl);
  if (!persistent_fits(h, b, ws_bytes)) return fail(h, HDC_ERR_WORKSPACE, "encode_rp: workspace too small");
  if (pl.tc) {
    const void* Xb = X;
    const void* Pb = P;
    int64_t ldxb = ldx, ldpb = ldp;
    if (!tc_ok_p) {
      if (do_prep(h)) {
        ce = launch_convert_bf16(P, pk, D_eff, F, ldp, (__nv_bfloat16*)pl.Ps, pl.ldps, st, &h->launches);
        if (ce != cudaSuccess) return cuda_fail(h, ce, "convert P");
      }
      Pb = pl.Ps;
      ldpb = pl.ldps;
    }
    if (prep_only(h)) return HDC_OK;
    if (!tc_ok_x) {
      ce = launch_convert_bf16(X, xk, N, F, ldx, (__nv_bfloat16*)pl.Xs, pl.ldxs, st, &h->launches);
      if (ce != cudaSuccess) return cuda_fail(h, ce, "convert X");
      Xb = pl.Xs;
      ldxb = pl.ldxs;
    }
    TcOperands o{Xb, Pb, OPK_BF16, ldxb, ldpb, F, F, F, 1, 0u, 0u, 0};
    int rc = contract_tc(o, "encode_rp bf16 tcgen05");
    if (rc <= 0) return rc;
  }
  if (prep_only(h)) return HDC_OK;
  const int xr = x_dtype == HDC_BF16 ? OPK_BF16 : OPK_F32_RBF16;
  const int pr = p_dtype == HDC_BF16 ? OPK_BF16 : OPK_F32_RBF16;
  ce = launch_gemm_simt(Operand{X, ldx, xr}, Operand{P, ldp, pr}, N, D_eff, F, false, e, st, &h->launches);
  return ce == cudaSuccess ? HDC_OK : cuda_fail(h, ce, "encode_rp bf16");
}

// Workspace of hdc_encode_rp: the compacted operands of a perforated contraction (upper bound: 4-byte
// elements) followed by the staging buffers of the contraction itself.
void encode_ws(const hdc_ctx* h, int64_t N, int F, int D_eff, const hdc_knobs_t* k, Bump& b, Bump& pm) {
  const Perf ef = enc_perf_of(k);
  if (perf_on(ef)) {
    F = perf_count(ef, F);
    const int64_t ldg = round_up(F, 16);
    b.take<float>((size_t)N * ldg);
    pm.take<float>((size_t)D_eff * ldg);
  }
  EncodePlan pl;
  plan_encode(h, N, F, D_eff, k, false, false, b, pm, pl);
}
void encode_ws(const hdc_ctx* h, int64_t N, int F, int D_eff, const hdc_knobs_t* k, Bump& b) {
  encode_ws(h, N, F, D_eff, k, b, b);
}

// hdc_encode_rp after argument checks.  A perforated F reduction (knobs enc_perf_*; PAPER.md L155,
// reading A18) is the same contraction over compacted copies of the visited columns, with the raw
// accumulators multiplied by F / F_visited afterwards (the sign bits do not depend on that scale).
int do_encode_rp(hdc_ctx* h, const void* X, int x_dtype, int64_t N, int F, int64_t ldx, const void* P,
                 int p_dtype, int D, int64_t ldp, const hdc_knobs_t* k, int out_kinds, uint32_t* Hbits,
                 int64_t ldh, void* Hraw, int64_t ldraw, Bump& b, size_t ws_bytes, cudaStream_t st) {
  (void)D;
  const Perf ef = enc_perf_of(k);
  if (!perf_on(ef))
    return encode_rp_core(h, X, x_dtype, N, F, ldx, P, p_dtype, ldp, k, out_kinds, Hbits, ldh, Hraw, ldraw, b,
                          ws_bytes, st);
  const int D_eff = k->D_eff;
  const int Fv = perf_count(ef, F);
  const int64_t ldg = round_up(Fv, 16);
  const int xs = x_dtype == HDC_BF16 ? 2 : 4;
  const int ps = p_dtype == HDC_BF16 ? 2 : (p_dtype == HDC_I8 ? 1 : 4);
  Bump& pm = persistent(h, b);
  void* Xg = b.take<uint8_t>((size_t)N * ldg * xs);
  void* Pg = pm.take<uint8_t>((size_t)D_eff * ldg * (h->model ? 4 : ps));  // a model reserves the 4-byte bound (encode_ws)
  {  // the whole workspace is checked before the first launch
    Bump dry(nullptr), dry_pm(nullptr);
    dry.off = b.off;
    dry_pm.off = pm.off;
    EncodePlan pl;
    plan_encode(h, N, Fv, D_eff, k, false, false, dry, h->model ? dry_pm : dry, pl);
    if (dry.off > ws_bytes || (h->model && dry_pm.off > h->model_cap))
      return fail(h, HDC_ERR_WORKSPACE, "encode_rp: workspace too small");
  }
  cudaError_t ce = cudaSuccess;
  if (!prep_only(h)) ce = launch_gather_cols(X, xs, N, ldx, ef, Fv, Xg, ldg, st, &h->launches);
  if (ce != cudaSuccess) return cuda_fail(h, ce, "gather X");
  if (do_prep(h)) ce = launch_gather_cols(P, ps, D_eff, ldp, ef, Fv, Pg, ldg, st, &h->launches);
  if (ce != cudaSuccess) return cuda_fail(h, ce, "gather P");
  int rc = encode_rp_core(h, Xg, x_dtype, N, Fv, ldg, Pg, p_dtype, ldg, k, out_kinds, Hbits, ldh, Hraw, ldraw, b,
                          ws_bytes, st);
  if (rc != HDC_OK || !(out_kinds & HDC_OUT_RAW) || prep_only(h)) return rc;
  const float scale = (float)((double)F / (double)Fv);
  ce = launch_scale_raw(Hraw, N, D_eff, ldraw, scale, k->precision == HDC_I8, st, &h->launches);
  return ce == cudaSuccess ? HDC_OK : cuda_fail(h, ce, "scale raw");
}

// ------------------------------------------------------------------------------------- similarity
// Shared by hdc_similarity (S != null), hdc_classify (labels != null) and hdc_train_epoch.
int do_similarity(hdc_ctx* h, const uint32_t* Hbits, int64_t N, int64_t ldh, const float* C_acc, int K,
                  int64_t ldc, const hdc_knobs_t* k, void* S, int s_i32, int64_t lds, int32_t* labels,
                  float* best, float* second, Bump& b, size_t ws_bytes, cudaStream_t st) {
  const int D_eff = k->D_eff;
  const int W = words_of(D_eff);
  const Perf pf = perf_of(k);
  const int n_vis = perf_count(pf, D_eff);  // dimensions the reduction visits (= D_eff unless perforated)
  cudaError_t ce;
  Bump& pm = persistent(h, b);   // class operand, scales, masks: per-call-invariant (prepared-model modes)
  bool prep = do_prep(h);
  auto too_small = [&]() { return fail(h, HDC_ERR_WORKSPACE, "similarity: workspace too small"); };
  if (wide_int(k)) {
    // 32- / 64-bit integer class codes (A22), exact 64-bit sums.
    const int cos = k->sim == HDC_SIM_COS;
    const int width = k->hv_bits == HDC_HV_I32 ? 32 : 64;
    Epilogue e{};
    if (labels) {
      e.kind = EPI_ARGMAX;
      e.labels = labels;
      e.best = best;
      e.second = second;
    } else {
      e.kind = EPI_SCORE;
      e.S = S;
      e.lds = lds;
      e.s_i32 = s_i32;
    }
    double* colscale = pm.take<double>((size_t)K);
    // Tensor-core route: the codes as balanced base-65536 pieces, each staged like an int16 operand (three base-128
    // digits on tcgen05 kind::i8, exact int32 scores per piece: D_eff * 32768 < 2^31) and contracted by sim_tc_kernel
    // over row chunks; the pieces' scores are recombined in 64 bits by wide_combine_kernel.
    if (use_tc(h, k) && D_eff <= 65535) {
      const int pieces = width / 16;
      const size_t cop_bytes = sim_tc_operand_bytes(K, HDC_HV_I16, D_eff);
      void* cop[4];
      for (int j = 0; j < pieces; ++j) cop[j] = pm.take<uint8_t>(cop_bytes);
      // live[j] = piece j holds a nonzero code.  Accumulators as training leaves them are small integers whose upper
      // pieces are all zero: their contractions return at once and the combine kernel skips them
      int* live = pm.take<int>(4);
      const int64_t rows_max = wide_chunk_rows(N, K);
      int32_t* Sp = b.take<int32_t>((size_t)pieces * (size_t)rows_max * (size_t)K);
      if (!persistent_fits(h, b, ws_bytes)) return too_small();
      bool ok = true;
      if (prep) {
        ce = launch_wide_prepare(C_acc, K, ldc, D_eff, k->hv_bits, pf, cos, nullptr, colscale, st, &h->launches, live);
        if (ce != cudaSuccess) return cuda_fail(h, ce, "wide-integer cosine scales");
        Epilogue none{};
        none.kind = EPI_SCORE;
        for (int j = 0; j < pieces && ok; ++j) {
          ce = launch_sim_tc(h->tc, Hbits, 0, ldh, C_acc, K, ldc, D_eff, HDC_HV_I16, cop[j], nullptr, none, pf, nullptr,
                             false, true, h->sm_count, tc_cta_group(k), st, &h->launches, j + 1, width, live + j);
          if (ce == cudaErrorNotSupported) ok = false;
          else if (ce != cudaSuccess) return cuda_fail(h, ce, "wide-integer class pieces");
        }
      }
      if (ok && prep_only(h)) return HDC_OK;
      if (ok) {
        Timed tm(h, HDC_K_SIM, st);
        for (int64_t r0 = 0; r0 < N && ok; r0 += rows_max) {
          const int64_t rows = N - r0 < rows_max ? N - r0 : rows_max;
          for (int j = 0; j < pieces && ok; ++j) {
            Epilogue es{};
            es.kind = EPI_SCORE;
            es.S = Sp + (size_t)j * (size_t)rows * (size_t)K;
            es.lds = K;
            es.s_i32 = 1;
            ce = launch_sim_tc(h->tc, Hbits + r0 * ldh, rows, ldh, C_acc, K, ldc, D_eff, HDC_HV_I16, cop[j], nullptr, es,
                               pf, nullptr, true, false, h->sm_count, tc_cta_group(k), st, &h->launches, j + 1, width,
                               live + j);
            if (ce == cudaErrorNotSupported && r0 == 0 && j == 0) ok = false;
            else if (ce != cudaSuccess) return cuda_fail(h, ce, "wide-integer similarity (tcgen05)");
          }
          if (!ok) break;
          Epilogue er = e;
          if (er.labels) er.labels += r0;
          if (er.best) er.best += r0;
          if (er.second) er.second += r0;
          if (er.S) er.S = static_cast<char*>(er.S) + (size_t)r0 * (size_t)lds * (s_i32 == 2 ? 8 : 4);
          ce = launch_wide_combine(Sp, pieces, rows, K, cos, colscale, live, er, st, &h->launches);
          if (ce != cudaSuccess) return cuda_fail(h, ce, "wide-integer combine");
        }
        if (ok) return HDC_OK;
      }
      ++h->stats[HDC_STAT_SIMT_FALLBACKS];
      h->err = "wide-integer similarity: tensor-core kernel refused the operands, dp4a kernel used";
      prep = true;   // the dp4a kernel takes another operand form (byte planes): stage it here
    }
    // CUDA-core route: byte planes + dp4a contraction (widedot.cu)
    uint32_t* planes = pm.take<uint32_t>(wide_operand_bytes(K, k->hv_bits, D_eff) / sizeof(uint32_t));
    if (!persistent_fits(h, b, ws_bytes)) return too_small();
    if (prep) {
      ce = launch_wide_prepare(C_acc, K, ldc, D_eff, k->hv_bits, pf, cos, planes, colscale, st, &h->launches);
      if (ce != cudaSuccess) return cuda_fail(h, ce, "wide-integer class operand");
    }
    if (prep_only(h)) return HDC_OK;
    {
      Timed tm(h, HDC_K_SIM, st);
      ce = launch_wide_dot(Hbits, N, ldh, K, D_eff, k->hv_bits, cos, planes, colscale, e, st, &h->launches);
    }
    return ce == cudaSuccess ? HDC_OK : cuda_fail(h, ce, "wide-integer similarity");
  }
  // tensor-core path from packed queries: DOT / COS at any K; Hamming once K is large enough that
  // the popcount pipe would bound it (dist = (D_eff - dot)/2 is exact in int32)
  if (use_tc(h, k) && (k->sim != HDC_SIM_HAMMING || K >= 64)) {
    double* colscale = nullptr;
    float* colscale_f = nullptr;
    if (k->sim == HDC_SIM_COS) {
      colscale = pm.take<double>((size_t)K);
      colscale_f = pm.take<float>((size_t)K);
    }
    float* amax = pm.take<float>(1);
    void* cop = pm.take<uint8_t>(sim_tc_operand_bytes(K, k->hv_bits, D_eff));
    const size_t pbytes = sim_tc_partial_bytes(N, K, k->hv_bits, D_eff, h->sm_count);
    double* partial = pbytes ? b.take<double>(pbytes / sizeof(double)) : nullptr;
    if (!persistent_fits(h, b, ws_bytes)) return too_small();
    // (the cosine scales -- norms over the operand as the contraction sees it -- are written by the kernel that
    // stages the class operand, inside launch_sim_tc)
    Epilogue e{};
    e.colscale = colscale;
    e.colscale_f = colscale_f;
    e.ham_D = k->sim == HDC_SIM_HAMMING ? n_vis : 0;
    if (labels) {
      e.kind = EPI_ARGMAX;
      e.labels = labels;
      e.best = best;
      e.second = second;
    } else {
      e.kind = EPI_SCORE;
      e.S = S;
      e.lds = lds;
      e.s_i32 = s_i32;
    }
    {
      Timed tm(h, HDC_K_SIM, st);
      ce = launch_sim_tc(h->tc, Hbits, N, ldh, C_acc, K, ldc, D_eff, k->hv_bits, cop, amax, e, pf, partial,
                         !prep, prep_only(h), h->sm_count, tc_cta_group(k), st, &h->launches);
    }
    if (ce == cudaSuccess) return HDC_OK;
    if (ce != cudaErrorNotSupported) return cuda_fail(h, ce, "similarity tcgen05");
    prep = true;  // the CUDA-core kernels below take other operand forms: prepare them here
  }
  if (k->sim == HDC_SIM_HAMMING) {
    uint32_t* cbits = pm.take<uint32_t>((size_t)K * W);
    uint32_t* pmask = perf_on(pf) ? pm.take<uint32_t>((size_t)W) : nullptr;
    if (!persistent_fits(h, b, ws_bytes)) return too_small();
    if (prep) {
      ce = launch_sign_bits(C_acc, K, D_eff, ldc, cbits, W, st, &h->launches);
      if (ce != cudaSuccess) return cuda_fail(h, ce, "sign_bits");
      if (pmask) {
        ce = launch_perf_mask(pmask, W, D_eff, pf, st, &h->launches);
        if (ce != cudaSuccess) return cuda_fail(h, ce, "perforation mask");
      }
    }
    if (prep_only(h)) return HDC_OK;
    {
      Timed tm(h, HDC_K_SIM, st);
      ce = launch_hamming(Hbits, N, ldh, cbits, K, W, D_eff, pmask, (int32_t*)S, lds, labels, best, second,
                          h->sm_count, h->smem_optin, st, &h->launches);
    }
    return ce == cudaSuccess ? HDC_OK : cuda_fail(h, ce, "hamming");
  }
  // DOT / COS: contraction of +-1 queries with the class operand at hv_bits (CUDA-core kernels)
  if (perf_on(pf)) return fail(h, HDC_ERR_UNSUPPORTED, "perforated DOT / COS needs the tensor-core path");
  Operand B{};
  bool int_acc = false;
  double* colscale = nullptr;
  if (k->sim == HDC_SIM_COS) colscale = pm.take<double>((size_t)K);
  if (k->hv_bits == 32) {
    B = Operand{C_acc, ldc, OPK_F32};
  } else if (k->hv_bits == 16) {
    B = Operand{C_acc, ldc, OPK_F32_RBF16};
  } else if (k->hv_bits == HDC_HV_F16) {
    B = Operand{C_acc, ldc, OPK_F32_RF16};
  } else if (k->hv_bits == 8) {
    const int64_t ldq = round_up(D_eff, 16);
    int8_t* Cq = pm.take<int8_t>((size_t)K * ldq);
    float* amax = pm.take<float>(1);
    if (!persistent_fits(h, b, ws_bytes)) return too_small();
    if (prep) {
      ce = launch_quantize_tensor_i8(C_acc, K, D_eff, ldc, pf, Cq, ldq, amax, st, &h->launches);
      if (ce != cudaSuccess) return cuda_fail(h, ce, "quantize C");
    }
    B = Operand{Cq, ldq, OPK_I8};
    int_acc = true;
  } else if (k->hv_bits == HDC_HV_I16) {
    const int64_t ldq = round_up(D_eff, 16);
    int16_t* Cq = reinterpret_cast<int16_t*>(pm.take<int8_t>((size_t)K * ldq * 2));
    float* amax = pm.take<float>(1);
    if (!persistent_fits(h, b, ws_bytes)) return too_small();
    if (prep) {
      ce = launch_quantize_tensor_i16(C_acc, K, D_eff, ldc, pf, Cq, ldq, amax, st, &h->launches);
      if (ce != cudaSuccess) return cuda_fail(h, ce, "quantize C");
    }
    B = Operand{Cq, ldq, OPK_I16};
    int_acc = true;
  } else {
    uint32_t* cbits = pm.take<uint32_t>((size_t)K * W);
    if (!persistent_fits(h, b, ws_bytes)) return too_small();
    if (prep) {
      ce = launch_sign_bits(C_acc, K, D_eff, ldc, cbits, W, st, &h->launches);
      if (ce != cudaSuccess) return cuda_fail(h, ce, "sign_bits");
    }
    B = Operand{cbits, W, OPK_BITS};
    int_acc = true;
  }
  if (!persistent_fits(h, b, ws_bytes)) return too_small();
  if (colscale && prep) {
    ce = launch_col_scale(B, K, D_eff, 1, pf, colscale, st, &h->launches);
    if (ce != cudaSuccess) return cuda_fail(h, ce, "col_scale");
  }
  if (prep_only(h)) return HDC_OK;
  Epilogue e{};
  e.colscale = colscale;
  if (labels) {
    e.kind = EPI_ARGMAX;
    e.labels = labels;
    e.best = best;
    e.second = second;
  } else {
    e.kind = EPI_SCORE;
    e.S = S;
    e.lds = lds;
    e.s_i32 = s_i32;
  }
  ce = launch_gemm_simt(Operand{Hbits, ldh, OPK_BITS}, B, N, K, D_eff, int_acc, e, st, &h->launches);
  return ce == cudaSuccess ? HDC_OK : cuda_fail(h, ce, "similarity contraction");
}

// persistent operands of do_similarity (upper bound over its paths)
void similarity_model_ws(int K, const hdc_knobs_t* k, Bump& pm) {
  const int W = words_of(k->D_eff);
  pm.take<double>((size_t)K);
  pm.take<float>((size_t)K);
  pm.take<float>(1);
  pm.take<int8_t>((size_t)K * round_up(k->D_eff, 16) * 2);   // int8 or int16 codes
  pm.take<uint32_t>((size_t)K * W);
  pm.take<uint32_t>((size_t)W);  // perforation mask
  pm.take<uint8_t>(wide_operand_bytes(K, k->hv_bits, k->D_eff));  // byte planes of 32- / 64-bit integer codes
  wide_tc_ws(0, K, k, &pm, nullptr);                              // ... and their 16-bit pieces (tensor-core route)
  pm.take<uint8_t>(sim_tc_operand_bytes(K, k->hv_bits == 32 || k->hv_bits == 16 || k->hv_bits == HDC_HV_F16 ||
                                               k->hv_bits == HDC_HV_I16 || k->hv_bits == 8 ? k->hv_bits : 1,
                                        k->D_eff));
}

size_t similarity_ws(int64_t N, int K, const hdc_knobs_t* k) {
  Bump b(nullptr);
  {  // split-D partial sums (simtc.cu): at most 8 splits and 64 MB, for any sub-batch of up to N queries
    size_t pb = (size_t)8 * (size_t)(N > 0 ? N : 1) * (size_t)K * sizeof(double);
    if (pb > ((size_t)64 << 20)) pb = (size_t)64 << 20;
    b.take<double>(pb / sizeof(double));
  }
  const int W = words_of(k->D_eff);
  b.take<double>((size_t)K);
  b.take<float>((size_t)K);
  b.take<int8_t>((size_t)K * round_up(k->D_eff, 16) * 2);   // int8 or int16 codes
  b.take<float>(1);
  b.take<uint32_t>((size_t)K * W);
  b.take<uint32_t>((size_t)W);  // perforation mask
  b.take<uint32_t>((size_t)((k->D_eff + 127) / 128) * 4 * K);  // [chunk][class] sign bits of hdc_similarity_adc
  b.take<uint8_t>(wide_operand_bytes(K, k->hv_bits, k->D_eff));  // byte planes of 32- / 64-bit integer codes
  wide_tc_ws(N, K, k, &b, &b);                                   // their 16-bit pieces and per-pass piece scores
  b.take<uint8_t>(sim_tc_operand_bytes(K, k->hv_bits == 32 || k->hv_bits == 16 || k->hv_bits == HDC_HV_F16 ||
                                               k->hv_bits == HDC_HV_I16 || k->hv_bits == 8 ? k->hv_bits : 1,
                                       k->D_eff));
  return b.off + 1024;
}

// rows per steady-state chunk of hdc_infer_rp_host: 74 CTA pairs x 256 rows (whole waves of the pair kernel)
constexpr int64_t HOST_CHUNK = 18944;
constexpr int64_t HOST_RAMP_START = 2048;

// ------------------------------------------------------------------------------------- fused inference
// hdc_infer_rp = hdc_encode_rp followed by hdc_classify, kernel for kernel.  Opt-in (HDC_FLAG_FUSED_INFER):
// encode + similarity + arg-max in ONE contraction kernel (gemm_tc.cu, EPI_INFER) when the class model is
// small enough to search on the CUDA cores beside the tensor-core tiles: K <= 32, the tensor path is on,
// CTA pairs are allowed, and there are enough row blocks to occupy the pairs (each pair owns 256 rows and
// walks all of D).  Measured slower than the two kernels (shared-memory bandwidth): off by default.
constexpr int INFER_MAX_K = 32;
constexpr int64_t INFER_MIN_N = 12288;  // 48 row blocks of 256: below it the two-kernel path spreads m x n tiles better

bool infer_fused_knobs(const hdc_ctx* h, const hdc_knobs_t* k, int K) {   // the part that does not depend on N
  // (int16 class codes: sums beyond 2^24, which the fp32 search of the fused epilogue does not hold exactly)
  return (k->flags & HDC_FLAG_FUSED_INFER) && k->hv_bits != HDC_HV_I16 && !wide_int(k) && use_tc(h, k) && !(k->flags & HDC_FLAG_TC_1CTA) && h->sm_count >= 2 &&
         K <= INFER_MAX_K && k->D_eff <= (1 << 17);
}
int infer_kc(int K) { return K <= 8 ? 8 : (K <= 16 ? 16 : 32); }

// workspace of the fused path after the encode staging: class operand, scales, amax
void infer_ws(int K, int D_eff, Bump& b) {
  b.take<float>((size_t)infer_kc(K) * (size_t)round_up(D_eff, 256));
  b.take<double>((size_t)K);
  b.take<float>(1);
}

// Shared by hdc_infer_rp and hdc_infer_rp_host (per chunk).  Hbits may be NULL on the fused path; the
// two-kernel path then keeps the hypervectors in the workspace.
int do_infer_rp(hdc_ctx* h, const void* X, int x_dtype, int64_t N, int F, int64_t ldx, const void* P, int p_dtype,
                int D, int64_t ldp, const float* C_acc, int K, int64_t ldc, const hdc_knobs_t* k, int32_t* labels,
                float* best, float* second, uint32_t* Hbits, int64_t ldh, Bump& b, size_t ws_bytes,
                cudaStream_t st) {
  const int D_eff = k->D_eff;
  const int W = words_of(D_eff);
  // Whether the fused kernel is an option for these knobs does not depend on N; whether THIS pass takes it does.
  // The persistent operands are therefore always carved -- and, when preparing, prepared -- in one fixed order:
  // [fused class operand, scales] [staged P] [class operand of the classify kernel], so that passes of any size
  // (the chunks of hdc_infer_rp_host, a prepared model) find what they need.
  const bool fused_ops = infer_fused_knobs(h, k, K) && !perf_on(enc_perf_of(k));
  const bool fused = fused_ops && N >= INFER_MIN_N;
  Epilogue e{};
  if (fused_ops) {
    const int KC = infer_kc(K);
    const int64_t ldcls = round_up(D_eff, 256);
    const Perf pf = perf_of(k);
    Bump& pm = persistent(h, b);
    float* cls = pm.take<float>((size_t)KC * (size_t)ldcls);
    double* colscale = pm.take<double>((size_t)K);
    float* amax = pm.take<float>(1);
    if (!persistent_fits(h, b, ws_bytes)) return fail(h, HDC_ERR_WORKSPACE, "infer_rp: workspace too small");
    cudaError_t ce = cudaSuccess;
    if (do_prep(h)) {
      if (k->hv_bits == 8) ce = launch_tensor_amax(C_acc, K, D_eff, ldc, pf, amax, st, &h->launches);
      if (ce == cudaSuccess)
        ce = launch_class_operand_f32(C_acc, K, D_eff, ldc, k->hv_bits, pf, amax, cls, KC, ldcls, st, &h->launches);
      if (ce == cudaSuccess && k->sim == HDC_SIM_COS)   // norms over the operand as the epilogue contracts it
        ce = launch_col_scale(Operand{cls, ldcls, OPK_F32}, K, D_eff, 1, pf, colscale, st, &h->launches);
      if (ce != cudaSuccess) return cuda_fail(h, ce, "infer_rp: class operand");
    }
    e.labels = labels;
    e.best = best;
    e.second = second;
    e.colscale = k->sim == HDC_SIM_COS ? colscale : nullptr;
    e.ham_D = k->sim == HDC_SIM_HAMMING ? perf_count(pf, D_eff) : 0;
    e.cls = cls;
    e.ldcls = ldcls;
    e.K = K;
  }
  if (fused) {
    int rc = encode_rp_core(h, X, x_dtype, N, F, ldx, P, p_dtype, ldp, k, HDC_OUT_BITS, Hbits, ldh, nullptr, 0, b,
                            ws_bytes, st, &e);
    if (rc == HDC_OK && do_prep(h)) {  // a later, smaller pass takes the classify kernel: prepare its operand too
      const int mode = h->prep_mode;
      h->prep_mode = PREP_ONLY;
      rc = do_similarity(h, nullptr, 1, W, C_acc, K, ldc, k, nullptr, 0, 0, nullptr, nullptr, nullptr, b, ws_bytes, st);
      h->prep_mode = mode;
    }
    if (rc == HDC_OK && !prep_only(h)) ++h->stats[HDC_STAT_INFER_FUSED];
    return rc;
  }
  uint32_t* Hd = Hbits;
  int64_t ldhd = ldh;
  if (!Hd && !prep_only(h)) {
    // rows of W words rounded up to 4: 16-byte aligned rows let the encode epilogue write 16-byte stores and the
    // small-tile similarity kernel fetch the words by TMA (as Handle.alloc_hbits does for caller-owned hypervectors)
    ldhd = round_up(W, 4);
    Hd = b.take<uint32_t>((size_t)N * (size_t)ldhd);
    if (b.off > ws_bytes) return fail(h, HDC_ERR_WORKSPACE, "infer_rp: workspace too small");
  }
  int rc = do_encode_rp(h, X, x_dtype, N, F, ldx, P, p_dtype, D, ldp, k, HDC_OUT_BITS, Hd, ldhd, nullptr, 0, b,
                        ws_bytes, st);
  if (rc == HDC_OK)
    rc = do_similarity(h, Hd, N, ldhd, C_acc, K, ldc, k, nullptr, 0, 0, labels, best, second, b, ws_bytes, st);
  if (rc == HDC_OK && !prep_only(h)) ++h->stats[HDC_STAT_INFER_UNFUSED];
  return rc;
}

// bytes of the persistent operands of encode (P staging) + similarity (class operand, scales, masks) + the
// fused inference epilogue (fp32 class operand) for these sizes and knobs: the prepared-model blob
size_t model_ws_bytes(const hdc_ctx* h, int F, int K, const hdc_knobs_t* k) {
  Bump scratch(nullptr), pm(nullptr);
  encode_ws(h, 0, F, k->D_eff, k, scratch, pm);
  similarity_model_ws(K, k, pm);
  infer_ws(K, k->D_eff, pm);
  return pm.off + 1024;
}

// Runs `fn` with the persistent operands directed at [blob, blob + cap) in the given mode.
template <typename Fn>
int with_model(hdc_ctx* h, void* blob, size_t cap, int mode, Fn fn) {
  Bump pm(blob);
  h->model = &pm;
  h->model_cap = cap;
  h->prep_mode = mode;
  const int rc = fn();
  h->model = nullptr;
  h->model_cap = 0;
  h->prep_mode = PREP_AND_RUN;
  return rc;
}

// upper bound of what do_infer_rp takes from the workspace for up to N rows
size_t infer_ws_bytes(const hdc_ctx* h, int64_t N, int F, int K, const hdc_knobs_t* k) {
  Bump b(nullptr);
  infer_ws(K, k->D_eff, b);
  b.take<uint32_t>((size_t)N * (size_t)round_up(words_of(k->D_eff), 4));
  encode_ws(h, N, F, k->D_eff, k, b);
  return b.off + 1024 + similarity_ws(N, K, k);
}

}  // namespace
}  // namespace hdc

using namespace hdc;

// =================================================================================== handle
extern "C" int32_t hdc_version(void) { return 105; }  // 1.5: + HDC_HV_I32 / HDC_HV_I64, HDC_I64 scores

extern "C" int32_t hdc_create(hdc_handle_t* out, int32_t device) {
  if (!out) return HDC_ERR_INVALID_ARG;
  *out = nullptr;
  int count = 0;
  if (cudaGetDeviceCount(&count) != cudaSuccess || device < 0 || device >= count) {
    (void)cudaGetLastError();
    return HDC_ERR_CUDA;
  }
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return HDC_ERR_CUDA;
  if (prop.major != 10 || prop.minor != 0) return HDC_ERR_ARCH;  // the library holds sm_100a code only (no forward compatibility)
  if (cudaSetDevice(device) != cudaSuccess) return HDC_ERR_CUDA;
  hdc_ctx* h = new hdc_ctx();
  h->device = device;
  h->sm_count = prop.multiProcessorCount;
  h->smem_optin = (int)prop.sharedMemPerBlockOptin;
  h->tc = tc_context_create();
  if (cudaStreamCreateWithFlags(&h->copy_stream, cudaStreamNonBlocking) != cudaSuccess) {
    delete h;
    return HDC_ERR_CUDA;
  }
  for (int i = 0; i < 2; ++i) {
    cudaEventCreateWithFlags(&h->ev_copied[i], cudaEventDisableTiming);
    cudaEventCreateWithFlags(&h->ev_done[i], cudaEventDisableTiming);
  }
  cudaEventCreateWithFlags(&h->ev_entry, cudaEventDisableTiming);
  *out = h;
  return HDC_OK;
}

extern "C" int32_t hdc_destroy(hdc_handle_t h) {
  if (!h) return HDC_ERR_INVALID_ARG;
  DeviceGuard device_guard(h->device);
  for (int i = 0; i < 2; ++i) {
    if (h->ev_copied[i]) cudaEventDestroy(h->ev_copied[i]);
    if (h->ev_done[i]) cudaEventDestroy(h->ev_done[i]);
  }
  if (h->ev_entry) cudaEventDestroy(h->ev_entry);
  if (h->copy_stream) cudaStreamDestroy(h->copy_stream);
  for (auto& v : h->tev)
    for (auto& pr : v) {
      cudaEventDestroy(pr.first);
      cudaEventDestroy(pr.second);
    }
  tc_context_destroy(h->tc);
  delete h;
  return HDC_OK;
}

extern "C" const char* hdc_last_error(hdc_handle_t h) { return h ? h->err.c_str() : "null handle"; }

extern "C" int64_t hdc_launch_count(hdc_handle_t h) { return h ? h->launches : -1; }

extern "C" int64_t hdc_stat(hdc_handle_t h, int32_t stat_id) {
  if (!h || stat_id < 0 || stat_id >= HDC_STAT_COUNT) return -1;
  return h->stats[stat_id];
}

extern "C" int32_t hdc_kernel_timing(hdc_handle_t h, int32_t enable) {
  if (!h) return HDC_ERR_INVALID_ARG;
  DeviceGuard device_guard(h->device);
  h->timing = enable != 0;
  for (auto& u : h->tused) u = 0;
  return HDC_OK;
}

extern "C" int32_t hdc_kernel_time(hdc_handle_t h, int32_t kernel_id, float* ms_total, int64_t* launches) {
  if (!h || kernel_id < 0 || kernel_id >= HDC_K_COUNT || !ms_total || !launches)
    return h ? fail(h, HDC_ERR_INVALID_ARG, "kernel_time: bad argument") : HDC_ERR_INVALID_ARG;
  float total = 0.0f;
  for (size_t i = 0; i < h->tused[kernel_id]; ++i) {
    auto& pr = h->tev[kernel_id][i];
    cudaError_t ce = cudaEventSynchronize(pr.second);
    float ms = 0.0f;
    if (ce == cudaSuccess) ce = cudaEventElapsedTime(&ms, pr.first, pr.second);
    if (ce != cudaSuccess) return cuda_fail(h, ce, "kernel_time");
    total += ms;
  }
  *ms_total = total;
  *launches = (int64_t)h->tused[kernel_id];
  h->tused[kernel_id] = 0;
  return HDC_OK;
}

// =================================================================================== workspace
extern "C" size_t hdc_workspace_bytes(hdc_handle_t h, int32_t op, int64_t N, int32_t F_or_Q, int32_t D,
                                      int32_t K, const hdc_knobs_t* knobs) {
  if (!h || !knobs || N < 0) return 0;
  hdc_knobs_t k = *knobs;
  if (k.D_eff < 1 || k.D_eff > D) k.D_eff = D;
  if (K < 1) K = 1;  // sizes only: a bad K is reported by the call itself
  if (k.D_eff < 1) return 0;
  Bump b(nullptr);
  switch (op) {
    case HDC_OP_ENCODE_RP: {
      encode_ws(h, N, F_or_Q, k.D_eff, &k, b);
      return b.off + 256;
    }
    case HDC_OP_ENCODE_LEVELID:
      return 0;
    case HDC_OP_SIMILARITY:
    case HDC_OP_CLASSIFY:
      return similarity_ws(N, K, &k);
    case HDC_OP_TRAIN_EPOCH: {
      b.take<int32_t>((size_t)K * words_of(k.D_eff) * 32);  // Delta
      b.take<int32_t>((size_t)N);                           // predictions of one mini-batch
      b.take<int32_t>((size_t)K);                           // members per cluster (HDC_TRAIN_KMEANS)
      return b.off + 256 + similarity_ws(N, K, &k);
    }
    case HDC_OP_INFER_RP:
      return infer_ws_bytes(h, N, F_or_Q, K, &k) + 256;
    case HDC_OP_INFER_RP_HOST: {
      const int64_t chunk = N < HOST_CHUNK ? N : HOST_CHUNK;
      b.take<float>((size_t)chunk * F_or_Q);  // two staging buffers for X (fp32 upper bound)
      b.take<float>((size_t)chunk * F_or_Q);
      b.take<int32_t>((size_t)N);
      b.take<uint8_t>(model_ws_bytes(h, F_or_Q, K, &k));
      return b.off + 512 + infer_ws_bytes(h, chunk, F_or_Q, K, &k);
    }
    default:
      return 0;
  }
}

// =================================================================================== (1a)
static int check_encode_rp_args(hdc_ctx* h, const void* X, int x_dtype, int64_t N, int F, int64_t ldx,
                                const void* P, int p_dtype, int D, int64_t ldp, const hdc_knobs_t* k) {
  if ((!X && N > 0) || !P) return fail(h, HDC_ERR_INVALID_ARG, "encode_rp: NULL operand");
  if (N < 0 || F < 1 || D < 1 || ldx < F || ldp < F) return fail(h, HDC_ERR_INVALID_ARG, "encode_rp: bad sizes");
  if (x_dtype != HDC_F32 && x_dtype != HDC_BF16) return fail(h, HDC_ERR_INVALID_ARG, "encode_rp: x_dtype");
  if (p_dtype != HDC_F32 && p_dtype != HDC_BF16 && p_dtype != HDC_I8)
    return fail(h, HDC_ERR_INVALID_ARG, "encode_rp: p_dtype");
  int rc = check_knobs(h, k, D);
  if (rc) return rc;
  if (k->precision != HDC_F32 && k->precision != HDC_BF16 && k->precision != HDC_I8 && k->precision != HDC_B1 &&
      k->precision != HDC_F16)
    return fail(h, HDC_ERR_INVALID_ARG, "encode_rp: precision");
  if (p_dtype == HDC_I8 && k->precision != HDC_I8)
    return fail(h, HDC_ERR_INVALID_ARG, "encode_rp: int8 P needs precision HDC_I8");
  if (k->enc_perf_stride < 0 || k->enc_perf_begin < 0 || k->enc_perf_begin >= F)
    return fail(h, HDC_ERR_INVALID_ARG, "encode_rp: need enc_perf_stride >= 0 and 0 <= enc_perf_begin < F");
  const size_t xa = x_dtype == HDC_BF16 ? 2 : 4, pa = p_dtype == HDC_BF16 ? 2 : (p_dtype == HDC_I8 ? 1 : 4);
  if ((reinterpret_cast<uintptr_t>(X) % xa) || (reinterpret_cast<uintptr_t>(P) % pa))
    return fail(h, HDC_ERR_ALIGNMENT, "encode_rp: operand not element aligned");
  return HDC_OK;
}

extern "C" int32_t hdc_encode_rp(hdc_handle_t h, const void* X, int32_t x_dtype, int64_t N, int32_t F,
                                 int64_t ldx, const void* P, int32_t p_dtype, int32_t D, int64_t ldp,
                                 const hdc_knobs_t* knobs, int32_t out_kinds, uint32_t* Hbits,
                                 int64_t ldh_words, void* Hraw, int64_t ldraw, void* ws, size_t ws_bytes,
                                 void* stream) {
  if (!h) return HDC_ERR_INVALID_ARG;
  DeviceGuard device_guard(h->device);
  int rc = check_encode_rp_args(h, X, x_dtype, N, F, ldx, P, p_dtype, D, ldp, knobs);
  if (rc) return rc;
  if (!(out_kinds & HDC_OUT_BITS) || (!Hbits && N > 0))
    return fail(h, HDC_ERR_INVALID_ARG, "encode_rp: Hbits required");
  if (ldh_words < words_of(knobs->D_eff)) return fail(h, HDC_ERR_INVALID_ARG, "encode_rp: ldh_words < W");
  if ((out_kinds & HDC_OUT_RAW) && ((!Hraw && N > 0) || ldraw < knobs->D_eff))
    return fail(h, HDC_ERR_INVALID_ARG, "encode_rp: Hraw / ldraw");
  if (reinterpret_cast<uintptr_t>(Hbits) & 3) return fail(h, HDC_ERR_ALIGNMENT, "encode_rp: Hbits alignment");
  if (N == 0) return HDC_OK;
  Bump b(ws);
  if (!ws) ws_bytes = 0;
  return do_encode_rp(h, X, x_dtype, N, F, ldx, P, p_dtype, D, ldp, knobs, out_kinds, Hbits, ldh_words, Hraw,
                      ldraw, b, ws_bytes, (cudaStream_t)stream);
}

// =================================================================================== (1b)
static int32_t encode_levelid_impl(hdc_handle_t h, const void* levels, int lvl16, int64_t N, int32_t F, int64_t ldl,
                                   const uint32_t* IDbits, int64_t ldid_words, const uint32_t* LVbits, int32_t Q,
                                   int64_t ldlv_words, int32_t D, const hdc_knobs_t* knobs, uint32_t* Hbits,
                                   int64_t ldh_words, void* stream) {
  if (!h) return HDC_ERR_INVALID_ARG;
  DeviceGuard device_guard(h->device);
  if (((!levels || !Hbits) && N > 0) || !IDbits || !LVbits)
    return fail(h, HDC_ERR_INVALID_ARG, "encode_levelid: NULL pointer");
  if (N < 0 || F < 1 || F > 65535 || Q < 1 || Q > (lvl16 ? 65535 : 256) || D < 1 || ldl < F)
    return fail(h, HDC_ERR_INVALID_ARG, "encode_levelid: bad sizes");
  int rc = check_knobs(h, knobs, D);
  if (rc) return rc;
  const int W = words_of(knobs->D_eff);
  if (ldid_words < W || ldlv_words < W || ldh_words < W)
    return fail(h, HDC_ERR_INVALID_ARG, "encode_levelid: leading dimension < W");
  if ((reinterpret_cast<uintptr_t>(IDbits) | reinterpret_cast<uintptr_t>(LVbits) |
       reinterpret_cast<uintptr_t>(Hbits)) & 3)
    return fail(h, HDC_ERR_ALIGNMENT, "encode_levelid: bit matrices must be 4-byte aligned");
  if (lvl16 && (reinterpret_cast<uintptr_t>(levels) & 1))
    return fail(h, HDC_ERR_ALIGNMENT, "encode_levelid_u16: levels must be 2-byte aligned");
  if (N == 0) return HDC_OK;
  cudaError_t ce;
  {
    Timed tm(h, HDC_K_LEVELID, (cudaStream_t)stream);
    ce = launch_levelid(levels, lvl16, N, F, ldl, IDbits, ldid_words, LVbits, Q, ldlv_words, knobs->D_eff, Hbits,
                        ldh_words, h->sm_count, h->smem_optin, (cudaStream_t)stream, &h->launches);
  }
  if (ce == cudaErrorNotSupported)
    return fail(h, HDC_ERR_UNSUPPORTED, "encode_levelid: F too large (a batch of level rows must fit in shared memory: "
                                        "about 7000 features with 8-bit, 3500 with 16-bit level indices)");
  return ce == cudaSuccess ? HDC_OK : cuda_fail(h, ce, "encode_levelid");
}

extern "C" int32_t hdc_encode_levelid(hdc_handle_t h, const uint8_t* levels, int64_t N, int32_t F,
                                      int64_t ldl, const uint32_t* IDbits, int64_t ldid_words,
                                      const uint32_t* LVbits, int32_t Q, int64_t ldlv_words, int32_t D,
                                      const hdc_knobs_t* knobs, uint32_t* Hbits, int64_t ldh_words, void* ws,
                                      size_t ws_bytes, void* stream) {
  (void)ws;
  (void)ws_bytes;
  return encode_levelid_impl(h, levels, 0, N, F, ldl, IDbits, ldid_words, LVbits, Q, ldlv_words, D, knobs, Hbits,
                             ldh_words, stream);
}

extern "C" int32_t hdc_encode_levelid_u16(hdc_handle_t h, const uint16_t* levels, int64_t N, int32_t F,
                                          int64_t ldl, const uint32_t* IDbits, int64_t ldid_words,
                                          const uint32_t* LVbits, int32_t Q, int64_t ldlv_words, int32_t D,
                                          const hdc_knobs_t* knobs, uint32_t* Hbits, int64_t ldh_words, void* ws,
                                          size_t ws_bytes, void* stream) {
  (void)ws;
  (void)ws_bytes;
  return encode_levelid_impl(h, levels, 1, N, F, ldl, IDbits, ldid_words, LVbits, Q, ldlv_words, D, knobs, Hbits,
                             ldh_words, stream);
}

// =================================================================================== (2), (2+3a)
static int check_sim_args(hdc_ctx* h, const uint32_t* Hbits, int64_t N, int64_t ldh, const float* C_acc,
                          int K, int64_t ldc, int D, const hdc_knobs_t* k) {
  if ((!Hbits && N > 0) || !C_acc) return fail(h, HDC_ERR_INVALID_ARG, "similarity: NULL operand");
  if (N < 0 || K < 1 || K > 65535 || D < 1 || ldc < D) return fail(h, HDC_ERR_INVALID_ARG, "similarity: bad sizes");
  int rc = check_knobs(h, k, D);
  if (rc) return rc;
  rc = check_sim_knobs(h, k);
  if (rc) return rc;
  if (ldh < words_of(k->D_eff)) return fail(h, HDC_ERR_INVALID_ARG, "similarity: ldh_words < W");
  if ((reinterpret_cast<uintptr_t>(Hbits) | reinterpret_cast<uintptr_t>(C_acc)) & 3)
    return fail(h, HDC_ERR_ALIGNMENT, "similarity: operands must be 4-byte aligned");
  return HDC_OK;
}

extern "C" int32_t hdc_similarity(hdc_handle_t h, const uint32_t* Hbits, int64_t N, int64_t ldh_words,
                                  const float* C_acc, int32_t K, int64_t ldc, int32_t D,
                                  const hdc_knobs_t* knobs, void* S, int32_t s_dtype, int64_t lds, void* ws,
                                  size_t ws_bytes, void* stream) {
  if (!h) return HDC_ERR_INVALID_ARG;
  DeviceGuard device_guard(h->device);
  int rc = check_sim_args(h, Hbits, N, ldh_words, C_acc, K, ldc, D, knobs);
  if (rc) return rc;
  if ((!S && N > 0) || lds < K) return fail(h, HDC_ERR_INVALID_ARG, "similarity: S / lds");
  if (knobs->sim == HDC_SIM_HAMMING && s_dtype != HDC_I32)
    return fail(h, HDC_ERR_INVALID_ARG, "similarity: HAMMING writes int32");
  if (knobs->sim == HDC_SIM_COS && s_dtype != HDC_F32) return fail(h, HDC_ERR_INVALID_ARG, "similarity: COS writes fp32");
  if (wide_int(knobs)) {
    if (s_dtype != HDC_F32 && !(s_dtype == HDC_I64 && knobs->sim == HDC_SIM_DOT))
      return fail(h, HDC_ERR_INVALID_ARG, "similarity: 32- / 64-bit integer classes write fp32, or int64 for DOT");
    if (s_dtype == HDC_I64 && (reinterpret_cast<uintptr_t>(S) & 7))
      return fail(h, HDC_ERR_ALIGNMENT, "similarity: int64 scores must be 8-byte aligned");
  } else if (knobs->sim == HDC_SIM_DOT) {
    if (s_dtype != HDC_F32 && s_dtype != HDC_I32) return fail(h, HDC_ERR_INVALID_ARG, "similarity: s_dtype");
    if (s_dtype == HDC_I32 && knobs->hv_bits != 8 && knobs->hv_bits != 1 && knobs->hv_bits != HDC_HV_I16)
      return fail(h, HDC_ERR_INVALID_ARG, "similarity: int32 DOT needs hv_bits 8, HDC_HV_I16 or 1");
  }
  if (N == 0) return HDC_OK;
  Bump b(ws);
  if (!ws) ws_bytes = 0;
  return do_similarity(h, Hbits, N, ldh_words, C_acc, K, ldc, knobs, S, s_dtype == HDC_I32 ? 1 : (s_dtype == HDC_I64 ? 2 : 0), lds, nullptr,
                       nullptr, nullptr, b, ws_bytes, (cudaStream_t)stream);
}

extern "C" int32_t hdc_similarity_adc(hdc_handle_t h, const uint32_t* Hbits, int64_t N, int64_t ldh_words,
                                      const float* C_acc, int32_t K, int64_t ldc, int32_t D,
                                      const hdc_knobs_t* knobs, const hdc_adc_t* adc, int32_t* S, int64_t lds,
                                      int32_t* labels, void* ws, size_t ws_bytes, void* stream) {
  if (!h) return HDC_ERR_INVALID_ARG;
  DeviceGuard device_guard(h->device);
  if ((!Hbits && N > 0) || !C_acc || !adc) return fail(h, HDC_ERR_INVALID_ARG, "similarity_adc: NULL operand");
  if (N < 0 || K < 1 || K > 65535 || D < 1 || ldc < D) return fail(h, HDC_ERR_INVALID_ARG, "similarity_adc: bad sizes");
  int rc = check_knobs(h, knobs, D);
  if (rc) return rc;
  if (ldh_words < words_of(knobs->D_eff)) return fail(h, HDC_ERR_INVALID_ARG, "similarity_adc: ldh_words < W");
  if (adc->res < 1 || adc->res > 16 || adc->step < 1 || adc->step > 65536 || adc->floor > adc->ceil ||
      adc->floor < -32768 || adc->ceil > 32768)
    return fail(h, HDC_ERR_INVALID_ARG, "similarity_adc: bad ADC window");
  if (!S && !labels && N > 0) return fail(h, HDC_ERR_INVALID_ARG, "similarity_adc: S or labels required");
  if (S && lds < K) return fail(h, HDC_ERR_INVALID_ARG, "similarity_adc: lds < K");
  if ((reinterpret_cast<uintptr_t>(Hbits) | reinterpret_cast<uintptr_t>(C_acc) | reinterpret_cast<uintptr_t>(S) |
       reinterpret_cast<uintptr_t>(labels)) & 3)
    return fail(h, HDC_ERR_ALIGNMENT, "similarity_adc: operands must be 4-byte aligned");
  if (N == 0) return HDC_OK;
  const int D_eff = knobs->D_eff;
  Bump b(ws);
  if (!ws) ws_bytes = 0;
  uint32_t* cls = b.take<uint32_t>(adc_class_bytes(K, D_eff) / sizeof(uint32_t));
  if (b.off > ws_bytes) return fail(h, HDC_ERR_WORKSPACE, "similarity_adc: workspace too small");
  // the transfer function, tabulated by the number of differing bits of a chunk of n dimensions
  AdcTables tab;
  const int n_tail = D_eff - 128 * ((D_eff + 127) / 128 - 1);
  const long long top = (1ll << adc->res) - 1;
  auto level = [&](int n, int diff) -> int {
    long long p = (long long)n - 2ll * diff;
    if (p < adc->floor) p = adc->floor;
    if (p > adc->ceil) p = adc->ceil;
    long long code = (p - adc->floor + adc->step / 2) / adc->step;
    if (code > top) code = top;
    return (int)(adc->floor + code * adc->step);
  };
  for (int i = 0; i <= 128; ++i) {
    tab.full[i] = level(128, i);
    tab.tail[i] = i <= n_tail ? level(n_tail, i) : 0;
  }
  cudaError_t ce;
  {
    Timed tm(h, HDC_K_SIM, (cudaStream_t)stream);
    ce = launch_adc_similarity(Hbits, N, ldh_words, C_acc, K, ldc, D_eff, tab, cls, S, lds, labels, h->sm_count,
                               h->smem_optin, (cudaStream_t)stream, &h->launches);
  }
  if (ce == cudaErrorNotSupported) return fail(h, HDC_ERR_UNSUPPORTED, "similarity_adc: D_eff too large for one CTA");
  return ce == cudaSuccess ? HDC_OK : cuda_fail(h, ce, "similarity_adc");
}

extern "C" int32_t hdc_classify(hdc_handle_t h, const uint32_t* Hbits, int64_t N, int64_t ldh_words,
                                const float* C_acc, int32_t K, int64_t ldc, int32_t D,
                                const hdc_knobs_t* knobs, int32_t* labels, float* best, float* second,
                                void* ws, size_t ws_bytes, void* stream) {
  if (!h) return HDC_ERR_INVALID_ARG;
  DeviceGuard device_guard(h->device);
  int rc = check_sim_args(h, Hbits, N, ldh_words, C_acc, K, ldc, D, knobs);
  if (rc) return rc;
  if (!labels && N > 0) return fail(h, HDC_ERR_INVALID_ARG, "classify: labels is NULL");
  if (N == 0) return HDC_OK;
  Bump b(ws);
  if (!ws) ws_bytes = 0;
  return do_similarity(h, Hbits, N, ldh_words, C_acc, K, ldc, knobs, nullptr, 0, 0, labels, best, second, b,
                       ws_bytes, (cudaStream_t)stream);
}

// =================================================================================== (3b, 3c)
extern "C" int32_t hdc_train_epoch(hdc_handle_t h, int32_t mode, const uint32_t* Hbits, int64_t N,
                                   int64_t ldh_words, const int32_t* y, float* C_acc, int32_t K, int64_t ldc,
                                   int32_t D, const hdc_knobs_t* knobs, float lr, int64_t batch, int32_t* pred,
                                   unsigned long long* n_wrong, void* ws, size_t ws_bytes, void* stream) {
  if (!h) return HDC_ERR_INVALID_ARG;
  DeviceGuard device_guard(h->device);
  if (mode != HDC_TRAIN_BUNDLE && mode != HDC_TRAIN_PERCEPTRON && mode != HDC_TRAIN_KMEANS)
    return fail(h, HDC_ERR_INVALID_ARG, "train: mode");
  if (!y && N > 0 && mode != HDC_TRAIN_KMEANS) return fail(h, HDC_ERR_INVALID_ARG, "train: y is NULL");
  if (batch < 0) return fail(h, HDC_ERR_INVALID_ARG, "train: batch < 0");
  hdc_knobs_t k;
  if (!knobs) return fail(h, HDC_ERR_INVALID_ARG, "knobs is NULL");
  k = *knobs;
  if (mode == HDC_TRAIN_BUNDLE) {  // only D_eff matters
    k.hv_bits = 32;
    k.sim = HDC_SIM_DOT;
  }
  int rc = check_sim_args(h, Hbits, N, ldh_words, C_acc, K, ldc, D, &k);
  if (rc) return rc;
  if (N == 0) return HDC_OK;
  cudaStream_t st = (cudaStream_t)stream;
  Bump b(ws);
  if (!ws) ws_bytes = 0;
  int32_t* delta = b.take<int32_t>((size_t)K * words_of(k.D_eff) * 32);
  if (b.off > ws_bytes) return fail(h, HDC_ERR_WORKSPACE, "train: workspace too small");
  cudaError_t ce;
  if (mode == HDC_TRAIN_BUNDLE) {
    ce = launch_class_update(Hbits, 0, N, ldh_words, y, nullptr, C_acc, K, ldc, k.D_eff, 1.0f, delta, nullptr,
                             h->sm_count, st, &h->launches);
    return ce == cudaSuccess ? HDC_OK : cuda_fail(h, ce, "bundle");
  }
  if (mode == HDC_TRAIN_KMEANS) {
    // assign every sample with the current accumulators, then re-bundle the clusters that have members
    int32_t* assign = pred ? pred : b.take<int32_t>((size_t)N);
    int32_t* members = b.take<int32_t>((size_t)K);
    if (b.off > ws_bytes) return fail(h, HDC_ERR_WORKSPACE, "train: workspace too small");
    rc = do_similarity(h, Hbits, N, ldh_words, C_acc, K, ldc, &k, nullptr, 0, 0, assign, nullptr, nullptr, b,
                       ws_bytes, st);
    if (rc) return rc;
    Timed tm(h, HDC_K_CLASS_UPDATE, st);
    ce = launch_kmeans_reset(assign, y, N, C_acc, K, ldc, k.D_eff, members, n_wrong, h->sm_count, st,
                             &h->launches);
    if (ce != cudaSuccess) return cuda_fail(h, ce, "kmeans reset");
    ce = launch_class_update(Hbits, 0, N, ldh_words, assign, nullptr, C_acc, K, ldc, k.D_eff, 1.0f, delta, nullptr,
                             h->sm_count, st, &h->launches);
    return ce == cudaSuccess ? HDC_OK : cuda_fail(h, ce, "kmeans bundle");
  }
  const int64_t B = (batch == 0 || batch > N) ? N : batch;
  int32_t* pbuf = pred;
  if (!pbuf) pbuf = b.take<int32_t>((size_t)B);
  if (b.off > ws_bytes) return fail(h, HDC_ERR_WORKSPACE, "train: workspace too small");
  const size_t base_off = b.off;
  for (int64_t n0 = 0; n0 < N; n0 += B) {
    const int64_t nb = (N - n0 < B) ? (N - n0) : B;
    int32_t* pb = pred ? pred + n0 : pbuf;
    Bump bs(ws);
    bs.off = base_off;
    rc = do_similarity(h, Hbits + n0 * ldh_words, nb, ldh_words, C_acc, K, ldc, &k, nullptr, 0, 0, pb, nullptr,
                       nullptr, bs, ws_bytes, st);
    if (rc) return rc;
    // class_update indexes y and pred with absolute sample numbers
    {
      Timed tm(h, HDC_K_CLASS_UPDATE, st);
      ce = launch_class_update(Hbits, n0, nb, ldh_words, y, pb - n0, C_acc, K, ldc, k.D_eff, lr, delta, n_wrong,
                               h->sm_count, st, &h->launches);
    }
    if (ce != cudaSuccess) return cuda_fail(h, ce, "class update");
  }
  return HDC_OK;
}

// =================================================================================== (3c) split for data-parallel training
extern "C" int32_t hdc_train_delta(hdc_handle_t h, const uint32_t* Hbits, int64_t N, int64_t ldh_words,
                                   const int32_t* y, const float* C_acc, int32_t K, int64_t ldc, int32_t D,
                                   const hdc_knobs_t* knobs, int32_t* delta, int32_t* pred,
                                   unsigned long long* n_wrong, void* ws, size_t ws_bytes, void* stream) {
  if (!h) return HDC_ERR_INVALID_ARG;
  DeviceGuard device_guard(h->device);
  if (!delta) return fail(h, HDC_ERR_INVALID_ARG, "train_delta: delta is NULL");
  if (!y && N > 0) return fail(h, HDC_ERR_INVALID_ARG, "train_delta: y is NULL");
  int rc = check_sim_args(h, Hbits, N, ldh_words, C_acc, K, ldc, D, knobs);
  if (rc) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  Bump b(ws);
  if (!ws) ws_bytes = 0;
  int32_t* pb = pred;
  if (!pb && N > 0) pb = b.take<int32_t>((size_t)N);
  if (b.off > ws_bytes) return fail(h, HDC_ERR_WORKSPACE, "train_delta: workspace too small");
  if (N > 0) {
    rc = do_similarity(h, Hbits, N, ldh_words, C_acc, K, ldc, knobs, nullptr, 0, 0, pb, nullptr, nullptr, b, ws_bytes,
                       st);
    if (rc) return rc;
  }
  Timed tm(h, HDC_K_CLASS_UPDATE, st);
  cudaError_t ce = launch_class_delta(Hbits, 0, N, ldh_words, y, pb, K, knobs->D_eff, delta, n_wrong, h->sm_count, st,
                                      &h->launches);
  return ce == cudaSuccess ? HDC_OK : cuda_fail(h, ce, "train_delta");
}

extern "C" int32_t hdc_train_apply(hdc_handle_t h, float* C_acc, int32_t K, int64_t ldc, int32_t D,
                                   const hdc_knobs_t* knobs, const int32_t* delta, float lr, void* stream) {
  if (!h) return HDC_ERR_INVALID_ARG;
  DeviceGuard device_guard(h->device);
  if (!C_acc || !delta) return fail(h, HDC_ERR_INVALID_ARG, "train_apply: NULL pointer");
  if (K < 1 || K > 65535 || D < 1 || ldc < D) return fail(h, HDC_ERR_INVALID_ARG, "train_apply: bad sizes");
  int rc = check_knobs(h, knobs, D);
  if (rc) return rc;
  cudaError_t ce = launch_apply_update(C_acc, K, ldc, knobs->D_eff, delta, lr, h->sm_count, (cudaStream_t)stream,
                                       &h->launches);
  return ce == cudaSuccess ? HDC_OK : cuda_fail(h, ce, "train_apply");
}

// =================================================================================== fused inference
extern "C" int32_t hdc_infer_rp(hdc_handle_t h, const void* X, int32_t x_dtype, int64_t N, int32_t F, int64_t ldx,
                                const void* P, int32_t p_dtype, int32_t D, int64_t ldp, const float* C_acc,
                                int32_t K, int64_t ldc, const hdc_knobs_t* knobs, int32_t* labels, float* best,
                                float* second, uint32_t* Hbits, int64_t ldh_words, void* ws, size_t ws_bytes,
                                void* stream) {
  if (!h) return HDC_ERR_INVALID_ARG;
  DeviceGuard device_guard(h->device);
  int rc = check_encode_rp_args(h, X, x_dtype, N, F, ldx, P, p_dtype, D, ldp, knobs);
  if (rc) return rc;
  if (!C_acc || (!labels && N > 0)) return fail(h, HDC_ERR_INVALID_ARG, "infer_rp: NULL pointer");
  if (K < 1 || K > 65535 || ldc < D) return fail(h, HDC_ERR_INVALID_ARG, "infer_rp: bad sizes");
  rc = check_sim_knobs(h, knobs);
  if (rc) return rc;
  if (Hbits && ldh_words < words_of(knobs->D_eff)) return fail(h, HDC_ERR_INVALID_ARG, "infer_rp: ldh_words < W");
  if ((reinterpret_cast<uintptr_t>(Hbits) | reinterpret_cast<uintptr_t>(C_acc) | reinterpret_cast<uintptr_t>(labels)) & 3)
    return fail(h, HDC_ERR_ALIGNMENT, "infer_rp: operands must be 4-byte aligned");
  if (N == 0) return HDC_OK;
  Bump b(ws);
  if (!ws) ws_bytes = 0;
  return do_infer_rp(h, X, x_dtype, N, F, ldx, P, p_dtype, D, ldp, C_acc, K, ldc, knobs, labels, best, second, Hbits,
                     ldh_words, b, ws_bytes, (cudaStream_t)stream);
}

// =================================================================================== prepared model
// The operands that do not depend on the queries -- the staged projection (bf16 / 3 x bf16 / half / int8 with
// its row scales) and the class operand at hv_bits with its cosine scales -- prepared ONCE into caller memory
// ("the one-time conversion of P and of the class model is not per-query work"); the *_m entry
// points then run only the per-query kernels.
constexpr uint32_t MODEL_MAGIC = 0x4D434448u;  // "HDCM"

static bool same_knobs(const hdc_knobs_t& a, const hdc_knobs_t& b) {
  return a.D_eff == b.D_eff && a.precision == b.precision && a.hv_bits == b.hv_bits && a.sim == b.sim &&
         a.flags == b.flags && a.perf_begin == b.perf_begin && a.perf_stride == b.perf_stride &&
         a.enc_perf_begin == b.enc_perf_begin && a.enc_perf_stride == b.enc_perf_stride;
}

extern "C" size_t hdc_model_bytes(hdc_handle_t h, int32_t F, int32_t D, int32_t K, const hdc_knobs_t* knobs) {
  if (!h || !knobs || F < 1 || D < 1 || K < 1) return 0;
  hdc_knobs_t k = *knobs;
  if (k.D_eff < 1 || k.D_eff > D) k.D_eff = D;
  return model_ws_bytes(h, F, K, &k);
}

extern "C" int32_t hdc_model_prepare(hdc_handle_t h, const void* P, int32_t p_dtype, int32_t F, int32_t D, int64_t ldp,
                                     const float* C_acc, int32_t K, int64_t ldc, const hdc_knobs_t* knobs, void* blob,
                                     size_t blob_bytes, hdc_model_t* out, void* stream) {
  if (!h) return HDC_ERR_INVALID_ARG;
  DeviceGuard device_guard(h->device);
  if (!out || !blob) return fail(h, HDC_ERR_INVALID_ARG, "model_prepare: NULL pointer");
  if (!P && !C_acc) return fail(h, HDC_ERR_INVALID_ARG, "model_prepare: neither P nor C_acc");
  int rc = check_knobs(h, knobs, D);
  if (rc) return rc;
  if (reinterpret_cast<uintptr_t>(blob) & 255) return fail(h, HDC_ERR_ALIGNMENT, "model_prepare: blob must be 256-byte aligned");
  if (P) {
    float dummy = 0.0f;  // X is not read when only preparing
    rc = check_encode_rp_args(h, &dummy, HDC_F32, 0, F, F, P, p_dtype, D, ldp, knobs);
    if (rc) return rc;
  }
  if (C_acc) {
    if (K < 1 || K > 65535 || ldc < D) return fail(h, HDC_ERR_INVALID_ARG, "model_prepare: bad sizes");
    rc = check_sim_knobs(h, knobs);
    if (rc) return rc;
    if (reinterpret_cast<uintptr_t>(C_acc) & 3) return fail(h, HDC_ERR_ALIGNMENT, "model_prepare: C_acc alignment");
  }
  if (blob_bytes < model_ws_bytes(h, P ? F : 1, C_acc ? K : 1, knobs))
    return fail(h, HDC_ERR_WORKSPACE, "model_prepare: blob smaller than hdc_model_bytes()");
  cudaStream_t st = (cudaStream_t)stream;
  rc = with_model(h, blob, blob_bytes, PREP_ONLY, [&]() {
    Bump none(nullptr);  // preparing takes nothing from a scratch workspace
    int r = HDC_OK;
    // the same order as do_infer_rp's two-kernel path carves them: encode, then similarity; the fused
    // epilogue's operand is prepared by hdc_model_prepare only when the knobs ask for that kernel
    if (P && C_acc && infer_fused_knobs(h, knobs, K))   // both operand sets, in do_infer_rp's order
      return do_infer_rp(h, nullptr, HDC_F32, INFER_MIN_N, F, F, P, p_dtype, D, ldp, C_acc, K, ldc, knobs, nullptr,
                         nullptr, nullptr, nullptr, 0, none, (size_t)-1, st);
    if (P) r = do_encode_rp(h, nullptr, HDC_F32, 1, F, F, P, p_dtype, D, ldp, knobs, HDC_OUT_BITS, nullptr, 0, nullptr, 0,
                            none, (size_t)-1, st);
    if (r == HDC_OK && C_acc)
      r = do_similarity(h, nullptr, 1, words_of(knobs->D_eff), C_acc, K, ldc, knobs, nullptr, 0, 0, nullptr, nullptr,
                        nullptr, none, (size_t)-1, st);
    return r;
  });
  if (rc) return rc;
  out->magic = MODEL_MAGIC;
  out->F = P ? F : 0;
  out->D = D;
  out->K = C_acc ? K : 0;
  out->p_dtype = p_dtype;
  out->ldp = ldp;
  out->ldc = ldc;
  out->P = P;
  out->C_acc = C_acc;
  out->blob = blob;
  out->blob_bytes = blob_bytes;
  out->knobs = *knobs;
  return HDC_OK;
}

static int check_model(hdc_ctx* h, const hdc_model_t* m, bool need_p, bool need_c) {
  if (!m || m->magic != MODEL_MAGIC || !m->blob) return fail(h, HDC_ERR_INVALID_ARG, "model: not prepared by hdc_model_prepare");
  if (need_p && !m->P) return fail(h, HDC_ERR_INVALID_ARG, "model: prepared without a projection");
  if (need_c && !m->C_acc) return fail(h, HDC_ERR_INVALID_ARG, "model: prepared without class accumulators");
  return HDC_OK;
}

extern "C" int32_t hdc_encode_rp_m(hdc_handle_t h, const void* X, int32_t x_dtype, int64_t N, int64_t ldx,
                                   const hdc_model_t* m, uint32_t* Hbits, int64_t ldh_words, void* ws, size_t ws_bytes,
                                   void* stream) {
  if (!h) return HDC_ERR_INVALID_ARG;
  DeviceGuard device_guard(h->device);
  int rc = check_model(h, m, true, false);
  if (rc) return rc;
  rc = check_encode_rp_args(h, X, x_dtype, N, m->F, ldx, m->P, m->p_dtype, m->D, m->ldp, &m->knobs);
  if (rc) return rc;
  if ((!Hbits && N > 0) || ldh_words < words_of(m->knobs.D_eff)) return fail(h, HDC_ERR_INVALID_ARG, "encode_rp_m: Hbits / ldh_words");
  if (reinterpret_cast<uintptr_t>(Hbits) & 3) return fail(h, HDC_ERR_ALIGNMENT, "encode_rp_m: Hbits alignment");
  if (N == 0) return HDC_OK;
  Bump b(ws);
  if (!ws) ws_bytes = 0;
  return with_model(h, m->blob, m->blob_bytes, RUN_ONLY, [&]() {
    return do_encode_rp(h, X, x_dtype, N, m->F, ldx, m->P, m->p_dtype, m->D, m->ldp, &m->knobs, HDC_OUT_BITS, Hbits,
                        ldh_words, nullptr, 0, b, ws_bytes, (cudaStream_t)stream);
  });
}

extern "C" int32_t hdc_classify_m(hdc_handle_t h, const uint32_t* Hbits, int64_t N, int64_t ldh_words,
                                  const hdc_model_t* m, int32_t* labels, float* best, float* second, void* ws,
                                  size_t ws_bytes, void* stream) {
  if (!h) return HDC_ERR_INVALID_ARG;
  DeviceGuard device_guard(h->device);
  int rc = check_model(h, m, false, true);
  if (rc) return rc;
  rc = check_sim_args(h, Hbits, N, ldh_words, m->C_acc, m->K, m->ldc, m->D, &m->knobs);
  if (rc) return rc;
  if (!labels && N > 0) return fail(h, HDC_ERR_INVALID_ARG, "classify_m: labels is NULL");
  if (N == 0) return HDC_OK;
  Bump b(ws);
  if (!ws) ws_bytes = 0;
  return with_model(h, m->blob, m->blob_bytes, RUN_ONLY, [&]() {
    // a model prepared with both halves holds the encode operands first: skip over them as hdc_model_prepare did
    Bump& pm = *static_cast<Bump*>(h->model);
    if (m->P) {
      Bump skip(nullptr);
      if (m->C_acc && infer_fused_knobs(h, &m->knobs, m->K) && !perf_on(enc_perf_of(&m->knobs))) infer_ws(m->K, m->knobs.D_eff, pm);
      encode_ws(h, 0, m->F, m->knobs.D_eff, &m->knobs, skip, pm);
    }
    return do_similarity(h, Hbits, N, ldh_words, m->C_acc, m->K, m->ldc, &m->knobs, nullptr, 0, 0, labels, best, second,
                         b, ws_bytes, (cudaStream_t)stream);
  });
}

extern "C" int32_t hdc_infer_rp_m(hdc_handle_t h, const void* X, int32_t x_dtype, int64_t N, int64_t ldx,
                                  const hdc_model_t* m, int32_t* labels, float* best, float* second, uint32_t* Hbits,
                                  int64_t ldh_words, void* ws, size_t ws_bytes, void* stream) {
  if (!h) return HDC_ERR_INVALID_ARG;
  DeviceGuard device_guard(h->device);
  int rc = check_model(h, m, true, true);
  if (rc) return rc;
  rc = check_encode_rp_args(h, X, x_dtype, N, m->F, ldx, m->P, m->p_dtype, m->D, m->ldp, &m->knobs);
  if (rc) return rc;
  if (!labels && N > 0) return fail(h, HDC_ERR_INVALID_ARG, "infer_rp_m: labels is NULL");
  if (Hbits && ldh_words < words_of(m->knobs.D_eff)) return fail(h, HDC_ERR_INVALID_ARG, "infer_rp_m: ldh_words < W");
  if ((reinterpret_cast<uintptr_t>(Hbits) | reinterpret_cast<uintptr_t>(labels)) & 3)
    return fail(h, HDC_ERR_ALIGNMENT, "infer_rp_m: operands must be 4-byte aligned");
  if (N == 0) return HDC_OK;
  Bump b(ws);
  if (!ws) ws_bytes = 0;
  return with_model(h, m->blob, m->blob_bytes, RUN_ONLY, [&]() {
    return do_infer_rp(h, X, x_dtype, N, m->F, ldx, m->P, m->p_dtype, m->D, m->ldp, m->C_acc, m->K, m->ldc, &m->knobs,
                       labels, best, second, Hbits, ldh_words, b, ws_bytes, (cudaStream_t)stream);
  });
}

// =================================================================================== host end-to-end
extern "C" int32_t hdc_infer_rp_host(hdc_handle_t h, const void* X_host, int32_t x_dtype, int64_t N, int32_t F,
                                     int64_t ldx, const void* P, int32_t p_dtype, int32_t D, int64_t ldp,
                                     const float* C_acc, int32_t K, int64_t ldc, const hdc_knobs_t* knobs,
                                     int32_t* labels_host, void* ws, size_t ws_bytes, void* stream) {
  if (!h) return HDC_ERR_INVALID_ARG;
  DeviceGuard device_guard(h->device);
  int rc = check_encode_rp_args(h, X_host, x_dtype, N, F, ldx, P, p_dtype, D, ldp, knobs);
  if (rc) return rc;
  if (!C_acc || !labels_host) return fail(h, HDC_ERR_INVALID_ARG, "infer_rp_host: NULL pointer");
  if (K < 1 || K > 65535 || ldc < D) return fail(h, HDC_ERR_INVALID_ARG, "infer_rp_host: bad sizes");
  rc = check_sim_knobs(h, knobs);
  if (rc) return rc;
  if (N == 0) return HDC_OK;
  cudaStream_t st = (cudaStream_t)stream;
  const size_t es = x_dtype == HDC_BF16 ? 2 : 4;
  const int64_t chunk = N < HOST_CHUNK ? N : HOST_CHUNK;
  Bump b(ws);
  if (!ws) ws_bytes = 0;
  char* Xd[2];
  Xd[0] = (char*)b.take<float>((size_t)chunk * F);
  Xd[1] = (char*)b.take<float>((size_t)chunk * F);
  int32_t* Ld = b.take<int32_t>((size_t)N);
  // the per-call-invariant operands (staged P, class operand, scales) are prepared by the first chunk into a
  // region of their own and used by every later one, whatever its size
  const size_t mbytes = model_ws_bytes(h, F, K, knobs);
  uint8_t* mblob = b.take<uint8_t>(mbytes);
  if (b.off > ws_bytes) return fail(h, HDC_ERR_WORKSPACE, "infer_rp_host: workspace too small");
  const size_t base_off = b.off;
  {  // dry run of the first (largest) chunk: workspace errors are reported before any copy is enqueued
    const size_t need = base_off + infer_ws_bytes(h, chunk, F, K, knobs);
    if (need > ws_bytes) return fail(h, HDC_ERR_WORKSPACE, "infer_rp_host: workspace too small");
  }
  cudaError_t ce = cudaEventRecord(h->ev_entry, st);
  if (ce == cudaSuccess) ce = cudaStreamWaitEvent(h->copy_stream, h->ev_entry, 0);
  if (ce != cudaSuccess) return cuda_fail(h, ce, "infer_rp_host: entry");
  // The copy of the first chunk is the one transfer no kernel overlaps, so the chunks ramp up: 2048 rows, then
  // x 1.5 per chunk up to HOST_CHUNK (the operands are prepared once, so a small chunk costs only its launches;
  // the copy is only ~15 % faster than the compute, so a steeper ramp would starve the kernels).  Measured at
  // 131072 C2 queries: 7.89 ms with constant 16384-row chunks, 7.4-7.6 ms with the ramp.
  int64_t c = 0;
  int64_t cur = chunk > HOST_RAMP_START ? HOST_RAMP_START : chunk;
  for (int64_t n0 = 0; n0 < N; ++c) {
    const int64_t nb = (N - n0 < cur) ? (N - n0) : cur;
    const int buf = (int)(c & 1);
    if (c >= 2) cudaStreamWaitEvent(h->copy_stream, h->ev_done[buf], 0);
    // rows are copied densely: device leading dimension is F
    if (ldx == F)
      ce = cudaMemcpyAsync(Xd[buf], (const char*)X_host + (size_t)n0 * ldx * es, (size_t)nb * F * es,
                           cudaMemcpyHostToDevice, h->copy_stream);
    else
      ce = cudaMemcpy2DAsync(Xd[buf], (size_t)F * es, (const char*)X_host + (size_t)n0 * ldx * es,
                             (size_t)ldx * es, (size_t)F * es, (size_t)nb, cudaMemcpyHostToDevice,
                             h->copy_stream);
    if (ce != cudaSuccess) {
      cudaStreamSynchronize(h->copy_stream);
      return cuda_fail(h, ce, "infer_rp_host: H2D");
    }
    cudaEventRecord(h->ev_copied[buf], h->copy_stream);
    cudaStreamWaitEvent(st, h->ev_copied[buf], 0);
    Bump be(ws);
    be.off = base_off;
    rc = with_model(h, mblob, mbytes, c == 0 ? PREP_AND_RUN : RUN_ONLY, [&]() {
      return do_infer_rp(h, Xd[buf], x_dtype, nb, F, F, P, p_dtype, D, ldp, C_acc, K, ldc, knobs, Ld + n0, nullptr,
                         nullptr, nullptr, 0, be, ws_bytes, st);
    });
    if (rc) {
      cudaStreamSynchronize(h->copy_stream);  // no copy into the caller's workspace outlives the call
      return rc;
    }
    cudaEventRecord(h->ev_done[buf], st);
    n0 += nb;
    {
      const int64_t nx = (cur * 3 / 2 + 255) / 256 * 256;   // x 1.5, whole 256-row tiles
      cur = nx < chunk ? nx : chunk;
    }
  }
  ce = cudaMemcpyAsync(labels_host, Ld, sizeof(int32_t) * (size_t)N, cudaMemcpyDeviceToHost, st);
  if (ce != cudaSuccess) return cuda_fail(h, ce, "infer_rp_host: D2H");
  ce = cudaStreamSynchronize(st);
  if (ce != cudaSuccess) return cuda_fail(h, ce, "infer_rp_host: sync");
  return HDC_OK;
}

// =================================================================================== no-allocation classify
// Scratch of hdc_classify_hamming_static: a fixed array in the library's device image (one copy per GPU that loads
// the library).  In host code the NAME below is only a stand-in for the symbol: the device address comes from
// cudaGetSymbolAddress, asked once per handle with the handle's device current, and that pointer is what the kernels
// receive.
static __device__ __align__(256) uint32_t g_static_scratch[HDC_STATIC_SCRATCH_BYTES / 4];

extern "C" int32_t hdc_classify_hamming_static(hdc_handle_t h, const uint32_t* Hbits, int64_t N, int64_t ldh_words,
                                               const float* C_acc, int32_t K, int64_t ldc, int32_t D,
                                               const hdc_knobs_t* knobs, int32_t* labels, float* best,
                                               float* second, void* stream) {
  if (!h) return HDC_ERR_INVALID_ARG;
  DeviceGuard device_guard(h->device);
  int rc = check_sim_args(h, Hbits, N, ldh_words, C_acc, K, ldc, D, knobs);
  if (rc) return rc;
  if (knobs->sim != HDC_SIM_HAMMING || knobs->hv_bits != 1)
    return fail(h, HDC_ERR_INVALID_ARG, "classify_hamming_static: needs sim = HDC_SIM_HAMMING, hv_bits = 1");
  if (!labels && N > 0) return fail(h, HDC_ERR_INVALID_ARG, "classify_hamming_static: labels is NULL");
  const int D_eff = knobs->D_eff;
  const int W = words_of(D_eff);
  if (K > 64 || ((size_t)K + 1) * (size_t)W * sizeof(uint32_t) > (size_t)HDC_STATIC_SCRATCH_BYTES)
    return fail(h, HDC_ERR_UNSUPPORTED,
                "classify_hamming_static: needs K <= 64 and (K + 1) * ceil(D_eff / 32) * 4 <= HDC_STATIC_SCRATCH_BYTES "
                "(1 MiB); use hdc_classify with a workspace");
  if (N == 0) return HDC_OK;
  cudaError_t ce;
  if (!h->static_scratch) {
    void* ptr = nullptr;
    ce = cudaGetSymbolAddress(&ptr, g_static_scratch);   // the current device is h->device (DeviceGuard)
    if (ce != cudaSuccess || !ptr) return cuda_fail(h, ce, "classify_hamming_static: cudaGetSymbolAddress");
    h->static_scratch = static_cast<uint32_t*>(ptr);
  }
  cudaStream_t st = (cudaStream_t)stream;
  const Perf pf = perf_of(knobs);
  uint32_t* cbits = h->static_scratch;                                         // [K][W], every word rewritten
  uint32_t* pmask = perf_on(pf) ? h->static_scratch + (size_t)K * W : nullptr;  // [W], every word rewritten
  ce = launch_sign_bits(C_acc, K, D_eff, ldc, cbits, W, st, &h->launches);
  if (ce != cudaSuccess) return cuda_fail(h, ce, "classify_hamming_static: sign_bits");
  if (pmask) {
    ce = launch_perf_mask(pmask, W, D_eff, pf, st, &h->launches);
    if (ce != cudaSuccess) return cuda_fail(h, ce, "classify_hamming_static: perforation mask");
  }
  ce = launch_hamming(Hbits, N, ldh_words, cbits, K, W, D_eff, pmask, nullptr, 0, labels, best, second, h->sm_count,
                      h->smem_optin, st, &h->launches);
  return ce == cudaSuccess ? HDC_OK : cuda_fail(h, ce, "classify_hamming_static: hamming");
}
