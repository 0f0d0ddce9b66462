// gemm_tc.cu -- tensor-core contraction C[m,n] = sum_k A[m,k] * B[n,k] for sm_100a: TMA ->
// shared memory (128-byte swizzle) -> tcgen05.mma -> TMEM -> tcgen05.ld epilogue, with the HDC
// epilogues fused: sign + pack (random-projection encode, Listing 1 L68-L70 + L161),
// scores (L110 cos_sim / L197 dot) and row arg-max (L79-L80).
//
// One persistent CTA per SM, 10 warps: warp 0 = TMA producer, warp 1 = MMA issuer (+ TMEM
// allocation), warps 2-9 = epilogue (warp w reads TMEM lanes 32*(w%4).., thread = accumulator
// row; two warps per lane quadrant split a tile's columns).  k-blocks of 128 bytes (64 bf16 / 128 int8), mbarrier ring between producer and issuer, two
// 256-column TMEM accumulators so that the epilogue of tile i overlaps the MMAs of tile i+1.
// Operands are K-contiguous ("K-major") for both A and B, which is the layout of X[N][F], P[D][F]
// and C[K][D] (include/hdc.h).
//
// CG = 2 (default for large problems): the two CTAs of a cluster (one TPC) share a 256 x 256 tile
// with tcgen05.mma.cta_group::2.  Each CTA loads its own 128 rows of A and HALF of the B tile, so a
// k-block costs 32 KB of shared-memory fill per SM instead of 48 KB (the 1-CTA kernel is bound by
// the L2 -> SM fill rate, profiles/r1_tcgen05_path.md) and the ring is 6 deep.  The even CTA issues
// the MMAs for both; barriers: `full` lives in the leader and counts the TMA bytes of both CTAs,
// `empty` and `tmem full` are signalled in both CTAs by a multicast tcgen05.commit, `tmem empty`
// lives in the leader and collects the epilogue warps of both CTAs.
// CG = 1: one CTA per 128 x 256 tile, 4-deep ring (small problems, HDC_FLAG_TC_1CTA).
//
// EPI_INFER (CTA pairs only; Listing 1 L63-L81 as ONE kernel): the epilogue warps, which idle for most of a tile
// while the tensor core works, also run the similarity search of the row they have just signed against K <= 32
// class hypervectors on the CUDA cores -- score[m,k] += sgn(acc[m,n]) * cls[k][n], one FFMA per (class,
// dimension), class tiles [KC][256] fp32 arriving by TMA through a two-slot ring of their own -- and the
// arg-max after the last n-tile of the row block, so the hypervectors never leave the SM unless asked for.
//
// The reduction axis is a list of SEGMENTS: k-block kb reads A columns a_seg[kb / nkb_seg] *
// seg_stride + (kb % nkb_seg) * BK and B columns b_seg[..] likewise.  One segment = a plain GEMM.
// Six segments over 3-way bf16-split operands [x1|x2|x3], [p1|p2|p3] give the fp32-precision
// contraction  x*p ~= x3p1 + x2p2 + x1p3 + x2p1 + x1p2 + x1p1  (smallest terms first, fp32
// accumulation in TMEM) without materialising the repeated operands (DESIGN.md "fp32 on tensor
// cores").
#include <cuda.h>
#include <cudaTypedefs.h>
#include <limits.h>

#include <type_traits>

#include "common.cuh"
#include "tc_ptx.cuh"

namespace hdc {

struct TcContext {
  PFN_cuTensorMapEncodeTiled_v12000 encode;
};

TcContext* tc_context_create() {
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult q;
  if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q) != cudaSuccess ||
      q != cudaDriverEntryPointSuccess || fn == nullptr) {
    (void)cudaGetLastError();
    return nullptr;
  }
  TcContext* tc = new TcContext();
  tc->encode = reinterpret_cast<PFN_cuTensorMapEncodeTiled_v12000>(fn);
  return tc;
}
void tc_context_destroy(TcContext* tc) { delete tc; }

// [rows][cols] matrix of `es`-byte elements, row stride ld elements, boxes of (128 bytes) x box_rows
// with the 128-byte swizzle; out-of-range elements read as zero.
bool tc_make_map(TcContext* tc, CUtensorMap* out, const void* ptr, bool int8, int64_t rows, int64_t cols,
                  int64_t ld, int box_rows) {
  const cuuint64_t es = int8 ? 1 : 2;
  cuuint64_t dims[2] = {(cuuint64_t)cols, (cuuint64_t)rows};
  cuuint64_t strides[1] = {(cuuint64_t)ld * es};
  cuuint32_t box[2] = {(cuuint32_t)(tcp::KB_BYTES / es), (cuuint32_t)box_rows};
  cuuint32_t estr[2] = {1, 1};
  return CUDA_SUCCESS == tc->encode(out, int8 ? CU_TENSOR_MAP_DATA_TYPE_UINT8 : CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2,
                    const_cast<void*>(ptr), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                    CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                    CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
}

// packed hypervector words [rows][cols] uint32, row stride ld words (ld % 4 == 0, 16-byte aligned base): boxes of
// 32 words x 128 rows with the 128-byte swizzle (16-byte piece j of row r sits at piece j ^ (r & 7): lane = row
// reads of one piece are conflict-free); out-of-range words and rows read as zero.
bool tc_make_map_words(TcContext* tc, CUtensorMap* out, const void* ptr, int64_t rows, int64_t cols, int64_t ld) {
  cuuint64_t dims[2] = {(cuuint64_t)cols, (cuuint64_t)rows};
  cuuint64_t strides[1] = {(cuuint64_t)ld * 4};
  cuuint32_t box[2] = {32, 128};
  cuuint32_t estr[2] = {1, 1};
  return CUDA_SUCCESS == tc->encode(out, CU_TENSOR_MAP_DATA_TYPE_UINT32, 2, const_cast<void*>(ptr), dims, strides,
                                    box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                                    CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
}

// fp32 [rows][cols] row-major, row stride ld elements: un-swizzled boxes of box_cols x box_rows
static bool tc_make_map_f32(TcContext* tc, CUtensorMap* out, const void* ptr, int64_t rows, int64_t cols, int64_t ld,
                            int box_cols, int box_rows) {
  cuuint64_t dims[2] = {(cuuint64_t)cols, (cuuint64_t)rows};
  cuuint64_t strides[1] = {(cuuint64_t)ld * 4};
  cuuint32_t box[2] = {(cuuint32_t)box_cols, (cuuint32_t)box_rows};
  cuuint32_t estr[2] = {1, 1};
  return CUDA_SUCCESS == tc->encode(out, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<void*>(ptr), dims, strides,
                                    box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                    CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
}

namespace {

using namespace tcp;

constexpr int BM = 128;            // rows of A per tile == TMEM lanes
constexpr int BN = 256;            // rows of B per tile == TMEM columns of one accumulator
constexpr int A_BYTES = BM * KB_BYTES;   // 16 KB
constexpr int EPI_WARPS = 8;            // two per TMEM lane quadrant: columns 0-127 and 128-255 of a tile
constexpr int NTHREADS = 64 + 32 * EPI_WARPS;
constexpr int TMEM_COLS = 512;
constexpr int MAX_STAGES = 6;
// KC = rows of the class tile of the fused inference epilogue (0: none).  The class tiles (two slots of
// KC x 256 floats) and the exchange buffer of the final arg-max (128 rows x KC floats) come out of the ring.
template <int CG, int KC = 0>
struct Cfg {
  static constexpr int STAGES = KC == 32 ? 4 : KC == 16 ? 5 : CG == 2 ? 6 : 4;
  static constexpr int B_ROWS = BN / CG;               // rows of B this CTA stages
  static constexpr int B_BYTES = B_ROWS * KB_BYTES;    // 32 KB / 16 KB
  static constexpr int STAGE_BYTES = A_BYTES + B_BYTES;
  static constexpr int CLS_BYTES = KC * BN * 4;        // one class tile
  static constexpr int XCH_BYTES = BM * KC * 4;
  static constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + 1024 /*alignment slack*/ + 256 /*barriers*/ +
                                    2 * CLS_BYTES + XCH_BYTES;
};

struct TcParams {
  int64_t M;
  int Nc;
  int m_tiles, n_tiles;
  int nseg, nkb_seg;            // number of reduction segments, k-blocks per segment
  int nk_last;                  // MMAs (32 bytes of the reduction axis each) the last k-block of a segment needs: 1..4
  uint32_t a_segs, b_segs;      // 4 bits per segment: which operand segment it reads
  int seg_stride;               // elements between operand segments
  int group_m;                  // m-tiles per rasterisation group (EPI_SIGN / EPI_SCORE)
  int f16;                      // 16-bit operands are IEEE half instead of bf16
  int bits_vec4;                // EPI_SIGN: rows of e.bits are 16-byte aligned (base and ldbits % 4 == 0)
  Epilogue e;
};

struct Top2 {
  double b1;
  int i1;
  double b2;
};
constexpr double NEG_BIG = -1.0e300;

// i-th tile of this CTA: EPI_ARGMAX owns whole m-tiles (n inner, so a thread sees every class of
// its row); the others walk groups of group_m m-tiles, m fastest, so that CTAs running at the same
// time share B tiles and reuse A tiles from L2.
// (CG = 2: the unit that walks the tiles is the cluster, and an m-tile is 256 rows.)
template <int EPI, int CG>
__device__ __forceinline__ bool tile_at(const TcParams& p, int i, int& mt, int& nt) {
  // 32-bit arithmetic (launch_gemm_tc bounds the tile count): every role calls this once per tile, and 64-bit
  // divisions cost the producer warp several hundred cycles of a 2560-cycle int8 tile
  const unsigned unit = blockIdx.x / CG, nunits = gridDim.x / CG;
  if (EPI == EPI_ARGMAX || EPI == EPI_INFER) {
    const unsigned q = (unsigned)i / (unsigned)p.n_tiles;
    const unsigned u = unit + q * nunits;
    if (u >= (unsigned)p.m_tiles) return false;
    mt = (int)u;
    nt = (int)((unsigned)i - q * (unsigned)p.n_tiles);
    return true;
  }
  const unsigned t = unit + (unsigned)i * nunits;
  if (t >= (unsigned)p.m_tiles * (unsigned)p.n_tiles) return false;
  const unsigned gsz = (unsigned)p.group_m * (unsigned)p.n_tiles;
  const unsigned g = t / gsz;
  const unsigned r = t - g * gsz;
  unsigned gm = (unsigned)p.m_tiles - g * (unsigned)p.group_m;
  if (gm > (unsigned)p.group_m) gm = (unsigned)p.group_m;
  const unsigned rq = r / gm;
  mt = (int)(g * (unsigned)p.group_m + (r - rq * gm));
  nt = (int)rq;
  return true;
}

template <bool INT8, int EPI, int CG, int KC>
__global__ void __launch_bounds__(NTHREADS, 1)
gemm_tc_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB,
               const __grid_constant__ CUtensorMap tmC, const TcParams p) {
  static_assert((EPI == EPI_INFER) == (KC != 0), "class tiles belong to the fused inference epilogue");
  constexpr int STAGES = Cfg<CG, KC>::STAGES;
  constexpr int STAGE_BYTES = Cfg<CG, KC>::STAGE_BYTES;
  constexpr int CLS_BYTES = Cfg<CG, KC>::CLS_BYTES;
  extern __shared__ uint8_t smem_raw[];
  const uint32_t base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  // barriers live after the stage ring (same offsets in both CTAs of a pair)
  const uint32_t bar0 = base + STAGES * STAGE_BYTES;
  auto full_bar = [&](int s) { return bar0 + 8u * s; };
  auto empty_bar = [&](int s) { return bar0 + 8u * (MAX_STAGES + s); };
  auto tfull_bar = [&](int s) { return bar0 + 8u * (2 * MAX_STAGES + s); };
  auto tempty_bar = [&](int s) { return bar0 + 8u * (2 * MAX_STAGES + 2 + s); };
  const uint32_t tmem_slot = bar0 + 8u * (2 * MAX_STAGES + 4);
  uint32_t* tmem_slot_ptr = reinterpret_cast<uint32_t*>(smem_raw + (tmem_slot - smem_u32(smem_raw)));
  // EPI_INFER: class-tile ring (two slots, barriers local to each CTA) and the arg-max exchange buffer
  auto cfull_bar = [&](int s) { return bar0 + 8u * (2 * MAX_STAGES + 6 + s); };
  auto cempty_bar = [&](int s) { return bar0 + 8u * (2 * MAX_STAGES + 8 + s); };
  const uint32_t cls0 = bar0 + 256u;
  const uint32_t xch0 = cls0 + 2u * CLS_BYTES;

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int rank = CG == 2 ? (int)cluster_ctarank() : 0;  // 0 = leader (issues the MMAs)
  constexpr int BK = INT8 ? 128 : 64;  // elements per k-block
  const int num_kb = p.nseg * p.nkb_seg;

  if (warp == 0 && lane == 0) {
    asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(&tmA)) : "memory");
    asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(&tmB)) : "memory");
    for (int s = 0; s < STAGES; ++s) {
      mbar_init(full_bar(s), 1);
      mbar_init(empty_bar(s), 1);
    }
    for (int s = 0; s < 2; ++s) {
      mbar_init(tfull_bar(s), 1);
      mbar_init(tempty_bar(s), EPI_WARPS * CG);
      mbar_init(cfull_bar(s), 1);
      mbar_init(cempty_bar(s), EPI_WARPS);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 1) {
    tmem_alloc<CG>(tmem_slot, TMEM_COLS);
  }
  tc_fence_before();
  if (CG == 2) cluster_sync_all(); else __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot_ptr;

  if (warp == 0) {
    // ================================================================= TMA producer
    int stage = 0;
    uint32_t phase = 0;
    int mt, nt;
    for (int i = 0; tile_at<EPI, CG>(p, i, mt, nt); ++i) {
      const int n0 = nt * BN;
      int nb = 0;
      if (CG == 2) {  // this CTA stages rows [rank * N/2, +N/2) of the tile's N (rounded to 16) columns
        int n_valid = p.Nc - n0;
        if (n_valid > BN) n_valid = BN;
        nb = rank * (((n_valid + 15) & ~15) >> 1);
      }
      const int m0 = (mt * CG + rank) * BM;
      if (EPI == EPI_INFER) {  // this tile's class tile: cls[0..KC)[n0, n0 + 256), own copy per CTA
        const int cs = (int)(i & 1);
        mbar_wait(cempty_bar(cs), (uint32_t)((i >> 1) & 1) ^ 1u);
        mbar_arrive_expect_tx_elect(cfull_bar(cs), CLS_BYTES);
        tma_load_2d_elect(cls0 + cs * CLS_BYTES, &tmC, cfull_bar(cs), n0, 0);
        __syncwarp();
      }
      // k-blocks in segment order (no division in this loop: the producer shares its scheduler with two
      // epilogue warps and has one k-block per 512 tensor cycles to issue)
      int seg = 0, j = 0;
      int acol = (int)(p.a_segs & 15u) * p.seg_stride, bcol = (int)(p.b_segs & 15u) * p.seg_stride;
      for (int kb = 0; kb < num_kb; ++kb) {
        mbar_wait(empty_bar(stage), phase ^ 1u);
        {
          const uint32_t sa = base + stage * STAGE_BYTES;
          if (CG == 2) {
            // both CTAs' bytes complete on the leader's barrier; only the leader arms it
            if (rank == 0) mbar_arrive_expect_tx_elect(full_bar(stage), 2 * STAGE_BYTES);
            tma_load_2d_2sm_elect(sa, &tmA, full_bar(stage) & PEER_MASK, acol, m0);
            tma_load_2d_2sm_elect(sa + A_BYTES, &tmB, full_bar(stage) & PEER_MASK, bcol, n0 + nb);
          } else {
            mbar_arrive_expect_tx_elect(full_bar(stage), STAGE_BYTES);
            tma_load_2d_elect(sa, &tmA, full_bar(stage), acol, m0);
            tma_load_2d_elect(sa + A_BYTES, &tmB, full_bar(stage), bcol, n0);
          }
        }
        __syncwarp();
        if (++stage == STAGES) {
          stage = 0;
          phase ^= 1u;
        }
        acol += BK;
        bcol += BK;
        if (++j == p.nkb_seg) {
          j = 0;
          ++seg;
          acol = (int)((p.a_segs >> (4 * seg)) & 15u) * p.seg_stride;
          bcol = (int)((p.b_segs >> (4 * seg)) & 15u) * p.seg_stride;
        }
      }
    }
  } else if (warp == 1) {
    // ================================================================= MMA issuer (leader CTA)
    int stage = 0;
    uint32_t phase = 0;
    int acc = 0;
    uint32_t acc_phase = 0;
    int mt, nt;
    for (int i = 0; rank == 0 && tile_at<EPI, CG>(p, i, mt, nt); ++i) {
      int n_valid = p.Nc - nt * BN;
      if (n_valid > BN) n_valid = BN;
      // kind::f16 operand formats (bits 7..9 A, 10..12 B): 1 = bf16, 0 = IEEE half
      const uint32_t idesc = instr_desc<INT8>(BM * CG, (n_valid + 15) & ~15) &
                             ((!INT8 && p.f16) ? ~((1u << 7) | (1u << 10)) : ~0u);
      mbar_wait(tempty_bar(acc), acc_phase ^ 1u);
      tc_fence_after();
      const uint32_t d_tmem = tmem_base + (uint32_t)(acc * BN);
      // The last k-block of a segment issues only the MMAs that reach valid columns (F = 617 bf16: 3 of 4, i.e. 39
      // instead of 40 MMAs per segment).  Two copies of the loop: the common case (every k-block full) must not pay
      // for the bookkeeping -- with five k-blocks per tile the int8 contraction follows this warp's issue rate
      // (measured: 0.470 -> 0.501 ms with the segment counter in its loop).
      auto issue_tile = [&](auto trimmed) {
        constexpr bool TRIM = decltype(trimmed)::value;
        int jseg = 0;   // k-block within its segment
        for (int kb = 0; kb < num_kb; ++kb) {
          mbar_wait(full_bar(stage), phase);
          tc_fence_after();
          {  // whole warp, converged: each call issues once (tc_ptx.cuh, *_elect)
            const uint32_t sa = base + stage * STAGE_BYTES;
            const uint64_t da = smem_desc(sa), db = smem_desc(sa + A_BYTES);
            bool full = true;
            if (TRIM && ++jseg == p.nkb_seg) {
              jseg = 0;
              full = false;
            }
            if (full) {
#pragma unroll
              for (int k = 0; k < KB_BYTES / 32; ++k)
                tc_mma_elect<INT8, CG>(d_tmem, da + 2u * k, db + 2u * k, idesc, (kb | k) != 0 ? 1u : 0u);
            } else {
#pragma unroll 1
              for (int k = 0; k < p.nk_last; ++k)
                tc_mma_elect<INT8, CG>(d_tmem, da + 2u * k, db + 2u * k, idesc, (kb | k) != 0 ? 1u : 0u);
            }
            tc_commit_elect<CG>(empty_bar(stage));            // frees the smem slot when these MMAs retire
            if (kb == num_kb - 1) tc_commit_elect<CG>(tfull_bar(acc));  // accumulator complete
          }
          __syncwarp();
          if (++stage == STAGES) {
            stage = 0;
            phase ^= 1u;
          }
        }
      };
      // (one-segment contractions -- bf16 / fp16 / int8 operands -- are not bound by the tensor pipe's power: there the
      // skipped MMA buys nothing and the bookkeeping costs 1 %)
      if (p.nk_last == KB_BYTES / 32 || p.nseg == 1) issue_tile(std::false_type{});
      else issue_tile(std::true_type{});
      if (++acc == 2) {
        acc = 0;
        acc_phase ^= 1u;
      }
    }
  } else {
    // ================================================================= epilogue (warps 2..9)
    using AccT = typename std::conditional<INT8, int, float>::type;
    const int q = warp & 3;  // TMEM lane quadrant this warp may read
    // EPI_SIGN: warps 2-5 drain chunks 0-3 of a tile, warps 6-9 chunks 4-7 (with few k-blocks per
    // tile the sign epilogue, not the MMAs, set the pace: profiles/r1_tcgen05_path.md, int8).  The
    // score / arg-max epilogues need every column of a row in one thread: warps 6-9 only hand the
    // accumulator back.
    const int ehalf = (warp - 2) >> 2;
    int acc = 0;
    uint32_t acc_phase = 0;
    Top2 run = Top2{NEG_BIG, INT_MAX, NEG_BIG};
    // EPI_INFER: running scores of this thread's row over its half of the columns.  fp32 holds them exactly
    // for the integer class operands (|score| <= 127 * D_eff < 2^24: launch_gemm_tc checks D_eff) and adds
    // one rounding per 32-column partial for the float ones.
    float irun[KC > 0 ? KC : 1];
#pragma unroll
    for (int k = 0; k < (KC > 0 ? KC : 1); ++k) irun[k] = 0.0f;
    int mt, nt;
    for (int i = 0; tile_at<EPI, CG>(p, i, mt, nt); ++i) {
      const int n0 = nt * BN;
      int n_valid = p.Nc - n0;
      if (n_valid > BN) n_valid = BN;
      const int64_t row = (int64_t)(mt * CG + rank) * BM + q * 32 + lane;
      const bool row_ok = row < p.M;
      mbar_wait(tfull_bar(acc), acc_phase);
      tc_fence_after();
      const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)(acc * BN);
      const int nchunks = (n_valid + 31) >> 5;
      if (EPI == EPI_SIGN) {
        // Two register buffers: the tcgen05.ld of chunk c+1 is in flight while chunk c is packed.
        // Sign + pack: one funnel shift per accumulator moves its sign bit into the word (last
        // column first, so column j lands in bit j); for floats x + (+0.0) first turns -0.0 into
        // +0.0 (reading A1: sgn(-0.0) = +1) on the FMA pipe, leaving the ALU pipe one op per value.
        uint32_t va[32], vb[32];
        uint32_t words[4] = {0u, 0u, 0u, 0u};   // this warp's (up to) four packed words of the row
        auto pack = [&](const uint32_t (&v)[32], int c) -> uint32_t {
          // four independent funnel-shift chains of eight (a single chain of 32 dependent shifts made the
          // epilogue latency, not its instruction count, the pace of short-reduction tiles)
          uint32_t w4[4] = {0u, 0u, 0u, 0u};
#pragma unroll
          for (int j = 7; j >= 0; --j) {
#pragma unroll
            for (int g = 0; g < 4; ++g) {
              const uint32_t x = v[8 * g + j];
              const uint32_t u = INT8 ? x : __float_as_uint(__fadd_rn(__uint_as_float(x), 0.0f));
              w4[g] = __funnelshift_l(u, w4[g], 1);
            }
          }
          uint32_t word = (w4[0] | (w4[1] << 8)) | ((w4[2] << 16) | (w4[3] << 24));
          const int valid = n_valid - c * 32;  // >= 1
          if (valid < 32) word &= (1u << valid) - 1u;
          if (row_ok && p.e.raw) {
            uint32_t* out = reinterpret_cast<uint32_t*>(p.e.raw) + row * p.e.ldraw + n0 + c * 32;
#pragma unroll
            for (int j = 0; j < 32; ++j)
              if (j < valid) out[j] = v[j];
          }
          return word;
        };
        const int c_begin = ehalf * 4;
        const int c_end = nchunks < c_begin + 4 ? nchunks : c_begin + 4;
        const int nleft = c_end - c_begin;   // 0..4 chunks for this warp
        if (nleft > 0) tmem_ld32(taddr + (uint32_t)(c_begin * 32), va);
#pragma unroll
        for (int i = 0; i < 4; i += 2) {
          if (i < nleft) {
            tmem_ld_wait();
            if (i + 1 < nleft) tmem_ld32(taddr + (uint32_t)((c_begin + i + 1) * 32), vb);
            words[i] = pack(va, c_begin + i);
            if (i + 1 < nleft) {
              tmem_ld_wait();
              if (i + 2 < nleft) tmem_ld32(taddr + (uint32_t)((c_begin + i + 2) * 32), va);
              words[i + 1] = pack(vb, c_begin + i + 1);
            }
          }
        }
        // one 16-byte store per thread when the row segment is aligned and complete (each warp of a lane
        // quadrant writes half of the row's 32-byte sector of this tile), else word by word
        if (row_ok && c_begin < c_end) {
          uint32_t* dst = p.e.bits + row * p.e.ldbits + (n0 >> 5) + c_begin;
          if (c_end - c_begin == 4 && p.bits_vec4) {
            *reinterpret_cast<uint4*>(dst) = make_uint4(words[0], words[1], words[2], words[3]);
          } else {
#pragma unroll
            for (int c = 0; c < 4; ++c)
              if (c_begin + c < c_end) dst[c] = words[c];
          }
        }
      }
      if (EPI == EPI_INFER) {
        // Fused similarity search.  Per 32-column chunk: sg[j] = +-1.0f from the sign of accumulator j, then one
        // FFMA per (class, column) against the class tile in shared memory (every lane reads the same 16 bytes:
        // a broadcast); each 32-column partial sum is added to the class's running score.
        const int cs = (int)(i & 1);
        mbar_wait(cfull_bar(cs), (uint32_t)((i >> 1) & 1));
        const float* ctile = reinterpret_cast<const float*>(smem_raw + (cls0 + cs * CLS_BYTES - smem_u32(smem_raw)));
        uint32_t words[4] = {0u, 0u, 0u, 0u};
        const int c_begin = ehalf * 4;
        const int c_end = nchunks < c_begin + 4 ? nchunks : c_begin + 4;
#pragma unroll 1
        for (int c = c_begin; c < c_end; ++c) {
          uint32_t v[32];
          tmem_ld32(taddr + (uint32_t)(c * 32), v);
          tmem_ld_wait();
          uint32_t w4[4] = {0u, 0u, 0u, 0u};
#pragma unroll
          for (int j = 7; j >= 0; --j) {
#pragma unroll
            for (int g = 0; g < 4; ++g) {
              const uint32_t x = v[8 * g + j];
              const uint32_t u = INT8 ? x : __float_as_uint(__fadd_rn(__uint_as_float(x), 0.0f));
              w4[g] = __funnelshift_l(u, w4[g], 1);
              v[8 * g + j] = (u & 0x80000000u) | 0x3F800000u;   // sgn as a float: -0.0 and 0 count as +1 (A1)
            }
          }
          uint32_t word = (w4[0] | (w4[1] << 8)) | ((w4[2] << 16) | (w4[3] << 24));
          const int valid = n_valid - c * 32;  // >= 1; columns beyond it meet zero class values
          if (valid < 32) word &= (1u << valid) - 1u;
          {
            const int ci = c - c_begin;   // static register selection (a dynamic index would go through local memory)
            if (ci == 0) words[0] = word;
            else if (ci == 1) words[1] = word;
            else if (ci == 2) words[2] = word;
            else words[3] = word;
          }
          const float4* crow = reinterpret_cast<const float4*>(ctile + c * 32);
#pragma unroll
          for (int k = 0; k < KC; ++k) {   // two chains of 16 per class, one add into the running score per chunk
            float t0 = 0.0f, t1 = 0.0f;
#pragma unroll
            for (int j4 = 0; j4 < 8; ++j4) {
              const float4 cv = crow[k * (BN / 4) + j4];
              t0 = __fmaf_rn(__uint_as_float(v[4 * j4 + 0]), cv.x, t0);
              t1 = __fmaf_rn(__uint_as_float(v[4 * j4 + 1]), cv.y, t1);
              t0 = __fmaf_rn(__uint_as_float(v[4 * j4 + 2]), cv.z, t0);
              t1 = __fmaf_rn(__uint_as_float(v[4 * j4 + 3]), cv.w, t1);
            }
            irun[k] = __fadd_rn(irun[k], __fadd_rn(t0, t1));
          }
        }
        if (p.e.bits && row_ok && c_begin < c_end) {
          uint32_t* dst = p.e.bits + row * p.e.ldbits + (n0 >> 5) + c_begin;
          if (c_end - c_begin == 4 && p.bits_vec4) {
            *reinterpret_cast<uint4*>(dst) = make_uint4(words[0], words[1], words[2], words[3]);
          } else {
#pragma unroll
            for (int c = 0; c < 4; ++c)
              if (c_begin + c < c_end) dst[c] = words[c];
          }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(cempty_bar(cs));   // class tile consumed
      }
      for (int c = 0; EPI != EPI_SIGN && EPI != EPI_INFER && ehalf == 0 && c < nchunks; ++c) {
        uint32_t v[32];
        tmem_ld32(taddr + (uint32_t)(c * 32), v);
        tmem_ld_wait();
        const int valid = n_valid - c * 32;  // >= 1
        if (EPI == EPI_SCORE) {
          if (row_ok) {
#pragma unroll
            for (int j = 0; j < 32; ++j) {
              if (j < valid) {
                const int col = n0 + c * 32 + j;
                const AccT a = INT8 ? (AccT)(int)v[j] : (AccT)__uint_as_float(v[j]);
                if (p.e.s_i32) {
                  reinterpret_cast<int32_t*>(p.e.S)[row * p.e.lds + col] = (int32_t)a;
                } else {
                  const float s = p.e.colscale ? (float)((double)a * p.e.colscale[col]) : (float)a;
                  reinterpret_cast<float*>(p.e.S)[row * p.e.lds + col] = s;
                }
              }
            }
          }
        } else {
#pragma unroll
          for (int j = 0; j < 32; ++j) {
            if (j < valid) {
              const int col = n0 + c * 32 + j;
              const AccT a = INT8 ? (AccT)(int)v[j] : (AccT)__uint_as_float(v[j]);
              const double s = p.e.colscale ? (double)a * p.e.colscale[col] : (double)a;
              if (s > run.b1) {  // columns arrive in increasing order: strict > keeps the lowest index
                run.b2 = run.b1;
                run.b1 = s;
                run.i1 = col;
              } else if (s > run.b2) {
                run.b2 = s;
              }
            }
          }
        }
      }
      // accumulator drained: hand it back to the MMA issuer
      tc_fence_before();
      __syncwarp();
      if (lane == 0) {
        if (CG == 2) mbar_arrive_cluster_relaxed(tempty_bar(acc) & PEER_MASK);  // the leader's barrier
        else mbar_arrive(tempty_bar(acc));
      }
      if (++acc == 2) {
        acc = 0;
        acc_phase ^= 1u;
      }
      if (EPI == EPI_ARGMAX && nt == p.n_tiles - 1) {
        if (row_ok && ehalf == 0) {
          double b1 = run.b1, b2 = run.b2;
          if (b2 == NEG_BIG) b2 = b1;  // K == 1
          if (p.e.ham_D > 0) {
            b1 = 0.5 * ((double)p.e.ham_D - b1);
            b2 = 0.5 * ((double)p.e.ham_D - b2);
          }
          p.e.labels[row] = run.i1;
          if (p.e.best) p.e.best[row] = (float)b1;
          if (p.e.second) p.e.second[row] = (float)b2;
        }
        run = Top2{NEG_BIG, INT_MAX, NEG_BIG};
      }
      if (EPI == EPI_INFER && nt == p.n_tiles - 1) {
        // the two warps of a lane quadrant hold the scores of the same rows over the two halves of every tile's
        // columns: the upper half hands its sums over through shared memory ([class][row]: conflict-free)
        float* xch = reinterpret_cast<float*>(smem_raw + (xch0 - smem_u32(smem_raw)));
        const int r = q * 32 + lane;
        if (ehalf == 1) {
#pragma unroll
          for (int k = 0; k < KC; ++k) xch[k * BM + r] = irun[k];
        }
        asm volatile("bar.sync %0, 64;" ::"r"(1 + q) : "memory");
        if (ehalf == 0) {
          Top2 t = Top2{NEG_BIG, INT_MAX, NEG_BIG};
#pragma unroll
          for (int k = 0; k < KC; ++k) {
            if (k < p.e.K) {
              const double a = (double)irun[k] + (double)xch[k * BM + r];
              const double sc = p.e.colscale ? a * p.e.colscale[k] : a;
              if (sc > t.b1) {  // increasing k: strict > keeps the lowest index
                t.b2 = t.b1;
                t.b1 = sc;
                t.i1 = k;
              } else if (sc > t.b2) {
                t.b2 = sc;
              }
            }
          }
          if (row_ok) {
            double b1 = t.b1, b2 = t.b2;
            if (b2 == NEG_BIG) b2 = b1;  // K == 1
            if (p.e.ham_D > 0) {
              b1 = 0.5 * ((double)p.e.ham_D - b1);
              b2 = 0.5 * ((double)p.e.ham_D - b2);
            }
            p.e.labels[row] = t.i1;
            if (p.e.best) p.e.best[row] = (float)b1;
            if (p.e.second) p.e.second[row] = (float)b2;
          }
        }
        asm volatile("bar.sync %0, 64;" ::"r"(1 + q) : "memory");   // buffer free for the next row block
#pragma unroll
        for (int k = 0; k < KC; ++k) irun[k] = 0.0f;
      }
    }
  }

  // ------------------------------------------------------------------- teardown
  tc_fence_before();
  if (CG == 2) cluster_sync_all(); else __syncthreads();
  if (warp == 1) {
    tc_fence_after();
    tmem_dealloc<CG>(tmem_base, TMEM_COLS);
  }
}

template <bool INT8, int EPI, int CG, int KC = 0>
cudaError_t launch_one(const CUtensorMap& tmA, const CUtensorMap& tmB, const CUtensorMap& tmC, const TcParams& p,
                       int grid, cudaStream_t st) {
  constexpr int SMEM_BYTES = Cfg<CG, KC>::SMEM_BYTES;
  static_assert(SMEM_BYTES <= 227 * 1024, "shared memory budget");
  // the opt-in is a per-device attribute of the function: set on every launch (a cheap host-side call), so
  // that handles on different devices of one process each get it
  cudaError_t e = cudaFuncSetAttribute(gemm_tc_kernel<INT8, EPI, CG, KC>,
                                       cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
  if (e != cudaSuccess) return e;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)grid);
  cfg.blockDim = dim3(NTHREADS);
  cfg.dynamicSmemBytes = SMEM_BYTES;
  cfg.stream = st;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeClusterDimension;
  at[0].val.clusterDim.x = CG;
  at[0].val.clusterDim.y = 1;
  at[0].val.clusterDim.z = 1;
  cfg.attrs = at;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, gemm_tc_kernel<INT8, EPI, CG, KC>, tmA, tmB, tmC, p);
}

template <int CG>
cudaError_t launch_cg(bool int8, int kind, const CUtensorMap& tmA, const CUtensorMap& tmB, const TcParams& p,
                      int grid, cudaStream_t st) {
  if (int8) {
    switch (kind) {
      case EPI_SIGN: return launch_one<true, EPI_SIGN, CG>(tmA, tmB, tmB, p, grid, st);
      case EPI_SCORE: return launch_one<true, EPI_SCORE, CG>(tmA, tmB, tmB, p, grid, st);
      default: return launch_one<true, EPI_ARGMAX, CG>(tmA, tmB, tmB, p, grid, st);
    }
  }
  switch (kind) {
    case EPI_SIGN: return launch_one<false, EPI_SIGN, CG>(tmA, tmB, tmB, p, grid, st);
    case EPI_SCORE: return launch_one<false, EPI_SCORE, CG>(tmA, tmB, tmB, p, grid, st);
    default: return launch_one<false, EPI_ARGMAX, CG>(tmA, tmB, tmB, p, grid, st);
  }
}

template <bool INT8>
cudaError_t launch_infer(int KC, const CUtensorMap& tmA, const CUtensorMap& tmB, const CUtensorMap& tmC,
                         const TcParams& p, int grid, cudaStream_t st) {
  switch (KC) {
    case 8: return launch_one<INT8, EPI_INFER, 2, 8>(tmA, tmB, tmC, p, grid, st);
    case 16: return launch_one<INT8, EPI_INFER, 2, 16>(tmA, tmB, tmC, p, grid, st);
    default: return launch_one<INT8, EPI_INFER, 2, 32>(tmA, tmB, tmC, p, grid, st);
  }
}

}  // namespace

cudaError_t launch_gemm_tc(TcContext* tc, const TcOperands& o, int64_t M, int Nc, const Epilogue& e,
                           int sm_count, int cta_group, cudaStream_t st, int64_t* nlaunch) {
  if (!tc) return cudaErrorNotSupported;
  if (M <= 0 || Nc <= 0) return cudaSuccess;
  const bool int8 = o.elem_kind == OPK_I8;
  const int es = int8 ? 1 : 2;
  const int BK = KB_BYTES / es;
  // TMA needs 16-byte aligned bases and row strides; segments must start on k-block boundaries
  if ((reinterpret_cast<uintptr_t>(o.A) & 15) || (reinterpret_cast<uintptr_t>(o.B) & 15) ||
      ((o.lda * es) & 15) || ((o.ldb * es) & 15) || o.nseg < 1 || o.nseg > 8 ||
      (o.nseg > 1 && (o.seg_stride % BK) != 0))
    return cudaErrorNotSupported;
  if (M > (int64_t)INT_MAX - 2 * BM || o.cols_a > INT_MAX || o.cols_b > INT_MAX) return cudaErrorNotSupported;
  const int n_tiles = (Nc + BN - 1) / BN;
  if ((M + BM - 1) / BM * (int64_t)n_tiles > (int64_t)INT_MAX / 2) return cudaErrorNotSupported;  // 32-bit tile indices
  const bool infer = e.kind == EPI_INFER;
  if (infer && (sm_count < 2 || e.K < 1 || e.K > 32 || Nc > (1 << 17) || !e.cls || (e.ldcls % BN) != 0 || e.ldcls < (int64_t)n_tiles * BN ||
                (reinterpret_cast<uintptr_t>(e.cls) & 15) || !e.labels))
    return cudaErrorNotSupported;
  const int64_t units1 = e.kind == EPI_ARGMAX ? (M + BM - 1) / BM : (M + BM - 1) / BM * n_tiles;
  // CTA pairs once every SM has a tile of its own either way; small problems keep the 1-CTA kernel
  // (twice as many independent tiles)
  int cg = cta_group;
  if (cg != 1 && cg != 2) cg = units1 >= 2 * (int64_t)sm_count ? 2 : 1;
  if (sm_count < 2) cg = 1;
  if (infer) cg = 2;
  TcParams p;
  p.M = M;
  p.Nc = Nc;
  p.m_tiles = (int)((M + BM * cg - 1) / (BM * cg));
  p.n_tiles = n_tiles;
  p.nseg = o.nseg;
  p.nkb_seg = (o.Kr + BK - 1) / BK;
  {
    const int kv = (o.Kvalid > 0 && o.Kvalid < o.Kr) ? o.Kvalid : o.Kr;
    const int last = kv - (p.nkb_seg - 1) * BK;                     // valid elements of a segment's last k-block
    const int per = 32 / (int8 ? 1 : 2);                            // elements per MMA
    p.nk_last = last <= 0 ? 1 : (last + per - 1) / per;
    if (p.nk_last > KB_BYTES / 32) p.nk_last = KB_BYTES / 32;
  }
  p.a_segs = o.a_segs;
  p.b_segs = o.b_segs;
  p.seg_stride = o.seg_stride;
  p.group_m = 16 / cg;
  p.f16 = o.elem_kind == OPK_F16;
  p.bits_vec4 = e.kind == EPI_SIGN && (reinterpret_cast<uintptr_t>(e.bits) & 15) == 0 && (e.ldbits & 3) == 0;
  p.e = e;
  CUtensorMap tmA, tmB;
  if (!tc_make_map(tc, &tmA, o.A, int8, M, o.cols_a, o.lda, BM)) return cudaErrorInvalidValue;
  if (!tc_make_map(tc, &tmB, o.B, int8, Nc, o.cols_b, o.ldb, BN / cg)) return cudaErrorInvalidValue;
  const int64_t units = (e.kind == EPI_ARGMAX || infer) ? p.m_tiles : (int64_t)p.m_tiles * p.n_tiles;
  const int max_units = sm_count / cg;
  const int grid = (int)(units < max_units ? units : max_units) * cg;
  ++*nlaunch;
  if (infer) {
    const int KC = e.K <= 8 ? 8 : (e.K <= 16 ? 16 : 32);
    CUtensorMap tmC;
    if (!tc_make_map_f32(tc, &tmC, e.cls, KC, e.ldcls, e.ldcls, BN, KC)) return cudaErrorInvalidValue;
    return int8 ? launch_infer<true>(KC, tmA, tmB, tmC, p, grid, st) : launch_infer<false>(KC, tmA, tmB, tmC, p, grid, st);
  }
  if (cg == 2) return launch_cg<2>(int8, e.kind, tmA, tmB, p, grid, st);
  return launch_cg<1>(int8, e.kind, tmA, tmB, p, grid, st);
}

}  // namespace hdc
