// simtc.cu -- similarity search on the tensor cores straight from PACKED query hypervectors
// (PAPER.md L110 cos_sim, L197 dot, L72-L74 Hamming via dist = (D_eff - dot)/2, L79-L80 arg-extremum):
//
//   S[n,k] = sum_{d<D_eff} v[n,d] * c[k,d],   v = 1 - 2*bit
//
// The +-1 query operand never exists in HBM: eight "expander" warps turn the packed words of a
// 128-query tile into the K-major, 128-byte-swizzled shared-memory tile that tcgen05.mma reads (the
// layout TMA would have written), while the class operand arrives by TMA.  Roles (14 warps, one
// persistent CTA per SM): warp 0 = TMA producer (class tiles), warp 1 = MMA issuer + TMEM
// allocation, warps 2-5 = epilogue (thread = query row), warps 6-13 = expanders (thread = query row
// x half of a k-block; the packed words reach each warp through a private cp.async ring).  Producer, expanders and
// issuer hand k-blocks over in groups (one full / empty barrier pair, one proxy fence, one commit per
// group); for small N the reduction axis is split over several CTAs per m-tile (split_reduce_kernel
// adds the partial sums in a fixed order).
//
// CG = 2 (large N, K >= 128): the two CTAs of a cluster share a 256-query x kc-class tile with
// tcgen05.mma.cta_group::2.  Each CTA expands its own 128 queries and stages HALF of the class tile, so per
// k-block an SM's shared memory takes 16 KB (expanders) + 16 KB (TMA) of writes and serves 32 KB of tensor-core
// reads instead of 16 + 32 and 48: the one-CTA kernel is bound by exactly that traffic (profiles/r2_simtc.md:
// tensor pipe 51 % active with the shared-memory data pipe saturated).  Barriers as in gemm_tc.cu: `full` lives in
// the leader (even CTA) and collects the TMA bytes and the expander warps of BOTH CTAs (the peer's warps arrive
// remotely after their proxy fence), `empty` / `tmem full` are signalled in both CTAs by multicast commits,
// `tmem empty` lives in the leader.
//
// Reduction-axis permutation.  A sum over d is invariant under any permutation of d applied to both
// operands, so the k-block position kappa <-> dimension map is chosen to make the expansion two or
// three ALU ops per 32-bit shared-memory word (perm_bf16 / perm_i8 below); the class operand is
// staged once per call in the same order by class_prepare_kernel (it is tiny: K x D_eff).
//
// Class operand precisions (S5): bf16 (hv_bits 16); fp32 (hv_bits 32) as three bf16 parts
// c1+c2+c3 stacked along the class axis of one tile -- the three partial accumulators are summed in
// the epilogue, so the queries are expanded once; int8 (hv_bits 8) and +-1 int8 (hv_bits 1) with
// int32 accumulation (exact).
#include <cuda_fp16.h>
#include <limits.h>

#include <type_traits>

#include "common.cuh"
#include "tc_ptx.cuh"

namespace hdc {
namespace {

using namespace tcp;

constexpr int BM = 128;
constexpr int BN_MAX = 256;
constexpr int MAX_STAGES = 10;  // ring depth is a runtime value: as many stages as fit in shared memory
constexpr int A_BYTES = BM * KB_BYTES;
constexpr int EXW = 8;                 // expander warps: two per 128-row tile half (4 of a k-block's 8 chunks each)
constexpr int NTHREADS = 192 + 32 * EXW;
constexpr int TMEM_COLS = 512;
constexpr int SMEM_LIMIT = 227 * 1024;
constexpr int SMEM_EXTRA = 1024 /*alignment slack*/ + 256 /*barriers*/;
// Query ring: every expander warp keeps a private 3-slot ring of [32 rows][8 words (+1 pad)] tiles holding just the
// packed words ITS threads expand (its 32 rows, its half of each k-block), filled by its own cp.async copies, so the
// ring needs no barrier between warps: a cp.async.wait_group and a __syncwarp per chunk.  (The round-1 ring was one
// [words][128 rows] tile shared by the eight warps behind a 256-thread named barrier per chunk: for int8 operands
// -- 4 k-blocks per chunk -- the warps spent 44 % of their samples in that hand-shake, profiles/r2_simtc.md.)
constexpr int CW = 8;                        // packed words per row and chunk in a warp's ring tile
constexpr int RLD = CW + 1;                  // row stride (words): conflict-free reads, lane = row
constexpr int WSLOT = 32 * RLD;              // words per slot and warp
constexpr int Q_SLOTS = 3;
constexpr int QRING_BYTES = 8 /*expander warps*/ * Q_SLOTS * WSLOT * 4;   // 27 648
__host__ __device__ constexpr int qring_bytes(int) { return QRING_BYTES; }

// dimension offset (within a k-block) of shared-memory K position kappa
__host__ __device__ __forceinline__ int perm_bf16(int kappa) {  // k-block = 64 dims = 2 words
  const int i = kappa >> 1;
  return 32 * (i >> 4) + (i & 15) + 16 * (kappa & 1);
}
__host__ __device__ __forceinline__ int perm_i8(int kappa) {  // k-block = 128 dims = 4 words
  const int i = kappa >> 2;
  return 32 * (i >> 3) + 8 * (kappa & 3) + (i & 7);
}

struct SimParams {
  const uint32_t* Hbits;
  int64_t N;
  int64_t ldh;
  int W;        // words holding d < D_eff
  int K;        // classes
  int kc;       // classes per n-tile (multiple of 16)
  int nparts;   // 1, or 3: the fp32 class operand as three bf16 parts / the int16 one as three base-128 digits
  int m_tiles, n_tiles;
  int num_kb;
  int splits;       // CTAs that share one m-tile, each reducing kbs k-blocks (split-D for small N)
  int kbs;          // k-blocks per split (multiple of 16)
  float* partial;   // [splits][K][N] partial sums when splits > 1 (fp32: exact for the integer paths, see sim_tc_splits)
  int kps;          // k-blocks per pipeline group
  int stages;       // ring depth
  int stage_bytes;  // A_BYTES + nparts*kc*KB_BYTES
  int f16;          // 16-bit operands are IEEE half instead of bf16 (hv code HDC_HV_F16)
  const int32_t* rowsum;   // INT8: sum of every staged class row (see the expanders), behind the staged operand
  const int* live;         // nullable: *live == 0 -> the staged class operand is all zero and nobody reads the scores
                           // (an all-zero 16-bit piece of 32- / 64-bit integer codes): the kernel returns at once
  int acc_cols, acc_bufs;  // sim_ts_kernel: TMEM columns of one accumulator and how many there are
  int ngroups;             // sim_ts_kernel: groups of 4 k-blocks in flight (class tiles in shared memory, expanded
                           // queries in tensor memory)
  Epilogue e;
};

struct Top2 {   // split_reduce_kernel (small N): double throughout
  double b1;
  int i1;
  double b2;
};
constexpr double NEG_BIG = -1.0e300;
// Running arg-max of the main kernel.  FP64 arithmetic is ~50 cycles per warp instruction and SM on this part
// (measured: with a double multiply, two double compares and a conversion per (query, class) the K = 1000
// classify spent every cycle of its epilogue warps there and the tensor pipe idled at 51 %), so the scores are
// compared in fp32 and the decision falls back to the exact double product only where two scores are within
// 2e-6 relative of each other -- which keeps the integer paths' labels (and exact ties -> lowest index)
// identical to an all-double comparison: an int32 / fp32 accumulator times the fp32-rounded scale is within
// 2^-23 relative of the double product.  a1 / a2: the accumulators of the best and the runner-up, from
// which their reported scores are recomputed in double once per row.
constexpr float NEG_BIG_F = -3.0e38f;
struct Top2f {
  float b1, b2;
  float a1, a2;
  int i1, i2;
  // a score below `lim` is neither a new best, nor a new runner-up, nor too close to the best for fp32: the sweep
  // over the classes tests one compare per class and enters the update logic behind a (mostly not taken) branch --
  // with 1000 classes the K-loop of the epilogue, not the tensor pipe, paced the int8 kernels (scaled arg-max
  // 1.20 ms against 0.79 ms unscaled per 65536 queries)
  float lim = NEG_BIG_F;
};

__device__ __forceinline__ uint32_t prmt_sign_bytes(uint32_t v) {
  uint32_t d;
  asm("prmt.b32 %0, %1, %1, 0xBA98;" : "=r"(d) : "r"(v));  // byte b <- 0xFF if msb of byte b of v else 0
  return d;
}

// Running best / runner-up of a query row: class k arrives with its accumulator (iv: integer kinds, a: as a float) and
// its fp32 score sc >= run.lim.  Classes arrive in increasing order: strict > keeps the lowest index.
template <bool INT8>
__device__ __forceinline__ void top2_update(const SimParams& p, Top2f& run, int k, int iv, float a, float sc,
                                            bool scaled) {
  bool better = sc > run.b1;
  bool second = sc > run.b2;
  if (scaled && fabsf(sc - run.b1) <= 2.0e-6f * fmaxf(fabsf(sc), fabsf(run.b1)) && run.i1 != INT_MAX) {
    // too close for fp32: the exact products decide (rare)
    const double ea = INT8 ? (double)iv : (double)a;
    const double e1 = INT8 ? (double)__float_as_int(run.a1) : (double)run.a1;
    better = ea * p.e.colscale[k] > e1 * p.e.colscale[run.i1];
  }
  if (INT8 && p.nparts == 3 && !scaled) {
    // int16 codes: sums beyond 2^24 are not exact as floats, the integers decide
    better = run.i1 == INT_MAX || iv > __float_as_int(run.a1);
    second = run.i2 == INT_MAX || iv > __float_as_int(run.a2);
  }
  const float araw = INT8 ? __int_as_float(iv) : a;   // integer accumulators are kept bit for bit
  if (better) {
    run.b2 = run.b1; run.a2 = run.a1; run.i2 = run.i1;
    run.b1 = sc; run.a1 = araw; run.i1 = k;
  } else if (second) {
    run.b2 = sc; run.a2 = araw; run.i2 = k;
  }
  // (superset of the ambiguity band |sc - b1| <= 2e-6 max(|sc|, |b1|) for sc < b1, and of sc > b2; the
  // integer compares of the int16 codes are covered by float conversion being monotonic: >= not >)
  run.lim = scaled ? fminf(run.b2, run.b1 - 2.1e-6f * fabsf(run.b1)) : run.b2;
}

// Epilogue of one accumulator tile for the query row of this thread (lane = TMEM lane of its warp's quarter): columns
// [0, k_valid) of the tile at taddr are classes k_base + c of n-tile nt; with nparts == 3 the three parts of class c
// sit kc columns apart.  sp: split of the reduction axis this CTA reduced (p.splits > 1: partial sums only).
template <bool INT8, int EPI, bool TS>
__device__ __forceinline__ void sim_epi_columns(const SimParams& p, uint32_t taddr, int nt, int k_base, int k_valid,
                                                int64_t row, bool row_ok, int sp, bool scaled, Top2f& run) {
  for (int c0 = 0; c0 < k_valid; c0 += 16) {
    uint32_t v0[16], v1[16], v2[16];
    tmem_ld16(taddr + (uint32_t)c0, v0);
    if (p.nparts == 3) {
      tmem_ld16(taddr + (uint32_t)(p.kc + c0), v1);
      tmem_ld16(taddr + (uint32_t)(2 * p.kc + c0), v2);
    }
    tmem_ld_wait();
    if constexpr (INT8 && EPI == EPI_ARGMAX && !TS) {
      // wide int8 tiles, sixteen valid classes: the sweep that paces the K = 1000 kernels -- scales by 16-byte loads,
      // no per-column bounds test, convert + multiply + one compare per class in front of the update logic
      if (p.nparts == 1 && p.splits == 1 && c0 + 16 <= k_valid) {
        float cs[16];
        if (scaled) {
          const float4* cp = reinterpret_cast<const float4*>(p.e.colscale_f + k_base + c0);   // 64-byte aligned
#pragma unroll
          for (int q4 = 0; q4 < 4; ++q4) {
            const float4 c4 = __ldg(cp + q4);
            cs[4 * q4] = c4.x; cs[4 * q4 + 1] = c4.y; cs[4 * q4 + 2] = c4.z; cs[4 * q4 + 3] = c4.w;
          }
        }
#pragma unroll
        for (int j = 0; j < 16; ++j) {
          const int iv = (int)v0[j];
          const float a = (float)iv;
          const float sc = scaled ? __fmul_rn(a, cs[j]) : a;
          if (sc < run.lim) continue;
          top2_update<INT8>(p, run, k_base + c0 + j, iv, a, sc, scaled);
        }
        continue;
      }
    }
#pragma unroll
    for (int j = 0; j < 16; ++j) {
      if (c0 + j < k_valid) {
        const int k = k_base + c0 + j;
        // the accumulator as a float: exact for the integer paths below 2^24, one rounding for the sum of
        // the three fp32-class parts
        float a;
        int iv = 0;
        if (INT8) {
          // TS: the expanders write the query bit b as the byte -128 b (one AND per word) instead of v = 1 - 2 b, so
          // the accumulator holds -128 sum_{b=1} c and  sum_d v c = sum_d c - 2 sum_{b=1} c = rowsum + (acc >> 6),
          // exactly (acc is a multiple of 128).  A split of the reduction axis adds the row sum once (split 0).
          int i0 = (int)v0[j], i1 = (int)v1[j], i2 = (int)v2[j];
          if constexpr (TS) {   // (wide class tiles keep +-1 bytes: one more load per column costs their epilogue more)
            const int32_t* rs = p.rowsum + (size_t)nt * p.nparts * p.kc + c0 + j;
            const bool first = sp == 0;
            i0 = (i0 >> 6) + (first ? __ldg(rs) : 0);
            if (p.nparts == 3) {
              i1 = (i1 >> 6) + (first ? __ldg(rs + p.kc) : 0);
              i2 = (i2 >> 6) + (first ? __ldg(rs + 2 * p.kc) : 0);
            }
          }
          // int16 class codes: three balanced base-128 digits, most significant first (exact in int32)
          iv = p.nparts == 3 ? i0 * 16384 + i1 * 128 + i2 : i0;
          a = (float)iv;
        } else if (p.nparts == 3) {
          a = __fadd_rn(__fadd_rn(__uint_as_float(v2[j]), __uint_as_float(v1[j])), __uint_as_float(v0[j]));
        } else {
          a = __uint_as_float(v0[j]);
        }
        if (p.splits > 1) {
          // partial sum of this split of the reduction axis; split_reduce_kernel adds the splits
          // in a fixed order and applies the epilogue
          if (row_ok) p.partial[((int64_t)sp * p.K + k) * p.N + row] = a;   // [split][class][query]: coalesced
        } else if (EPI == EPI_SCORE) {
          if (row_ok) {
            if (p.e.s_i32) {
              if (p.e.ham_D > 0) iv = (p.e.ham_D - iv) >> 1;
              reinterpret_cast<int32_t*>(p.e.S)[row * p.e.lds + k] = iv;
            } else {
              reinterpret_cast<float*>(p.e.S)[row * p.e.lds + k] = scaled ? __fmul_rn(a, p.e.colscale_f[k]) : a;
            }
          }
        } else {
          // classes arrive in increasing order: strict > keeps the lowest index
          const float sc = scaled ? __fmul_rn(a, p.e.colscale_f[k]) : a;
          if (sc < run.lim) continue;
          top2_update<INT8>(p, run, k, iv, a, sc, scaled);
        }
      }
    }
  }
}

// End of a query row's class sweep (EPI_ARGMAX): label, best and runner-up scores.
template <bool INT8>
__device__ __forceinline__ void sim_epi_finish(const SimParams& p, int64_t row, bool row_ok, bool scaled, Top2f& run) {
  if (row_ok) {
    // reported scores: the exact double products of the two winners (one conversion per row)
    const double e1 = INT8 ? (double)__float_as_int(run.a1) : (double)run.a1;
    const double e2 = INT8 ? (double)__float_as_int(run.a2) : (double)run.a2;
    double b1 = scaled ? e1 * p.e.colscale[run.i1] : e1;
    double b2 = run.i2 == INT_MAX ? b1 : (scaled ? e2 * p.e.colscale[run.i2] : e2);  // K == 1
    if (p.e.ham_D > 0) {
      b1 = 0.5 * ((double)p.e.ham_D - b1);
      b2 = 0.5 * ((double)p.e.ham_D - b2);
    }
    p.e.labels[row] = run.i1;
    if (p.e.best) p.e.best[row] = (float)b1;
    if (p.e.second) p.e.second[row] = (float)b2;
  }
  run = Top2f{NEG_BIG_F, NEG_BIG_F, 0.0f, 0.0f, INT_MAX, INT_MAX};
}

// TS: the expanded query tile lives in TENSOR memory instead of shared memory (tcgen05.mma with the A operand in
// TMEM): expanders write their rows with tcgen05.st into a ring of 8 k-block slots (32 columns each) beside two
// 128-column accumulators, the ring stages hold only the class tile.  For class tiles of <= 128 rows, where the
// shared-memory traffic of the A tile (16 KB written + 16 KB read per k-block against 2..12 KB of class rows)
// was the bound.  One CTA per tile.
constexpr int TS_ACC_COLS = 128;
constexpr int TS_A_COL0 = 2 * TS_ACC_COLS;
constexpr int TS_STAGES = (TMEM_COLS - TS_A_COL0) / 32;   // 8

template <bool INT8, int EPI, int CG, bool TS = false>
__global__ void __launch_bounds__(NTHREADS, 1)
sim_tc_kernel(const __grid_constant__ CUtensorMap tmB, const SimParams p) {
  static_assert(!TS || CG == 1, "the tensor-memory A ring is a one-CTA layout");
  if (p.live && *p.live == 0) return;   // (uniform over the grid: every CTA of a cluster leaves)
  constexpr uint32_t B_OFF = TS ? 0u : (uint32_t)A_BYTES;     // class tile within a ring stage
  constexpr int ACC_STRIDE = TS ? TS_ACC_COLS : BN_MAX;       // TMEM columns between the two accumulators
  extern __shared__ uint8_t smem_raw[];
  const uint32_t base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const int STAGES = p.stages;  // k-block slots in the ring
  const int G = p.kps;          // k-blocks per pipeline group (one full / empty barrier pair per group)
  const int NG = STAGES / G;
  const uint32_t STAGE_BYTES = (uint32_t)p.stage_bytes;
  const uint32_t bar0 = base + STAGES * STAGE_BYTES;
  auto full_bar = [&](int s) { return bar0 + 8u * s; };
  auto empty_bar = [&](int s) { return bar0 + 8u * (MAX_STAGES + s); };
  auto tfull_bar = [&](int s) { return bar0 + 8u * (2 * MAX_STAGES + s); };
  auto tempty_bar = [&](int s) { return bar0 + 8u * (2 * MAX_STAGES + 2 + s); };
  const uint32_t tmem_slot = bar0 + 8u * (2 * MAX_STAGES + 4);
  uint32_t* tmem_slot_ptr = reinterpret_cast<uint32_t*>(smem_raw + (tmem_slot - smem_u32(smem_raw)));

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int rank = CG == 2 ? (int)cluster_ctarank() : 0;   // 0 = leader: issues the MMAs, owns `full` / `tmem empty`
  constexpr int BK = INT8 ? 128 : 64;
  const int nb_rows = p.nparts * p.kc;      // class rows of a tile (the MMA's N)
  const int nb_half = nb_rows / CG;         // ... of which this CTA stages this many

  if (warp == 0 && lane == 0) {
    asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(&tmB)) : "memory");
    for (int s = 0; s < NG; ++s) {
      // leader's producer (with the TMA byte count of both CTAs) + one arrival per expander warp of each CTA
      mbar_init(full_bar(s), 1 + EXW * CG);
      mbar_init(empty_bar(s), 1);
    }
    for (int s = 0; s < 2; ++s) {
      mbar_init(tfull_bar(s), 1);
      mbar_init(tempty_bar(s), 4 * CG);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 1) tmem_alloc<CG>(tmem_slot, TMEM_COLS);
  tc_fence_before();
  if (CG == 2) cluster_sync_all(); else __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot_ptr;

  // work item = (m-tile of BM * CG queries, split of the reduction axis); a CTA (pair) walks items unit, +nunits, ...
  const int64_t unit = blockIdx.x / CG, nunits = gridDim.x / CG;
  const int64_t n_items = (int64_t)p.m_tiles * p.splits;
  const int64_t tiles_per_cta = (n_items > unit) ? ((n_items - 1 - unit) / nunits + 1) * p.n_tiles : 0;
  auto item_of = [&](int64_t i, int& mt, int& sp, int& kb_lo, int& kb_hi) {
    const int64_t item = unit + (i / p.n_tiles) * nunits;
    mt = (int)(item / p.splits);
    sp = (int)(item - (int64_t)mt * p.splits);
    kb_lo = sp * p.kbs;
    kb_hi = kb_lo + p.kbs < p.num_kb ? kb_lo + p.kbs : p.num_kb;
  };

  if (warp == 0) {
    // ================================================================= TMA producer (class tiles)
    int grp = 0;
    uint32_t phase = 0;
    for (int64_t i = 0; i < tiles_per_cta; ++i) {
      const int nt = (int)(i % p.n_tiles);
      int mt, sp, kb_lo, kb_hi;
      item_of(i, mt, sp, kb_lo, kb_hi);
      for (int kb0 = kb_lo; kb0 < kb_hi; kb0 += G) {
        const int n = kb_hi - kb0 < G ? kb_hi - kb0 : G;
        mbar_wait(empty_bar(grp), phase ^ 1u);
        if (CG == 2) {
          // both CTAs' halves complete on the leader's barrier; only the leader arms it
          if (rank == 0) mbar_arrive_expect_tx_elect(full_bar(grp), (uint32_t)(n * nb_rows) * KB_BYTES);
          for (int u = 0; u < n; ++u)
            tma_load_2d_2sm_elect(base + (grp * G + u) * STAGE_BYTES + B_OFF, &tmB, full_bar(grp) & PEER_MASK,
                                  (kb0 + u) * BK, nt * nb_rows + rank * nb_half);
        } else {
          mbar_arrive_expect_tx_elect(full_bar(grp), (uint32_t)(n * nb_rows) * KB_BYTES);
          for (int u = 0; u < n; ++u)
            tma_load_2d_elect(base + (grp * G + u) * STAGE_BYTES + B_OFF, &tmB, full_bar(grp), (kb0 + u) * BK,
                              nt * nb_rows);
        }
        __syncwarp();
        if (++grp == NG) {
          grp = 0;
          phase ^= 1u;
        }
      }
    }
  } else if (warp == 1) {
    // ================================================================= MMA issuer
    int grp = 0;
    uint32_t phase = 0;
    int acc = 0;
    uint32_t acc_phase = 0;
    // kind::f16 operand formats (bits 7..9 A, 10..12 B): 1 = bf16, 0 = IEEE half
    const uint32_t idesc = instr_desc<INT8>(BM * CG, nb_rows) & ((!INT8 && p.f16) ? ~((1u << 7) | (1u << 10)) : ~0u);
    for (int64_t i = 0; rank == 0 && i < tiles_per_cta; ++i) {
      mbar_wait(tempty_bar(acc), acc_phase ^ 1u);
      tc_fence_after();
      const uint32_t d_tmem = tmem_base + (uint32_t)(acc * ACC_STRIDE);
      int mt, sp, kb_lo, kb_hi;
      item_of(i, mt, sp, kb_lo, kb_hi);
      for (int kb0 = kb_lo; kb0 < kb_hi; kb0 += G) {
        const int n = kb_hi - kb0 < G ? kb_hi - kb0 : G;
        mbar_wait(full_bar(grp), phase);
        tc_fence_after();
        // whole warp, converged: each call issues once (tc_ptx.cuh, *_elect)
        if (TS && n == 4 && G == 4) {
          const uint32_t sa = base + (grp * G) * STAGE_BYTES;
          tc_mma_ts_group_elect<INT8>(d_tmem, tmem_base + (uint32_t)(TS_A_COL0 + grp * G * 32),
                                      ((sa & 0x3FFFFu) >> 4) | (1u << 16), (STAGE_BYTES >> 4) - 6u, idesc,
                                      kb0 != kb_lo ? 1u : 0u);
        } else
        for (int u = 0; u < n; ++u) {
          const uint32_t sa = base + (grp * G + u) * STAGE_BYTES;
          if constexpr (TS) {
            // (16..128-column MMAs take 8..64 tensor cycles: the issue sequence sets the pace, so the four MMAs of
            // a k-block go out of one asm block with one election and 32-bit descriptor arithmetic)
            const uint32_t b_lo = ((sa & 0x3FFFFu) >> 4) | (1u << 16);   // lower half of smem_desc(sa)
            const uint32_t at = tmem_base + (uint32_t)(TS_A_COL0 + (grp * G + u) * 32);
            tc_mma_ts_kblock_elect<INT8>(d_tmem, at, b_lo, idesc, kb0 + u != kb_lo ? 1u : 0u);
          } else {
            const uint64_t da = smem_desc(sa), db = smem_desc(sa + A_BYTES);
#pragma unroll
            for (int k = 0; k < KB_BYTES / 32; ++k)
              tc_mma_elect<INT8, CG>(d_tmem, da + 2u * k, db + 2u * k, idesc, (kb0 + u != kb_lo || k != 0) ? 1u : 0u);
          }
        }
        tc_commit_elect<CG>(empty_bar(grp));  // frees the group's slots (in both CTAs) when these MMAs retire
        if (kb0 + n == kb_hi) tc_commit_elect<CG>(tfull_bar(acc));
        __syncwarp();
        if (++grp == NG) {
          grp = 0;
          phase ^= 1u;
        }
      }
      if (++acc == 2) {
        acc = 0;
        acc_phase ^= 1u;
      }
    }
  } else if (warp < 6) {
    // ================================================================= epilogue (warps 2..5)
    const int q = warp & 3;
    int acc = 0;
    uint32_t acc_phase = 0;
    Top2f run = Top2f{NEG_BIG_F, NEG_BIG_F, 0.0f, 0.0f, INT_MAX, INT_MAX};
    const bool scaled = p.e.colscale != nullptr;
    for (int64_t i = 0; i < tiles_per_cta; ++i) {
      int mt, sp, kb_lo, kb_hi;
      item_of(i, mt, sp, kb_lo, kb_hi);
      const int nt = (int)(i % p.n_tiles);
      const int64_t row = (int64_t)(mt * CG + rank) * BM + q * 32 + lane;
      const bool row_ok = row < p.N;
      mbar_wait(tfull_bar(acc), acc_phase);
      tc_fence_after();
      const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)(acc * ACC_STRIDE);
      const int k_base = nt * p.kc;
      int k_valid = p.K - k_base;
      if (k_valid > p.kc) k_valid = p.kc;
      sim_epi_columns<INT8, EPI, TS>(p, taddr, nt, k_base, k_valid, row, row_ok, sp, scaled, run);
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
      if (EPI == EPI_ARGMAX && nt == p.n_tiles - 1 && p.splits == 1) sim_epi_finish<INT8>(p, row, row_ok, scaled, run);
    }
  } else {
    // ================================================================= expanders (warps 6..13)
    // Query words reach each expander warp through its private 3-deep cp.async ring (see CW above): nothing is
    // staged in registers, and a copy instruction covers 4 rows x 8 words whatever ldh is.
    const int et = (int)threadIdx.x - 192;    // 0..255
    // row of the tile; TS: a warp reaches only the TMEM lanes of ITS quarter (warp index mod 4)
    const int t = TS ? ((warp & 3) * 32 + lane) : (et & (BM - 1));
    const int part_id = et / BM;              // which half of a row's eight 16-byte chunks (warp-uniform)
    const int ew = et >> 5;                   // expander warp 0..7
    constexpr int C_PER = 8 / (EXW / 4);
    static_assert(EXW == 8, "two expander threads per row");
    constexpr int WPK = INT8 ? 4 : 2;         // packed words per k-block
    constexpr int WPP = WPK / 2;              // words of a k-block this thread's half needs
    constexpr int KPC = CW / WPP;             // k-blocks per ring chunk (8 / 4)
    const uint32_t sw = (uint32_t)(t & 7);
    const uint32_t q_smem = bar0 + 256u + (uint32_t)ew * (Q_SLOTS * WSLOT * 4);   // this warp's ring (after the barriers)
    const uint32_t* q_ptr = reinterpret_cast<const uint32_t*>(smem_raw + (q_smem - smem_u32(smem_raw)));
    int64_t is_i = 0;   // copy cursor: tile, chunk of the tile's k-block range, ring slot
    int is_c = 0, is_slot = 0;
    // geometry of the tile the cursor is in (item_of divides: once per tile, not once per chunk)
    int is_kb_lo = 0, is_nch = 0, is_rows = 0;
    const uint32_t* is_row0 = p.Hbits;
    auto issue_tile = [&]() {
      if (is_i >= tiles_per_cta) return;
      int mt, sp, kb_hi;
      item_of(is_i, mt, sp, is_kb_lo, kb_hi);
      is_nch = (kb_hi - is_kb_lo + KPC - 1) / KPC;
      const int64_t m0 = (int64_t)(mt * CG + rank) * BM + (t & ~31);   // first row of this warp
      const int64_t rows_left = p.N - m0;
      is_rows = rows_left < 32 ? (rows_left < 0 ? 0 : (int)rows_left) : 32;
      is_row0 = p.Hbits + (is_rows > 0 ? m0 : 0) * p.ldh;
    };
    issue_tile();
    auto issue = [&]() {
      if (is_i >= tiles_per_cta) return;
      const int lw = lane & (CW - 1), sub = lane >> 3;                  // word of the chunk, row within a group of 4
      // word lw of the chunk = word (lw % WPP) of this half of k-block kb_lo + is_c * KPC + lw / WPP
      const int w = (is_kb_lo + is_c * KPC + lw / WPP) * WPK + part_id * WPP + (lw % WPP);
      const int nrow = w < p.W ? is_rows : 0;
      const uint32_t* src = is_row0 + (int64_t)sub * p.ldh + w;
      uint32_t dst = q_smem + (uint32_t)(is_slot * WSLOT + sub * RLD + lw) * 4u;
#pragma unroll
      for (int rr = sub; rr < 32; rr += 4) {
        const bool ok = rr < nrow;
        asm volatile("cp.async.ca.shared.global [%0], [%1], 4, %2;" ::"r"(dst), "l"(ok ? src : p.Hbits),
                     "r"(ok ? 4 : 0)
                     : "memory");
        src += 4 * p.ldh;
        dst += 4 * RLD * 4u;
      }
      if (++is_slot == Q_SLOTS) is_slot = 0;
      if (++is_c == is_nch) {
        is_c = 0;
        ++is_i;
        issue_tile();
      }
    };
    for (int s0 = 0; s0 < Q_SLOTS - 1; ++s0) {
      issue();
      asm volatile("cp.async.commit_group;" ::: "memory");
    }

    int grp = 0;
    uint32_t phase = 0;
    int slot = 0;
    int64_t step = 0;
    // one k-block of this thread's row half: WPP packed words -> C_PER 16-byte chunks of the A tile
    const uint32_t one2 = p.f16 ? 0x3C003C00u : 0x3F803F80u;  // two +1.0 in half / bf16; the sign bit makes -1.0
    auto expand = [&](auto part, const uint32_t* qk, uint32_t a_row) {
      constexpr int PART = decltype(part)::value;
      constexpr int C0 = PART * C_PER;
      uint32_t wq[WPP];
#pragma unroll
      for (int v = 0; v < WPP; ++v) wq[v] = qk[v];
      uint32_t o[4 * C_PER];
#pragma unroll
      for (int cc = 0; cc < C_PER; ++cc) {  // 16-byte chunk cidx of the row = 4 words
        const int cidx = C0 + cc;
#pragma unroll
        for (int e = 0; e < 4; ++e) {
          const int iw = 4 * cidx + e;  // word index within the k-block's 32 output words
          if (INT8) {
            const uint32_t w = wq[(iw >> 3) - PART * WPP];
            // TS: byte = -128 * bit, one ALU instruction per word (the epilogue adds the class row sum: the ALU pipe
            // bounds the small-tile kernel); else byte = 1 - 2 * bit
            o[4 * cc + e] = TS ? ((w << (7 - (iw & 7))) & 0x80808080u)
                               : (prmt_sign_bytes(w << (7 - (iw & 7))) | 0x01010101u);
          } else {
            const uint32_t w = wq[(iw >> 4) - PART * WPP];
            o[4 * cc + e] = ((w << (15 - (iw & 15))) & 0x80008000u) | one2;
          }
        }
        if constexpr (!TS) {
          const uint32_t dst = a_row + ((((uint32_t)cidx) ^ sw) << 4);
          asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(dst), "r"(o[4 * cc]), "r"(o[4 * cc + 1]),
                       "r"(o[4 * cc + 2]), "r"(o[4 * cc + 3])
                       : "memory");
        }
      }
      // TS: a_row is the k-block's TMEM slot (this warp's lane quarter); word iw of the row = column iw
      if constexpr (TS) tmem_st16(a_row + (uint32_t)(4 * C0), o);
    };
    for (int64_t i = 0; i < tiles_per_cta; ++i) {
      int mt, sp, kb_lo, kb_hi;
      item_of(i, mt, sp, kb_lo, kb_hi);
      const int nch = (kb_hi - kb_lo + KPC - 1) / KPC;
      for (int c = 0; c < nch; ++c, ++step) {
        asm volatile("cp.async.wait_group %0;" ::"n"(Q_SLOTS - 2) : "memory");
        __syncwarp();   // this warp's tile is complete; its lanes are done with the slot about to be refilled
        issue();
        asm volatile("cp.async.commit_group;" ::: "memory");
        // this thread's words of the chunk's first k-block (groups never straddle a chunk: G | KPC)
        const uint32_t* qk = q_ptr + slot * WSLOT + lane * RLD;
        int left = (kb_hi - kb_lo) - c * KPC;
        if (left > KPC) left = KPC;
        while (left > 0) {
          const int n = left < G ? left : G;
          mbar_wait(empty_bar(grp), phase ^ 1u);
          uint32_t a_row;
          if constexpr (TS) {
            tc_fence_after();   // the MMAs that read these TMEM slots have retired (tcgen05.commit -> empty)
            a_row = tmem_base + ((uint32_t)(t & ~31) << 16) + (uint32_t)(TS_A_COL0 + grp * G * 32);
          } else {
            a_row = base + (uint32_t)(grp * G) * STAGE_BYTES + (uint32_t)t * KB_BYTES;
          }
#pragma unroll 1
          for (int u = 0; u < n; ++u) {
            if (part_id == 0) expand(std::integral_constant<int, 0>{}, qk, a_row);
            else expand(std::integral_constant<int, 1>{}, qk, a_row);
            qk += WPP;
            a_row += TS ? 32u : STAGE_BYTES;
          }
          // the group is published with one fence and one arrival per warp
          if constexpr (TS) {
            tmem_st_wait();
            tc_fence_before();
          } else {
            fence_proxy_async_smem();
          }
          __syncwarp();
          if (lane == 0) {
            if (CG == 2) mbar_arrive_remote(full_bar(grp) & PEER_MASK);   // the leader's barrier, from either CTA
            else mbar_arrive(full_bar(grp));
          }
          if (++grp == NG) {
            grp = 0;
            phase ^= 1u;
          }
          left -= n;
        }
        if (++slot == Q_SLOTS) slot = 0;
      }
    }
    asm volatile("cp.async.wait_group 0;" ::: "memory");
  }

  tc_fence_before();
  if (CG == 2) cluster_sync_all(); else __syncthreads();
  if (warp == 1) {
    tc_fence_after();
    tmem_dealloc<CG>(tmem_base, TMEM_COLS);
  }
}

// ---------------------------------------------------------------------------------- class operand
// Stages the class operand of sim_tc_kernel from the fp32 accumulators: staged row r holds class
// k = tile*kc + (r % (nparts*kc)) % kc, part (r % (nparts*kc)) / kc of tile r / (nparts*kc); staged
// column kb*BK + kappa holds dimension kb*BK + perm(kappa), zero for d >= D_eff or k >= K.
// mode: 32 -> bf16 part j of the 3-way split; 16 -> bf16 RNE; HDC_HV_F16 -> IEEE half RNE; 8 -> int8
// with scale 127/amax; HDC_HV_I16 -> digit 2 - j (balanced, base 128, each in [-64, 63]; the top one in
// [-2, 2]) of the int16 code with scale 32767/amax: q = 16384*part0 + 128*part1 + part2; 1 -> +-1 int8 from
// the sign.
__device__ __forceinline__ int quant_i8_c(float x, float s) {
  float q = rintf(__fmul_rn(x, s));
  q = fminf(fmaxf(q, -127.0f), 127.0f);
  return (int)q;
}

// One block per (padded) class: writes the class's nparts staged rows and, in the same pass, what the epilogue
// needs of it -- the cosine scale colscale[k] = 1 / (sqrt(n_vis) * |operand row|) (0 for a zero row; double, and
// rounded to fp32 in colscale_f; both nullable = no cosine) and, for the int8 kinds, the integer sum of every staged
// row (rowsum, see the expanders of sim_tc_kernel).  Fixed reduction order: thread-strided partial sums, then a
// shuffle / shared-memory tree (deterministic).  The norm is taken over the operand as the contraction sees it:
// the fp32 value (its three parts add up to it exactly), the rounded bf16 / half value, the integer code, +-1.
// FP64 instructions retire at ~1 per 53 cycles and SM on this part, and a DFMA per element made this kernel (and
// col_scale_kernel before it) 9 us of a 55 us retraining epoch: the per-thread partial sums are exact integers for
// the integer kinds and fp32 for the float kinds (<= 40 terms per thread at D = 10^4: ~1e-7 relative, inside the
// float paths' tolerance); the 1024 partials are added in double.
constexpr int CP_THREADS = 1024;   // (the kernel is a chain of load latencies: many short chains)
template <bool INT8>
__global__ void __launch_bounds__(CP_THREADS)
class_prepare_kernel(const float* __restrict__ C, int K, int D_eff, int64_t ldc, int mode, int kc, int nparts,
                     int num_kb, const float* __restrict__ amax, Perf pf, int n_vis, void* __restrict__ dst,
                     int32_t* __restrict__ rowsum, double* __restrict__ colscale, float* __restrict__ colscale_f,
                     int piece, int width, int* __restrict__ live) {
  constexpr int BK = INT8 ? 128 : 64;
  const int ld = num_kb * BK;
  const int k = blockIdx.x;                                   // class (rows k >= K are zero padding)
  const int64_t r0 = (int64_t)(k / kc) * (nparts * kc) + k % kc;   // staged row of part 0; part p: + p * kc
  float s = 1.0f;
  if (mode == 8 || (mode == HDC_HV_I16 && piece == 0)) {
    const float a = *amax;
    s = a > 0.0f ? __fdiv_rn(mode == 8 ? 127.0f : 32767.0f, a) : 1.0f;
  }
  float nrm2f = 0.0f;                // float kinds
  unsigned long long nrm2i = 0ull;   // integer kinds: exact
  int sum0 = 0, sum1 = 0, sum2 = 0;
#pragma unroll 4
  for (int col = threadIdx.x; col < ld; col += CP_THREADS) {
    const int kb = col / BK, kappa = col % BK;
    const int d = kb * BK + (INT8 ? perm_i8(kappa) : perm_bf16(kappa));
    const bool live = k < K && d < D_eff && perf_visits(pf, d);  // unvisited dimensions contribute 0
    const float x = live ? __ldg(C + (int64_t)k * ldc + d) : 0.0f;
    if (INT8) {
      int8_t* o = reinterpret_cast<int8_t*>(dst) + r0 * ld + col;
      if (mode == HDC_HV_I16) {
        int q;
        if (piece > 0) {
          // 32- / 64-bit integer codes (HDC_HV_I32 / _I64, reading A22): w = rint(x) saturated to `width` bits,
          // written as balanced base-65536 pieces w = sum_j p_j 65536^j (p_j in [-32768, 32767], the top one in
          // [-32768, 32768]); this call stages piece `piece - 1` like an int16 code
          long long w = live ? __float2ll_rn(x) : 0ll;
          const long long lim = width == 32 ? 2147483647ll : 9223372036854775807ll;
          w = w > lim ? lim : (w < -lim ? -lim : w);
          q = 0;
          for (int j = 1; j <= piece; ++j) {
            if (j * 16 == width) {
              q = (int)w;
            } else {
              const int low = (int)(w & 0xFFFFll);
              q = low >= 32768 ? low - 65536 : low;
              w = (w >> 16) + (low >= 32768 ? 1 : 0);
            }
          }
        } else {
          q = live ? (int)fminf(fmaxf(rintf(__fmul_rn(x, s)), -32767.0f), 32767.0f) : 0;
        }
        const int d0 = ((q + 64) & 127) - 64;
        const int r1 = (q - d0) >> 7;                  // exact: q - d0 is a multiple of 128
        const int d1 = ((r1 + 64) & 127) - 64;
        const int d2 = (r1 - d1) >> 7;
        o[0] = (int8_t)d2;
        o[(int64_t)kc * ld] = (int8_t)d1;
        o[(int64_t)2 * kc * ld] = (int8_t)d0;
        sum0 += d2; sum1 += d1; sum2 += d0;
        nrm2i += (unsigned long long)(q * q);
      } else {
        const int qv = !live ? 0 : (mode == 8 ? quant_i8_c(x, s) : (x < 0.0f ? -1 : 1));
        o[0] = (int8_t)qv;
        sum0 += qv;
        nrm2i += (unsigned long long)(qv * qv);
      }
    } else if (mode == HDC_HV_F16) {
      const __half hv = __float2half_rn(x);
      reinterpret_cast<__half*>(dst)[r0 * ld + col] = hv;
      const float v = __half2float(hv);
      nrm2f = __fmaf_rn(v, v, nrm2f);
    } else {
      __nv_bfloat16* o = reinterpret_cast<__nv_bfloat16*>(dst) + r0 * ld + col;
      const __nv_bfloat16 b1 = __float2bfloat16_rn(x);
      o[0] = b1;
      float v = __bfloat162float(b1);
      if (mode == 32) {
        const float r1 = __fsub_rn(x, __bfloat162float(b1));
        const __nv_bfloat16 b2 = __float2bfloat16_rn(r1);
        const float r2 = __fsub_rn(r1, __bfloat162float(b2));
        o[(int64_t)kc * ld] = b2;
        o[(int64_t)2 * kc * ld] = __float2bfloat16_rn(r2);
        v = x;
      }
      nrm2f = __fmaf_rn(v, v, nrm2f);
    }
  }
  if (INT8 && live) {   // piece mode: does this piece hold any nonzero code?  (live[] zeroed by wide_prepare_kernel)
    if (__syncthreads_or(nrm2i != 0ull) && threadIdx.x == 0) atomicOr(live, 1);
  }
  double nrm2 = INT8 ? (double)nrm2i : (double)nrm2f;   // (integers below 2^53: exact)
  __shared__ double sh_n[CP_THREADS / 32];
  __shared__ int sh_s[3][CP_THREADS / 32];
#pragma unroll
  for (int off = 16; off; off >>= 1) {
    nrm2 += __shfl_xor_sync(0xffffffffu, nrm2, off);
    if (INT8) {
      sum0 += __shfl_xor_sync(0xffffffffu, sum0, off);
      sum1 += __shfl_xor_sync(0xffffffffu, sum1, off);
      sum2 += __shfl_xor_sync(0xffffffffu, sum2, off);
    }
  }
  const int warp = threadIdx.x >> 5;
  if ((threadIdx.x & 31) == 0) {
    sh_n[warp] = nrm2;
    sh_s[0][warp] = sum0; sh_s[1][warp] = sum1; sh_s[2][warp] = sum2;
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    double t = 0.0;
    int t0 = 0, t1 = 0, t2 = 0;
    for (int i = 0; i < CP_THREADS / 32; ++i) {
      t += sh_n[i];
      t0 += sh_s[0][i]; t1 += sh_s[1][i]; t2 += sh_s[2][i];
    }
    if (INT8) {
      rowsum[r0] = t0;
      if (nparts == 3) {
        rowsum[r0 + kc] = t1;
        rowsum[r0 + 2 * kc] = t2;
      }
    }
    if (colscale && k < K) {
      const double nrm = sqrt(t);
      const double cs = nrm > 0.0 ? 1.0 / (sqrt((double)n_vis) * nrm) : 0.0;
      colscale[k] = cs;
      if (colscale_f) colscale_f[k] = (float)cs;
    }
  }
}

// Adds the split partial sums in split order (fixed: deterministic) and applies the epilogue of
// sim_tc_kernel: scores (S) or arg-max with best / runner-up, with the same fp32 comparison + exact double
// tie-break.  One thread per query row; [split][class][query] layout: coalesced.  int_acc: the partial sums are
// integers (exact in fp32 below 2^24, which sim_tc_splits guarantees).
template <int SU>   // SU >= splits: 2, 4 or 8
__global__ void split_reduce_kernel(const float* __restrict__ partial, int splits, int64_t N, int K, Epilogue e) {
  const int64_t n = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (n >= N) return;
  const bool scaled = e.colscale != nullptr;
  Top2f run = Top2f{NEG_BIG_F, NEG_BIG_F, 0.0f, 0.0f, INT_MAX, INT_MAX};
  constexpr int KU = 64 / SU;   // classes whose partial sums are fetched together (64 independent loads in flight)
  for (int k0 = 0; k0 < K; k0 += KU) {
    // all splits of the KU classes are fetched before the first add (at most 8 splits: sim_tc_splits): one memory
    // round trip per KU classes instead of one per (KU classes, split) -- the kernel is nothing but load latency
    float t[SU][KU];
#pragma unroll
    for (int sp = 0; sp < SU; ++sp)
#pragma unroll
      for (int j = 0; j < KU; ++j)
        t[sp][j] = (sp < splits && k0 + j < K) ? __ldg(partial + ((int64_t)sp * K + k0 + j) * N + n) : 0.0f;
    float av[KU];
#pragma unroll
    for (int j = 0; j < KU; ++j) {
      av[j] = t[0][j];
#pragma unroll
      for (int sp = 1; sp < SU; ++sp)
        if (sp < splits) av[j] = __fadd_rn(av[j], t[sp][j]);   // split order: deterministic
    }
#pragma unroll
    for (int j = 0; j < KU; ++j) {
    const int k = k0 + j;
    if (k >= K) break;
    const float a = av[j];
    if (e.kind == EPI_SCORE) {
      if (e.s_i32) {
        int iv = (int)a;
        if (e.ham_D > 0) iv = (e.ham_D - iv) >> 1;
        reinterpret_cast<int32_t*>(e.S)[n * e.lds + k] = iv;
      } else {
        reinterpret_cast<float*>(e.S)[n * e.lds + k] = scaled ? __fmul_rn(a, e.colscale_f[k]) : a;
      }
    } else {
      const float sc = scaled ? __fmul_rn(a, e.colscale_f[k]) : a;
      bool better = sc > run.b1;
      if (scaled && fabsf(sc - run.b1) <= 2.0e-6f * fmaxf(fabsf(sc), fabsf(run.b1)) && run.i1 != INT_MAX)
        better = (double)a * e.colscale[k] > (double)run.a1 * e.colscale[run.i1];
      if (better) {
        run.b2 = run.b1; run.a2 = run.a1; run.i2 = run.i1;
        run.b1 = sc; run.a1 = a; run.i1 = k;
      } else if (sc > run.b2) {
        run.b2 = sc; run.a2 = a; run.i2 = k;
      }
    }
    }
  }
  if (e.kind == EPI_ARGMAX) {
    double b1 = scaled ? (double)run.a1 * e.colscale[run.i1] : (double)run.a1;
    double b2 = run.i2 == INT_MAX ? b1 : (scaled ? (double)run.a2 * e.colscale[run.i2] : (double)run.a2);  // K == 1
    if (e.ham_D > 0) {
      b1 = 0.5 * ((double)e.ham_D - b1);
      b2 = 0.5 * ((double)e.ham_D - b2);
    }
    e.labels[n] = run.i1;
    if (e.best) e.best[n] = (float)b1;
    if (e.second) e.second[n] = (float)b2;
  }
}

// ---------------------------------------------------------------------------------- small class tiles, TMA-fed
// sim_ts_kernel: the small-tile kernel (query tile in tensor memory, see TS above) for query rows that are 16-byte
// aligned (what Handle.alloc_hbits / hdc_encode_* give): the packed words arrive by TMA -- boxes of 128 rows x 32
// words = 1024 dimensions, 128-byte swizzle, one elected lane of a producer warp per box -- instead of through the
// expander warps' private cp.async rings, whose refill (8 four-byte copies per lane and chunk plus addresses) was a
// quarter of an expander warp's time per group (profiles/r2_simtc.md 4.1).  Roles (16 warps, one persistent CTA per
// SM): warp 0 = TMA producer of the class tiles, warp 1 = MMA issuer + TMEM allocation, warp 2 = TMA producer of the
// query words, warps 4-7 = epilogue, warps 8-15 = expanders: warp w serves the TMEM lane quarter w % 4 (the only one
// it can reach); the two warps of a quarter take alternate 16-byte pieces of every row = whole k-blocks (one int8
// k-block of 128 dimensions or two 16-bit k-blocks of 64).  Groups and barriers as in the TS variant of
// sim_tc_kernel; TMEM: acc_bufs accumulators of acc_cols columns, then ngroups x 4 k-block slots of 32 columns.
constexpr int TSQ_THREADS = 512;
constexpr int TSQ_SLOTS = 4;                       // query chunks in flight
constexpr int TSQ_WORDS = 32;                      // packed words of a row per chunk
constexpr int TSQ_BYTES = BM * TSQ_WORDS * 4;      // 16 KB
constexpr int TSQ_G = 4;                           // k-blocks per group
constexpr int TSQ_MAXG = 3;                        // groups in flight

template <bool INT8, int EPI>
__global__ void __launch_bounds__(TSQ_THREADS, 1)
sim_ts_kernel(const __grid_constant__ CUtensorMap tmB, const __grid_constant__ CUtensorMap tmQ, const SimParams p) {
  if (p.live && *p.live == 0) return;
  extern __shared__ uint8_t smem_raw[];
  constexpr int BK = INT8 ? 128 : 64;
  constexpr int WPK = INT8 ? 4 : 2;          // packed words per k-block
  constexpr int KPC = TSQ_WORDS / WPK;       // k-blocks per query chunk (8 / 16)
  constexpr int KPP = 4 / WPK;               // k-blocks per 16-byte piece of a row (1 / 2)
  constexpr int G = TSQ_G, MG = TSQ_MAXG;
  const int NG = p.ngroups;
  const uint32_t base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const int nb_rows = p.nparts * p.kc;
  const uint32_t B_BYTES = (uint32_t)nb_rows * KB_BYTES;
  const uint32_t q_base = base + (uint32_t)(NG * G) * B_BYTES;
  const uint32_t bar0 = q_base + TSQ_SLOTS * TSQ_BYTES;
  auto full_bar = [&](int s) { return bar0 + 8u * s; };
  auto empty_bar = [&](int s) { return bar0 + 8u * (MG + s); };
  auto qfull_bar = [&](int s) { return bar0 + 8u * (2 * MG + s); };
  auto qempty_bar = [&](int s) { return bar0 + 8u * (2 * MG + TSQ_SLOTS + s); };
  auto tfull_bar = [&](int s) { return bar0 + 8u * (2 * MG + 2 * TSQ_SLOTS + s); };
  auto tempty_bar = [&](int s) { return bar0 + 8u * (2 * MG + 2 * TSQ_SLOTS + 2 + s); };
  const uint32_t tmem_slot = bar0 + 8u * (2 * MG + 2 * TSQ_SLOTS + 4);
  const int A_COL0 = p.acc_bufs * p.acc_cols;   // first TMEM column of the query slots
  uint32_t* tmem_slot_ptr = reinterpret_cast<uint32_t*>(smem_raw + (tmem_slot - smem_u32(smem_raw)));

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (warp == 0 && lane == 0) {
    asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(&tmB)) : "memory");
    asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(&tmQ)) : "memory");
    for (int s = 0; s < NG; ++s) {
      mbar_init(full_bar(s), 1 + EXW);   // class tiles (producer + bytes) and one arrival per expander warp
      mbar_init(empty_bar(s), 1);
    }
    for (int s = 0; s < TSQ_SLOTS; ++s) {
      mbar_init(qfull_bar(s), 1);
      mbar_init(qempty_bar(s), EXW);
    }
    for (int s = 0; s < 2; ++s) {
      mbar_init(tfull_bar(s), 1);
      mbar_init(tempty_bar(s), 4);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 1) tmem_alloc<1>(tmem_slot, TMEM_COLS);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot_ptr;

  // work item = (m-tile of 128 queries, split of the reduction axis); a CTA walks items blockIdx.x, +gridDim.x, ...
  const int64_t n_items = (int64_t)p.m_tiles * p.splits;
  auto item_of = [&](int64_t item, int& mt, int& sp, int& kb_lo, int& kb_hi) {
    mt = (int)(item / p.splits);
    sp = (int)(item - (int64_t)mt * p.splits);
    kb_lo = sp * p.kbs;
    kb_hi = kb_lo + p.kbs < p.num_kb ? kb_lo + p.kbs : p.num_kb;
  };

  if (warp == 0) {
    // ================================================================= TMA producer: class tiles
    int grp = 0;
    uint32_t phase = 0;
    for (int64_t item = blockIdx.x; item < n_items; item += gridDim.x) {
      int mt, sp, kb_lo, kb_hi;
      item_of(item, mt, sp, kb_lo, kb_hi);
      for (int kb0 = kb_lo; kb0 < kb_hi; kb0 += G) {
        const int n = kb_hi - kb0 < G ? kb_hi - kb0 : G;
        mbar_wait(empty_bar(grp), phase ^ 1u);
        mbar_arrive_expect_tx_elect(full_bar(grp), (uint32_t)n * B_BYTES);
        for (int u = 0; u < n; ++u)
          tma_load_2d_elect(base + (uint32_t)(grp * G + u) * B_BYTES, &tmB, full_bar(grp), (kb0 + u) * BK, 0);
        __syncwarp();
        if (++grp == NG) {
          grp = 0;
          phase ^= 1u;
        }
      }
    }
  } else if (warp == 2) {
    // ================================================================= TMA producer: packed query words
    int qs = 0;
    uint32_t qphase = 0;
    for (int64_t item = blockIdx.x; item < n_items; item += gridDim.x) {
      int mt, sp, kb_lo, kb_hi;
      item_of(item, mt, sp, kb_lo, kb_hi);
      const int nch = (kb_hi - kb_lo + KPC - 1) / KPC;
      for (int c = 0; c < nch; ++c) {
        mbar_wait(qempty_bar(qs), qphase ^ 1u);
        mbar_arrive_expect_tx_elect(qfull_bar(qs), TSQ_BYTES);
        tma_load_2d_elect(q_base + (uint32_t)qs * TSQ_BYTES, &tmQ, qfull_bar(qs), kb_lo * WPK + c * TSQ_WORDS, mt * BM);
        __syncwarp();
        if (++qs == TSQ_SLOTS) {
          qs = 0;
          qphase ^= 1u;
        }
      }
    }
  } else if (warp == 1) {
    // ================================================================= MMA issuer
    int grp = 0;
    uint32_t phase = 0;
    int acc = 0;
    uint32_t acc_phase = 0;
    // kind::f16 operand formats (bits 7..9 A, 10..12 B): 1 = bf16, 0 = IEEE half
    const uint32_t idesc = instr_desc<INT8>(BM, nb_rows) & ((!INT8 && p.f16) ? ~((1u << 7) | (1u << 10)) : ~0u);
    for (int64_t item = blockIdx.x; item < n_items; item += gridDim.x) {
      int mt, sp, kb_lo, kb_hi;
      item_of(item, mt, sp, kb_lo, kb_hi);
      mbar_wait(tempty_bar(acc), acc_phase ^ 1u);
      tc_fence_after();
      const uint32_t d_tmem = tmem_base + (uint32_t)(acc * p.acc_cols);
      for (int kb0 = kb_lo; kb0 < kb_hi; kb0 += G) {
        const int n = kb_hi - kb0 < G ? kb_hi - kb0 : G;
        mbar_wait(full_bar(grp), phase);
        tc_fence_after();
        const uint32_t sa = base + (uint32_t)(grp * G) * B_BYTES;
        const uint32_t b_lo = ((sa & 0x3FFFFu) >> 4) | (1u << 16);   // lower half of smem_desc(sa)
        const uint32_t at = tmem_base + (uint32_t)(A_COL0 + grp * G * 32);
        if (n == G) {
          tc_mma_ts_group_elect<INT8>(d_tmem, at, b_lo, (B_BYTES >> 4) - 6u, idesc, kb0 != kb_lo ? 1u : 0u);
        } else {
          for (int u = 0; u < n; ++u)
            tc_mma_ts_kblock_elect<INT8>(d_tmem, at + 32u * u, b_lo + (B_BYTES >> 4) * u, idesc,
                                         kb0 + u != kb_lo ? 1u : 0u);
        }
        tc_commit_elect<1>(empty_bar(grp));  // frees the group's class tiles and TMEM slots when these MMAs retire
        if (kb0 + n == kb_hi) tc_commit_elect<1>(tfull_bar(acc));
        __syncwarp();
        if (++grp == NG) {
          grp = 0;
          phase ^= 1u;
        }
      }
      if (++acc == p.acc_bufs) {
        acc = 0;
        acc_phase ^= 1u;
      }
    }
  } else if (warp >= 4 && warp < 8) {
    // ================================================================= epilogue (warps 4..7)
    const int q = warp & 3;
    int acc = 0;
    uint32_t acc_phase = 0;
    Top2f run = Top2f{NEG_BIG_F, NEG_BIG_F, 0.0f, 0.0f, INT_MAX, INT_MAX};
    const bool scaled = p.e.colscale != nullptr;
    for (int64_t item = blockIdx.x; item < n_items; item += gridDim.x) {
      int mt, sp, kb_lo, kb_hi;
      item_of(item, mt, sp, kb_lo, kb_hi);
      const int64_t row = (int64_t)mt * BM + q * 32 + lane;
      const bool row_ok = row < p.N;
      mbar_wait(tfull_bar(acc), acc_phase);
      tc_fence_after();
      const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)(acc * p.acc_cols);
      sim_epi_columns<INT8, EPI, true>(p, taddr, 0, 0, p.K, row, row_ok, sp, scaled, run);
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(tempty_bar(acc));
      if (++acc == p.acc_bufs) {
        acc = 0;
        acc_phase ^= 1u;
      }
      if (EPI == EPI_ARGMAX && p.splits == 1) sim_epi_finish<INT8>(p, row, row_ok, scaled, run);
    }
  } else if (warp >= 8) {
    // ================================================================= expanders (warps 8..15)
    const int q = warp & 3;            // TMEM lane quarter of this warp
    const int hsel = (warp - 8) >> 2;  // the two warps of a quarter take alternate 16-byte pieces of every row
    const int t = q * 32 + lane;       // row of the tile
    // row t of a query slot: 128 bytes, piece j at ((j ^ (t & 7)) << 4) (128-byte swizzle: conflict-free, lane = row)
    const uint32_t q_row = (uint32_t)t * 128u;
    const uint32_t sw = (uint32_t)(t & 7);
    const uint32_t one2 = p.f16 ? 0x3C003C00u : 0x3F803F80u;  // two +1.0 in half / bf16; the sign bit makes -1.0
    const uint32_t lane_base = tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)A_COL0;
    int grp = 0, qs = 0;
    uint32_t phase = 0, qphase = 0;
    // group hand-off of this warp: published with one fence and one arrival
    auto publish = [&]() {
      tmem_st_wait();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(full_bar(grp));
      if (++grp == NG) {
        grp = 0;
        phase ^= 1u;
      }
    };
    auto acquire = [&]() {
      mbar_wait(empty_bar(grp), phase ^ 1u);
      tc_fence_after();   // the MMAs that read these TMEM slots have retired (tcgen05.commit -> empty)
    };
    for (int64_t item = blockIdx.x; item < n_items; item += gridDim.x) {
      int mt, sp, kb_lo, kb_hi;
      item_of(item, mt, sp, kb_lo, kb_hi);
      const int nkb = kb_hi - kb_lo;
      const int ngr = (nkb + G - 1) / G;
      const int nch = (nkb + KPC - 1) / KPC;
      int cur_g = 0;   // group (of this item) whose TMEM slots this warp is filling
      acquire();
      for (int c = 0; c < nch; ++c) {
        mbar_wait(qfull_bar(qs), qphase);
        const uint32_t q_slot = q_base + (uint32_t)qs * TSQ_BYTES + q_row;
#pragma unroll
        for (int jj = 0; jj < 4; ++jj) {
          const int j = 2 * jj + hsel;               // piece of the chunk
          const int kb = (c * 8 + j) * KPP;          // its first k-block (relative to kb_lo)
          if (kb >= nkb) break;
          const int g = kb / G;
          while (cur_g < g) {                        // (a warp's pieces never skip a group: one step)
            publish();
            acquire();
            ++cur_g;
          }
          uint32_t w[4];
          asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];"
                       : "=r"(w[0]), "=r"(w[1]), "=r"(w[2]), "=r"(w[3])
                       : "r"(q_slot + ((((uint32_t)j) ^ sw) << 4))
                       : "memory");
          const uint32_t a_grp = lane_base + (uint32_t)(grp * G * 32);
          if (INT8) {
            // one k-block of 128 dimensions: 4 words -> 32 words of bytes -128 * bit (see sim_epi_columns)
            const uint32_t dst = a_grp + (uint32_t)((kb - g * G) * 32);
#pragma unroll
            for (int hh = 0; hh < 2; ++hh) {
              uint32_t o[16];
#pragma unroll
              for (int i = 0; i < 16; ++i) {
                const int iw = 16 * hh + i;
                o[i] = (w[iw >> 3] << (7 - (iw & 7))) & 0x80808080u;
              }
              tmem_st16(dst + 16u * hh, o);
            }
          } else {
            // two k-blocks of 64 dimensions: 2 words -> 32 words of +-1.0 pairs, each
#pragma unroll
            for (int kk = 0; kk < 2; ++kk) {
              if (kb + kk < nkb) {
                const uint32_t dst = a_grp + (uint32_t)((kb + kk - g * G) * 32);
#pragma unroll
                for (int hh = 0; hh < 2; ++hh) {
                  uint32_t o[16];
#pragma unroll
                  for (int i = 0; i < 16; ++i) o[i] = ((w[2 * kk + hh] << (15 - i)) & 0x80008000u) | one2;
                  tmem_st16(dst + 16u * hh, o);
                }
              }
            }
          }
        }
        __syncwarp();   // every lane holds its words in registers: the slot may be refilled
        if (lane == 0) mbar_arrive(qempty_bar(qs));
        if (++qs == TSQ_SLOTS) {
          qs = 0;
          qphase ^= 1u;
        }
      }
      // groups this warp has no piece in (the item's last k-blocks) still take its arrival
      while (cur_g < ngr - 1) {
        publish();
        acquire();
        ++cur_g;
      }
      publish();
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 1) {
    tc_fence_after();
    tmem_dealloc<1>(tmem_base, TMEM_COLS);
  }
}

template <bool INT8, int EPI>
cudaError_t launch_ts(const CUtensorMap& tmB, const CUtensorMap& tmQ, SimParams p, int grid, cudaStream_t st) {
  // per-device attribute of the function: set on every launch (handles on several devices of one process)
  cudaError_t e = cudaFuncSetAttribute(sim_ts_kernel<INT8, EPI>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                       SMEM_LIMIT);
  if (e != cudaSuccess) return e;
  const int nb_rows = p.nparts * p.kc;
  const int group_bytes = TSQ_G * nb_rows * KB_BYTES;
  // Two groups in flight beside two 128-column accumulators.  Measured alternatives: three groups with two
  // accumulators of 32 columns (K = 6 int8: 0.105 against 0.104 ms per 131072 queries), three groups with ONE
  // 128-column accumulator (K = 26 fp32: 0.234 against 0.218 ms; int16 0.171 against 0.130).
  p.ngroups = 2;
  p.acc_cols = TS_ACC_COLS;
  p.acc_bufs = 2;
  const int smem = p.ngroups * group_bytes + TSQ_SLOTS * TSQ_BYTES + SMEM_EXTRA;
  sim_ts_kernel<INT8, EPI><<<grid, TSQ_THREADS, smem, st>>>(tmB, tmQ, p);
  return cudaGetLastError();
}

template <bool INT8, int EPI, int CG, bool TS = false>
cudaError_t launch_cg(const CUtensorMap& tmB, const SimParams& p, int grid, cudaStream_t st) {
  // per-device attribute of the function: set on every launch (handles on several devices of one process)
  cudaError_t e = cudaFuncSetAttribute(sim_tc_kernel<INT8, EPI, CG, TS>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                       SMEM_LIMIT);
  if (e != cudaSuccess) return e;
  const int smem = p.stages * p.stage_bytes + SMEM_EXTRA + qring_bytes(CG);
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)grid);
  cfg.blockDim = dim3(NTHREADS);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeClusterDimension;
  at[0].val.clusterDim.x = CG;
  at[0].val.clusterDim.y = 1;
  at[0].val.clusterDim.z = 1;
  cfg.attrs = at;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, sim_tc_kernel<INT8, EPI, CG, TS>, tmB, p);
}
template <bool INT8, int EPI>
cudaError_t launch_one(const CUtensorMap& tmB, const CUtensorMap* tmQ, const SimParams& p, int cg, bool ts, int grid,
                       cudaStream_t st) {
  if (ts && tmQ) return launch_ts<INT8, EPI>(tmB, *tmQ, p, grid, st);
  if (ts) return launch_cg<INT8, EPI, 1, true>(tmB, p, grid, st);
  return cg == 2 ? launch_cg<INT8, EPI, 2>(tmB, p, grid, st) : launch_cg<INT8, EPI, 1>(tmB, p, grid, st);
}

void sim_tc_shape(int K, int hv_bits, int D_eff, int& kc, int& nparts, int& n_tiles, int& num_kb, bool& int8) {
  int8 = hv_bits == 8 || hv_bits == 1 || hv_bits == HDC_HV_I16;
  nparts = (hv_bits == 32 || hv_bits == HDC_HV_I16) ? 3 : 1;
  const int kc_max = nparts == 3 ? 80 : 256;
  kc = (K + 15) & ~15;
  if (kc > kc_max) kc = kc_max;
  n_tiles = (K + kc - 1) / kc;
  const int BK = int8 ? 128 : 64;
  num_kb = (D_eff + BK - 1) / BK;
}

}  // namespace

size_t sim_tc_operand_bytes(int K, int hv_bits, int D_eff) {
  int kc, nparts, n_tiles, num_kb;
  bool int8;
  sim_tc_shape(K, hv_bits, D_eff, kc, nparts, n_tiles, num_kb, int8);
  // staged rows (a multiple of 128 bytes), then for the int8 kinds one int32 sum per staged row
  return (size_t)n_tiles * nparts * kc * num_kb * KB_BYTES + (int8 ? (size_t)n_tiles * nparts * kc * 4 : 0);
}

// Split-D for small N: with fewer m-tiles than half the SMs, `splits` CTAs share an m-tile, each
// reducing kbs k-blocks (a multiple of 16, so that splits start on ring-chunk boundaries); their
// partial sums go through a [splits][K][N] fp32 buffer (integer class operands: only while every score stays
// below 2^24, i.e. exact in fp32).  Returns 1 when not worth it.
int sim_tc_splits(int64_t N, int K, int hv_bits, int D_eff, int sm_count, int* kbs_out) {
  int kc, nparts, n_tiles, num_kb;
  bool int8;
  sim_tc_shape(K, hv_bits, D_eff, kc, nparts, n_tiles, num_kb, int8);
  const int64_t m_tiles = (N + BM - 1) / BM;
  int splits = 1, kbs = num_kb;
  const bool exact_ok = !int8 || (int64_t)D_eff * 3 * (hv_bits == 8 ? 127 : (hv_bits == 1 ? 1 : 32767)) < (1 << 24);   // (small tiles: row sum + 2 x the split's share)
  if (n_tiles == 1 && m_tiles * 2 <= sm_count && num_kb >= 32 && exact_ok) {
    int want = (int)(sm_count / m_tiles);
    if (want > 8) want = 8;
    if (want > num_kb / 16) want = num_kb / 16;
    if (want >= 2 && (size_t)want * (size_t)N * K * sizeof(double) <= ((size_t)64 << 20)) {
      kbs = (int)round_up((num_kb + want - 1) / want, 16);
      splits = (num_kb + kbs - 1) / kbs;
      if (splits < 2) {
        splits = 1;
        kbs = num_kb;
      }
    }
  }
  if (kbs_out) *kbs_out = kbs;
  return splits;
}
size_t sim_tc_partial_bytes(int64_t N, int K, int hv_bits, int D_eff, int sm_count) {
  const int splits = sim_tc_splits(N, K, hv_bits, D_eff, sm_count, nullptr);
  return splits > 1 ? (size_t)splits * (size_t)N * K * sizeof(double) : 0;
}

cudaError_t launch_sim_tc(TcContext* tc, const uint32_t* Hbits, int64_t N, int64_t ldh, const float* C_acc,
                          int K, int64_t ldc, int D_eff, int hv_bits, void* cop, float* amax_scratch,
                          const Epilogue& e, Perf pf, double* partial, bool cop_ready, bool prep_only, int sm_count,
                          int force_cg, cudaStream_t st, int64_t* nlaunch, int piece, int width, int* live) {
  if (!tc) return cudaErrorNotSupported;
  if (N <= 0 && !prep_only) return cudaSuccess;
  if ((reinterpret_cast<uintptr_t>(cop) & 15) != 0) return cudaErrorNotSupported;
  int kc, nparts, n_tiles, num_kb;
  bool int8;
  sim_tc_shape(K, hv_bits, D_eff, kc, nparts, n_tiles, num_kb, int8);
  const int rows_total = n_tiles * nparts * kc;
  const int BK = int8 ? 128 : 64;
  const int64_t ld = (int64_t)num_kb * BK;
  cudaError_t ce;
  if ((hv_bits == 8 || (hv_bits == HDC_HV_I16 && piece == 0)) && !cop_ready) {
    ce = launch_tensor_amax(C_acc, K, D_eff, ldc, pf, amax_scratch, st, nlaunch);
    if (ce != cudaSuccess) return ce;
  }
  int32_t* rowsum = int8 ? reinterpret_cast<int32_t*>(static_cast<char*>(cop) + (size_t)rows_total * ld) : nullptr;
  if (!cop_ready) {
    const int n_vis = perf_count(pf, D_eff);
    // (the scales are the caller's e.colscale / e.colscale_f: written here, read by the kernels below)
    double* cs = const_cast<double*>(e.colscale);
    float* csf = const_cast<float*>(e.colscale_f);
    if (int8)
      class_prepare_kernel<true><<<(unsigned)(n_tiles * kc), CP_THREADS, 0, st>>>(C_acc, K, D_eff, ldc, hv_bits, kc, nparts, num_kb,
                                                                          amax_scratch, pf, n_vis, cop, rowsum, cs, csf, piece, width, live);
    else
      class_prepare_kernel<false><<<(unsigned)(n_tiles * kc), CP_THREADS, 0, st>>>(C_acc, K, D_eff, ldc, hv_bits, kc, nparts,
                                                                           num_kb, amax_scratch, pf, n_vis, cop, nullptr, cs,
                                                                           csf, 0, 0, nullptr);
    ++*nlaunch;
    ce = cudaGetLastError();
    if (ce != cudaSuccess) return ce;
  }
  if (prep_only) return cudaSuccess;
  // CTA pairs once every pair has a 256-query tile of its own and the class tile is wide enough for the
  // shared-memory traffic to matter: K >= 128, or the three-part fp32 class operand (measured at K = 26: 0.338 ->
  // 0.294 ms per 131072 queries; bf16 / int8 classes at small K are bound by the expansion itself and lose 5-15 %)
  int cg = (sm_count >= 2 && (K >= 128 || nparts == 3) && (N + 2 * BM - 1) / (2 * BM) >= sm_count / 2) ? 2 : 1;
  if (force_cg == 1 || (force_cg == 2 && sm_count >= 2)) cg = force_cg;
  // class tiles of <= 128 rows: the one-CTA kernel with the query tile in tensor memory (unless pairs are forced)
  const bool ts = nparts * kc <= TS_ACC_COLS && force_cg != 2;
  if (ts) cg = 1;
  CUtensorMap tmB;
  if (!tc_make_map(tc, &tmB, cop, int8, rows_total, ld, ld, nparts * kc / cg)) return cudaErrorInvalidValue;
  // small tiles with 16-byte aligned query rows: the packed words by TMA (sim_ts_kernel)
  CUtensorMap tmQ;
  const CUtensorMap* tq = nullptr;
  if (ts && (ldh & 3) == 0 && (reinterpret_cast<uintptr_t>(Hbits) & 15) == 0) {
    if (!tc_make_map_words(tc, &tmQ, Hbits, N, words_of(D_eff), ldh)) return cudaErrorInvalidValue;
    tq = &tmQ;
  }
  SimParams p;
  p.Hbits = Hbits;
  p.N = N;
  p.ldh = ldh;
  p.W = words_of(D_eff);
  p.K = K;
  p.kc = kc;
  p.nparts = nparts;
  p.m_tiles = (int)((N + BM * cg - 1) / (BM * cg));
  p.n_tiles = n_tiles;
  p.num_kb = num_kb;
  p.f16 = hv_bits == HDC_HV_F16;
  p.rowsum = rowsum;
  p.live = live;
  p.stage_bytes = (ts ? 0 : A_BYTES) + nparts * kc / cg * KB_BYTES;
  p.stages = (SMEM_LIMIT - SMEM_EXTRA - qring_bytes(cg)) / p.stage_bytes;
  if (p.stages > MAX_STAGES) p.stages = MAX_STAGES;
  if (ts && p.stages > TS_STAGES) p.stages = TS_STAGES;
  // k-blocks per pipeline group: every hand-off through the full / empty barriers costs several hundred
  // cycles whatever the k-block holds, so short k-blocks (few class rows) travel in groups
  p.kps = p.stages >= 8 ? 4 : (p.stages >= 4 ? 2 : 1);   // (divides the k-blocks of a ring tile: 16 / 8 / 4)
  p.stages -= p.stages % p.kps;
  p.e = e;
  p.splits = (partial && cg == 1) ? sim_tc_splits(N, K, hv_bits, D_eff, sm_count, &p.kbs) : 1;
  if (p.splits == 1) p.kbs = num_kb;
  p.partial = reinterpret_cast<float*>(partial);
  const int64_t items = (int64_t)p.m_tiles * p.splits;
  const int max_units = sm_count / cg;
  const int grid = (int)(items < max_units ? items : max_units) * cg;
  ++*nlaunch;
  if (p.splits > 1) {
    ce = int8 ? launch_one<true, EPI_SCORE>(tmB, tq, p, 1, ts, grid, st)
              : launch_one<false, EPI_SCORE>(tmB, tq, p, 1, ts, grid, st);
    if (ce != cudaSuccess) return ce;
    const unsigned rg = (unsigned)((N + 63) / 64);
    if (p.splits <= 2) split_reduce_kernel<2><<<rg, 64, 0, st>>>(p.partial, p.splits, N, K, e);
    else if (p.splits <= 4) split_reduce_kernel<4><<<rg, 64, 0, st>>>(p.partial, p.splits, N, K, e);
    else split_reduce_kernel<8><<<rg, 64, 0, st>>>(p.partial, p.splits, N, K, e);
    ++*nlaunch;
    return cudaGetLastError();
  }
  if (int8)
    return e.kind == EPI_SCORE ? launch_one<true, EPI_SCORE>(tmB, tq, p, cg, ts, grid, st)
                               : launch_one<true, EPI_ARGMAX>(tmB, tq, p, cg, ts, grid, st);
  return e.kind == EPI_SCORE ? launch_one<false, EPI_SCORE>(tmB, tq, p, cg, ts, grid, st)
                             : launch_one<false, EPI_ARGMAX>(tmB, tq, p, cg, ts, grid, st);
}

}  // namespace hdc
