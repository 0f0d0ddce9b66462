// hamming.cu -- packed XOR + popcount similarity (Listing 1 L72-L74
// `__hetero_hdc_hamming_distance`, L161 "xor and popcount") with the arg-min (L79-L80) fused.
//
//   dist[n,k] = popcount( (h[n] xor c[k]) restricted to bits d < D_eff )
//
// Mapping: one thread owns one query and keeps the distances to a group of KC classes in
// registers (KC is a template parameter chosen from K, so no popcount is spent on classes that do
// not exist), so no cross-lane reduction is needed.  A CTA of QT threads stages a [WC words][QT
// queries] tile of query bits in shared memory (transposed, stride QT+1: conflict-free both ways)
// and the matching [KC][WC] tile of class bits, which every thread then reads as a broadcast
// (one 16-byte LDS feeds four words).  For K > KC the query tile is re-staged per class group (it
// comes from L2).
//
// Pipe balance (DESIGN.md kernel table): POPC issues on the XU pipe at 16 lanes/clk/SM, LOP3 on the
// ALU pipe at 64 lanes/clk/SM, so a plain XOR+POPC loop is XU-bound at 8 clk per word per warp.  A
// block of 8 words is therefore reduced Harley-Seal style: seven XORed words go through four
// carry-save adders (8 LOP3) into a ones / twos / fours word and the eighth is counted directly:
//   sum_{i<8} popc(x_i) = popc(ones) + 2 popc(twos) + 4 popc(fours) + popc(x_7)
// = 16 LOP3 (32 ALU clk) + 4 POPC (32 XU clk) per 8 words: both pipes level at 4 clk per word.
#include <limits.h>

#include "common.cuh"

namespace hdc {
namespace {

constexpr int QT = 128;  // queries per CTA == threads per CTA
constexpr int WC = 32;   // words per staged chunk
constexpr int KC_MAX = 32;

// carry-save adder: (hi, lo) = a + b + c per bit
__device__ __forceinline__ void csa(uint32_t& hi, uint32_t& lo, uint32_t a, uint32_t b, uint32_t c) {
  lo = a ^ b ^ c;
  hi = (a & b) | ((a ^ b) & c);
}

constexpr int NST = 2;                      // cp.async ring depth
constexpr int HQ_WORDS = WC * (QT + 1);     // transposed query tile, stride QT+1: conflict-free
__host__ __device__ constexpr int stage_words(int KC) { return HQ_WORDS + (KC + 1) * WC; }  // + mask row

__device__ __forceinline__ void cp_async4(uint32_t dst_smem, const void* src, bool ok) {
  // 4-byte asynchronous copy global -> shared; src-size 0 writes zeros (rows >= N, words >= W)
  asm volatile("cp.async.ca.shared.global [%0], [%1], 4, %2;" ::"r"(dst_smem), "l"(src), "r"(ok ? 4 : 0)
               : "memory");
}

// Work of a CTA = its query tiles (grid-stride) x class groups x chunks, flattened into steps; the
// query / class words of step s+2 are in flight (cp.async, no registers) while step s is counted.
// PERF: a mask row (the visited dimensions of a perforated reduction) travels with the
// class tile and is ANDed into every XORed word -- the AND folds into the same LOP3 as the XOR.
template <int KC, bool PERF>
__global__ void __launch_bounds__(QT)
hamming_kernel(const uint32_t* __restrict__ Hbits, int64_t N, int64_t ldh,
               const uint32_t* __restrict__ Cbits, int K, int W, int D_eff,
               const uint32_t* __restrict__ mask, int32_t* __restrict__ dist, int64_t lds, int32_t* __restrict__ labels,
               float* __restrict__ best, float* __restrict__ second) {
  extern __shared__ __align__(16) uint32_t sm[];
  constexpr int STW = stage_words(KC);
  const int tid = threadIdx.x;
  const int lane = tid & 31, warp = tid >> 5;
  const uint32_t tail_mask = (D_eff & 31) ? ((1u << (D_eff & 31)) - 1u) : 0xffffffffu;
  const int nchunks = (W + WC - 1) / WC;
  const int ngroups = (K + KC - 1) / KC;
  const int spt = ngroups * nchunks;  // steps per query tile
  const int64_t tiles = (N + QT - 1) / QT;
  const int64_t my_tiles = tiles > blockIdx.x ? (tiles - 1 - blockIdx.x) / gridDim.x + 1 : 0;
  const int64_t total = my_tiles * spt;
  const uint32_t sm_base = (uint32_t)__cvta_generic_to_shared(sm);

  // producer-side cursor (tile, class group, chunk, ring stage) advanced step by step: no divisions
  int64_t is_q0 = (int64_t)blockIdx.x * QT;
  int is_g = 0, is_ch = 0, is_st = 0;
  auto issue = [&]() {
    const int w0 = is_ch * WC, k0 = is_g * KC;
    const uint32_t st = sm_base + (uint32_t)(is_st * STW) * 4u;
    const int w = w0 + lane;
    const int64_t rows_left = N - is_q0;                    // rows of this tile that exist
    const int nrow = w < W ? (rows_left < QT ? (int)rows_left : QT) : 0;
    const uint32_t* src = Hbits + (is_q0 + warp) * ldh + w;
    uint32_t dst = st + (uint32_t)(lane * (QT + 1) + warp) * 4u;
#pragma unroll 8
    for (int rr = warp; rr < QT; rr += QT / 32) {
      const bool ok = rr < nrow;
      cp_async4(dst, ok ? src : Hbits, ok);
      src += (QT / 32) * ldh;
      dst += (QT / 32) * 4u;
    }
    for (int idx = tid; idx < KC * WC; idx += QT) {
      const int k = idx / WC, wl = idx % WC;
      const bool ok = k0 + k < K && w0 + wl < W;
      cp_async4(st + (uint32_t)(HQ_WORDS + idx) * 4u, ok ? Cbits + (int64_t)(k0 + k) * W + w0 + wl : Cbits, ok);
    }
    if (PERF && tid < WC) {
      const bool ok = w0 + tid < W;
      cp_async4(st + (uint32_t)(HQ_WORDS + KC * WC + tid) * 4u, ok ? mask + w0 + tid : mask, ok);
    }
    if (++is_st == NST) is_st = 0;
    if (++is_ch == nchunks) {
      is_ch = 0;
      if (++is_g == ngroups) {
        is_g = 0;
        is_q0 += (int64_t)gridDim.x * QT;
      }
    }
  };
  for (int s0 = 0; s0 < NST - 1; ++s0) {
    if (s0 < total) issue();
    asm volatile("cp.async.commit_group;" ::: "memory");
  }

  int acc[KC];
  int b1 = INT_MAX, i1 = INT_MAX, b2 = INT_MAX;
  int64_t i = 0;
  int g = 0, ch = 0, cs_st = 0;
  for (int64_t step = 0; step < total; ++step) {
    asm volatile("cp.async.wait_group %0;" ::"n"(NST - 2) : "memory");
    __syncthreads();  // step's words visible to all; everyone is done counting step-1
    if (step + NST - 1 < total) issue();
    asm volatile("cp.async.commit_group;" ::: "memory");

    uint32_t* hq = sm + cs_st * STW;
    const uint32_t* cs = hq + HQ_WORDS;
    const int w0 = ch * WC, k0 = g * KC;
    if (ch == 0) {
#pragma unroll
      for (int k = 0; k < KC; ++k) acc[k] = 0;
    }
    if (!PERF && w0 + WC >= W && tail_mask != 0xffffffffu)
      hq[(W - 1 - w0) * (QT + 1) + tid] &= tail_mask;  // own column (the perforation mask covers the tail)
#pragma unroll 1
    for (int w = 0; w < WC; w += 8) {
      uint32_t h[8];
#pragma unroll
      for (int j = 0; j < 8; ++j) h[j] = hq[(w + j) * (QT + 1) + tid];
      uint4 ma = make_uint4(~0u, ~0u, ~0u, ~0u), mb = ma;
      if (PERF) {
        ma = *reinterpret_cast<const uint4*>(&cs[KC * WC + w]);
        mb = *reinterpret_cast<const uint4*>(&cs[KC * WC + w + 4]);
      }
#pragma unroll
      for (int k = 0; k < KC; ++k) {
        const uint4 ca = *reinterpret_cast<const uint4*>(&cs[k * WC + w]);
        const uint4 cb = *reinterpret_cast<const uint4*>(&cs[k * WC + w + 4]);
        uint32_t a1, s1, a2, s2, a3, ones, fours, twos;
        csa(a1, s1, (h[0] ^ ca.x) & ma.x, (h[1] ^ ca.y) & ma.y, (h[2] ^ ca.z) & ma.z);
        csa(a2, s2, (h[3] ^ ca.w) & ma.w, (h[4] ^ cb.x) & mb.x, (h[5] ^ cb.y) & mb.y);
        csa(a3, ones, s1, s2, (h[6] ^ cb.z) & mb.z);
        csa(fours, twos, a1, a2, a3);
        acc[k] += (__popc(ones) + __popc((h[7] ^ cb.w) & mb.w)) + 2 * __popc(twos) + 4 * __popc(fours);
      }
    }
    if (ch == nchunks - 1) {
      const int64_t n = ((int64_t)blockIdx.x + i * gridDim.x) * QT + tid;
      if (n < N) {
        if (dist) {
#pragma unroll
          for (int k = 0; k < KC; ++k)
            if (k0 + k < K) dist[n * lds + k0 + k] = acc[k];
        }
#pragma unroll
        for (int k = 0; k < KC; ++k) {
          if (k0 + k < K) {
            const int v = acc[k];
            if (v < b1) {  // strict: ties keep the lower (earlier) class index
              b2 = b1;
              b1 = v;
              i1 = k0 + k;
            } else if (v < b2) {
              b2 = v;
            }
          }
        }
        if (g == ngroups - 1 && labels) {
          labels[n] = i1;
          if (b2 == INT_MAX) b2 = b1;  // K == 1
          if (best) best[n] = (float)b1;
          if (second) second[n] = (float)b2;
        }
      }
      if (g == ngroups - 1) {
        b1 = INT_MAX;
        i1 = INT_MAX;
        b2 = INT_MAX;
      }
    }
    if (++cs_st == NST) cs_st = 0;
    if (++ch == nchunks) {
      ch = 0;
      if (++g == ngroups) {
        g = 0;
        ++i;
      }
    }
  }
  asm volatile("cp.async.wait_group 0;" ::: "memory");
}

template <int KC, bool PERF>
cudaError_t launch_ham2(int grid, cudaStream_t st, const uint32_t* Hbits, int64_t N, int64_t ldh,
                        const uint32_t* Cbits, int K, int W, int D_eff, const uint32_t* mask, int32_t* dist,
                        int64_t lds, int32_t* labels, float* best, float* second) {
  constexpr int SMEM = NST * stage_words(KC) * 4;
  // per-device attribute of the function: set on every launch (handles on several devices of one process)
  cudaError_t e = cudaFuncSetAttribute(hamming_kernel<KC, PERF>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM);
  if (e != cudaSuccess) return e;
  hamming_kernel<KC, PERF><<<grid, QT, SMEM, st>>>(Hbits, N, ldh, Cbits, K, W, D_eff, mask, dist, lds, labels,
                                                   best, second);
  return cudaGetLastError();
}
template <int KC>
cudaError_t launch_ham(int grid, cudaStream_t st, const uint32_t* Hbits, int64_t N, int64_t ldh,
                       const uint32_t* Cbits, int K, int W, int D_eff, const uint32_t* mask, int32_t* dist,
                       int64_t lds, int32_t* labels, float* best, float* second) {
  if (mask)
    return launch_ham2<KC, true>(grid, st, Hbits, N, ldh, Cbits, K, W, D_eff, mask, dist, lds, labels, best, second);
  return launch_ham2<KC, false>(grid, st, Hbits, N, ldh, Cbits, K, W, D_eff, mask, dist, lds, labels, best, second);
}

}  // namespace


cudaError_t launch_hamming(const uint32_t* Hbits, int64_t N, int64_t ldh, const uint32_t* Cbits, int K,
                           int W, int D_eff, const uint32_t* mask, int32_t* dist, int64_t lds, int32_t* labels,
                           float* best, float* second, int sm_count, int, cudaStream_t st, int64_t* nlaunch) {
  if (N <= 0) return cudaSuccess;
  int64_t tiles = (N + QT - 1) / QT;
  const int64_t cap = (int64_t)sm_count * 64;  // one tile per CTA up to here: the block scheduler balances the SMs
  const int grid = (int)(tiles < cap ? tiles : cap);
  cudaError_t ce;
#define HDC_HAM(KC_) \
  ce = launch_ham<KC_>(grid, st, Hbits, N, ldh, Cbits, K, W, D_eff, mask, dist, lds, labels, best, second)
  // smallest register group that covers K in one pass; K > 32 walks groups of 32
  if (K <= 2) HDC_HAM(2);
  else if (K <= 4) HDC_HAM(4);
  else if (K <= 6) HDC_HAM(6);
  else if (K <= 8) HDC_HAM(8);
  else if (K <= 10) HDC_HAM(10);
  else if (K <= 12) HDC_HAM(12);
  else if (K <= 16) HDC_HAM(16);
  else if (K <= 20) HDC_HAM(20);
  else if (K <= 24) HDC_HAM(24);
  else if (K <= 28) HDC_HAM(28);
  else HDC_HAM(KC_MAX);
#undef HDC_HAM
  ++*nlaunch;
  return ce;
}

}  // namespace hdc
