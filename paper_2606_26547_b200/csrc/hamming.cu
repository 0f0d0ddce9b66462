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

template <int KC>
__global__ void __launch_bounds__(QT)
hamming_kernel(const uint32_t* __restrict__ Hbits, int64_t N, int64_t ldh,
               const uint32_t* __restrict__ Cbits, int K, int W, int D_eff,
               int32_t* __restrict__ dist, int64_t lds, int32_t* __restrict__ labels,
               float* __restrict__ best, float* __restrict__ second) {
  __shared__ uint32_t hq[WC][QT + 1];
  __shared__ __align__(16) uint32_t cs[KC][WC];
  const int tid = threadIdx.x;
  const int lane = tid & 31, warp = tid >> 5;
  const uint32_t tail_mask = (D_eff & 31) ? ((1u << (D_eff & 31)) - 1u) : 0xffffffffu;
  const int nchunks = (W + WC - 1) / WC;

  for (int64_t q0 = (int64_t)blockIdx.x * QT; q0 < N; q0 += (int64_t)gridDim.x * QT) {
    const int64_t n = q0 + tid;
    int b1 = INT_MAX, i1 = INT_MAX, b2 = INT_MAX;
    for (int k0 = 0; k0 < K; k0 += KC) {
      int acc[KC];
#pragma unroll
      for (int k = 0; k < KC; ++k) acc[k] = 0;
      for (int ch = 0; ch < nchunks; ++ch) {
        const int w0 = ch * WC;
        __syncthreads();  // previous chunk fully consumed
        // queries: each warp stages QT/4 rows, one coalesced 128-byte read per row
        {
          const int w = w0 + lane;
          const bool w_ok = w < W;
          const uint32_t m = (w == W - 1) ? tail_mask : 0xffffffffu;
#pragma unroll 8
          for (int r = warp; r < QT; r += QT / 32) {
            const int64_t row = q0 + r;
            uint32_t v = 0;
            if (row < N && w_ok) v = __ldg(Hbits + row * ldh + w) & m;
            hq[lane][r] = v;
          }
        }
        // classes: KC rows of WC words
        for (int i = tid; i < KC * WC; i += QT) {
          const int k = i / WC, wl = i % WC;
          const int w = w0 + wl;
          uint32_t v = 0;
          if (k0 + k < K && w < W) {
            v = __ldg(Cbits + (int64_t)(k0 + k) * W + w);
            if (w == W - 1) v &= tail_mask;
          }
          cs[k][wl] = v;
        }
        __syncthreads();
#pragma unroll 1
        for (int w = 0; w < WC; w += 8) {
          uint32_t h[8];
#pragma unroll
          for (int i = 0; i < 8; ++i) h[i] = hq[w + i][tid];
#pragma unroll
          for (int k = 0; k < KC; ++k) {
            const uint4 ca = *reinterpret_cast<const uint4*>(&cs[k][w]);
            const uint4 cb = *reinterpret_cast<const uint4*>(&cs[k][w + 4]);
            uint32_t a1, s1, a2, s2, a3, ones, fours, twos;
            csa(a1, s1, h[0] ^ ca.x, h[1] ^ ca.y, h[2] ^ ca.z);
            csa(a2, s2, h[3] ^ ca.w, h[4] ^ cb.x, h[5] ^ cb.y);
            csa(a3, ones, s1, s2, h[6] ^ cb.z);
            csa(fours, twos, a1, a2, a3);
            acc[k] += (__popc(ones) + __popc(h[7] ^ cb.w)) + 2 * __popc(twos) + 4 * __popc(fours);
          }
        }
      }
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
      }
    }
    if (n < N && labels) {
      labels[n] = i1;
      if (b2 == INT_MAX) b2 = b1;  // K == 1
      if (best) best[n] = (float)b1;
      if (second) second[n] = (float)b2;
    }
  }
}

}  // namespace

bool hamming_smem_fits(int, int, int) { return true; }

cudaError_t launch_hamming(const uint32_t* Hbits, int64_t N, int64_t ldh, const uint32_t* Cbits, int K,
                           int W, int D_eff, int32_t* dist, int64_t lds, int32_t* labels, float* best,
                           float* second, int sm_count, int, cudaStream_t st, int64_t* nlaunch) {
  if (N <= 0) return cudaSuccess;
  int64_t tiles = (N + QT - 1) / QT;
  const int64_t cap = (int64_t)sm_count * 8;
  const int grid = (int)(tiles < cap ? tiles : cap);
#define HDC_HAM(KC_)                                                                                         \
  hamming_kernel<KC_><<<grid, QT, 0, st>>>(Hbits, N, ldh, Cbits, K, W, D_eff, dist, lds, labels, best, second)
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
  return cudaGetLastError();
}

}  // namespace hdc
