// hamming.cu -- packed XOR + popcount similarity (Listing 1 L72-L74
// `__hetero_hdc_hamming_distance`, L161 "xor and popcount") with the arg-min (L79-L80) fused.
//
//   dist[n,k] = popcount( (h[n] xor c[k]) restricted to bits d < D_eff )
//
// Mapping: one thread owns one query and keeps the distances to a group of KC classes in
// registers, so no cross-lane reduction is needed.  A CTA of QT threads stages a [WC words][QT
// queries] tile of query bits in shared memory (transposed, stride QT+1: conflict-free both ways)
// and the matching [KC][WC] tile of class bits, which every thread then reads as a broadcast
// (one 16-byte LDS feeds four XOR+POPC).  For K > KC the query tile is re-staged per class group
// (it comes from L2; 32 popcounts are done per word staged).  The bound at K >= 3 is the POPC
// pipe, not HBM (kernel table).
#include <limits.h>

#include "common.cuh"

namespace hdc {
namespace {

constexpr int QT = 128;  // queries per CTA == threads per CTA
constexpr int WC = 32;   // words per staged chunk
constexpr int KC = 32;   // classes per register group

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
        for (int r = warp; r < QT; r += QT / 32) {
          const int64_t row = q0 + r;
          const int w = w0 + lane;
          uint32_t v = 0;
          if (row < N && w < W) {
            v = __ldg(Hbits + row * ldh + w);
            if (w == W - 1) v &= tail_mask;
          }
          hq[lane][r] = v;
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
#pragma unroll 2
        for (int w = 0; w < WC; w += 4) {
          const uint32_t h0 = hq[w][tid], h1 = hq[w + 1][tid], h2 = hq[w + 2][tid], h3 = hq[w + 3][tid];
#pragma unroll
          for (int k = 0; k < KC; ++k) {
            const uint4 c = *reinterpret_cast<const uint4*>(&cs[k][w]);
            acc[k] += (__popc(h0 ^ c.x) + __popc(h1 ^ c.y)) + (__popc(h2 ^ c.z) + __popc(h3 ^ c.w));
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
  hamming_kernel<<<grid, QT, 0, st>>>(Hbits, N, ldh, Cbits, K, W, D_eff, dist, lds, labels, best, second);
  ++*nlaunch;
  return cudaGetLastError();
}

}  // namespace hdc
