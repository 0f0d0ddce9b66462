// adc.cu -- chunked, ADC-quantised dot-product similarity of the SpecPCM simulator (PAPER.md L273:
// "The SpecPCM simulator computes dot-product similarity over 128-element array chunks, with each
// partial dot product quantized by the ADC before accumulation"; knobs ADC_RES, ADC_STEP, ADC_FLOOR,
// ADC_CEIL; MLC = 1: +-1 hypervectors; reading A19 for the transfer function).
//
//   s[n,k] = sum_j adc( sum_{d in chunk j} v[n,d] * c[k,d] ),   chunk j = [128 j, 128 (j+1)) /\ [0, D_eff)
//
// With bipolar operands a chunk's partial dot is n_j - 2 * popc(q ^ c) over its 128 (last chunk:
// n_tail) bits, so the ADC is a table indexed by the popcount: 129 entries for full chunks, a second
// table for the ragged last chunk.  Lanes of a warp hold classes, the warp walks the chunks of one
// query: the query chunk is a shared-memory broadcast, the class chunks are one coalesced 16-byte
// load per lane from the [chunk][class] layout (L1-resident: K*W words), 4 XOR + 4 POPC + one table
// read per (query, class, chunk).  POPC-pipe bound like the Hamming kernel; no carry-save tree here
// because every 128-bit chunk needs its own count.
#include "common.cuh"

namespace hdc {
namespace {

constexpr int ADC_WARPS = 8;

// One thread per output word: bits of class k, dims [32 w, 32 w + 32) /\ [0, D_eff), bit = [C_acc < 0].
// Layout out[(w >> 2) * K + k] (uint4), component w & 3; words beyond W are zero.
__global__ void adc_class_kernel(const float* __restrict__ C, int K, int D_eff, int64_t ldc,
                                 uint32_t* __restrict__ out, int nch) {
  const int64_t total = (int64_t)nch * 4 * K;
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < total;
       i += (int64_t)gridDim.x * blockDim.x) {
    const int w = (int)(i / K);
    const int k = (int)(i - (int64_t)w * K);
    uint32_t bits = 0;
#pragma unroll 8
    for (int b = 0; b < 32; ++b) {
      const int d = w * 32 + b;
      if (d < D_eff && __ldg(C + (int64_t)k * ldc + d) < 0.0f) bits |= 1u << b;
    }
    out[((int64_t)(w >> 2) * K + k) * 4 + (w & 3)] = bits;
  }
}

__global__ void __launch_bounds__(ADC_WARPS * 32)
adc_sim_kernel(const uint32_t* __restrict__ H, int64_t N, int64_t ldh, const uint4* __restrict__ C4, int K,
               int nch, int W, uint32_t last_word_mask, AdcTables tab,
               int32_t* __restrict__ S, int64_t lds, int32_t* __restrict__ labels) {
  extern __shared__ __align__(16) uint32_t smem[];
  int* lutF = reinterpret_cast<int*>(smem);            // [129] full chunk
  int* lutT = lutF + 132;                              // [129] last chunk
  uint32_t* sQ = smem + 264;                           // [ADC_WARPS][nch * 4]
  for (int i = threadIdx.x; i < 129; i += blockDim.x) {
    lutF[i] = tab.full[i];
    lutT[i] = tab.tail[i];
  }
  __syncthreads();
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  uint32_t* q = sQ + (size_t)warp * nch * 4;
  const uint4* q4 = reinterpret_cast<const uint4*>(q);
  for (int64_t n = (int64_t)blockIdx.x * ADC_WARPS + warp; n < N; n += (int64_t)gridDim.x * ADC_WARPS) {
    __syncwarp();
    for (int w = lane; w < nch * 4; w += 32) {
      uint32_t v = w < W ? __ldg(H + n * ldh + w) : 0u;
      if (w == W - 1) v &= last_word_mask;
      q[w] = v;
    }
    __syncwarp();
    int best = INT_MIN, best_k = 0;
    for (int k0 = 0; k0 < K; k0 += 32) {
      const int k = k0 + lane;
      const bool on = k < K;
      const uint4* cp = C4 + (on ? k : 0);
      int acc = 0;
#pragma unroll 2
      for (int c = 0; c < nch - 1; ++c) {
        const uint4 a = q4[c];
        const uint4 b = __ldg(cp + (int64_t)c * K);
        const int diff = __popc(a.x ^ b.x) + __popc(a.y ^ b.y) + __popc(a.z ^ b.z) + __popc(a.w ^ b.w);
        acc += lutF[diff];
      }
      {
        const int c = nch - 1;
        const uint4 a = q4[c];
        const uint4 b = __ldg(cp + (int64_t)c * K);
        const int diff = __popc(a.x ^ b.x) + __popc(a.y ^ b.y) + __popc(a.z ^ b.z) + __popc(a.w ^ b.w);
        acc += lutT[diff];
      }
      if (on) {
        if (S) S[n * lds + k] = acc;
        if (acc > best) {  // k ascends within a lane: strict > keeps the lowest index
          best = acc;
          best_k = k;
        }
      }
    }
    if (labels) {
#pragma unroll
      for (int off = 16; off; off >>= 1) {
        const int ob = __shfl_xor_sync(0xffffffffu, best, off);
        const int ok = __shfl_xor_sync(0xffffffffu, best_k, off);
        if (ob > best || (ob == best && ok < best_k)) {
          best = ob;
          best_k = ok;
        }
      }
      if (lane == 0) labels[n] = best_k;
    }
  }
}

}  // namespace

size_t adc_class_bytes(int K, int D_eff) { return (size_t)((D_eff + 127) / 128) * K * sizeof(uint4); }

cudaError_t launch_adc_similarity(const uint32_t* H, int64_t N, int64_t ldh, const float* C_acc, int K,
                                  int64_t ldc, int D_eff, const AdcTables& tab, uint32_t* class_ws, int32_t* S,
                                  int64_t lds, int32_t* labels, int sm_count, int smem_optin, cudaStream_t st,
                                  int64_t* nlaunch) {
  const int W = (D_eff + 31) / 32;
  const int nch = (D_eff + 127) / 128;
  const size_t smem = (size_t)(264 + ADC_WARPS * nch * 4) * sizeof(uint32_t);
  if (smem > (size_t)smem_optin) return cudaErrorNotSupported;
  {
    const int64_t total = (int64_t)nch * 4 * K;
    int64_t g = (total + 255) / 256;
    if (g > sm_count * 16) g = sm_count * 16;
    adc_class_kernel<<<(int)g, 256, 0, st>>>(C_acc, K, D_eff, ldc, class_ws, nch);
    ++*nlaunch;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
  }
  if (smem > 48 * 1024) {
    cudaError_t e = cudaFuncSetAttribute(adc_sim_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin);
    if (e != cudaSuccess) return e;
  }
  int64_t blocks = (N + ADC_WARPS - 1) / ADC_WARPS;
  const int64_t cap = (int64_t)sm_count * 8;
  if (blocks > cap) blocks = cap;
  const uint32_t last_mask = (D_eff & 31) ? ((1u << (D_eff & 31)) - 1u) : 0xffffffffu;
  adc_sim_kernel<<<(int)blocks, ADC_WARPS * 32, smem, st>>>(H, N, ldh, reinterpret_cast<const uint4*>(class_ws), K,
                                                           nch, W, last_mask, tab, S, lds, labels);
  ++*nlaunch;
  return cudaGetLastError();
}

}  // namespace hdc
