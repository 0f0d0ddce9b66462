// train.cu -- class-hypervector update ("vector addition" of same-class hypervectors;
// L181 TRAIN_ITERATIONS; perceptron-style rule = DESIGN.md reading S9/A9):
//
//   bundle      Delta[k,d] = sum_{n: y_n = k} v[n,d]
//   perceptron  Delta[k,d] = sum_{n: yhat_n != y_n} ([k = y_n] - [k = yhat_n]) * v[n,d]
//   then        C_acc[k,d] = fl32( C_acc[k,d] + fl32( lr * (float)Delta[k,d] ) )      (two rounded ops)
//
// with v = 1 - 2*bit.  Delta is an exact int32 segmented reduction per class: a CTA owns (class k,
// 128 word-columns, a segment of the samples); a thread owns one word-column and 32 signed counters
// in registers, walks the samples of its segment that touch class k (compacted through shared memory;
// word reads are coalesced) and finally adds its 32 partial sums into Delta with integer atomics -- integer
// addition commutes, so the result is deterministic; there are no floating-point atomics.
#include "common.cuh"

namespace hdc {
namespace {

constexpr int WT = 128;  // word-columns per CTA

constexpr int LCH = 1024;  // samples scanned per compaction round

__global__ void __launch_bounds__(WT)
class_delta_kernel(const uint32_t* __restrict__ Hbits, int64_t n0, int64_t nb, int64_t ldh,
                   const int32_t* __restrict__ y, const int32_t* __restrict__ pred, int W,
                   int32_t* __restrict__ delta, int64_t ldd, int64_t seg_len) {
  // Samples that touch class k are first compacted into shared memory (coalesced label reads, one
  // atomic per hit), then only those are walked: a CTA no longer pays two dependent label loads
  // for each of the (K-2)/K samples that do not concern its class.  The list order is arbitrary;
  // the sums are integers, so the result does not depend on it.
  __shared__ int s_list[LCH];  // (sample offset from c0) * 2 + (sign < 0)
  __shared__ int s_cnt;
  const int k = blockIdx.y;
  const int w = blockIdx.x * WT + threadIdx.x;
  const int64_t s0 = n0 + (int64_t)blockIdx.z * seg_len;
  int64_t s1 = s0 + seg_len;
  if (s1 > n0 + nb) s1 = n0 + nb;
  int cnt[32];
#pragma unroll
  for (int b = 0; b < 32; ++b) cnt[b] = 0;
  int m = 0;  // signed number of contributing samples
  for (int64_t c0 = s0; c0 < s1; c0 += LCH) {
    const int len = (int)(s1 - c0 < LCH ? s1 - c0 : LCH);
    if (threadIdx.x == 0) s_cnt = 0;
    __syncthreads();
    for (int i = threadIdx.x; i < len; i += WT) {
      const int yn = __ldg(y + c0 + i);
      int sg;
      if (pred) {
        const int pn = __ldg(pred + c0 + i);
        sg = (pn != yn) ? ((yn == k) - (pn == k)) : 0;
      } else {
        sg = (yn == k);
      }
      if (sg != 0) s_list[atomicAdd(&s_cnt, 1)] = i * 2 + (sg < 0);
    }
    __syncthreads();
    const int n_hit = s_cnt;
    const uint32_t* hcol = Hbits + c0 * ldh + (w < W ? w : 0);
#pragma unroll 4
    for (int j = 0; j < n_hit; ++j) {
      const int e = s_list[j];
      const int sg = 1 - 2 * (e & 1);
      const uint32_t word = (w < W) ? __ldg(hcol + (int64_t)(e >> 1) * ldh) : 0u;
      m += sg;
#pragma unroll
      for (int b = 0; b < 32; ++b) cnt[b] += sg * (int)((word >> b) & 1u);
    }
    __syncthreads();  // the list is rewritten in the next round
  }
  if (w < W) {
    int32_t* out = delta + (int64_t)k * ldd + (int64_t)w * 32;
#pragma unroll
    for (int b = 0; b < 32; ++b) {
      const int v = m - 2 * cnt[b];
      if (v != 0) atomicAdd(out + b, v);
    }
  }
}

__global__ void apply_update_kernel(float* __restrict__ C, int K, int D_eff, int64_t ldc,
                                    const int32_t* __restrict__ delta, int64_t ldd, float lr) {
  const int64_t total = (int64_t)K * D_eff;
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < total;
       i += (int64_t)gridDim.x * blockDim.x) {
    const int64_t k = i / D_eff;
    const int d = (int)(i - k * D_eff);
    const int dv = delta[k * ldd + d];
    if (dv != 0) {
      float* c = C + k * ldc + d;
      *c = __fadd_rn(*c, __fmul_rn(lr, (float)dv));
    }
  }
}

__global__ void count_wrong_kernel(const int32_t* __restrict__ y, const int32_t* __restrict__ pred,
                                   int64_t n0, int64_t nb, unsigned long long* __restrict__ n_wrong) {
  unsigned int c = 0;
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < nb;
       i += (int64_t)gridDim.x * blockDim.x)
    c += (y[n0 + i] != pred[n0 + i]);
#pragma unroll
  for (int off = 16; off; off >>= 1) c += __shfl_xor_sync(0xffffffffu, c, off);
  if ((threadIdx.x & 31) == 0 && c) atomicAdd(n_wrong, (unsigned long long)c);
}

// HD-Clustering (reading A16): members per cluster and, when the
// previous assignment is given, the number of samples that moved.
__global__ void assign_stats_kernel(const int32_t* __restrict__ assign, const int32_t* __restrict__ prev,
                                    int64_t N, int32_t* __restrict__ members,
                                    unsigned long long* __restrict__ n_changed) {
  unsigned int c = 0;
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < N;
       i += (int64_t)gridDim.x * blockDim.x) {
    const int a = assign[i];
    atomicAdd(members + a, 1);
    if (prev) c += (prev[i] != a);
  }
#pragma unroll
  for (int off = 16; off; off >>= 1) c += __shfl_xor_sync(0xffffffffu, c, off);
  if (n_changed && (threadIdx.x & 31) == 0 && c) atomicAdd(n_changed, (unsigned long long)c);
}

// clusters that received members are rebuilt from scratch; empty ones keep their accumulator
__global__ void zero_member_rows_kernel(float* __restrict__ C, int K, int D_eff, int64_t ldc,
                                        const int32_t* __restrict__ members) {
  const int64_t total = (int64_t)K * D_eff;
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < total;
       i += (int64_t)gridDim.x * blockDim.x) {
    const int64_t k = i / D_eff;
    if (members[k] > 0) C[k * ldc + (i - k * D_eff)] = 0.0f;
  }
}

}  // namespace

// members: int32 [K] workspace (zeroed here)
cudaError_t launch_kmeans_reset(const int32_t* assign, const int32_t* prev, int64_t N, float* C_acc, int K,
                                int64_t ldc, int D_eff, int32_t* members, unsigned long long* n_changed,
                                int sm_count, cudaStream_t st, int64_t* nlaunch) {
  cudaError_t e = cudaMemsetAsync(members, 0, sizeof(int32_t) * (size_t)K, st);
  if (e != cudaSuccess) return e;
  int64_t g = (N + 255) / 256;
  if (g > sm_count * 4) g = sm_count * 4;
  if (g < 1) g = 1;
  assign_stats_kernel<<<(unsigned)g, 256, 0, st>>>(assign, prev, N, members, n_changed);
  ++*nlaunch;
  e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  const int64_t total = (int64_t)K * D_eff;
  g = (total + 255) / 256;
  if (g > sm_count * 8) g = sm_count * 8;
  zero_member_rows_kernel<<<(unsigned)g, 256, 0, st>>>(C_acc, K, D_eff, ldc, members);
  ++*nlaunch;
  return cudaGetLastError();
}

// delta: int32 [K][W*32] (zeroed here, then filled): the exact integer class update of samples
// [n0, n0+nb); n_wrong (nullable) is incremented by the mispredictions among them.
cudaError_t launch_class_delta(const uint32_t* Hbits, int64_t n0, int64_t nb, int64_t ldh, const int32_t* y,
                               const int32_t* pred, int K, int D_eff, int32_t* delta,
                               unsigned long long* n_wrong, int sm_count, cudaStream_t st, int64_t* nlaunch) {
  const int W = words_of(D_eff);
  const int64_t ldd = (int64_t)W * 32;
  cudaError_t e = cudaMemsetAsync(delta, 0, sizeof(int32_t) * (size_t)K * ldd, st);
  if (e != cudaSuccess || nb <= 0) return e;
  const int gx = (W + WT - 1) / WT;
  // split the samples into segments so that about 4 CTAs per SM exist; each segment >= 64 samples
  int64_t segs = ((int64_t)sm_count * 4 + (int64_t)gx * K - 1) / ((int64_t)gx * K);
  const int64_t max_segs = (nb + 63) / 64;
  if (segs > max_segs) segs = max_segs;
  if (segs < 1) segs = 1;
  if (segs > 65535) segs = 65535;
  const int64_t seg_len = (nb + segs - 1) / segs;
  segs = (nb + seg_len - 1) / seg_len;
  if (K > 65535) return cudaErrorNotSupported;  // class index is blockIdx.y (checked by the API too)
  dim3 grid(gx, K, (unsigned)segs);
  class_delta_kernel<<<grid, WT, 0, st>>>(Hbits, n0, nb, ldh, y, pred, W, delta, ldd, seg_len);
  ++*nlaunch;
  e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  if (n_wrong && pred) {
    int64_t gw = (nb + 255) / 256;
    if (gw > sm_count * 4) gw = sm_count * 4;
    count_wrong_kernel<<<(unsigned)gw, 256, 0, st>>>(y, pred, n0, nb, n_wrong);
    ++*nlaunch;
    e = cudaGetLastError();
  }
  return e;
}

// C_acc[k,d] = fl32(C_acc[k,d] + fl32(lr * (float)delta[k,d])) for d < D_eff
cudaError_t launch_apply_update(float* C_acc, int K, int64_t ldc, int D_eff, const int32_t* delta, float lr,
                                int sm_count, cudaStream_t st, int64_t* nlaunch) {
  const int64_t ldd = (int64_t)words_of(D_eff) * 32;
  const int64_t total = (int64_t)K * D_eff;
  int64_t g = (total + 255) / 256;
  if (g > sm_count * 8) g = sm_count * 8;
  apply_update_kernel<<<(unsigned)g, 256, 0, st>>>(C_acc, K, D_eff, ldc, delta, ldd, lr);
  ++*nlaunch;
  return cudaGetLastError();
}

cudaError_t launch_class_update(const uint32_t* Hbits, int64_t n0, int64_t nb, int64_t ldh,
                                const int32_t* y, const int32_t* pred, float* C_acc, int K,
                                int64_t ldc, int D_eff, float lr, int32_t* delta,
                                unsigned long long* n_wrong, int sm_count, cudaStream_t st,
                                int64_t* nlaunch) {
  if (nb <= 0) return cudaSuccess;
  cudaError_t e = launch_class_delta(Hbits, n0, nb, ldh, y, pred, K, D_eff, delta, n_wrong, sm_count, st, nlaunch);
  if (e != cudaSuccess) return e;
  return launch_apply_update(C_acc, K, ldc, D_eff, delta, lr, sm_count, st, nlaunch);
}

}  // namespace hdc
