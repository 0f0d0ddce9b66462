// convert.cu -- operand preparation kernels ("element type representation"; DESIGN.md
// readings S1, S5, A7): fp32 -> bf16 staging, per-row / per-tensor symmetric int8 quantisation,
// sign bits of the class accumulators, cosine column scales.  All HBM-bound elementwise / row
// reductions; every rounding step is a single correctly rounded fp32 operation (__fdiv_rn,
// __fmul_rn, rintf) so that the integers produced are the ones the definition fixes.
#include "common.cuh"

namespace hdc {
namespace {

__device__ __forceinline__ float load_as_f32(const void* p, int kind, int64_t idx) {
  if (kind == OPK_BF16) return __bfloat162float(((const __nv_bfloat16*)p)[idx]);
  return __ldg((const float*)p + idx);
}

// ---------------------------------------------------------------------------------- bf16 staging
// One thread produces 8 consecutive bf16 (one 16-byte store); columns >= cols are zero.
__global__ void convert_bf16_kernel(const void* __restrict__ src, int src_kind, int64_t rows, int cols,
                                    int64_t ld_src, __nv_bfloat16* __restrict__ dst, int64_t ld_dst) {
  const int chunks = (int)(ld_dst >> 3);
  const int64_t total = rows * chunks;
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < total;
       i += (int64_t)gridDim.x * blockDim.x) {
    const int64_t r = i / chunks;
    const int c0 = (int)(i - r * chunks) << 3;
    __align__(16) __nv_bfloat16 v[8];
    const int64_t base = r * ld_src + c0;
    if (src_kind == OPK_F32 && c0 + 8 <= cols && ((ld_src & 3) == 0) &&
        ((reinterpret_cast<uintptr_t>(src) & 15) == 0)) {
      const float4 a = __ldg(reinterpret_cast<const float4*>((const float*)src + base));
      const float4 b = __ldg(reinterpret_cast<const float4*>((const float*)src + base) + 1);
      v[0] = __float2bfloat16_rn(a.x); v[1] = __float2bfloat16_rn(a.y);
      v[2] = __float2bfloat16_rn(a.z); v[3] = __float2bfloat16_rn(a.w);
      v[4] = __float2bfloat16_rn(b.x); v[5] = __float2bfloat16_rn(b.y);
      v[6] = __float2bfloat16_rn(b.z); v[7] = __float2bfloat16_rn(b.w);
    } else {
#pragma unroll
      for (int j = 0; j < 8; ++j)
        v[j] = (c0 + j < cols) ? __float2bfloat16_rn(load_as_f32(src, src_kind, base + j))
                               : __float2bfloat16_rn(0.0f);
    }
    *reinterpret_cast<uint4*>(dst + r * ld_dst + c0) = *reinterpret_cast<const uint4*>(v);
  }
}

// ---------------------------------------------------------------------------------- fp16 staging
// Same layout as convert_bf16_kernel with IEEE half RNE (precision HDC_F16).
__global__ void convert_f16_kernel(const void* __restrict__ src, int src_kind, int64_t rows, int cols,
                                   int64_t ld_src, __half* __restrict__ dst, int64_t ld_dst) {
  const int chunks = (int)(ld_dst >> 3);
  const int64_t total = rows * chunks;
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < total;
       i += (int64_t)gridDim.x * blockDim.x) {
    const int64_t r = i / chunks;
    const int c0 = (int)(i - r * chunks) << 3;
    __align__(16) __half v[8];
    const int64_t base = r * ld_src + c0;
#pragma unroll
    for (int j = 0; j < 8; ++j)
      v[j] = __float2half_rn((c0 + j < cols) ? load_as_f32(src, src_kind, base + j) : 0.0f);
    *reinterpret_cast<uint4*>(dst + r * ld_dst + c0) = *reinterpret_cast<const uint4*>(v);
  }
}

// ---------------------------------------------------------------------------------- bf16 x3 split
// x = x1 + x2 + x3 (+ O(2^-25 |x|)): x1 = bf16(x), x2 = bf16(x - x1), x3 = bf16(x - x1 - x2); both
// residuals are exact fp32 subtractions.  dst [rows][3*seg]: segment s holds x_{s+1}; columns >=
// cols of every segment are zero.  One thread = 8 consecutive columns of all three segments.
__global__ void split3_bf16_kernel(const void* __restrict__ src, int src_kind, int64_t rows, int cols,
                                   int64_t ld_src, __nv_bfloat16* __restrict__ dst, int seg) {
  const int chunks = seg >> 3;
  const int64_t total = rows * chunks;
  const bool vec = src_kind == OPK_F32 && ((ld_src & 3) == 0) && ((reinterpret_cast<uintptr_t>(src) & 15) == 0);
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < total;
       i += (int64_t)gridDim.x * blockDim.x) {
    const int64_t r = i / chunks;
    const int c0 = (int)(i - r * chunks) << 3;
    float x[8];
    const int64_t base = r * ld_src + c0;
    if (vec && c0 + 8 <= cols) {
      const float4 a = __ldg(reinterpret_cast<const float4*>((const float*)src + base));
      const float4 b = __ldg(reinterpret_cast<const float4*>((const float*)src + base) + 1);
      x[0] = a.x; x[1] = a.y; x[2] = a.z; x[3] = a.w;
      x[4] = b.x; x[5] = b.y; x[6] = b.z; x[7] = b.w;
    } else {
#pragma unroll
      for (int j = 0; j < 8; ++j) x[j] = (c0 + j < cols) ? load_as_f32(src, src_kind, base + j) : 0.0f;
    }
    __align__(16) __nv_bfloat16 v1[8], v2[8], v3[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) {
      v1[j] = __float2bfloat16_rn(x[j]);
      const float r1 = __fsub_rn(x[j], __bfloat162float(v1[j]));
      v2[j] = __float2bfloat16_rn(r1);
      const float r2 = __fsub_rn(r1, __bfloat162float(v2[j]));
      v3[j] = __float2bfloat16_rn(r2);
    }
    __nv_bfloat16* o = dst + r * (int64_t)(3 * seg) + c0;
    *reinterpret_cast<uint4*>(o) = *reinterpret_cast<const uint4*>(v1);
    *reinterpret_cast<uint4*>(o + seg) = *reinterpret_cast<const uint4*>(v2);
    *reinterpret_cast<uint4*>(o + 2 * seg) = *reinterpret_cast<const uint4*>(v3);
  }
}

// ---------------------------------------------------------------------------------- fp16 x2 split
// HDC_FLAG_F32_FAST: x * 2^e = h1 + h2 (+ O(2^-22 |x|)), h1 = half(x 2^e), h2 = half(x 2^e - h1), with the
// per-row exponent e chosen so that the row maximum lands in [2^14, 2^15): every element within 2^-18
// of the row maximum keeps 22 mantissa bits, smaller ones are held to 2^-25 absolute (half subnormals),
// i.e. 2^-40 of the row maximum.  Power-of-two row scales change no sign and are undone exactly on
// the optional raw accumulators.  dst [rows][2*seg]: segment 0 = h1, segment 1 = h2; columns >= cols
// are zero.  One warp per row.
__global__ void split2_f16_rows_kernel(const void* __restrict__ src, int src_kind, int64_t rows, int cols,
                                       int64_t ld_src, __half* __restrict__ dst, int seg,
                                       int* __restrict__ expo) {
  const int lane = threadIdx.x & 31;
  const int64_t warp = (blockIdx.x * (int64_t)blockDim.x + threadIdx.x) >> 5;
  const int64_t nwarps = ((int64_t)gridDim.x * blockDim.x) >> 5;
  for (int64_t r = warp; r < rows; r += nwarps) {
    float a = 0.0f;
    for (int c = lane; c < cols; c += 32) a = fmaxf(a, fabsf(load_as_f32(src, src_kind, r * ld_src + c)));
#pragma unroll
    for (int off = 16; off; off >>= 1) a = fmaxf(a, __shfl_xor_sync(0xffffffffu, a, off));
    const int e = a > 0.0f ? 14 - ilogbf(a) : 0;
    if (lane == 0) expo[r] = e;
    __half* o = dst + r * (int64_t)(2 * seg);
    for (int c0 = lane * 8; c0 < seg; c0 += 256) {  // seg is a multiple of 64: whole 16-byte stores
      __align__(16) __half v1[8], v2[8];
#pragma unroll
      for (int j = 0; j < 8; ++j) {
        float xs = 0.0f;
        if (c0 + j < cols) xs = scalbnf(load_as_f32(src, src_kind, r * ld_src + c0 + j), e);
        v1[j] = __float2half_rn(xs);
        v2[j] = __float2half_rn(__fsub_rn(xs, __half2float(v1[j])));
      }
      *reinterpret_cast<uint4*>(o + c0) = *reinterpret_cast<const uint4*>(v1);
      *reinterpret_cast<uint4*>(o + seg + c0) = *reinterpret_cast<const uint4*>(v2);
    }
  }
}

// raw[n,d] = raw[n,d] * 2^-(ex[n] + ep[d])   (exact)
__global__ void unscale_raw_kernel(float* __restrict__ raw, int64_t rows, int cols, int64_t ld,
                                   const int* __restrict__ ex, const int* __restrict__ ep) {
  const int64_t total = rows * cols;
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < total;
       i += (int64_t)gridDim.x * blockDim.x) {
    const int64_t r = i / cols;
    const int d = (int)(i - r * cols);
    raw[r * ld + d] = scalbnf(raw[r * ld + d], -(ex[r] + ep[d]));
  }
}

// ---------------------------------------------------------------------------------- int8 per row
__device__ __forceinline__ int quant_i8(float x, float s) {
  float q = rintf(__fmul_rn(x, s));  // round-half-even, one rounded multiply (no FMA contraction)
  q = fminf(fmaxf(q, -127.0f), 127.0f);
  return (int)q;
}

// One warp per row: a = max|x|, s = fl32(127/a) (1 if a == 0), q = clamp(rint(fl32(x*s)), +-127).
__global__ void quantize_rows_i8_kernel(const void* __restrict__ src, int src_kind, int64_t rows, int cols,
                                        int64_t ld_src, int8_t* __restrict__ dst, int64_t ld_dst) {
  const int lane = threadIdx.x & 31;
  const int64_t warp = (blockIdx.x * (int64_t)blockDim.x + threadIdx.x) >> 5;
  const int64_t nwarps = ((int64_t)gridDim.x * blockDim.x) >> 5;
  for (int64_t r = warp; r < rows; r += nwarps) {
    float a = 0.0f;
    for (int c = lane; c < cols; c += 32) a = fmaxf(a, fabsf(load_as_f32(src, src_kind, r * ld_src + c)));
#pragma unroll
    for (int off = 16; off; off >>= 1) a = fmaxf(a, __shfl_xor_sync(0xffffffffu, a, off));
    const float s = a > 0.0f ? __fdiv_rn(127.0f, a) : 1.0f;
    for (int c = lane; c < (int)ld_dst; c += 32) {
      int q = 0;
      if (c < cols) q = quant_i8(load_as_f32(src, src_kind, r * ld_src + c), s);
      dst[r * ld_dst + c] = (int8_t)q;
    }
  }
}

// ---------------------------------------------------------------------------------- int8 per tensor
// max |C[k][d]| over k < K, d < D_eff; non-negative floats order as unsigned ints.
__global__ void tensor_amax_kernel(const float* __restrict__ C, int K, int D_eff, int64_t ldc, Perf pf,
                                   float* __restrict__ amax) {
  // blockIdx.y = class row, blockIdx.x = slice of its columns (no division per element)
  const float* row = C + (int64_t)blockIdx.y * ldc;
  float a = 0.0f;
  for (int d = blockIdx.x * blockDim.x + threadIdx.x; d < D_eff; d += gridDim.x * blockDim.x)
    if (perf_visits(pf, d)) a = fmaxf(a, fabsf(__ldg(row + d)));
#pragma unroll
  for (int off = 16; off; off >>= 1) a = fmaxf(a, __shfl_xor_sync(0xffffffffu, a, off));
  if ((threadIdx.x & 31) == 0 && a > 0.0f) atomicMax(reinterpret_cast<unsigned int*>(amax), __float_as_uint(a));
}

__global__ void quantize_tensor_i8_kernel(const float* __restrict__ C, int K, int D_eff, int64_t ldc,
                                          int8_t* __restrict__ dst, int64_t ld_dst,
                                          const float* __restrict__ amax) {
  const float a = *amax;
  const float s = a > 0.0f ? __fdiv_rn(127.0f, a) : 1.0f;
  const int64_t total = (int64_t)K * ld_dst;
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < total;
       i += (int64_t)gridDim.x * blockDim.x) {
    const int64_t k = i / ld_dst;
    const int d = (int)(i - k * ld_dst);
    dst[i] = (int8_t)(d < D_eff ? quant_i8(__ldg(C + k * ldc + d), s) : 0);
  }
}

__global__ void quantize_tensor_i16_kernel(const float* __restrict__ C, int K, int D_eff, int64_t ldc,
                                           int16_t* __restrict__ dst, int64_t ld_dst,
                                           const float* __restrict__ amax) {
  const float a = *amax;
  const float s = a > 0.0f ? __fdiv_rn(32767.0f, a) : 1.0f;
  const int64_t total = (int64_t)K * ld_dst;
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < total;
       i += (int64_t)gridDim.x * blockDim.x) {
    const int64_t k = i / ld_dst;
    const int d = (int)(i - k * ld_dst);
    float q = 0.0f;
    if (d < D_eff) q = fminf(fmaxf(rintf(__fmul_rn(__ldg(C + k * ldc + d), s)), -32767.0f), 32767.0f);
    dst[i] = (int16_t)(int)q;
  }
}

// ---------------------------------------------------------------------------------- fp32 class operand
// Class operand of the fused inference epilogue (gemm_tc.cu, EPI_INFER), S5: the value the
// similarity contracts at hv_bits, as a float (int8 codes and +-1 are exact in fp32).
__global__ void class_operand_f32_kernel(const float* __restrict__ C, int K, int D_eff, int64_t ldc, int hv_bits,
                                         Perf pf, const float* __restrict__ amax, float* __restrict__ dst, int KC,
                                         int64_t ld_dst) {
  float s = 1.0f;
  if (hv_bits == 8) {
    const float a = *amax;
    s = a > 0.0f ? __fdiv_rn(127.0f, a) : 1.0f;
  }
  const int64_t total = (int64_t)KC * ld_dst;
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < total;
       i += (int64_t)gridDim.x * blockDim.x) {
    const int k = (int)(i / ld_dst);
    const int d = (int)(i - (int64_t)k * ld_dst);
    float v = 0.0f;
    if (k < K && d < D_eff && perf_visits(pf, d)) {
      const float x = __ldg(C + (int64_t)k * ldc + d);
      switch (hv_bits) {
        case 32: v = x; break;
        case 16: v = __bfloat162float(__float2bfloat16_rn(x)); break;
        case HDC_HV_F16: v = __half2float(__float2half_rn(x)); break;
        case 8: v = (float)quant_i8(x, s); break;
        default: v = x < 0.0f ? -1.0f : 1.0f; break;
      }
    }
    dst[i] = v;
  }
}

// ---------------------------------------------------------------------------------- sign bits
// One warp produces 32 words (1024 dims) of one class row: coalesced loads, one ballot per word.
__global__ void sign_bits_kernel(const float* __restrict__ C, int K, int D_eff, int64_t ldc,
                                 uint32_t* __restrict__ cbits, int W) {
  const int lane = threadIdx.x & 31;
  const int groups = (W + 31) >> 5;
  const int64_t warp = (blockIdx.x * (int64_t)blockDim.x + threadIdx.x) >> 5;
  if (warp >= (int64_t)K * groups) return;
  const int k = (int)(warp / groups);
  const int g = (int)(warp - (int64_t)k * groups);
  uint32_t mine = 0;
#pragma unroll 4
  for (int i = 0; i < 32; ++i) {
    const int d = (g * 32 + i) * 32 + lane;
    const float v = d < D_eff ? __ldg(C + (int64_t)k * ldc + d) : 0.0f;
    const uint32_t b = __ballot_sync(0xffffffffu, v < 0.0f);
    if (i == lane) mine = b;
  }
  const int w = g * 32 + lane;
  if (w < W) cbits[(int64_t)k * W + w] = mine;
}

// ---------------------------------------------------------------------------------- cosine scales
// colscale[k] = cos ? (nrm > 0 ? 1 / (sqrt(D_eff) * nrm) : 0) : 1, nrm^2 = sum_d c[k,d]^2 in double
// over the operand as the contraction loads it.  One block per class, fixed reduction order.
__global__ void col_scale_kernel(Operand C, int K, int D_eff, int cos, Perf pf, int n_vis,
                                 double* __restrict__ colscale, float* __restrict__ colscale_f) {
  const int k = blockIdx.x;
  __shared__ double part[32];
  double s = 0.0;
  if (cos) {
#pragma unroll 4
    for (int d = threadIdx.x; d < D_eff; d += blockDim.x) {
      if (!perf_visits(pf, d)) continue;
      double v;
      const int64_t idx = (int64_t)k * C.ld + d;
      switch (C.kind) {
        case OPK_F32: v = (double)__ldg((const float*)C.p + idx); break;
        case OPK_BF16: v = (double)__bfloat162float(((const __nv_bfloat16*)C.p)[idx]); break;
        case OPK_F32_RBF16:
          v = (double)__bfloat162float(__float2bfloat16_rn(__ldg((const float*)C.p + idx)));
          break;
        case OPK_F32_RF16: v = (double)__half2float(__float2half_rn(__ldg((const float*)C.p + idx))); break;
        case OPK_BITS: v = 1.0; break;
        case OPK_I16: v = (double)((const int16_t*)C.p)[idx]; break;
        default: v = (double)((const int8_t*)C.p)[idx]; break;
      }
      s += v * v;
    }
#pragma unroll
    for (int off = 16; off; off >>= 1) s += __shfl_xor_sync(0xffffffffu, s, off);
    if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = s;
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    if (!cos) {
      colscale[k] = 1.0;
    } else {
      double t = 0.0;
      for (int i = 0; i < (int)(blockDim.x >> 5); ++i) t += part[i];
      const double nrm = sqrt(t);
      colscale[k] = nrm > 0.0 ? 1.0 / (sqrt((double)n_vis) * nrm) : 0.0;
    }
    if (colscale_f) colscale_f[k] = (float)colscale[k];
  }
}

inline int grid_for(int64_t work_items, int threads, int cap) {
  int64_t g = (work_items + threads - 1) / threads;
  if (g < 1) g = 1;
  if (g > cap) g = cap;
  return (int)g;
}

}  // namespace

cudaError_t launch_convert_bf16(const void* src, int src_kind, int64_t rows, int cols, int64_t ld_src,
                                __nv_bfloat16* dst, int64_t ld_dst, cudaStream_t st, int64_t* nlaunch) {
  if (rows <= 0) return cudaSuccess;
  const int64_t total = rows * (ld_dst >> 3);
  convert_bf16_kernel<<<grid_for(total, 256, 148 * 16), 256, 0, st>>>(src, src_kind, rows, cols, ld_src,
                                                                     dst, ld_dst);
  ++*nlaunch;
  return cudaGetLastError();
}

cudaError_t launch_convert_f16(const void* src, int src_kind, int64_t rows, int cols, int64_t ld_src,
                               __half* dst, int64_t ld_dst, cudaStream_t st, int64_t* nlaunch) {
  if (rows <= 0) return cudaSuccess;
  const int64_t total = rows * (ld_dst >> 3);
  convert_f16_kernel<<<grid_for(total, 256, 148 * 16), 256, 0, st>>>(src, src_kind, rows, cols, ld_src, dst, ld_dst);
  ++*nlaunch;
  return cudaGetLastError();
}

cudaError_t launch_split3_bf16(const void* src, int src_kind, int64_t rows, int cols, int64_t ld_src,
                               __nv_bfloat16* dst, int seg, cudaStream_t st, int64_t* nlaunch) {
  if (rows <= 0) return cudaSuccess;
  const int64_t total = rows * (seg >> 3);
  split3_bf16_kernel<<<grid_for(total, 256, 148 * 16), 256, 0, st>>>(src, src_kind, rows, cols, ld_src, dst, seg);
  ++*nlaunch;
  return cudaGetLastError();
}

cudaError_t launch_split2_f16(const void* src, int src_kind, int64_t rows, int cols, int64_t ld_src, __half* dst,
                              int seg, int* expo, cudaStream_t st, int64_t* nlaunch) {
  if (rows <= 0) return cudaSuccess;
  split2_f16_rows_kernel<<<grid_for(rows * 32, 256, 148 * 16), 256, 0, st>>>(src, src_kind, rows, cols, ld_src, dst,
                                                                            seg, expo);
  ++*nlaunch;
  return cudaGetLastError();
}

cudaError_t launch_unscale_raw(float* raw, int64_t rows, int cols, int64_t ld, const int* ex, const int* ep,
                               cudaStream_t st, int64_t* nlaunch) {
  if (rows <= 0) return cudaSuccess;
  unscale_raw_kernel<<<grid_for(rows * cols, 256, 148 * 16), 256, 0, st>>>(raw, rows, cols, ld, ex, ep);
  ++*nlaunch;
  return cudaGetLastError();
}

namespace {
// Same result, one pass over HBM: the row (<= 1024 columns) is read once into registers with coalesced
// loads, its codes go through a per-warp shared-memory line and leave as 16-byte stores (the plain kernel
// reads the row twice and stores single bytes: 3x off the HBM time of the C4 int8 point's 294 MB of features).
constexpr int QR_WARPS = 8;
constexpr int QR_MAXC = 1024;
__global__ void __launch_bounds__(QR_WARPS * 32)
quantize_rows_i8_reg_kernel(const void* __restrict__ src, int src_kind, int64_t rows, int cols, int64_t ld_src,
                            int8_t* __restrict__ dst, int64_t ld_dst) {
  __shared__ __align__(16) int8_t line[QR_WARPS][QR_MAXC + 64];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const int64_t warp = (int64_t)blockIdx.x * QR_WARPS + wid;
  const int64_t nwarps = (int64_t)gridDim.x * QR_WARPS;
  const int nvec = (int)(ld_dst >> 4);  // ld_dst is a multiple of 16
  for (int64_t r = warp; r < rows; r += nwarps) {
    float v[QR_MAXC / 32];
    float a = 0.0f;
#pragma unroll
    for (int i = 0; i < QR_MAXC / 32; ++i) {
      const int c = i * 32 + lane;
      v[i] = c < cols ? load_as_f32(src, src_kind, r * ld_src + c) : 0.0f;
      a = fmaxf(a, fabsf(v[i]));
    }
#pragma unroll
    for (int off = 16; off; off >>= 1) a = fmaxf(a, __shfl_xor_sync(0xffffffffu, a, off));
    const float s = a > 0.0f ? __fdiv_rn(127.0f, a) : 1.0f;
#pragma unroll
    for (int i = 0; i < QR_MAXC / 32; ++i) {
      const int c = i * 32 + lane;
      if (c < (int)ld_dst) line[wid][c] = (int8_t)(c < cols ? quant_i8(v[i], s) : 0);
    }
    __syncwarp();
    for (int j = lane; j < nvec; j += 32)
      reinterpret_cast<uint4*>(dst + r * ld_dst)[j] = reinterpret_cast<const uint4*>(line[wid])[j];
    __syncwarp();
  }
}
}  // namespace

cudaError_t launch_quantize_rows_i8(const void* src, int src_kind, int64_t rows, int cols, int64_t ld_src,
                                    int8_t* dst, int64_t ld_dst, cudaStream_t st, int64_t* nlaunch) {
  if (rows <= 0) return cudaSuccess;
  if (cols <= QR_MAXC && ld_dst <= QR_MAXC + 64 && (ld_dst & 15) == 0 && (reinterpret_cast<uintptr_t>(dst) & 15) == 0) {
    quantize_rows_i8_reg_kernel<<<grid_for(rows, QR_WARPS, 148 * 8), QR_WARPS * 32, 0, st>>>(src, src_kind, rows, cols,
                                                                                          ld_src, dst, ld_dst);
    ++*nlaunch;
    return cudaGetLastError();
  }
  quantize_rows_i8_kernel<<<grid_for(rows * 32, 256, 148 * 16), 256, 0, st>>>(src, src_kind, rows, cols,
                                                                             ld_src, dst, ld_dst);
  ++*nlaunch;
  return cudaGetLastError();
}

namespace {
__global__ void perf_mask_kernel(uint32_t* __restrict__ mask, int W, int D_eff, Perf pf) {
  const int w = blockIdx.x * blockDim.x + threadIdx.x;
  if (w >= W) return;
  uint32_t m = 0;
  for (int b = 0; b < 32; ++b) {
    const int d = w * 32 + b;
    if (d < D_eff && perf_visits(pf, d)) m |= 1u << b;
  }
  mask[w] = m;
}

}  // namespace

namespace {
// Perforated encode contraction (reading A18): compacts the visited columns
// f = begin + j*stride of a row-major matrix; columns >= n_vis of the copy are zero.
template <typename T>
__global__ void gather_cols_kernel(const T* __restrict__ src, int64_t rows, int64_t ld_src, Perf pf, int n_vis,
                                   T* __restrict__ dst, int64_t ld_dst) {
  const int64_t total = rows * ld_dst;
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < total;
       i += (int64_t)gridDim.x * blockDim.x) {
    const int64_t r = i / ld_dst;
    const int j = (int)(i - r * ld_dst);
    T v = T(0);
    if (j < n_vis) v = src[r * ld_src + pf.begin + (int64_t)j * pf.stride];
    dst[i] = v;
  }
}

// raw[n,d] = fl32( fl32(acc[n,d]) * scale ), in place (int32 accumulators are converted first).
__global__ void scale_raw_kernel(void* __restrict__ raw, int64_t rows, int cols, int64_t ld, float scale,
                                 int from_i32) {
  const int64_t total = rows * cols;
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < total;
       i += (int64_t)gridDim.x * blockDim.x) {
    const int64_t r = i / cols;
    const int64_t idx = r * ld + (i - r * cols);
    const float a = from_i32 ? (float)reinterpret_cast<const int32_t*>(raw)[idx]
                             : reinterpret_cast<const float*>(raw)[idx];
    reinterpret_cast<float*>(raw)[idx] = __fmul_rn(a, scale);
  }
}
}  // namespace

cudaError_t launch_gather_cols(const void* src, int esize, int64_t rows, int64_t ld_src, Perf pf, int n_vis,
                               void* dst, int64_t ld_dst, cudaStream_t st, int64_t* nlaunch) {
  if (rows <= 0) return cudaSuccess;
  const int g = grid_for(rows * ld_dst, 256, 148 * 16);
  if (esize == 4)
    gather_cols_kernel<uint32_t><<<g, 256, 0, st>>>((const uint32_t*)src, rows, ld_src, pf, n_vis, (uint32_t*)dst, ld_dst);
  else if (esize == 2)
    gather_cols_kernel<uint16_t><<<g, 256, 0, st>>>((const uint16_t*)src, rows, ld_src, pf, n_vis, (uint16_t*)dst, ld_dst);
  else
    gather_cols_kernel<uint8_t><<<g, 256, 0, st>>>((const uint8_t*)src, rows, ld_src, pf, n_vis, (uint8_t*)dst, ld_dst);
  ++*nlaunch;
  return cudaGetLastError();
}

cudaError_t launch_scale_raw(void* raw, int64_t rows, int cols, int64_t ld, float scale, int from_i32,
                             cudaStream_t st, int64_t* nlaunch) {
  if (rows <= 0) return cudaSuccess;
  scale_raw_kernel<<<grid_for(rows * cols, 256, 148 * 16), 256, 0, st>>>(raw, rows, cols, ld, scale, from_i32);
  ++*nlaunch;
  return cudaGetLastError();
}

cudaError_t launch_perf_mask(uint32_t* mask, int W, int D_eff, Perf pf, cudaStream_t st, int64_t* nlaunch) {
  perf_mask_kernel<<<(W + 255) / 256, 256, 0, st>>>(mask, W, D_eff, pf);
  ++*nlaunch;
  return cudaGetLastError();
}

cudaError_t launch_tensor_amax(const float* C, int K, int D_eff, int64_t ldc, Perf pf, float* amax,
                               cudaStream_t st, int64_t* nlaunch) {
  cudaError_t e = cudaMemsetAsync(amax, 0, sizeof(float), st);
  if (e != cudaSuccess) return e;
  // K rows x slices of up to 2048 columns (8 per thread); K <= 65535 (checked at the API)
  const int slices = (D_eff + 2047) / 2048;
  tensor_amax_kernel<<<dim3((unsigned)slices, (unsigned)K), 256, 0, st>>>(C, K, D_eff, ldc, pf, amax);
  ++*nlaunch;
  return cudaGetLastError();
}

cudaError_t launch_quantize_tensor_i8(const float* C, int K, int D_eff, int64_t ldc, Perf pf, int8_t* dst,
                                      int64_t ld_dst, float* amax_scratch, cudaStream_t st,
                                      int64_t* nlaunch) {
  cudaError_t e = launch_tensor_amax(C, K, D_eff, ldc, pf, amax_scratch, st, nlaunch);
  if (e != cudaSuccess) return e;
  quantize_tensor_i8_kernel<<<grid_for((int64_t)K * ld_dst, 256, 148 * 8), 256, 0, st>>>(
      C, K, D_eff, ldc, dst, ld_dst, amax_scratch);
  ++*nlaunch;
  return cudaGetLastError();
}

cudaError_t launch_quantize_tensor_i16(const float* C, int K, int D_eff, int64_t ldc, Perf pf, int16_t* dst,
                                       int64_t ld_dst, float* amax_scratch, cudaStream_t st,
                                       int64_t* nlaunch) {
  cudaError_t e = launch_tensor_amax(C, K, D_eff, ldc, pf, amax_scratch, st, nlaunch);
  if (e != cudaSuccess) return e;
  quantize_tensor_i16_kernel<<<grid_for((int64_t)K * ld_dst, 256, 148 * 8), 256, 0, st>>>(
      C, K, D_eff, ldc, dst, ld_dst, amax_scratch);
  ++*nlaunch;
  return cudaGetLastError();
}

cudaError_t launch_sign_bits(const float* C, int K, int D_eff, int64_t ldc, uint32_t* cbits, int W,
                             cudaStream_t st, int64_t* nlaunch) {
  const int64_t warps = (int64_t)K * ((W + 31) >> 5);
  sign_bits_kernel<<<(unsigned)((warps * 32 + 255) / 256), 256, 0, st>>>(C, K, D_eff, ldc, cbits, W);
  ++*nlaunch;
  return cudaGetLastError();
}

cudaError_t launch_class_operand_f32(const float* C, int K, int D_eff, int64_t ldc, int hv_bits, Perf pf,
                                     const float* amax, float* dst, int KC, int64_t ld_dst, cudaStream_t st,
                                     int64_t* nlaunch) {
  class_operand_f32_kernel<<<grid_for((int64_t)KC * ld_dst, 256, 148 * 8), 256, 0, st>>>(C, K, D_eff, ldc, hv_bits, pf,
                                                                                        amax, dst, KC, ld_dst);
  ++*nlaunch;
  return cudaGetLastError();
}

cudaError_t launch_col_scale(const Operand& C, int K, int D_eff, int cos, Perf pf, double* colscale,
                             cudaStream_t st, int64_t* nlaunch, float* colscale_f) {
  col_scale_kernel<<<K, 1024, 0, st>>>(C, K, D_eff, cos, pf, perf_count(pf, D_eff), colscale, colscale_f);
  ++*nlaunch;
  return cudaGetLastError();
}

}  // namespace hdc
