// widedot.cu -- DOT / COS similarity and arg-max of packed queries against class operands held as 32- or
// 64-bit integers (hv codes HDC_HV_I32 / HDC_HV_I64; "integer data types (8, 16, 32, or
// 64-bit)"; reading A22: q = rint(C_acc), no scale, symmetric saturation).
//
//   s[n,k] = sum_{d visited, d < D_eff} (1 - 2 b[n,d]) * q[k,d]        exact, in 64-bit integers
//
// The contraction runs on the integer dot-product instruction: the two's-complement bytes of the codes are
// staged once per model as BYTE PLANES -- for every group of four dimensions ("quad": dimensions 32 w + j + 8 i,
// i < 4, so that the four query bits of quad j of word w are (word >> j) & 0x01010101, two ALU operations and no
// multiply on the pipe the dp4a needs) P = 4 or 8 words, word p holding byte p of the four codes -- so that one dp4a multiplies four +-1 query bytes with four code bytes
// (unsigned for the lower planes, signed for the top one) into an int32 per-plane sum (|.| <= 255 * D_eff),
// and the sums of the planes are recombined as sum_p acc_p << 8p in 64 bits when a class is finished.
// Unvisited (perforated) dimensions and the padding beyond D_eff are staged as zero codes: no masks in the loop.
//
// A thread owns QT queries; a CTA of 128 threads walks the reduction axis in chunks of 512 dimensions (16 query
// words per row through a padded shared-memory tile, 128 quads of KC classes as broadcast 16-byte reads) with
// QT x KC x P accumulators in registers; classes beyond KC take further passes over the query rows (L2-resident).
// dp4a and IMAD share one pipe (ncu: fmaheavy 89 % busy in the first version, dp4a 62 % of it): the kernel keeps
// everything else off it.  The query bytes are 0 / 1 (bit set = -1): sum (1 - 2b) q = rowsum - 2 sum b q, the row
// sums of the codes staged with the planes.  QT = 1, KC = 8 (4 for 64-bit codes) measured best: more queries per
// thread halve the shared-memory wavefronts per dp4a but spend the pipe on more expansions per class word.
// Bound: the dp4a issue rate -- N * K * D_eff * P / 4 instructions per call.
#include <limits.h>

#include "common.cuh"

namespace hdc {
namespace {

constexpr int WQ = 128;        // queries per CTA
constexpr int CHUNK_W = 16;    // query words per chunk (512 dimensions = 128 quads)
constexpr int CHUNK_Q = CHUNK_W * 8;

__device__ __forceinline__ int dp4a_uu(uint32_t a, uint32_t b, int c) {   // unsigned a bytes x unsigned b bytes
  int d;
  asm("dp4a.u32.u32 %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(b), "r"(c));
  return d;
}
__device__ __forceinline__ int dp4a_us(uint32_t a, uint32_t b, int c) {   // unsigned a bytes x signed b bytes
  int d;
  asm("dp4a.u32.s32 %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(b), "r"(c));
  return d;
}

// ---------------------------------------------------------------------------------- preparation
// One block per class: codes -> byte planes [K][quads_ld][P] words, and the cosine scale
// 1 / (sqrt(n_vis) * |q|) (0 for a zero row; 1 for DOT), norm summed in double in a fixed order.
__global__ void wide_prepare_kernel(const float* __restrict__ C, int D_eff, int64_t ldc, Perf pf, int P,
                                    uint32_t* __restrict__ planes, int quads_ld, int cos, int n_vis,
                                    double* __restrict__ colscale, long long* __restrict__ rowsum,
                                    int* __restrict__ live) {
  const int k = blockIdx.x;
  if (live && k == 0 && threadIdx.x < 4) live[threadIdx.x] = 0;   // the pieces' preparation (next launches) sets them
  const long long lim = P == 4 ? 2147483647LL : 9223372036854775807LL;
  __shared__ double part[32];
  __shared__ unsigned long long part_s[32];
  double ss = 0.0;
  unsigned long long rs = 0;   // sum of the codes (wraps beyond the contract, like the scores)
  for (int qd = threadIdx.x; qd < quads_ld; qd += blockDim.x) {
    unsigned long long code[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const int d = (qd >> 3) * 32 + (qd & 7) + 8 * i;   // quad j of query word w: dimensions 32 w + j + 8 i
      long long q = 0;
      if (d < D_eff && perf_visits(pf, d)) {
        q = __float2ll_rn(__ldg(C + (int64_t)k * ldc + d));   // round half to even, saturates at the int64 range
        q = q > lim ? lim : (q < -lim ? -lim : q);
      }
      code[i] = (unsigned long long)q;
      rs += (unsigned long long)q;
      const double v = (double)q;
      ss += v * v;
    }
    if (!planes) continue;   // tensor-core route: only the cosine scales are wanted
    uint32_t* dst = planes + ((int64_t)k * quads_ld + qd) * P;
    for (int p = 0; p < P; ++p) {
      const int sh = 8 * p;
      dst[p] = (uint32_t)((code[0] >> sh) & 0xFFu) | (uint32_t)((code[1] >> sh) & 0xFFu) << 8 |
               (uint32_t)((code[2] >> sh) & 0xFFu) << 16 | (uint32_t)((code[3] >> sh) & 0xFFu) << 24;
    }
  }
#pragma unroll
  for (int off = 16; off; off >>= 1) {
    ss += __shfl_xor_sync(0xffffffffu, ss, off);
    rs += __shfl_xor_sync(0xffffffffu, rs, off);
  }
  if ((threadIdx.x & 31) == 0) {
    part[threadIdx.x >> 5] = ss;
    part_s[threadIdx.x >> 5] = rs;
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    double t = 0.0;
    unsigned long long ts = 0;
    for (int i = 0; i < (int)(blockDim.x >> 5); ++i) {
      t += part[i];
      ts += part_s[i];
    }
    if (rowsum) rowsum[k] = (long long)ts;
    const double nrm = sqrt(t);
    colscale[k] = !cos ? 1.0 : (nrm > 0.0 ? 1.0 / (sqrt((double)n_vis) * nrm) : 0.0);
  }
}

// Epilogue shared by the dp4a kernel and the tensor-core route's combine kernel: exact integer arg-max for DOT
// (ties keep the lower index: classes arrive in ascending order), the cosine compared in double; or scores.
struct WideOut {
  const double* colscale;
  int cos;
  int32_t* labels;
  float* best;
  float* second;
  void* S;
  int64_t lds;
  int s_mode;   // 0 fp32, 2 int64
};
struct WideTop2 {   // best / runner-up as raw 64-bit patterns: long long for DOT, double for COS
  long long b1, b2;
  int lab;
};
__device__ __forceinline__ WideTop2 wide_top2_init(const WideOut& o) {
  const long long lo = o.cos ? __double_as_longlong(-1.0e300) : LLONG_MIN;
  return WideTop2{lo, lo, 0};
}
__device__ __forceinline__ void wide_push(const WideOut& o, WideTop2& t, int64_t n, int cls, long long s) {
  if (o.labels) {
    if (o.cos) {
      const double v = (double)s * o.colscale[cls];
      if (v > __longlong_as_double(t.b1)) {
        t.b2 = t.b1;
        t.b1 = __double_as_longlong(v);
        t.lab = cls;
      } else if (v > __longlong_as_double(t.b2)) {
        t.b2 = __double_as_longlong(v);
      }
    } else {
      if (s > t.b1) {
        t.b2 = t.b1;
        t.b1 = s;
        t.lab = cls;
      } else if (s > t.b2) {
        t.b2 = s;
      }
    }
  } else if (o.s_mode == 2) {
    reinterpret_cast<long long*>(o.S)[n * o.lds + cls] = s;
  } else {
    reinterpret_cast<float*>(o.S)[n * o.lds + cls] = o.cos ? (float)((double)s * o.colscale[cls]) : (float)s;
  }
}
__device__ __forceinline__ void wide_finish(const WideOut& o, const WideTop2& t, int64_t n, int K) {
  if (!o.labels) return;
  o.labels[n] = t.lab;
  const float b1 = o.cos ? (float)__longlong_as_double(t.b1) : (float)t.b1;
  const float b2 = K > 1 ? (o.cos ? (float)__longlong_as_double(t.b2) : (float)t.b2) : b1;
  if (o.best) o.best[n] = b1;
  if (o.second) o.second[n] = b2;
}

// ---------------------------------------------------------------------------------- contraction
struct WideParams {
  const uint32_t* H;
  int64_t N, ldh;
  int W;                      // query words per row that carry visited dimensions
  const uint32_t* planes;
  const long long* rowsum;    // [K] sums of the codes
  int quads_ld;
  int K;
  WideOut o;                  // arg-max outputs (labels != NULL) or scores
};

template <int P>
__device__ __forceinline__ long long recombine(const int (&a)[P]) {
  unsigned long long s = 0;
#pragma unroll
  for (int p = 0; p < P; ++p) s += (unsigned long long)(long long)a[p] << (8 * p);
  return (long long)s;
}

template <int P, int KC, int QT>
__global__ void __launch_bounds__(WQ) wide_dot_kernel(const WideParams p) {
  constexpr int V = P / 4;                                  // 16-byte vectors per quad
  constexpr int ROWS = WQ * QT;                             // queries per CTA: thread t owns rows t + WQ * j
  __shared__ uint32_t sq[ROWS][CHUNK_W + 1];
  __shared__ uint4 sc[KC][CHUNK_Q][V];
  const int t = threadIdx.x;
  const int64_t n0 = (int64_t)blockIdx.x * ROWS;

  WideTop2 top[QT];   // running arg-max state of this thread's queries
#pragma unroll
  for (int q = 0; q < QT; ++q) top[q] = wide_top2_init(p.o);

  for (int kg = 0; kg < p.K; kg += KC) {
    int acc[QT][KC][P];
#pragma unroll
    for (int q = 0; q < QT; ++q)
#pragma unroll
      for (int k = 0; k < KC; ++k)
#pragma unroll
        for (int j = 0; j < P; ++j) acc[q][k][j] = 0;

    for (int c0 = 0; c0 < p.W; c0 += CHUNK_W) {
      __syncthreads();   // the previous chunk's readers are done
#pragma unroll 4
      for (int j = 0; j < CHUNK_W * QT; ++j) {
        const int i = t + WQ * j;
        const int r = i / CHUNK_W, w = i % CHUNK_W;
        int64_t row = n0 + r;
        if (row >= p.N) row = p.N - 1;
        sq[r][w] = (c0 + w < p.W) ? __ldg(p.H + row * p.ldh + c0 + w) : 0u;
      }
      for (int i = t; i < KC * CHUNK_Q * V; i += WQ) {
        const int k = i / (CHUNK_Q * V), rem = i % (CHUNK_Q * V);
        uint4 v = make_uint4(0u, 0u, 0u, 0u);
        if (kg + k < p.K)
          v = __ldg(reinterpret_cast<const uint4*>(p.planes + ((int64_t)(kg + k) * p.quads_ld + (int64_t)c0 * 8) * P) + rem);
        (&sc[k][0][0])[rem] = v;
      }
      __syncthreads();
#pragma unroll 1
      for (int w = 0; w < CHUNK_W; ++w) {
        uint32_t qw[QT];
#pragma unroll
        for (int q = 0; q < QT; ++q) qw[q] = sq[t + WQ * q][w];
#pragma unroll
        for (int nib = 0; nib < 8; ++nib) {
          uint32_t a[QT];   // bits nib, nib + 8, nib + 16, nib + 24 of the word -> bytes 0..3 (0 or 1)
#pragma unroll
          for (int q = 0; q < QT; ++q) a[q] = (qw[q] >> nib) & 0x01010101u;
#pragma unroll
          for (int k = 0; k < KC; ++k) {
#pragma unroll
            for (int v = 0; v < V; ++v) {
              const uint4 c = sc[k][w * 8 + nib][v];
              const bool last = v == V - 1;
#pragma unroll
              for (int q = 0; q < QT; ++q) {
                acc[q][k][4 * v + 0] = dp4a_uu(a[q], c.x, acc[q][k][4 * v + 0]);
                acc[q][k][4 * v + 1] = dp4a_uu(a[q], c.y, acc[q][k][4 * v + 1]);
                acc[q][k][4 * v + 2] = dp4a_uu(a[q], c.z, acc[q][k][4 * v + 2]);
                acc[q][k][4 * v + 3] = last ? dp4a_us(a[q], c.w, acc[q][k][4 * v + 3])
                                            : dp4a_uu(a[q], c.w, acc[q][k][4 * v + 3]);
              }
            }
          }
        }
      }
    }

#pragma unroll
    for (int k = 0; k < KC; ++k) {
      const int cls = kg + k;
      if (cls >= p.K) break;
      const unsigned long long rs = (unsigned long long)__ldg(p.rowsum + cls);
#pragma unroll
      for (int q = 0; q < QT; ++q) {
        const int64_t n = n0 + t + WQ * q;
        // sum (1 - 2b) code = rowsum - 2 * sum over the set bits
        const long long s = (long long)(rs - 2ull * (unsigned long long)recombine<P>(acc[q][k]));
        if (n < p.N) wide_push(p.o, top[q], n, cls, s);
      }
    }
  }
#pragma unroll
  for (int q = 0; q < QT; ++q) {
    const int64_t n = n0 + t + WQ * q;
    if (n < p.N) wide_finish(p.o, top[q], n, p.K);
  }
}

// Tensor-core route: recombines the int32 scores of the 16-bit pieces, S_j [rows][K] at Sp + j * rows * K.
// One warp per query row (lanes = classes: coalesced reads of the piece scores and writes of the scores), the
// lanes' running best / runner-up merged by a butterfly with the index tie-break (ties -> lowest class index).
__device__ __forceinline__ bool wide_gt(int cos, long long a, long long b) {
  return cos ? __longlong_as_double(a) > __longlong_as_double(b) : a > b;
}
__device__ __forceinline__ long long wide_max(int cos, long long a, long long b) { return wide_gt(cos, b, a) ? b : a; }

constexpr int WC_WARPS = 8;
__global__ void __launch_bounds__(WC_WARPS * 32)
wide_combine_kernel(const int32_t* __restrict__ Sp, int pieces, int64_t rows, int K, const int* __restrict__ live,
                    WideOut o) {
  const int lane = threadIdx.x & 31;
  int on = 0;   // pieces that hold a nonzero code (the others' scores are zero and were never written)
  for (int j = 0; j < pieces; ++j) on |= (__ldg(live + j) != 0) << j;
  const int64_t warp0 = (int64_t)blockIdx.x * WC_WARPS + (threadIdx.x >> 5);
  for (int64_t n = warp0; n < rows; n += (int64_t)gridDim.x * WC_WARPS) {
    WideTop2 top = wide_top2_init(o);
    top.lab = INT_MAX;   // lanes without a class never win a tie
    if ((K & 3) == 0) {
      // four classes per lane and load: a row is a chain of load latencies, 16-byte loads put 4x the bytes in flight
      // (rows of K int32 are 16-byte aligned when K is a multiple of 4)
      for (int k = 4 * lane; k < K; k += 128) {
        unsigned long long s0 = 0, s1 = 0, s2 = 0, s3 = 0;
        for (int j = 0; j < pieces; ++j) {
          if (!(on >> j & 1)) continue;
          const int4 v = __ldg(reinterpret_cast<const int4*>(Sp + ((int64_t)j * rows + n) * K + k));
          s0 += (unsigned long long)(long long)v.x << (16 * j);
          s1 += (unsigned long long)(long long)v.y << (16 * j);
          s2 += (unsigned long long)(long long)v.z << (16 * j);
          s3 += (unsigned long long)(long long)v.w << (16 * j);
        }
        wide_push(o, top, n, k, (long long)s0);
        wide_push(o, top, n, k + 1, (long long)s1);
        wide_push(o, top, n, k + 2, (long long)s2);
        wide_push(o, top, n, k + 3, (long long)s3);
      }
    } else {
      for (int k = lane; k < K; k += 32) {
        unsigned long long s = 0;
        for (int j = 0; j < pieces; ++j)
          if (on >> j & 1) s += (unsigned long long)(long long)__ldg(Sp + ((int64_t)j * rows + n) * K + k) << (16 * j);
        wide_push(o, top, n, k, (long long)s);
      }
    }
    if (!o.labels) continue;
#pragma unroll
    for (int off = 16; off; off >>= 1) {
      const long long ob1 = __shfl_xor_sync(0xffffffffu, top.b1, off);
      const long long ob2 = __shfl_xor_sync(0xffffffffu, top.b2, off);
      const int olab = __shfl_xor_sync(0xffffffffu, top.lab, off);
      const bool other = wide_gt(o.cos, ob1, top.b1) || (!wide_gt(o.cos, top.b1, ob1) && olab < top.lab);
      const long long rest = wide_max(o.cos, top.b2, ob2);
      if (other) {
        top.b2 = wide_max(o.cos, top.b1, rest);
        top.b1 = ob1;
        top.lab = olab;
      } else {
        top.b2 = wide_max(o.cos, ob1, rest);
      }
    }
    if (lane == 0) wide_finish(o, top, n, K);
  }
}

// Few classes: one thread per query row (a warp per row leaves lanes idle and pays the butterfly per row; measured
// at K = 26: 24 us against 58 us per 131072 rows; at K = 1000 the strided reads of this form cost 0.5 ms per pass).
__global__ void wide_combine_rows_kernel(const int32_t* __restrict__ Sp, int pieces, int64_t rows, int K,
                                         const int* __restrict__ live, WideOut o) {
  const int64_t n = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (n >= rows) return;
  int on = 0;
  for (int j = 0; j < pieces; ++j) on |= (__ldg(live + j) != 0) << j;
  WideTop2 top = wide_top2_init(o);
  if ((K & 1) == 0) {   // rows of an even number of int32 are 8-byte aligned: two classes per load
#pragma unroll 4
    for (int k = 0; k < K; k += 2) {
      unsigned long long s0 = 0, s1 = 0;
      for (int j = 0; j < pieces; ++j) {
        if (!(on >> j & 1)) continue;
        const int2 v = __ldg(reinterpret_cast<const int2*>(Sp + ((int64_t)j * rows + n) * K + k));
        s0 += (unsigned long long)(long long)v.x << (16 * j);
        s1 += (unsigned long long)(long long)v.y << (16 * j);
      }
      wide_push(o, top, n, k, (long long)s0);
      wide_push(o, top, n, k + 1, (long long)s1);
    }
  } else {
    for (int k = 0; k < K; ++k) {
      unsigned long long s = 0;
      for (int j = 0; j < pieces; ++j)
        if (on >> j & 1) s += (unsigned long long)(long long)__ldg(Sp + ((int64_t)j * rows + n) * K + k) << (16 * j);
      wide_push(o, top, n, k, (long long)s);
    }
  }
  wide_finish(o, top, n, K);
}

}  // namespace

static inline int wide_planes(int hv_bits) { return hv_bits == HDC_HV_I32 ? 4 : (hv_bits == HDC_HV_I64 ? 8 : 0); }
static inline int wide_quads_ld(int D_eff) { return (int)round_up((D_eff + 3) / 4, CHUNK_Q); }

size_t wide_operand_bytes(int K, int hv_bits, int D_eff) {
  const int P = wide_planes(hv_bits);
  // byte planes, then one 64-bit sum of the codes per class
  return P ? (size_t)K * (size_t)wide_quads_ld(D_eff) * P * sizeof(uint32_t) + (size_t)K * sizeof(long long) : 0;
}
static inline long long* wide_rowsum(uint32_t* planes, int K, int hv_bits, int D_eff) {
  return reinterpret_cast<long long*>(planes + (size_t)K * (size_t)wide_quads_ld(D_eff) * wide_planes(hv_bits));
}

static WideOut wide_out(const Epilogue& e, int cos, const double* colscale) {
  WideOut o{};
  o.colscale = colscale;
  o.cos = cos;
  if (e.kind == EPI_ARGMAX) {
    o.labels = e.labels;
    o.best = e.best;
    o.second = e.second;
  } else {
    o.S = e.S;
    o.lds = e.lds;
    o.s_mode = e.s_i32;
  }
  return o;
}

cudaError_t launch_wide_combine(const int32_t* Sp, int pieces, int64_t rows, int K, int cos, const double* colscale,
                                const int* live, const Epilogue& e, cudaStream_t st, int64_t* nlaunch) {
  if (rows <= 0) return cudaSuccess;
  if (K < 64) {
    wide_combine_rows_kernel<<<(unsigned)((rows + 127) / 128), 128, 0, st>>>(Sp, pieces, rows, K, live, wide_out(e, cos, colscale));
    *nlaunch += 1;
    return cudaGetLastError();
  }
  int64_t grid = (rows + WC_WARPS - 1) / WC_WARPS;
  if (grid > 148 * 16) grid = 148 * 16;
  wide_combine_kernel<<<(unsigned)grid, WC_WARPS * 32, 0, st>>>(Sp, pieces, rows, K, live, wide_out(e, cos, colscale));
  *nlaunch += 1;
  return cudaGetLastError();
}

cudaError_t launch_wide_prepare(const float* C_acc, int K, int64_t ldc, int D_eff, int hv_bits, Perf pf, int cos,
                                uint32_t* planes, double* colscale, cudaStream_t st, int64_t* nlaunch, int* live) {
  const int P = wide_planes(hv_bits);
  if (!P) return cudaErrorInvalidValue;
  wide_prepare_kernel<<<K, 256, 0, st>>>(C_acc, D_eff, ldc, pf, P, planes, wide_quads_ld(D_eff), cos,
                                         perf_count(pf, D_eff), colscale,
                                         planes ? wide_rowsum(planes, K, hv_bits, D_eff) : nullptr, live);
  *nlaunch += 1;
  return cudaGetLastError();
}

cudaError_t launch_wide_dot(const uint32_t* Hbits, int64_t N, int64_t ldh, int K, int D_eff, int hv_bits, int cos,
                            const uint32_t* planes, const double* colscale, const Epilogue& e, cudaStream_t st,
                            int64_t* nlaunch) {
  const int P = wide_planes(hv_bits);
  if (!P) return cudaErrorInvalidValue;
  if (N <= 0) return cudaSuccess;
  WideParams p{};
  p.H = Hbits;
  p.N = N;
  p.ldh = ldh;
  p.W = words_of(D_eff);
  p.planes = planes;
  p.rowsum = wide_rowsum(const_cast<uint32_t*>(planes), K, hv_bits, D_eff);
  p.quads_ld = wide_quads_ld(D_eff);
  p.K = K;
  p.o = wide_out(e, cos, colscale);
#ifndef WD_QT
#define WD_QT 1
#define WD_KC4 8
#define WD_KC8 4
#endif
  const int64_t blocks = (N + WQ * WD_QT - 1) / (WQ * WD_QT);
  if (blocks > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
  if (P == 4)
    wide_dot_kernel<4, WD_KC4, WD_QT><<<(unsigned)blocks, WQ, 0, st>>>(p);
  else
    wide_dot_kernel<8, WD_KC8, WD_QT><<<(unsigned)blocks, WQ, 0, st>>>(p);
  *nlaunch += 1;
  return cudaGetLastError();
}

}  // namespace hdc
