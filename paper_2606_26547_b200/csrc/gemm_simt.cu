// gemm_simt.cu -- CUDA-core contraction C[m,n] = sum_k A[m,k] * B[n,k] (both operands reduction-axis
// contiguous) with the HDC epilogues fused: sign+pack (random-projection encode, Listing 1
// L68-L70 + L161), scores (L110 cos_sim / L197 dot) and row arg-max (L79-L80).
//
// This is the fp32 path (no fp32 tensor-core mode exists; TF32 would break the sign contract) and
// the always-available path for every other precision (HDC_FLAG_SIMT): bf16 operands are exact in
// fp32, products of two bf16 are exact in fp32, and integer operands accumulate in int32.
//
// Tiling: 256 threads as a 16x16 grid; CTA tile 128 x (16*TN); each thread an 8 x TN register tile;
// 16-deep k-slices staged through shared memory (transposed, so the inner loop reads float4 /
// broadcast), register-prefetch double buffering: one __syncthreads per k-slice.
#include <float.h>
#include <limits.h>

#include "common.cuh"

namespace hdc {
namespace {

constexpr int BM = 128;
constexpr int BK = 16;
constexpr int TM = 8;
constexpr int NTHREADS = 256;
constexpr int PAD = 4;

struct GemmParams {
  Operand A, B;
  int64_t M;
  int Nc, Kr;
  int n_tiles;
  Epilogue e;
};

template <typename T>
__device__ __forceinline__ T load_elem(const Operand& o, int64_t row, int k) {
  switch (o.kind) {
    case OPK_F32:
      return (T)__ldg((const float*)o.p + row * o.ld + k);
    case OPK_BF16:
      return (T)__bfloat162float(((const __nv_bfloat16*)o.p)[row * o.ld + k]);
    case OPK_F32_RBF16:
      return (T)__bfloat162float(__float2bfloat16_rn(__ldg((const float*)o.p + row * o.ld + k)));
    case OPK_F32_RF16:
      return (T)__half2float(__float2half_rn(__ldg((const float*)o.p + row * o.ld + k)));
    case OPK_BF16_RF16:
      return (T)__half2float(__float2half_rn(__bfloat162float(((const __nv_bfloat16*)o.p)[row * o.ld + k])));
    case OPK_BITS: {
      uint32_t w = __ldg((const uint32_t*)o.p + row * o.ld + (k >> 5));
      return (T)(1 - 2 * (int)((w >> (k & 31)) & 1u));
    }
    case OPK_I16:
      return (T)((const int16_t*)o.p)[row * o.ld + k];
    default:  // OPK_I8
      return (T)((const int8_t*)o.p)[row * o.ld + k];
  }
}

// Running best / runner-up of one row.  Scores are compared in double: an int32 or fp32
// accumulator widens exactly and the cosine scale is a double, so integer paths decide exactly
// as the definition does (ties to the lowest class index).
struct Top2 {
  double b1;
  int i1;
  double b2;
};
constexpr double NEG_BIG = -1.0e300;
__device__ __forceinline__ void top2_push(Top2& s, double v, int i) {
  if (v > s.b1 || (v == s.b1 && i < s.i1)) {
    s.b2 = s.b1;
    s.b1 = v;
    s.i1 = i;
  } else {
    s.b2 = fmax(s.b2, v);
  }
}
__device__ __forceinline__ void top2_merge(Top2& a, const Top2& b) {
  if (b.b1 > a.b1 || (b.b1 == a.b1 && b.i1 < a.i1)) {
    double l = a.b1;
    a.b1 = b.b1;
    a.i1 = b.i1;
    a.b2 = fmax(fmax(a.b2, b.b2), l);
  } else {
    a.b2 = fmax(fmax(a.b2, b.b2), b.b1);
  }
}

// column owned by register j of thread tx: groups of G = min(TN,4) contiguous columns
template <int TN>
__device__ __forceinline__ int col_of(int tx, int j) {
  constexpr int G = TN < 4 ? TN : 4;
  return (j / G) * (16 * G) + tx * G + (j % G);
}

template <typename AccT, int TN, int EPI>
__global__ void __launch_bounds__(NTHREADS) gemm_simt_kernel(const GemmParams p) {
  constexpr int BN = 16 * TN;
  constexpr int G = TN < 4 ? TN : 4;
  constexpr int A_PER = BM * BK / NTHREADS;                       // 8
  constexpr int B_PER = (BN * BK + NTHREADS - 1) / NTHREADS;      // 8 (TN=8) or 2 (TN=2)
  __shared__ __align__(16) AccT As[2][BK][BM + PAD];
  __shared__ __align__(16) AccT Bs[2][BK][BN + PAD];
  __shared__ uint32_t sbits[EPI == EPI_SIGN ? BM * ((BN + 31) / 32) : 1];

  const int tid = threadIdx.x;
  const int tx = tid & 15, ty = tid >> 4;
  const int64_t m0 = (int64_t)blockIdx.y * BM;
  const int lk = tid & (BK - 1);   // k within slice owned by this thread in the loaders
  const int lr = tid >> 4;         // first row owned in the loaders (stride 16)

  Top2 run[TM];
  if (EPI == EPI_ARGMAX) {
#pragma unroll
    for (int i = 0; i < TM; ++i) run[i] = Top2{NEG_BIG, INT_MAX, NEG_BIG};
  }

  for (int nt = blockIdx.x; nt < p.n_tiles; nt += gridDim.x) {
    const int n0 = nt * BN;
    AccT acc[TM][TN];
#pragma unroll
    for (int i = 0; i < TM; ++i)
#pragma unroll
      for (int j = 0; j < TN; ++j) acc[i][j] = 0;

    AccT ra[A_PER], rb[B_PER];
    auto gload = [&](int k0) {
      const int k = k0 + lk;
#pragma unroll
      for (int i = 0; i < A_PER; ++i) {
        int64_t r = m0 + lr + 16 * i;
        ra[i] = (k < p.Kr && r < p.M) ? load_elem<AccT>(p.A, r, k) : (AccT)0;
      }
#pragma unroll
      for (int i = 0; i < B_PER; ++i) {
        int rr = lr + 16 * i;
        int r = n0 + rr;
        rb[i] = (rr < BN && k < p.Kr && r < p.Nc) ? load_elem<AccT>(p.B, r, k) : (AccT)0;
      }
    };
    auto sstore = [&](int buf) {
#pragma unroll
      for (int i = 0; i < A_PER; ++i) As[buf][lk][lr + 16 * i] = ra[i];
#pragma unroll
      for (int i = 0; i < B_PER; ++i)
        if (lr + 16 * i < BN) Bs[buf][lk][lr + 16 * i] = rb[i];
    };

    const int nk = (p.Kr + BK - 1) / BK;
    __syncthreads();  // previous tile's readers are done with smem
    gload(0);
    sstore(0);
    __syncthreads();
    for (int kt = 0; kt < nk; ++kt) {
      const int buf = kt & 1;
      if (kt + 1 < nk) gload((kt + 1) * BK);
#pragma unroll
      for (int k = 0; k < BK; ++k) {
        AccT a[TM], b[TN];
#pragma unroll
        for (int i = 0; i < TM; i += 4) {
          const float4 v = *reinterpret_cast<const float4*>(&As[buf][k][ty * TM + i]);
          a[i] = reinterpret_cast<const AccT&>(v.x);
          a[i + 1] = reinterpret_cast<const AccT&>(v.y);
          a[i + 2] = reinterpret_cast<const AccT&>(v.z);
          a[i + 3] = reinterpret_cast<const AccT&>(v.w);
        }
#pragma unroll
        for (int j = 0; j < TN; j += G) {
          if (G == 4) {
            const float4 v = *reinterpret_cast<const float4*>(&Bs[buf][k][col_of<TN>(tx, j)]);
            b[j] = reinterpret_cast<const AccT&>(v.x);
            b[j + 1] = reinterpret_cast<const AccT&>(v.y);
            b[j + 2] = reinterpret_cast<const AccT&>(v.z);
            b[j + 3] = reinterpret_cast<const AccT&>(v.w);
          } else {
#pragma unroll
            for (int g = 0; g < G; ++g) b[j + g] = Bs[buf][k][col_of<TN>(tx, j + g)];
          }
        }
#pragma unroll
        for (int i = 0; i < TM; ++i)
#pragma unroll
          for (int j = 0; j < TN; ++j) acc[i][j] += a[i] * b[j];
      }
      if (kt + 1 < nk) {
        sstore(buf ^ 1);
        __syncthreads();
      }
    }

    // ---------------------------------------------------------------- epilogues
    if (EPI == EPI_SIGN) {
      constexpr int WPT = (BN + 31) / 32;  // words per row of this tile
      for (int i = tid; i < BM * WPT; i += NTHREADS) sbits[i] = 0;
      __syncthreads();
#pragma unroll
      for (int i = 0; i < TM; ++i) {
        const int r = ty * TM + i;
#pragma unroll
        for (int j = 0; j < TN; j += G) {
          uint32_t nib = 0;
#pragma unroll
          for (int g = 0; g < G; ++g) nib |= (acc[i][j + g] < (AccT)0 ? 1u : 0u) << g;
          const int c = col_of<TN>(tx, j);
          if (nib) atomicOr(&sbits[r * WPT + (c >> 5)], nib << (c & 31));
        }
      }
      __syncthreads();
      const int W = (p.Nc + 31) >> 5;
      for (int i = tid; i < BM * WPT; i += NTHREADS) {
        const int r = i / WPT, w = i % WPT;
        const int gw = (n0 >> 5) + w;
        if (m0 + r < p.M && gw < W) p.e.bits[(m0 + r) * p.e.ldbits + gw] = sbits[i];
      }
      if (p.e.raw) {
#pragma unroll
        for (int i = 0; i < TM; ++i) {
          const int64_t r = m0 + ty * TM + i;
          if (r < p.M) {
#pragma unroll
            for (int j = 0; j < TN; ++j) {
              const int c = n0 + col_of<TN>(tx, j);
              if (c < p.Nc) reinterpret_cast<AccT*>(p.e.raw)[r * p.e.ldraw + c] = acc[i][j];
            }
          }
        }
      }
    } else if (EPI == EPI_SCORE) {
#pragma unroll
      for (int i = 0; i < TM; ++i) {
        const int64_t r = m0 + ty * TM + i;
        if (r >= p.M) continue;
#pragma unroll
        for (int j = 0; j < TN; ++j) {
          const int c = n0 + col_of<TN>(tx, j);
          if (c >= p.Nc) continue;
          if (p.e.s_i32) {
            reinterpret_cast<int32_t*>(p.e.S)[r * p.e.lds + c] = (int32_t)acc[i][j];
          } else {
            float v = p.e.colscale ? (float)((double)acc[i][j] * p.e.colscale[c]) : (float)acc[i][j];
            reinterpret_cast<float*>(p.e.S)[r * p.e.lds + c] = v;
          }
        }
      }
    } else {  // EPI_ARGMAX: fold this class tile into the running top-2 of each owned row
#pragma unroll
      for (int j = 0; j < TN; ++j) {
        const int c = n0 + col_of<TN>(tx, j);
        if (c >= p.Nc) continue;
        const double sc = p.e.colscale ? p.e.colscale[c] : 1.0;
#pragma unroll
        for (int i = 0; i < TM; ++i) {
          top2_push(run[i], (double)acc[i][j] * sc, c);
        }
      }
    }
  }

  if (EPI == EPI_ARGMAX) {
    // the 16 threads sharing a row are the 16 lanes of one half-warp: butterfly over 1,2,4,8
#pragma unroll
    for (int i = 0; i < TM; ++i) {
#pragma unroll
      for (int off = 1; off < 16; off <<= 1) {
        Top2 o;
        o.b1 = __shfl_xor_sync(0xffffffffu, run[i].b1, off);
        o.i1 = __shfl_xor_sync(0xffffffffu, run[i].i1, off);
        o.b2 = __shfl_xor_sync(0xffffffffu, run[i].b2, off);
        top2_merge(run[i], o);
      }
      const int64_t r = m0 + ty * TM + i;
      if (tx == 0 && r < p.M) {
        double b1 = run[i].b1, b2 = run[i].b2;
        if (b2 == NEG_BIG) b2 = b1;  // K == 1
        if (p.e.ham_D > 0) {
          b1 = 0.5 * ((double)p.e.ham_D - b1);
          b2 = 0.5 * ((double)p.e.ham_D - b2);
        }
        p.e.labels[r] = run[i].i1;
        if (p.e.best) p.e.best[r] = (float)b1;
        if (p.e.second) p.e.second[r] = (float)b2;
      }
    }
  }
}

template <typename AccT, int TN>
cudaError_t launch_tn(const GemmParams& p, cudaStream_t st) {
  constexpr int BN = 16 * TN;
  GemmParams q = p;
  q.n_tiles = (p.Nc + BN - 1) / BN;
  const int64_t m_tiles = (p.M + BM - 1) / BM;
  // grid.y is limited to 65535: split very tall problems into row bands
  const int64_t band = 65535;
  for (int64_t t0 = 0; t0 < m_tiles; t0 += band) {
    const int64_t nt = (m_tiles - t0 < band) ? (m_tiles - t0) : band;
    GemmParams b = q;
    const int64_t roff = t0 * BM;
    b.M = p.M - roff;
    if (b.M > nt * BM) b.M = nt * BM;
    auto adv = [&](Operand o) {
      size_t es = (o.kind == OPK_BF16 || o.kind == OPK_BF16_RF16 || o.kind == OPK_I16) ? 2 : (o.kind == OPK_I8 ? 1 : 4);
      o.p = (const char*)o.p + (size_t)roff * o.ld * es;
      return o;
    };
    b.A = adv(p.A);
    if (b.e.bits) b.e.bits += roff * b.e.ldbits;
    if (b.e.raw) b.e.raw = (char*)b.e.raw + (size_t)roff * b.e.ldraw * 4;
    if (b.e.S) b.e.S = (char*)b.e.S + (size_t)roff * b.e.lds * 4;
    if (b.e.labels) b.e.labels += roff;
    if (b.e.best) b.e.best += roff;
    if (b.e.second) b.e.second += roff;
    dim3 grid(p.e.kind == EPI_ARGMAX ? 1 : q.n_tiles, (unsigned)nt);
    switch (p.e.kind) {
      case EPI_SIGN:
        gemm_simt_kernel<AccT, TN, EPI_SIGN><<<grid, NTHREADS, 0, st>>>(b);
        break;
      case EPI_SCORE:
        gemm_simt_kernel<AccT, TN, EPI_SCORE><<<grid, NTHREADS, 0, st>>>(b);
        break;
      default:
        gemm_simt_kernel<AccT, TN, EPI_ARGMAX><<<grid, NTHREADS, 0, st>>>(b);
        break;
    }
    cudaError_t err = cudaGetLastError();
    if (err != cudaSuccess) return err;
  }
  return cudaSuccess;
}

}  // namespace

cudaError_t launch_gemm_simt(const Operand& A, const Operand& B, int64_t M, int Nc, int Kr,
                             bool int_acc, const Epilogue& e, cudaStream_t st, int64_t* nlaunch) {
  if (M <= 0 || Nc <= 0) return cudaSuccess;
  GemmParams p;
  p.A = A;
  p.B = B;
  p.M = M;
  p.Nc = Nc;
  p.Kr = Kr;
  p.n_tiles = 0;
  p.e = e;
  const bool narrow = Nc <= 32;  // few classes: 128x32 tiles waste less
  *nlaunch += (M + (int64_t)BM * 65535 - 1) / ((int64_t)BM * 65535);
  if (int_acc) return narrow ? launch_tn<int, 2>(p, st) : launch_tn<int, 8>(p, st);
  return narrow ? launch_tn<float, 2>(p, st) : launch_tn<float, 8>(p, st);
}

}  // namespace hdc
