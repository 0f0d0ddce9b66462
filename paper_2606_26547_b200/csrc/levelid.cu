// levelid.cu -- level-ID record encoding ("ID-based encoding", L183 N_LEVELS, L239
// "Level-ID encoding"; bind = XOR, bundle = majority per BASELINE.json north_star):
//
//   cnt[n,d] = sum_{f<F} ( ID[f,d] xor LV[levels[n,f], d] ),   bit[n,d] = [ 2*cnt[n,d] > F ]
//
// Bound: integer ALU (LOP3), not HBM -- a sample reads F bytes and writes W words but needs
// ~3.4*F*W logic ops (DESIGN.md kernel table).  Design: a CTA owns a 1024-bit slice of the
// hypervector (32 words, lane <-> word) and keeps that slice of the ID table and of the level
// table in shared memory; each warp encodes S samples at a time so that an ID word is loaded once
// per S samples.  The per-dimension count lives in a bit-sliced (vertical) counter: 16 bound
// words are folded with a carry-save-adder tree (15 CSA = 30 LOP3) and the carry-out ripples into
// the upper planes; the counter starts at 2^p - (floor(F/2)+1) so that plane p of the final sum IS
// the majority bit (no compare).  Work units are (slice, batch of samples), slice-major, split
// contiguously over a persistent grid so a CTA re-stages its tables only when its slice changes.
#include "common.cuh"

namespace hdc {
namespace {

constexpr int SW = 32;        // words per slice == lanes
constexpr int NWARPS = 8;
constexpr int NTHREADS = NWARPS * 32;

#define HDC_CSA(h, l, a, b, c)            \
  {                                       \
    const uint32_t u_ = (a) ^ (b);        \
    const uint32_t c_ = (c);              \
    (h) = ((a) & (b)) | (u_ & c_);        \
    (l) = u_ ^ c_;                        \
  }

struct LevelIdParams {
  const uint8_t* levels;
  int64_t N;
  int F;
  int64_t ldl;
  const uint32_t* ID;
  int64_t ldid;
  const uint32_t* LV;
  int Q;
  int64_t ldlv;
  int D_eff, W;
  uint32_t* Hbits;
  int64_t ldh;
  int n_slices;
  int64_t n_batches;
  int Fpad;     // staged level row stride (bytes), multiple of 16
  int tables_in_smem;
};

// NP = number of counter planes (p + 1 with 2^p > F); S = samples per warp iteration
template <int NP, int S>
__global__ void __launch_bounds__(NTHREADS, 1) levelid_kernel(const LevelIdParams p) {
  extern __shared__ __align__(16) uint8_t smem[];
  uint32_t* sID = reinterpret_cast<uint32_t*>(smem);                 // [F][SW]
  uint32_t* sLV = sID + (p.tables_in_smem ? (size_t)p.F * SW : 0);    // [Q][SW]
  uint8_t* sLvl = reinterpret_cast<uint8_t*>(sLV + (p.tables_in_smem ? (size_t)p.Q * SW : 0));

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  constexpr int SB = NWARPS * S;  // samples per batch
  constexpr int P = NP - 1;
  const uint32_t init = (1u << P) - (uint32_t)(p.F / 2 + 1);

  const int64_t units = (int64_t)p.n_slices * p.n_batches;
  const int64_t u_begin = units * blockIdx.x / gridDim.x;
  const int64_t u_end = units * (blockIdx.x + 1) / gridDim.x;
  int cur_slice = -1;

  for (int64_t u = u_begin; u < u_end; ++u) {
    const int slice = (int)(u / p.n_batches);
    const int64_t batch = u - (int64_t)slice * p.n_batches;
    const int w_glob = slice * SW + lane;
    __syncthreads();  // everyone is done with the previous unit's staged data
    if (slice != cur_slice && p.tables_in_smem) {
      for (int f = warp; f < p.F; f += NWARPS)
        sID[f * SW + lane] = w_glob < p.W ? __ldg(p.ID + (int64_t)f * p.ldid + w_glob) : 0u;
      for (int q = warp; q < p.Q; q += NWARPS)
        sLV[q * SW + lane] = w_glob < p.W ? __ldg(p.LV + (int64_t)q * p.ldlv + w_glob) : 0u;
    }
    cur_slice = slice;
    // stage the level bytes of this batch (rows past N read as level 0 and are never stored)
    const int64_t n0 = batch * SB;
    for (int s = warp; s < SB; s += NWARPS) {
      const int64_t n = n0 + s;
      for (int f = lane; f < p.Fpad; f += 32)
        sLvl[s * p.Fpad + f] = (n < p.N && f < p.F) ? __ldg(p.levels + n * p.ldl + f) : (uint8_t)0;
    }
    __syncthreads();

    uint32_t pl[S][NP];
#pragma unroll
    for (int j = 0; j < S; ++j)
#pragma unroll
      for (int i = 0; i < NP; ++i) pl[j][i] = ((init >> i) & 1u) ? 0xffffffffu : 0u;

    const uint8_t* myl = sLvl + (size_t)(warp * S) * p.Fpad;
    const uint32_t* idp = p.tables_in_smem ? sID + lane : p.ID + w_glob;
    const uint32_t* lvp = p.tables_in_smem ? sLV + lane : p.LV + w_glob;
    const int64_t idstride = p.tables_in_smem ? SW : p.ldid;
    const int64_t lvstride = p.tables_in_smem ? SW : p.ldlv;
    const bool live = p.tables_in_smem || w_glob < p.W;

    int f = 0;
    for (; f + 16 <= p.F; f += 16) {
      uint32_t x[S][16];
#pragma unroll
      for (int i = 0; i < 16; ++i) {
        const uint32_t idw = live ? idp[(int64_t)(f + i) * idstride] : 0u;
#pragma unroll
        for (int j = 0; j < S; ++j) {
          const uint32_t l = myl[j * p.Fpad + f + i];
          x[j][i] = idw ^ (live ? lvp[(int64_t)l * lvstride] : 0u);
        }
      }
#pragma unroll
      for (int j = 0; j < S; ++j) {
        uint32_t tA, tB, fA, fB, eA, eB, sx;
        HDC_CSA(tA, pl[j][0], pl[j][0], x[j][0], x[j][1]);
        HDC_CSA(tB, pl[j][0], pl[j][0], x[j][2], x[j][3]);
        HDC_CSA(fA, pl[j][1], pl[j][1], tA, tB);
        HDC_CSA(tA, pl[j][0], pl[j][0], x[j][4], x[j][5]);
        HDC_CSA(tB, pl[j][0], pl[j][0], x[j][6], x[j][7]);
        HDC_CSA(fB, pl[j][1], pl[j][1], tA, tB);
        HDC_CSA(eA, pl[j][2], pl[j][2], fA, fB);
        HDC_CSA(tA, pl[j][0], pl[j][0], x[j][8], x[j][9]);
        HDC_CSA(tB, pl[j][0], pl[j][0], x[j][10], x[j][11]);
        HDC_CSA(fA, pl[j][1], pl[j][1], tA, tB);
        HDC_CSA(tA, pl[j][0], pl[j][0], x[j][12], x[j][13]);
        HDC_CSA(tB, pl[j][0], pl[j][0], x[j][14], x[j][15]);
        HDC_CSA(fB, pl[j][1], pl[j][1], tA, tB);
        HDC_CSA(eB, pl[j][2], pl[j][2], fA, fB);
        HDC_CSA(sx, pl[j][3], pl[j][3], eA, eB);
#pragma unroll
        for (int i = 4; i < NP; ++i) {  // ripple the weight-16 carry into the upper planes
          const uint32_t t = pl[j][i] & sx;
          pl[j][i] ^= sx;
          sx = t;
        }
      }
    }
    for (; f < p.F; ++f) {  // remainder features: plain ripple add
      const uint32_t idw = live ? idp[(int64_t)f * idstride] : 0u;
#pragma unroll
      for (int j = 0; j < S; ++j) {
        const uint32_t l = myl[j * p.Fpad + f];
        uint32_t c = idw ^ (live ? lvp[(int64_t)l * lvstride] : 0u);
#pragma unroll
        for (int i = 0; i < NP; ++i) {
          const uint32_t t = pl[j][i] & c;
          pl[j][i] ^= c;
          c = t;
        }
      }
    }

    if (w_glob < p.W) {
      const uint32_t mask = (w_glob == p.W - 1 && (p.D_eff & 31)) ? ((1u << (p.D_eff & 31)) - 1u) : 0xffffffffu;
#pragma unroll
      for (int j = 0; j < S; ++j) {
        const int64_t n = n0 + warp * S + j;
        if (n < p.N) p.Hbits[n * p.ldh + w_glob] = pl[j][P] & mask;
      }
    }
  }
}

template <int NP, int S>
cudaError_t launch_t(const LevelIdParams& p, int grid, size_t smem, cudaStream_t st) {
  cudaError_t e = cudaFuncSetAttribute(levelid_kernel<NP, S>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                       (int)smem);
  if (e != cudaSuccess) return e;
  levelid_kernel<NP, S><<<grid, NTHREADS, smem, st>>>(p);
  return cudaGetLastError();
}

}  // namespace

cudaError_t launch_levelid(const uint8_t* levels, int64_t N, int F, int64_t ldl, const uint32_t* ID,
                           int64_t ldid, const uint32_t* LV, int Q, int64_t ldlv, int D_eff,
                           uint32_t* Hbits, int64_t ldh, int sm_count, int smem_optin, cudaStream_t st,
                           int64_t* nlaunch) {
  if (N <= 0) return cudaSuccess;
  constexpr int S = 4;
  LevelIdParams p;
  p.levels = levels; p.N = N; p.F = F; p.ldl = ldl;
  p.ID = ID; p.ldid = ldid; p.LV = LV; p.Q = Q; p.ldlv = ldlv;
  p.D_eff = D_eff; p.W = words_of(D_eff);
  p.Hbits = Hbits; p.ldh = ldh;
  p.n_slices = (p.W + SW - 1) / SW;
  const int SB = NWARPS * S;
  p.n_batches = (N + SB - 1) / SB;
  p.Fpad = (int)round_up(F, 16);
  const size_t lvl_bytes = (size_t)SB * p.Fpad;
  const size_t tab_bytes = ((size_t)F + Q) * SW * 4;
  p.tables_in_smem = (tab_bytes + lvl_bytes <= (size_t)smem_optin) ? 1 : 0;
  const size_t smem = lvl_bytes + (p.tables_in_smem ? tab_bytes : 0);
  if (smem > (size_t)smem_optin) return cudaErrorInvalidConfiguration;
  const int64_t units = (int64_t)p.n_slices * p.n_batches;
  const int grid = (int)(units < sm_count ? units : sm_count);
  ++*nlaunch;
  if (F < 1024) return launch_t<11, S>(p, grid, smem, st);
  return launch_t<17, S>(p, grid, smem, st);
}

}  // namespace hdc
