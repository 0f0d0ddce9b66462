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
  const void* levels;  // uint8_t (Q <= 256) or uint16_t level indices
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
  uint32_t mul_hi16;  // 0x0101: the dp2a selectors, passed at run time so that they are not strength-reduced
  uint32_t mul128;    // 0x8080: dp2a selectors "times 128" of the sparse path
  int rows_aligned;   // F % 4 == 0, ldl % 4 == 0 and a 4-byte aligned base: level rows are read as words
  int chunk;          // 16-bit levels on the fast kernel: features staged per pass (multiple of 64)
};

// NP = number of counter planes (p + 1 with 2^p > F); S = samples per warp iteration; LT = type of the
// level indices (uint16_t for Q > 256: PAPER.md L255 tunes the number of levels up to 814)
template <int NP, int S, typename LT>
__global__ void __launch_bounds__(NTHREADS, 1) levelid_kernel(const LevelIdParams p) {
  extern __shared__ __align__(16) uint8_t smem[];
  uint32_t* sID = reinterpret_cast<uint32_t*>(smem);                 // [F][SW]
  uint32_t* sLV = sID + (p.tables_in_smem ? (size_t)p.F * SW : 0);    // [Q][SW]
  LT* sLvl = reinterpret_cast<LT*>(sLV + (p.tables_in_smem ? (size_t)p.Q * SW : 0));

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
        sLvl[s * p.Fpad + f] = (n < p.N && f < p.F) ? __ldg(static_cast<const LT*>(p.levels) + n * p.ldl + f) : (LT)0;
    }
    __syncthreads();

    uint32_t pl[S][NP];
#pragma unroll
    for (int j = 0; j < S; ++j)
#pragma unroll
      for (int i = 0; i < NP; ++i) pl[j][i] = ((init >> i) & 1u) ? 0xffffffffu : 0u;

    const LT* myl = sLvl + (size_t)(warp * S) * p.Fpad;
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

// ---------------------------------------------------------------------------------------------
// Fast path (uint8 levels, F < 1024, tables + one batch fit in shared memory; word loads of the level
// rows): same mapping (CTA = 1024-bit slice, lane = word, warp = FS samples at a time) with the
// instruction stream cut to what the counter needs:
//   * levels are staged as 16-bit table byte-offsets (level << 7), two per word, read by the warp
//     as broadcast 16-byte loads; the LV address is one LOP3 (low half) or one IMAD.HI (high half,
//     FMA pipe) -- no 64-bit address arithmetic, no predication in the loop;
//   * features go in blocks of 64 (then 32, 16, 1): four 16-input CSA trees (30 LOP3 each) whose
//     weight-16 carries meet in three more CSAs, so the ripple into the upper planes runs once per
//     64 features;
//   * the next batch's level bytes are prefetched into registers before the block loop, so the
//     only exposed staging cost is the conversion between two barriers.
// ALU ops per (feature, sample, word): 1 bind XOR + 1.875 + 0.25 counter = 3.1 (addresses are dp2a).
constexpr int FS = 4;                   // samples per warp
constexpr int FWARPS = 12;              // warps per CTA (3 per scheduler; 166 registers x 384 threads fit)
constexpr int FTHREADS = FWARPS * 32;
constexpr int FSB = FWARPS * FS;        // samples per batch (48)
constexpr int PF_ROW = 8;               // prefetched level words per lane per sample row (F <= 1024)
constexpr int PF_MAX = FS * PF_ROW;

// 16 inputs of weight 2^OFF into planes OFF..OFF+3; returns the carry of weight 2^(OFF+4)
template <int NP, int OFF>
__device__ __forceinline__ uint32_t tree16o(uint32_t (&q)[NP], const uint32_t (&x)[16]) {
  uint32_t tA, tB, fA, fB, eA, eB, sx;
  HDC_CSA(tA, q[OFF], q[OFF], x[0], x[1]);
  HDC_CSA(tB, q[OFF], q[OFF], x[2], x[3]);
  HDC_CSA(fA, q[OFF + 1], q[OFF + 1], tA, tB);
  HDC_CSA(tA, q[OFF], q[OFF], x[4], x[5]);
  HDC_CSA(tB, q[OFF], q[OFF], x[6], x[7]);
  HDC_CSA(fB, q[OFF + 1], q[OFF + 1], tA, tB);
  HDC_CSA(eA, q[OFF + 2], q[OFF + 2], fA, fB);
  HDC_CSA(tA, q[OFF], q[OFF], x[8], x[9]);
  HDC_CSA(tB, q[OFF], q[OFF], x[10], x[11]);
  HDC_CSA(fA, q[OFF + 1], q[OFF + 1], tA, tB);
  HDC_CSA(tA, q[OFF], q[OFF], x[12], x[13]);
  HDC_CSA(tB, q[OFF], q[OFF], x[14], x[15]);
  HDC_CSA(fB, q[OFF + 1], q[OFF + 1], tA, tB);
  HDC_CSA(eB, q[OFF + 2], q[OFF + 2], fA, fB);
  HDC_CSA(sx, q[OFF + 3], q[OFF + 3], eA, eB);
  return sx;
}
template <int NP>
__device__ __forceinline__ uint32_t tree16(uint32_t (&q)[NP], const uint32_t (&x)[16]) {
  return tree16o<NP, 0>(q, x);
}
// adds the word c at weight 2^from into the bit-sliced counter
template <int NP>
__device__ __forceinline__ void ripple(uint32_t (&q)[NP], uint32_t c, int from) {
#pragma unroll
  for (int i = 0; i < NP; ++i) {
    if (i >= from) {
      const uint32_t t = q[i] & c;
      q[i] ^= c;
      c = t;
    }
  }
}

// VEC: level rows are word-aligned and F % 4 == 0 (plain word loads); otherwise aligned words are
// prefetched and re-aligned by fixup() (any F, any row alignment)
// L16: 16-bit level indices (PAPER.md L245 / L255: up to 1024 levels; the Micro-HD comparison tunes 814).  The staged
// offsets are then the raw indices, two per word, and the "* 128" of the table address moves into the dp2a
// selector.  A 1024-bit slice of an 814-level table is 104 KB, so the level rows of the 12 warps are staged in
// chunks of p.chunk features by plain loads behind an L1 prefetch of the next chunk issued one chunk earlier (a
// register prefetch costs 40 registers for rows that are only 2-byte aligned -- two halves per word -- and spills);
// the sparse path is left out.
template <int NP, bool VEC, bool L16, int NW>
__global__ void __launch_bounds__(NW * 32, 1) levelid_fast_kernel(const LevelIdParams p) {
  constexpr int FSB = NW * FS;      // samples per batch (shadows the 12-warp constant)
  constexpr int FWARPS = NW;
  constexpr int PFR = PF_ROW;                      // prefetched words per lane per row (8-bit levels only)
  constexpr int LB = L16 ? 2 : 1;                  // bytes per level index
  extern __shared__ __align__(16) uint8_t smem[];
  uint32_t* sID = reinterpret_cast<uint32_t*>(smem);          // [F][SW]
  uint32_t* sLV = sID + (size_t)p.F * SW;                      // [Q][SW]
  uint32_t* sOff = sLV + (size_t)p.Q * SW;                     // [FSB][Fp2] packed 16-bit offsets
  const int Fp2 = p.Fpad;                                      // words per staged row (multiple of 8)
  uint32_t* sBase = sOff + (size_t)FSB * Fp2;                  // [NP][SW] counter planes of the all-level-0 sample

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  constexpr int P = NP - 1;
  const uint32_t init = (1u << P) - (uint32_t)(p.F / 2 + 1);
  const uint32_t lane4 = (uint32_t)lane * 4u;
  const uint32_t sel_id = p.mul128 & 0x0080u, sel_lv = p.mul128 & 0x8000u;      // (16-bit half) * 128
  // dp2a byte selectors (run-time: not folded): staged half * 1 (8-bit levels, pre-multiplied) or * 128 (L16)
  const uint32_t sel_lo = L16 ? sel_id : (p.mul_hi16 & 0x0001u), sel_hi = L16 ? sel_lv : (p.mul_hi16 & 0x0100u);
  const int RB = p.F * LB;                                     // bytes of a level row
  const int F4 = (RB + 3) >> 2;                                // level words per sample row (last one zero-padded)

  const int64_t units = (int64_t)p.n_slices * p.n_batches;
  const int64_t u_begin = units * blockIdx.x / gridDim.x;
  const int64_t u_end = units * (blockIdx.x + 1) / gridDim.x;
  int cur_slice = -1;

  // Each warp stages the level rows of its own FS samples (lanes stride over the row's words), so
  // a unit needs no block-wide barrier unless the slice -- and with it the tables -- changes.
  uint32_t pf[FS * PFR];
  auto prefetch = [&](int64_t u) {
    const int64_t n0 = (u % p.n_batches) * FSB + warp * FS;
#pragma unroll
    for (int j = 0; j < FS; ++j) {
      const int64_t n = n0 + j;
      if (VEC) {
        const uint32_t* row = reinterpret_cast<const uint32_t*>(static_cast<const uint8_t*>(p.levels) +
                                                                (n < p.N ? n : 0) * p.ldl);
#pragma unroll
        for (int i = 0; i < PF_ROW; ++i) {
          const int g = lane + 32 * i;
          pf[j * PF_ROW + i] = (g < F4 && n < p.N) ? __ldg(row + g) : 0u;
        }
        continue;
      }
      // raw ALIGNED words covering the row (the loads have no dependants here: they stay in flight
      // during the previous unit's arithmetic); row-relative words are formed by fixup() a unit later
      const uint8_t* rowb = static_cast<const uint8_t*>(p.levels) + (n < p.N ? n : 0) * p.ldl * LB;
      const uint32_t off = (uint32_t)(reinterpret_cast<uintptr_t>(rowb) & 3u);
      const uint32_t* row = reinterpret_cast<const uint32_t*>(rowb - off);
      const int nwords = (int)((off + (uint32_t)RB + 3u) >> 2);   // aligned words that hold the row
#pragma unroll
      for (int i = 0; i < PFR; ++i) {
        const int g = lane + 32 * i;
        uint32_t v = 0u;
        if (g < nwords && n < p.N) {
          if (g + 1 < nwords || n + 1 < p.N || ((off + (uint32_t)RB) & 3u) == 0u) {
            v = __ldg(row + g);
          } else {  // last word of the last row: do not read past the end of the caller's buffer
            const int nb = (int)((off + (uint32_t)RB) & 3u);
            for (int b2 = 0; b2 < nb; ++b2)
              v |= (uint32_t)__ldg(reinterpret_cast<const uint8_t*>(row + g) + b2) << (8 * b2);
          }
        }
        pf[j * PFR + i] = v;
      }
    }
  };
  // pf[] of sample j: aligned words -> words relative to the row start, bytes >= F zeroed (level 0)
  auto fixup = [&](int64_t u) {
    if (VEC) return;
    const int64_t n0 = (u % p.n_batches) * FSB + warp * FS;
#pragma unroll
    for (int j = 0; j < FS; ++j) {
      const int64_t n = n0 + j;
      const uint8_t* rowb = static_cast<const uint8_t*>(p.levels) + (n < p.N ? n : 0) * p.ldl * LB;
      const uint32_t sh = (uint32_t)(reinterpret_cast<uintptr_t>(rowb) & 3u) * 8u;  // warp-uniform
      if (sh != 0u) {
#pragma unroll
        for (int i = 0; i < PFR; ++i) {
          const uint32_t lo = pf[j * PFR + i];
          uint32_t hi = __shfl_down_sync(0xffffffffu, lo, 1);                       // word of lane + 1
          const uint32_t nxt = i + 1 < PFR ? pf[j * PFR + (i + 1 < PFR ? i + 1 : i)] : 0u;
          const uint32_t wrap = __shfl_sync(0xffffffffu, nxt, 0);                   // lane 0 of the next round
          if (lane == 31) hi = wrap;
          pf[j * PFR + i] = __funnelshift_r(lo, hi, sh);
        }
      }
      if (RB & 3) {
#pragma unroll
        for (int i = 0; i < PFR; ++i) {
          const int g = lane + 32 * i;
          if (4 * g + 4 > RB) pf[j * PFR + i] &= (4 * g < RB) ? ((1u << (8 * (RB - 4 * g))) - 1u) : 0u;
        }
      }
    }
  };
  if (!L16 && u_begin < u_end) prefetch(u_begin);

  for (int64_t u = u_begin; u < u_end; ++u) {
    const int slice = (int)(u / p.n_batches);
    const int64_t batch = u - (int64_t)slice * p.n_batches;
    const int w_glob = slice * SW + lane;
    if (slice != cur_slice) {
      __syncthreads();  // everyone is done with the previous slice's tables
      for (int f = warp; f < p.F; f += FWARPS)
        sID[f * SW + lane] = w_glob < p.W ? __ldg(p.ID + (int64_t)f * p.ldid + w_glob) : 0u;
      for (int q = warp; q < p.Q; q += FWARPS)
        sLV[q * SW + lane] = w_glob < p.W ? __ldg(p.LV + (int64_t)q * p.ldlv + w_glob) : 0u;
      cur_slice = slice;
      __syncthreads();
      if (warp == 0) {  // counter planes of a sample whose features are all at level 0 (sparse path)
        uint32_t bp[NP];
#pragma unroll
        for (int i = 0; i < NP; ++i) bp[i] = 0u;
        const uint32_t l0 = sLV[lane];
        int f = 0;
        for (; f + 16 <= p.F; f += 16) {
          uint32_t x[16];
#pragma unroll
          for (int i = 0; i < 16; ++i) x[i] = sID[(f + i) * SW + lane] ^ l0;
          ripple(bp, tree16(bp, x), 4);
        }
        for (; f < p.F; ++f) ripple(bp, sID[f * SW + lane] ^ l0, 0);
#pragma unroll
        for (int i = 0; i < NP; ++i) sBase[i * SW + lane] = bp[i];
      }
      __syncthreads();
    }
    __syncwarp();  // this warp is done reading its rows of the previous unit
    if (!L16) fixup(u);

    // ---- sparse path (level 0 is the common level: C3's images are ~80 % zeros) ------------------
    // cnt = sum_f b(f, x_f) = base + sum_{f in L} (b(f, x_f) - b(f, 0)) for any list L holding every
    // feature with x_f != 0, base = sum_f b(f, 0).  With a = b(f, x), z = b(f, 0):
    // a - z = (a + ~z) - 1 and a + ~z = E + 2 G, E = ~(LV_x ^ LV_0) (the ID word cancels),
    // G = (ID ^ LV_x) & ~(ID ^ LV_0): one weight-1 and one weight-2 input per listed feature, and
    // the counter starts at base + init - |L|.  Exact for every input; chosen per warp when fewer
    // than 40 % of its FS samples' features are nonzero (the dense path costs 3.1 LOP3 per
    // feature, this one 6.3 per listed feature).
    if (!L16) {
      int nz = 0, nz_max = 0;
#pragma unroll
      for (int j = 0; j < FS; ++j) {
        int cj = 0;
#pragma unroll
        for (int i = 0; i < PF_ROW; ++i) {
          const uint32_t v = pf[j * PF_ROW + i];
          cj += __popc((v | ((v & 0x7f7f7f7fu) + 0x7f7f7f7fu)) & 0x80808080u);
        }
#pragma unroll
        for (int off = 16; off; off >>= 1) cj += __shfl_xor_sync(0xffffffffu, cj, off);
        nz += cj;
        nz_max = cj > nz_max ? cj : nz_max;
      }
      // (a padded list must also fit the F words set aside for it)
      if (nz * 5 < 2 * FS * p.F && nz_max + 32 <= p.F) {
        uint32_t* raw = sOff + (size_t)(warp * FS) * Fp2;   // this warp's region: FS*F4 raw words ...
        uint32_t* list = raw + FS * F4;                      // ... then one list of up to F entries
#pragma unroll
        for (int j = 0; j < FS; ++j)
#pragma unroll
          for (int i = 0; i < PF_ROW; ++i) {
            const int g = lane + 32 * i;
            if (g < F4) raw[j * F4 + g] = pf[j * PF_ROW + i];
          }
        __syncwarp();
        if (u + 1 < u_end) prefetch(u + 1);
        const uint32_t l0 = sLV[lane];
        const char* idb = reinterpret_cast<const char*>(sID);
        const char* lvb2 = reinterpret_cast<const char*>(sLV);
        const uint32_t omask =
            (w_glob == p.W - 1 && (p.D_eff & 31)) ? ((1u << (p.D_eff & 31)) - 1u) : 0xffffffffu;
#pragma unroll 1
        for (int j = 0; j < FS; ++j) {
          const int64_t n = batch * FSB + warp * FS + j;
          if (n >= p.N) break;
          // list of (feature | level << 16) of the nonzero features, padded with level-0 entries
          uint32_t wv[PF_ROW];
          int c = 0;
#pragma unroll
          for (int i = 0; i < PF_ROW; ++i) {
            const int g = lane + 32 * i;
            wv[i] = g < F4 ? raw[j * F4 + g] : 0u;
            c += __popc((wv[i] | ((wv[i] & 0x7f7f7f7fu) + 0x7f7f7f7fu)) & 0x80808080u);
          }
          int pos = c;
#pragma unroll
          for (int off = 1; off < 32; off <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, pos, off);
            if (lane >= off) pos += t;
          }
          const int nnz = __shfl_sync(0xffffffffu, pos, 31);
          pos -= c;  // exclusive
#pragma unroll
          for (int i = 0; i < PF_ROW; ++i) {
#pragma unroll
            for (int b = 0; b < 4; ++b) {
              const uint32_t lvl = (wv[i] >> (8 * b)) & 0xffu;
              if (lvl) list[pos++] = (uint32_t)(4 * (lane + 32 * i) + b) | (lvl << 16);
            }
          }
          const int nl = (nnz + 31) & ~31;
          for (int k2 = nnz + lane; k2 < nl; k2 += 32) list[k2] = 0u;   // feature 0 at level 0: contributes 0
          __syncwarp();
          // counter = base + (init - nl)
          uint32_t q[NP];
          {
            const uint32_t kc = (init - (uint32_t)nl) & ((1u << NP) - 1u);
            uint32_t carry = 0u;
#pragma unroll
            for (int i = 0; i < NP; ++i) {
              const uint32_t bw = sBase[i * SW + lane];
              const uint32_t kb = ((kc >> i) & 1u) ? 0xffffffffu : 0u;
              q[i] = bw ^ kb ^ carry;
              carry = (bw & kb) | ((bw ^ kb) & carry);
            }
          }
#pragma unroll 1
          for (int e0 = 0; e0 < nl; e0 += 32) {
            uint32_t sxE[2], sxG[2];
#pragma unroll
            for (int hf = 0; hf < 2; ++hf) {
              uint32_t E[16], G[16];
              const uint4* lp = reinterpret_cast<const uint4*>(list + e0 + 16 * hf);
#pragma unroll
              for (int v4 = 0; v4 < 4; ++v4) {
                const uint4 en = lp[v4];
                const uint32_t ent[4] = {en.x, en.y, en.z, en.w};
#pragma unroll
                for (int t = 0; t < 4; ++t) {
                  const uint32_t idw = *reinterpret_cast<const uint32_t*>(idb + __dp2a_lo(ent[t], sel_id, lane4));
                  const uint32_t lvw = *reinterpret_cast<const uint32_t*>(lvb2 + __dp2a_lo(ent[t], sel_lv, lane4));
                  E[4 * v4 + t] = ~(lvw ^ l0);
                  G[4 * v4 + t] = (idw ^ lvw) & ~(idw ^ l0);
                }
              }
              sxE[hf] = tree16o<NP, 0>(q, E);   // weight-1 inputs: carry of weight 16
              sxG[hf] = tree16o<NP, 1>(q, G);   // weight-2 inputs: carry of weight 32
            }
            uint32_t c32, c64a, s32, c128;
            HDC_CSA(c32, q[4], q[4], sxE[0], sxE[1]);
            HDC_CSA(c64a, s32, c32, sxG[0], sxG[1]);
            const uint32_t c64b = q[5] & s32;
            q[5] ^= s32;
            HDC_CSA(c128, q[6], q[6], c64a, c64b);
            ripple(q, c128, 7);
          }
          if (w_glob < p.W) p.Hbits[n * p.ldh + w_glob] = q[P] & omask;
          __syncwarp();  // the list is rebuilt for the next sample
        }
        continue;
      }
    }

    if (!L16) {
      // four level bytes -> two words of 16-bit offsets (level * 128)
#pragma unroll
      for (int j = 0; j < FS; ++j) {
#pragma unroll
        for (int i = 0; i < PF_ROW; ++i) {
          const int g = lane + 32 * i;
          if (g < F4) {
            const uint32_t v = pf[j * PF_ROW + i];
            uint2 o;
            o.x = ((v & 0xffu) << 7) | ((v & 0xff00u) << 15);
            o.y = ((v >> 9) & 0x7f80u) | ((v >> 1) & 0x7f800000u);
            *reinterpret_cast<uint2*>(sOff + (size_t)(warp * FS + j) * Fp2 + 2 * g) = o;
          }
        }
      }
      __syncwarp();
      if (u + 1 < u_end) prefetch(u + 1);
    }

    uint32_t pl[FS][NP];
#pragma unroll
    for (int j = 0; j < FS; ++j)
#pragma unroll
      for (int i = 0; i < NP; ++i) pl[j][i] = ((init >> i) & 1u) ? 0xffffffffu : 0u;

    const char* lvb = reinterpret_cast<const char*>(sLV);
    const uint32_t* myo = sOff + (size_t)(warp * FS) * Fp2;

    // bound words of 16 features of sample j starting at (chunk-relative) feature f (f % 16 == 0)
    auto bind16 = [&](int f, int j, const uint32_t (&idw)[16], uint32_t (&x)[16]) {
      const uint4* op = reinterpret_cast<const uint4*>(myo + (size_t)j * Fp2 + (f >> 1));
      const uint4 oa = op[0], ob = op[1];
      const uint32_t o[8] = {oa.x, oa.y, oa.z, oa.w, ob.x, ob.y, ob.z, ob.w};
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        // byte offset of the level row + lane word: 16-bit half of o times 1 (times 128 for raw 16-bit indices)
        // plus lane4 as one dp2a (integer dot-product pipe, not the ALU pipe that the LOP3s saturate)
        const uint32_t a_lo = __dp2a_lo(o[i], sel_lo, lane4);
        const uint32_t a_hi = __dp2a_lo(o[i], sel_hi, lane4);
        x[2 * i] = idw[2 * i] ^ *reinterpret_cast<const uint32_t*>(lvb + a_lo);
        x[2 * i + 1] = idw[2 * i + 1] ^ *reinterpret_cast<const uint32_t*>(lvb + a_hi);
      }
    };
    // 8-bit levels: the whole row is staged (one chunk).  16-bit levels: the rows are staged in chunks of
    // p.chunk features (a multiple of 64) straight from global memory, so that 12 warps' rows fit beside an
    // up-to-1024-level table slice; the other warps of the scheduler cover the load latency.
    const int CH = L16 ? p.chunk : p.F;
#pragma unroll 1
    for (int f0 = 0; f0 < p.F; f0 += CH) {
      const int fc = p.F - f0 < CH ? p.F - f0 : CH;   // features of this chunk
      if (L16) {
        __syncwarp();  // the previous chunk's offsets have been read
        const int64_t n0 = batch * FSB + warp * FS;
#pragma unroll
        for (int j = 0; j < FS; ++j) {
          const int64_t n = n0 + j;
          const uint16_t* row = static_cast<const uint16_t*>(p.levels) + (n < p.N ? n : 0) * p.ldl + f0;
          const bool word_ok = (reinterpret_cast<uintptr_t>(row) & 3u) == 0u;   // warp-uniform
          for (int g = lane; g < Fp2; g += 32) {
            uint32_t v = 0u;
            if (n < p.N) {
              if (word_ok && 2 * g + 1 < fc) {
                v = __ldg(reinterpret_cast<const uint32_t*>(row) + g);
              } else {
                if (2 * g < fc) v = __ldg(row + 2 * g);
                if (2 * g + 1 < fc) v |= (uint32_t)__ldg(row + 2 * g + 1) << 16;
              }
            }
            sOff[(size_t)(warp * FS + j) * Fp2 + g] = v;
          }
        }
        __syncwarp();
        // The next chunk of this warp's rows (of this unit or the next) is pulled into L1 / L2 while this one is
        // computed: every warp of the CTA reaches its staging loads at the same time (equal work per batch), so the
        // other warps do not cover their latency (ncu: a third of the stall samples sat behind those loads).
        {
          const bool same = f0 + CH < p.F;
          if (same || u + 1 < u_end) {
            const int64_t nb = same ? batch : (u + 1) % p.n_batches;
            const int nf0 = same ? f0 + CH : 0;
            const int nfc = p.F - nf0 < CH ? p.F - nf0 : CH;
            const int j = lane >> 3, ln = lane & 7;                  // 8 lanes per row, one 128-byte line each
            const int64_t n = nb * FSB + warp * FS + j;
            if (j < FS && n < p.N && ln * 64 < nfc + 64) {   // (rows are not line-aligned: the last element's line too)
              const int e = ln * 64 < nfc ? ln * 64 : nfc - 1;
              const uint16_t* a = static_cast<const uint16_t*>(p.levels) + n * p.ldl + nf0 + e;
              asm volatile("prefetch.global.L1 [%0];" ::"l"(a));
            }
          }
        }
      }
      const uint32_t* idp = sID + (size_t)f0 * SW + lane;
      int f = 0;
      // 64 features: four 16-input trees, their weight-16 carries folded by three more CSAs, so the
      // ripple into the upper planes runs once per 64 features
#pragma unroll 1
      for (; f + 64 <= fc; f += 64) {
        uint32_t sxs[FS][3];
#pragma unroll
        for (int q4 = 0; q4 < 4; ++q4) {
          uint32_t idw[16];
#pragma unroll
          for (int i = 0; i < 16; ++i) idw[i] = idp[(f + 16 * q4 + i) * SW];
#pragma unroll
          for (int j = 0; j < FS; ++j) {
            uint32_t x[16];
            bind16(f + 16 * q4, j, idw, x);
            const uint32_t sx = tree16(pl[j], x);
            if (q4 < 3) {
              sxs[j][q4] = sx;
            } else {
              uint32_t ca, cb, c64;
              HDC_CSA(ca, pl[j][4], pl[j][4], sxs[j][0], sxs[j][1]);
              HDC_CSA(cb, pl[j][4], pl[j][4], sxs[j][2], sx);
              HDC_CSA(c64, pl[j][5], pl[j][5], ca, cb);
              ripple(pl[j], c64, 6);
            }
          }
        }
      }
#pragma unroll 1
      for (; f + 32 <= fc; f += 32) {
        uint32_t sxa[FS];
        {
          uint32_t idw[16];
#pragma unroll
          for (int i = 0; i < 16; ++i) idw[i] = idp[(f + i) * SW];
#pragma unroll
          for (int j = 0; j < FS; ++j) {
            uint32_t x[16];
            bind16(f, j, idw, x);
            sxa[j] = tree16(pl[j], x);
          }
        }
        {
          uint32_t idw[16];
#pragma unroll
          for (int i = 0; i < 16; ++i) idw[i] = idp[(f + 16 + i) * SW];
#pragma unroll
          for (int j = 0; j < FS; ++j) {
            uint32_t x[16];
            bind16(f + 16, j, idw, x);
            const uint32_t sxb = tree16(pl[j], x);
            uint32_t c32;
            HDC_CSA(c32, pl[j][4], pl[j][4], sxa[j], sxb);
            ripple(pl[j], c32, 5);
          }
        }
      }
      if (f + 16 <= fc) {
        uint32_t idw[16];
#pragma unroll
        for (int i = 0; i < 16; ++i) idw[i] = idp[(f + i) * SW];
#pragma unroll
        for (int j = 0; j < FS; ++j) {
          uint32_t x[16];
          bind16(f, j, idw, x);
          ripple(pl[j], tree16(pl[j], x), 4);
        }
        f += 16;
      }
      for (; f < fc; ++f) {  // remainder features: plain ripple add
        const uint32_t idw = idp[f * SW];
#pragma unroll
        for (int j = 0; j < FS; ++j) {
          const uint32_t o = myo[(size_t)j * Fp2 + (f >> 1)];
          const uint32_t hv = ((f & 1) ? (o >> 16) : o) & 0xffffu;
          const uint32_t a = L16 ? (hv * 128u + lane4) : (hv | lane4);
          ripple(pl[j], idw ^ *reinterpret_cast<const uint32_t*>(lvb + a), 0);
        }
      }
    }

    if (w_glob < p.W) {
      const uint32_t mask = (w_glob == p.W - 1 && (p.D_eff & 31)) ? ((1u << (p.D_eff & 31)) - 1u) : 0xffffffffu;
      const int64_t n0 = batch * FSB;
#pragma unroll
      for (int j = 0; j < FS; ++j) {
        const int64_t n = n0 + warp * FS + j;
        if (n < p.N) p.Hbits[n * p.ldh + w_glob] = pl[j][P] & mask;
      }
    }
  }
}

template <int NP, int S, typename LT>
cudaError_t launch_t(const LevelIdParams& p, int grid, size_t smem, cudaStream_t st) {
  cudaError_t e = cudaFuncSetAttribute(levelid_kernel<NP, S, LT>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                       (int)smem);
  if (e != cudaSuccess) return e;
  levelid_kernel<NP, S, LT><<<grid, NTHREADS, smem, st>>>(p);
  return cudaGetLastError();
}

}  // namespace

cudaError_t launch_levelid(const void* levels, int lvl16, int64_t N, int F, int64_t ldl, const uint32_t* ID,
                           int64_t ldid, const uint32_t* LV, int Q, int64_t ldlv, int D_eff,
                           uint32_t* Hbits, int64_t ldh, int sm_count, int smem_optin, cudaStream_t st,
                           int64_t* nlaunch) {
  if (N <= 0) return cudaSuccess;
  constexpr int S = 4;
  {  // fast path
    const size_t fp2 = (size_t)round_up((F + 1) / 2, 8);
    const size_t smem_fast = ((size_t)F + Q) * SW * 4 + (size_t)FSB * fp2 * 4 + (size_t)11 * SW * 4;
    if (!lvl16 && F <= 1020 && smem_fast <= (size_t)smem_optin) {  // (+3 bytes of row misalignment fit the prefetch)
      LevelIdParams p;
      p.levels = levels; p.N = N; p.F = F; p.ldl = ldl;
      p.ID = ID; p.ldid = ldid; p.LV = LV; p.Q = Q; p.ldlv = ldlv;
      p.D_eff = D_eff; p.W = words_of(D_eff);
      p.Hbits = Hbits; p.ldh = ldh;
      p.n_slices = (p.W + SW - 1) / SW;
      p.n_batches = (N + FSB - 1) / FSB;
      p.Fpad = (int)fp2;
      p.tables_in_smem = 1;
      p.mul_hi16 = 0x0101u;
      p.mul128 = 0x8080u;
      p.rows_aligned = (F % 4 == 0 && (ldl & 3) == 0 && (reinterpret_cast<uintptr_t>(levels) & 3) == 0) ? 1 : 0;
      p.chunk = F;
      const int64_t units = (int64_t)p.n_slices * p.n_batches;
      const int grid = (int)(units < sm_count ? units : sm_count);
      cudaError_t e = cudaFuncSetAttribute(levelid_fast_kernel<11, true, false, FWARPS>,
                                           cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_fast);
      if (e == cudaSuccess)
        e = cudaFuncSetAttribute(levelid_fast_kernel<11, false, false, FWARPS>,
                                 cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_fast);
      if (e != cudaSuccess) return e;
      ++*nlaunch;
      if (p.rows_aligned) levelid_fast_kernel<11, true, false, FWARPS><<<grid, FTHREADS, smem_fast, st>>>(p);
      else levelid_fast_kernel<11, false, false, FWARPS><<<grid, FTHREADS, smem_fast, st>>>(p);
      return cudaGetLastError();
    }
    // 16-bit level indices: same kernel, dense path only, level rows staged in chunks of `chunk` features --
    // the largest multiple of 64 (up to 320) whose 48 rows fit beside the table slices
    if (lvl16 && F <= 1020 && Q <= 1024) {
      const size_t tab = ((size_t)F + Q) * SW * 4 + (size_t)11 * SW * 4;
      int chunk = 0;
      for (int c = 320; c >= 64 && !chunk; c -= 64)
        if (tab + (size_t)FSB * (c / 2) * 4 <= (size_t)smem_optin) chunk = c;
      if (chunk) {
        LevelIdParams p;
        p.levels = levels; p.N = N; p.F = F; p.ldl = ldl;
        p.ID = ID; p.ldid = ldid; p.LV = LV; p.Q = Q; p.ldlv = ldlv;
        p.D_eff = D_eff; p.W = words_of(D_eff);
        p.Hbits = Hbits; p.ldh = ldh;
        p.n_slices = (p.W + SW - 1) / SW;
        p.n_batches = (N + FSB - 1) / FSB;
        p.Fpad = chunk / 2;   // words per staged row
        p.chunk = chunk;
        p.tables_in_smem = 1;
        p.mul_hi16 = 0x0101u;
        p.mul128 = 0x8080u;
        p.rows_aligned = 0;
        const size_t smem_16 = tab + (size_t)FSB * p.Fpad * 4;
        const int64_t units = (int64_t)p.n_slices * p.n_batches;
        const int grid = (int)(units < sm_count ? units : sm_count);
        cudaError_t e = cudaFuncSetAttribute(levelid_fast_kernel<11, false, true, FWARPS>,
                                             cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_16);
        if (e != cudaSuccess) return e;
        ++*nlaunch;
        levelid_fast_kernel<11, false, true, FWARPS><<<grid, FTHREADS, smem_16, st>>>(p);
        return cudaGetLastError();
      }
    }
  }
  LevelIdParams p;
  p.levels = levels; p.N = N; p.F = F; p.ldl = ldl;
  p.ID = ID; p.ldid = ldid; p.LV = LV; p.Q = Q; p.ldlv = ldlv;
  p.D_eff = D_eff; p.W = words_of(D_eff);
  p.Hbits = Hbits; p.ldh = ldh;
  p.n_slices = (p.W + SW - 1) / SW;
  const int SB = NWARPS * S;
  p.n_batches = (N + SB - 1) / SB;
  p.Fpad = (int)round_up(F, 16);
  const size_t lvl_bytes = (size_t)SB * p.Fpad * (lvl16 ? 2 : 1);
  const size_t tab_bytes = ((size_t)F + Q) * SW * 4;
  p.tables_in_smem = (tab_bytes + lvl_bytes <= (size_t)smem_optin) ? 1 : 0;
  const size_t smem = lvl_bytes + (p.tables_in_smem ? tab_bytes : 0);
  if (smem > (size_t)smem_optin) return cudaErrorNotSupported;  // the staged level rows alone exceed one CTA's shared memory
  const int64_t units = (int64_t)p.n_slices * p.n_batches;
  const int grid = (int)(units < sm_count ? units : sm_count);
  ++*nlaunch;
  if (lvl16) {
    if (F < 1024) return launch_t<11, S, uint16_t>(p, grid, smem, st);
    return launch_t<17, S, uint16_t>(p, grid, smem, st);
  }
  if (F < 1024) return launch_t<11, S, uint8_t>(p, grid, smem, st);
  return launch_t<17, S, uint8_t>(p, grid, smem, st);
}

}  // namespace hdc
