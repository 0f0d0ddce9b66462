// tc_ptx.cuh -- inline-PTX wrappers of the sm_100a tensor-core path shared by gemm_tc.cu and
// simtc.cu: mbarrier, TMA (cp.async.bulk.tensor), tcgen05 alloc / mma / commit / ld / fences, and
// the shared-memory / instruction descriptors of K-major 128-byte-swizzled operand tiles.
#pragma once
#include <cuda.h>
#include <stdint.h>

namespace hdc {
namespace tcp {

constexpr int KB_BYTES = 128;  // bytes of the reduction axis per k-block (one swizzle row)

// ------------------------------------------------------------------------------------ PTX
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
  return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
// Spins on the phase parity.  A wait that lasts ~2 s of SM clocks is a protocol bug: trap instead
// of hanging the device.
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  uint32_t done = 0;
  long long t0 = 0;
  for (uint32_t it = 0;; ++it) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(done)
        : "r"(bar), "r"(parity)
        : "memory");
    if (done) return;
    if ((it & 1023u) == 1023u) {
      const long long t = clock64();
      if (t0 == 0) t0 = t;
      else if (t - t0 > 4000000000LL) __trap();
    }
  }
}
// Same, polling with test_wait (never suspends the thread: lowest wake-up latency; for roles whose
// hand-offs are short compared with try_wait's suspend quantum).
__device__ __forceinline__ void mbar_wait_spin(uint32_t bar, uint32_t parity) {
  uint32_t done = 0;
  long long t0 = 0;
  for (uint32_t it = 0;; ++it) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(done)
        : "r"(bar), "r"(parity)
        : "memory");
    if (done) return;
    if ((it & 4095u) == 4095u) {
      const long long t = clock64();
      if (t0 == 0) t0 = t;
      else if (t - t0 > 4000000000LL) __trap();
    }
  }
}
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap* tm, uint32_t bar, int c0, int c1) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];"
      ::"r"(dst), "l"(reinterpret_cast<uint64_t>(tm)), "r"(bar), "r"(c0), "r"(c1)
      : "memory");
}
// ---- CTA pairs (cta_group::2) --------------------------------------------------------------
// A shared::cta address is also the shared::cluster address of the same location in the executing
// CTA; clearing bit 24 gives the same offset in the even (leader) CTA of the pair.
constexpr uint32_t PEER_MASK = 0xFEFFFFFFu;
__device__ __forceinline__ uint32_t cluster_ctarank() {
  // the compiler intrinsic (not inline asm): the value is known to be warp-uniform, which keeps the
  // code it guards on the uniform datapath
  return __clusterRelativeBlockRank();
}
__device__ __forceinline__ void cluster_sync_all() {
  asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
  asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive_cluster(uint32_t cluster_addr) {
  asm volatile("mbarrier.arrive.release.cluster.shared::cluster.b64 _, [%0];" ::"r"(cluster_addr) : "memory");
}
// Arrival on a barrier of another CTA of the cluster with the default semantics (release at CTA scope): for a
// hand-off whose data was written to THIS CTA's shared memory and made visible to the async proxy by
// fence.proxy.async (the tensor core that reads it is this SM's own, driven by the pair's leader), so that no
// cluster- or GPU-scope memory barrier is needed in front of the arrive.
__device__ __forceinline__ void mbar_arrive_remote(uint32_t cluster_addr) {
  asm volatile("mbarrier.arrive.shared::cluster.b64 _, [%0];" ::"r"(cluster_addr) : "memory");
}
// Same without memory ordering.  For hand-offs that publish no generic-proxy memory: an epilogue warp
// returning a TMEM accumulator has already waited for its tcgen05.ld (tcgen05.wait::ld) and fenced the
// tensor proxy (tcgen05.fence::before_thread_sync).  The .release.cluster form compiles to MEMBAR.ALL.GPU +
// ERRBAR in front of the arrive, which makes the warp wait for the acknowledgement of its global stores of
// the tile on every hand-off (measured: profiles/r2_encode_epilogue.md).
__device__ __forceinline__ void mbar_arrive_cluster_relaxed(uint32_t cluster_addr) {
  asm volatile("mbarrier.arrive.relaxed.cluster.shared::cluster.b64 _, [%0];" ::"r"(cluster_addr) : "memory");
}
// each CTA of the pair loads into its own shared memory; the bytes complete on `bar` (a
// shared::cluster address, normally the leader's barrier)
__device__ __forceinline__ void tma_load_2d_2sm(uint32_t dst, const CUtensorMap* tm, uint32_t bar, int c0, int c1) {
  asm volatile(
      "cp.async.bulk.tensor.2d.cta_group::2.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];"
      ::"r"(dst), "l"(reinterpret_cast<uint64_t>(tm)), "r"(bar), "r"(c0), "r"(c1)
      : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
template <int CG = 1>
__device__ __forceinline__ void tc_commit(uint32_t bar) {
  if (CG == 2) {  // arrives on the barrier at this offset in both CTAs of the pair
    asm volatile(
        "tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;"
        ::"r"(bar), "h"((uint16_t)3)
        : "memory");
  } else {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
  }
}
template <bool INT8, int CG = 1>
__device__ __forceinline__ void tc_mma(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc,
                                       uint32_t accumulate) {
  if (CG == 2) {
    if (INT8) {
      asm volatile(
          "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
          "tcgen05.mma.cta_group::2.kind::i8 [%0], %1, %2, %3, p;\n\t}"
          ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate)
          : "memory");
    } else {
      asm volatile(
          "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
          "tcgen05.mma.cta_group::2.kind::f16 [%0], %1, %2, %3, p;\n\t}"
          ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate)
          : "memory");
    }
    return;
  }
  if (INT8) {
    asm volatile(
        "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::i8 [%0], %1, %2, %3, p;\n\t}"
        ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate)
        : "memory");
  } else {
    asm volatile(
        "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
        ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate)
        : "memory");
  }
}
// ---- warp-converged single-issue forms -------------------------------------------------------
// tcgen05.mma / tcgen05.commit / cp.async.bulk.tensor execute once per warp (uniform datapath).
// Written under `if (lane == 0)` ptxas wraps each one in an ELECT / R2UR.BROADCAST / BRA.U.ANY
// loop (~100 issue cycles apiece, measured: profiles/r1_tcgen05_path.md); predicated by the result
// of elect.sync inside the same asm block, in a fully converged warp, it emits the bare
// instruction.  All *_elect functions must be called by all 32 lanes of a converged warp with
// warp-uniform arguments.
__device__ __forceinline__ void mbar_arrive_expect_tx_elect(uint32_t bar, uint32_t bytes) {
  asm volatile(
      "{\n\t.reg .pred q;\n\telect.sync _|q, 0xffffffff;\n\t"
      "@q mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n\t}" ::"r"(bar), "r"(bytes)
      : "memory");
}
__device__ __forceinline__ void tma_load_2d_elect(uint32_t dst, const CUtensorMap* tm, uint32_t bar, int c0, int c1) {
  asm volatile(
      "{\n\t.reg .pred q;\n\telect.sync _|q, 0xffffffff;\n\t"
      "@q cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];\n\t}"
      ::"r"(dst), "l"(reinterpret_cast<uint64_t>(tm)), "r"(bar), "r"(c0), "r"(c1)
      : "memory");
}
__device__ __forceinline__ void tma_load_2d_2sm_elect(uint32_t dst, const CUtensorMap* tm, uint32_t bar, int c0,
                                                      int c1) {
  asm volatile(
      "{\n\t.reg .pred q;\n\telect.sync _|q, 0xffffffff;\n\t"
      "@q cp.async.bulk.tensor.2d.cta_group::2.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];\n\t}"
      ::"r"(dst), "l"(reinterpret_cast<uint64_t>(tm)), "r"(bar), "r"(c0), "r"(c1)
      : "memory");
}
template <int CG = 1>
__device__ __forceinline__ void tc_commit_elect(uint32_t bar) {
  if (CG == 2) {
    asm volatile(
        "{\n\t.reg .pred q;\n\telect.sync _|q, 0xffffffff;\n\t"
        "@q tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;\n\t}"
        ::"r"(bar), "h"((uint16_t)3)
        : "memory");
  } else {
    asm volatile(
        "{\n\t.reg .pred q;\n\telect.sync _|q, 0xffffffff;\n\t"
        "@q tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];\n\t}" ::"r"(bar)
        : "memory");
  }
}
#define HDC_MMA_ELECT(CGS, KIND)                                                                     \
  asm volatile(                                                                                      \
      "{\n\t.reg .pred p, q;\n\telect.sync _|q, 0xffffffff;\n\tsetp.ne.b32 p, %4, 0;\n\t"            \
      "@q tcgen05.mma.cta_group::" CGS ".kind::" KIND " [%0], %1, %2, %3, p;\n\t}" ::"r"(d_tmem),    \
      "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate)                                            \
      : "memory")
template <bool INT8, int CG = 1>
__device__ __forceinline__ void tc_mma_elect(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc,
                                             uint32_t accumulate) {
  if (CG == 2) {
    if (INT8) HDC_MMA_ELECT("2", "i8");
    else HDC_MMA_ELECT("2", "f16");
  } else {
    if (INT8) HDC_MMA_ELECT("1", "i8");
    else HDC_MMA_ELECT("1", "f16");
  }
}
#undef HDC_MMA_ELECT
// A operand in tensor memory (lane = row of the 128-row tile, each 32-bit column = 32 bits of the row's K-major
// elements; one MMA reads 8 columns), B from shared memory; one CTA
#define HDC_MMA_TS_ELECT(KIND)                                                                       \
  asm volatile(                                                                                      \
      "{\n\t.reg .pred p, q;\n\telect.sync _|q, 0xffffffff;\n\tsetp.ne.b32 p, %4, 0;\n\t"            \
      "@q tcgen05.mma.cta_group::1.kind::" KIND " [%0], [%1], %2, %3, p;\n\t}" ::"r"(d_tmem),           \
      "r"(a_tmem), "l"(bdesc), "r"(idesc), "r"(accumulate)                                           \
      : "memory")
template <bool INT8>
__device__ __forceinline__ void tc_mma_ts_elect(uint32_t d_tmem, uint32_t a_tmem, uint64_t bdesc, uint32_t idesc,
                                                uint32_t accumulate) {
  if (INT8) HDC_MMA_TS_ELECT("i8");
  else HDC_MMA_TS_ELECT("f16");
}
#undef HDC_MMA_TS_ELECT
// The four MMAs of one k-block (4 x 32 bytes of the reduction axis) in one block: one election, the descriptors of
// the class tile built from the 32-bit address field (the upper half of a 128-byte-swizzled K-major descriptor is the
// constant 0x40004040: SBO 1024, version 1, SWIZZLE_128B), A advancing 8 TMEM columns per MMA.  b_lo = lower half of
// smem_desc() of the k-block; first == 0: the first MMA overwrites the accumulator.
#define HDC_MMA_TS_KB(KIND)                                                                             \
  asm volatile(                                                                                         \
      "{\n\t.reg .pred p, q;\n\t.reg .b64 d0, d1, d2, d3;\n\t.reg .b32 l1, l2, l3, a1, a2, a3;\n\t"        \
      "elect.sync _|q, 0xffffffff;\n\tsetp.ne.b32 p, %4, 0;\n\t"                                         \
      "add.u32 l1, %2, 2;\n\tadd.u32 l2, %2, 4;\n\tadd.u32 l3, %2, 6;\n\t"                              \
      "add.u32 a1, %1, 8;\n\tadd.u32 a2, %1, 16;\n\tadd.u32 a3, %1, 24;\n\t"                            \
      "mov.b64 d0, {%2, 0x40004040};\n\tmov.b64 d1, {l1, 0x40004040};\n\t"                              \
      "mov.b64 d2, {l2, 0x40004040};\n\tmov.b64 d3, {l3, 0x40004040};\n\t"                              \
      "@q tcgen05.mma.cta_group::1.kind::" KIND " [%0], [%1], d0, %3, p;\n\t"                            \
      "@q tcgen05.mma.cta_group::1.kind::" KIND " [%0], [a1], d1, %3, 1;\n\t"                            \
      "@q tcgen05.mma.cta_group::1.kind::" KIND " [%0], [a2], d2, %3, 1;\n\t"                            \
      "@q tcgen05.mma.cta_group::1.kind::" KIND " [%0], [a3], d3, %3, 1;\n\t}" ::"r"(d_tmem),            \
      "r"(a_tmem), "r"(b_lo), "r"(idesc), "r"(first)                                                   \
      : "memory")
template <bool INT8>
__device__ __forceinline__ void tc_mma_ts_kblock_elect(uint32_t d_tmem, uint32_t a_tmem, uint32_t b_lo, uint32_t idesc,
                                                       uint32_t first) {
  if (INT8) HDC_MMA_TS_KB("i8");
  else HDC_MMA_TS_KB("f16");
}
#undef HDC_MMA_TS_KB
// A whole group of four k-blocks (16 MMAs) in one block.  b_step = (bytes between the class tiles of consecutive
// k-blocks) / 16 - 6: what takes the descriptor address field from the last MMA of a k-block to the first of the next.
#define HDC_MMA_TS_GROUP(KIND)                                                                          \
  asm volatile(                                                                                         \
      "{\n\t.reg .pred p, q;\n\t.reg .b64 d;\n\t.reg .b32 lo, a;\n\t" \
      "elect.sync _|q, 0xffffffff;\n\tsetp.ne.b32 p, %5, 0;\n\t" \
      "mov.b32 lo, %2;\n\tmov.b32 a, %1;\n\t" \
      "mov.b64 d, {lo, 0x40004040};\n\t" \
      "@q tcgen05.mma.cta_group::1.kind::" KIND " [%0], [a], d, %4, p;\n\t" \
      "add.u32 lo, lo, 2;\n\tadd.u32 a, a, 8;\n\t" \
      "mov.b64 d, {lo, 0x40004040};\n\t" \
      "@q tcgen05.mma.cta_group::1.kind::" KIND " [%0], [a], d, %4, 1;\n\t" \
      "add.u32 lo, lo, 2;\n\tadd.u32 a, a, 8;\n\t" \
      "mov.b64 d, {lo, 0x40004040};\n\t" \
      "@q tcgen05.mma.cta_group::1.kind::" KIND " [%0], [a], d, %4, 1;\n\t" \
      "add.u32 lo, lo, 2;\n\tadd.u32 a, a, 8;\n\t" \
      "mov.b64 d, {lo, 0x40004040};\n\t" \
      "@q tcgen05.mma.cta_group::1.kind::" KIND " [%0], [a], d, %4, 1;\n\t" \
      "add.u32 lo, lo, %3;\n\tadd.u32 a, a, 8;\n\t" \
      "mov.b64 d, {lo, 0x40004040};\n\t" \
      "@q tcgen05.mma.cta_group::1.kind::" KIND " [%0], [a], d, %4, 1;\n\t" \
      "add.u32 lo, lo, 2;\n\tadd.u32 a, a, 8;\n\t" \
      "mov.b64 d, {lo, 0x40004040};\n\t" \
      "@q tcgen05.mma.cta_group::1.kind::" KIND " [%0], [a], d, %4, 1;\n\t" \
      "add.u32 lo, lo, 2;\n\tadd.u32 a, a, 8;\n\t" \
      "mov.b64 d, {lo, 0x40004040};\n\t" \
      "@q tcgen05.mma.cta_group::1.kind::" KIND " [%0], [a], d, %4, 1;\n\t" \
      "add.u32 lo, lo, 2;\n\tadd.u32 a, a, 8;\n\t" \
      "mov.b64 d, {lo, 0x40004040};\n\t" \
      "@q tcgen05.mma.cta_group::1.kind::" KIND " [%0], [a], d, %4, 1;\n\t" \
      "add.u32 lo, lo, %3;\n\tadd.u32 a, a, 8;\n\t" \
      "mov.b64 d, {lo, 0x40004040};\n\t" \
      "@q tcgen05.mma.cta_group::1.kind::" KIND " [%0], [a], d, %4, 1;\n\t" \
      "add.u32 lo, lo, 2;\n\tadd.u32 a, a, 8;\n\t" \
      "mov.b64 d, {lo, 0x40004040};\n\t" \
      "@q tcgen05.mma.cta_group::1.kind::" KIND " [%0], [a], d, %4, 1;\n\t" \
      "add.u32 lo, lo, 2;\n\tadd.u32 a, a, 8;\n\t" \
      "mov.b64 d, {lo, 0x40004040};\n\t" \
      "@q tcgen05.mma.cta_group::1.kind::" KIND " [%0], [a], d, %4, 1;\n\t" \
      "add.u32 lo, lo, 2;\n\tadd.u32 a, a, 8;\n\t" \
      "mov.b64 d, {lo, 0x40004040};\n\t" \
      "@q tcgen05.mma.cta_group::1.kind::" KIND " [%0], [a], d, %4, 1;\n\t" \
      "add.u32 lo, lo, %3;\n\tadd.u32 a, a, 8;\n\t" \
      "mov.b64 d, {lo, 0x40004040};\n\t" \
      "@q tcgen05.mma.cta_group::1.kind::" KIND " [%0], [a], d, %4, 1;\n\t" \
      "add.u32 lo, lo, 2;\n\tadd.u32 a, a, 8;\n\t" \
      "mov.b64 d, {lo, 0x40004040};\n\t" \
      "@q tcgen05.mma.cta_group::1.kind::" KIND " [%0], [a], d, %4, 1;\n\t" \
      "add.u32 lo, lo, 2;\n\tadd.u32 a, a, 8;\n\t" \
      "mov.b64 d, {lo, 0x40004040};\n\t" \
      "@q tcgen05.mma.cta_group::1.kind::" KIND " [%0], [a], d, %4, 1;\n\t" \
      "add.u32 lo, lo, 2;\n\tadd.u32 a, a, 8;\n\t" \
      "mov.b64 d, {lo, 0x40004040};\n\t" \
      "@q tcgen05.mma.cta_group::1.kind::" KIND " [%0], [a], d, %4, 1;\n\t" \
      "}" ::"r"(d_tmem), "r"(a_tmem), "r"(b_lo), "r"(b_step), "r"(idesc), "r"(first)           \
      : "memory")
template <bool INT8>
__device__ __forceinline__ void tc_mma_ts_group_elect(uint32_t d_tmem, uint32_t a_tmem, uint32_t b_lo, uint32_t b_step,
                                                      uint32_t idesc, uint32_t first) {
  if (INT8) HDC_MMA_TS_GROUP("i8");
  else HDC_MMA_TS_GROUP("f16");
}
#undef HDC_MMA_TS_GROUP
// 32 lanes x 16 consecutive 32-bit columns, registers -> tensor memory: thread t of the warp writes lane (base + t)
__device__ __forceinline__ void tmem_st16(uint32_t taddr, const uint32_t (&v)[16]) {
  asm volatile(
      "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], "
      "{%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16};" ::"r"(taddr),
      "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]), "r"(v[8]), "r"(v[9]),
      "r"(v[10]), "r"(v[11]), "r"(v[12]), "r"(v[13]), "r"(v[14]), "r"(v[15])
      : "memory");
}
__device__ __forceinline__ void tmem_st_wait() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

// 32 lanes x 32 consecutive 32-bit columns: thread t of the warp gets lane (base + t), v[j] = column j
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&v)[32]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
      "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
      "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
      : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
        "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]),
        "=r"(v[16]), "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]),
        "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
      : "r"(taddr)
      : "memory");
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

// Shared-memory matrix descriptor of a K-major tile stored as rows of 128 bytes with the 128-byte
// swizzle (what TMA writes for SWIZZLE_128B): 8-row groups are 1024 bytes apart (SBO), the
// leading-dimension offset is unused for swizzled K-major layouts, descriptor version 1 (sm_100),
// layout type 2 = SWIZZLE_128B.  Advancing by one MMA along K (32 bytes) adds 2 to the address field.
__device__ __forceinline__ uint64_t smem_desc(uint32_t saddr) {
  uint64_t d = 0;
  d |= (uint64_t)((saddr & 0x3FFFFu) >> 4);
  d |= (uint64_t)1 << 16;                 // LBO (ignored)
  d |= (uint64_t)(1024 >> 4) << 32;       // SBO
  d |= (uint64_t)1 << 46;                 // version
  d |= (uint64_t)2 << 61;                 // SWIZZLE_128B
  return d;
}
// Instruction descriptor: D format (1 = f32, 2 = s32) bits 4-5, A/B format bits 7-9 / 10-12
// (kind::f16: 1 = bf16; kind::i8: 1 = signed), both operands K-major (bits 15, 16 = 0),
// N >> 3 at bit 17, M >> 4 at bit 24.
template <bool INT8>
__device__ __forceinline__ uint32_t instr_desc(int m, int n) {
  uint32_t d = 0;
  d |= (INT8 ? 2u : 1u) << 4;
  d |= 1u << 7;
  d |= 1u << 10;
  d |= (uint32_t)(n >> 3) << 17;
  d |= (uint32_t)(m >> 4) << 24;
  return d;
}

// 32 lanes x 16 consecutive 32-bit columns
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t (&v)[16]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 "
      "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
      : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
        "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
      : "r"(taddr)
      : "memory");
}
// makes this thread's generic-proxy shared-memory writes visible to the async proxy (tcgen05.mma)
__device__ __forceinline__ void fence_proxy_async_smem() {
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
// CG = 2: issued by the same warp of both CTAs of the pair, same slot offset in both
template <int CG = 1>
__device__ __forceinline__ void tmem_alloc(uint32_t slot_smem, uint32_t cols) {
  if (CG == 2) {
    asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(slot_smem), "r"(cols)
                 : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
  } else {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(slot_smem), "r"(cols)
                 : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
}
template <int CG = 1>
__device__ __forceinline__ void tmem_dealloc(uint32_t taddr, uint32_t cols) {
  if (CG == 2)
    asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(cols) : "memory");
  else
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(cols) : "memory");
}

}  // namespace tcp

// host: [rows][cols] matrix of 1-byte (int8) or 2-byte (bf16) elements, row stride ld elements, TMA
// boxes of 128 bytes x box_rows with the 128-byte swizzle; out-of-range elements read as zero.
struct TcContext;
bool tc_make_map(TcContext* tc, CUtensorMap* out, const void* ptr, bool int8, int64_t rows, int64_t cols,
                 int64_t ld, int box_rows);
// host: packed hypervector words [rows][cols] uint32, row stride ld words (ld % 4 == 0, 16-byte aligned base): TMA
// boxes of 32 words x 128 rows with the 128-byte swizzle; out-of-range words and rows read as zero.
bool tc_make_map_words(TcContext* tc, CUtensorMap* out, const void* ptr, int64_t rows, int64_t cols, int64_t ld);

}  // namespace hdc
