// common.cuh -- device helpers shared by the CUDA kernels of libdfemul (sm_100a).
// Nothing here is shared with oracle/: the digit arithmetic below is written
// from the definition in DESIGN.md section 2 (R2), not from the oracle's code.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace dfe {

// ---------------------------------------------------------------------------
// Status word bits (include/df_emul.h)
// ---------------------------------------------------------------------------
constexpr int kStatusNonFinite = 1;
constexpr int kStatusRange = 2;

// ---------------------------------------------------------------------------
// Scale index and fixed-point digits (R2)
// ---------------------------------------------------------------------------

// hi = upper 32 bits of |m| (sign cleared), m the row/column maximum.
// m = f 2^E with f in [0.5,1)  <=>  biased exponent field = E + 1022.
// e = E + 1 when the top 6 stored mantissa bits are all ones (f >= 127/128),
// rows with m < 2^-1000 (E <= -1000) are zero rows: e = 0.
__device__ __forceinline__ int scale_index_from_hi(uint32_t hi) {
  const int eb = (int)(hi >> 20);  // biased exponent (sign bit already cleared)
  if (eb <= 22) return 0;          // E = eb - 1022 <= -1000
  const int bump = ((hi >> 14) & 0x3Fu) == 0x3Fu;
  return eb - 1022 + bump;
}

// Status bits for a row/column maximum given by its hi word.
__device__ __forceinline__ int status_from_hi(uint32_t hi) {
  const int eb = (int)(hi >> 20);
  if (eb == 0x7FF) return kStatusNonFinite;
  if (eb <= 22) return 0;  // zero row
  const int E = eb - 1022;
  return (E > 450 || E < -449) ? kStatusRange : 0;
}

// 2^p as a double for p in the normal range.
__device__ __forceinline__ double pow2_double(int p) {
  return __hiloint2double((1023 + p) << 20, 0);
}

// Balanced base-256 digits of Q = rint(x * 2^(63-e)), all 8 at once.
// Adding 0x80 to each of the 7 low bytes lets the hardware carry chain do the
// "v >= 128 -> v -= 256, carry 1" rule; xor 0x80 takes the bias off again.
// Byte (8 - t) of the result is digit d_t as a signed int8 (byte 7 = d_1).
__device__ __forceinline__ uint64_t balanced_digits(double x, double scale /* 2^(63-e) */) {
  const long long Q = __double2ll_rn(x * scale);
  const uint64_t bias = 0x0080808080808080ull;
  return ((uint64_t)Q + bias) ^ bias;
}

// digit d_{t+1} (t = 0..7) of a packed digit word, as an unsigned byte value.
__device__ __forceinline__ uint32_t digit_byte(uint64_t dg, int t) {
  return (uint32_t)(dg >> (8 * (7 - t))) & 0xFFu;
}

// Four consecutive elements' digit words (upper or lower halves) -> the packed plane word of
// digit byte `b` (0..3 within the half): three byte permutes instead of twelve shift/mask/or.
__device__ __forceinline__ uint32_t pack4_digit(uint32_t h0, uint32_t h1, uint32_t h2, uint32_t h3, int b) {
  const uint32_t sel = (uint32_t)b | ((uint32_t)(4 + b) << 4);
  return __byte_perm(__byte_perm(h0, h1, sel), __byte_perm(h2, h3, sel), 0x5410);
}

// out[b] = byte b of h[0], h[1], h[2], h[3] (a 4 x 4 byte transpose): eight byte permutes for the
// four plane words of four consecutive elements.
__device__ __forceinline__ void transpose4x4_bytes(const uint32_t (&h)[4], uint32_t (&out)[4]) {
  const uint32_t a01 = __byte_perm(h[0], h[1], 0x5140), b01 = __byte_perm(h[0], h[1], 0x7362);
  const uint32_t a23 = __byte_perm(h[2], h[3], 0x5140), b23 = __byte_perm(h[2], h[3], 0x7362);
  out[0] = __byte_perm(a01, a23, 0x5410);
  out[1] = __byte_perm(a01, a23, 0x7632);
  out[2] = __byte_perm(b01, b23, 0x5410);
  out[3] = __byte_perm(b01, b23, 0x7632);
}

__device__ __forceinline__ uint32_t abs_hi_word(double x) {
  return (uint32_t)__double2hiint(x) & 0x7FFFFFFFu;
}

// ---------------------------------------------------------------------------
// PTX wrappers: mbarrier, TMA, tcgen05 (sm_100a)
// ---------------------------------------------------------------------------

__device__ __forceinline__ uint32_t smem_u32(const void* p) {
  return (uint32_t)__cvta_generic_to_shared(p);
}

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void fence_barrier_init() {
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void fence_proxy_async() {
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes)
               : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t* bar, uint32_t parity) {
  uint32_t ok;
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
      "selp.u32 %0, 1, 0, p;\n\t}"
      : "=r"(ok)
      : "r"(smem_u32(bar)), "r"(parity)
      : "memory");
  return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  while (!mbar_try_wait(bar, parity)) {
  }
}

// true in exactly one (elected) lane of a converged warp
__device__ __forceinline__ bool elect_one() {
  uint32_t pred = 0;
  asm volatile(
      "{\n\t.reg .b32 rx;\n\t.reg .pred px;\n\t"
      "elect.sync rx|px, 0xffffffff;\n\t"
      "@px mov.s32 %0, 1;\n\t}"
      : "+r"(pred));
  return pred != 0;
}

__device__ __forceinline__ void prefetch_tensormap(const void* tmap) {
  asm volatile("prefetch.tensormap [%0];" ::"l"(tmap) : "memory");
}

// 3-D tiled TMA load, completion on an mbarrier of this CTA.
__device__ __forceinline__ void tma_load_3d(void* smem_dst, const void* tmap, uint64_t* bar, int c0, int c1,
                                            int c2) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes"
      " [%0], [%1, {%3, %4, %5}], [%2];" ::"r"(smem_u32(smem_dst)),
      "l"(tmap), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2)
      : "memory");
}

// Same load, delivered to the same shared-memory offset (and mbarrier) of every CTA in `mask`.
__device__ __forceinline__ void tma_load_3d_mcast(void* smem_dst, const void* tmap, uint64_t* bar, int c0, int c1,
                                                  int c2, uint16_t mask) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes.multicast::cluster"
      " [%0], [%1, {%3, %4, %5}], [%2], %6;" ::"r"(smem_u32(smem_dst)),
      "l"(tmap), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2), "h"(mask)
      : "memory");
}

__device__ __forceinline__ uint32_t cluster_ctarank() {
  uint32_t r;
  asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
  return r;
}
__device__ __forceinline__ void cluster_sync_all() {
  asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
  asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
}

__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

// One warp allocates `ncols` (power of two >= 32) TMEM columns; base address -> *slot (smem).
__device__ __forceinline__ void tmem_alloc(uint32_t* slot, uint32_t ncols) {
  asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(slot)),
               "r"(ncols)
               : "memory");
  asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(uint32_t addr, uint32_t ncols) {
  asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(addr), "r"(ncols) : "memory");
}

// D[tmem] (+)= A[smem] . B[smem]^T, INT8 x INT8 -> INT32, issued by ONE thread.
__device__ __forceinline__ void mma_i8_ss(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc,
                                          uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::i8 [%0], %1, %2, %3, p;\n\t}" ::"r"(d_tmem),
      "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate));
  // no "memory" clobber: volatile asm keeps its order against the barrier waits, fences and
  // commits around it, while the compiler may hoist the next pair-table loads over this MMA
}

// All MMAs issued so far by this thread arrive on `bar` when they complete.
__device__ __forceinline__ void mma_commit(uint64_t* bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(
                   smem_u32(bar))
               : "memory");
}

// Same, arriving on the barrier at this offset in every CTA of `mask` (stage release in a cluster
// whose CTAs multicast operand tiles into each other's shared memory).
__device__ __forceinline__ void mma_commit_mcast(uint64_t* bar, uint16_t mask) {
  asm volatile(
      "tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;" ::"r"(
          smem_u32(bar)),
      "h"(mask)
      : "memory");
}

// ---- cta_group::2: two CTAs (an SM pair) run one MMA of M = 256; each holds its own 128 rows of A
// and half of the N rows of B in its shared memory, the leader CTA issues ----
__device__ __forceinline__ void tmem_alloc_pair(uint32_t* slot, uint32_t ncols) {
  asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(slot)),
               "r"(ncols)
               : "memory");
  asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc_pair(uint32_t addr, uint32_t ncols) {
  asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(addr), "r"(ncols) : "memory");
}
__device__ __forceinline__ void mma_i8_ss_pair(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc,
                                               uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::2.kind::i8 [%0], %1, %2, %3, p;\n\t}" ::"r"(d_tmem),
      "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate));
}
// arrives on the barrier at this offset in every CTA of `mask` when the pair's MMAs complete
__device__ __forceinline__ void mma_commit_pair(uint64_t* bar, uint16_t mask) {
  asm volatile(
      "tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;" ::"r"(
          smem_u32(bar)),
      "h"(mask)
      : "memory");
}
// TMA load into this CTA's shared memory whose bytes are counted on a barrier given by its
// shared::cluster address (the leader CTA's full barrier)
__device__ __forceinline__ void tma_load_3d_pair(void* smem_dst, const void* tmap, uint32_t bar_cluster_addr, int c0,
                                                 int c1, int c2) {
  asm volatile(
      "cp.async.bulk.tensor.3d.cta_group::2.shared::cluster.global.mbarrier::complete_tx::bytes"
      " [%0], [%1, {%3, %4, %5}], [%2];" ::"r"(smem_u32(smem_dst)),
      "l"(tmap), "r"(bar_cluster_addr), "r"(c0), "r"(c1), "r"(c2)
      : "memory");
}
__device__ __forceinline__ uint32_t mapa_shared(uint32_t local_addr, uint32_t rank) {
  uint32_t r;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(local_addr), "r"(rank));
  return r;
}
__device__ __forceinline__ void mbar_arrive_cluster(uint32_t cluster_addr) {
  asm volatile("mbarrier.arrive.release.cluster.shared::cluster.b64 _, [%0];" ::"r"(cluster_addr) : "memory");
}

// The same without the release: the arrival only says "these TMEM columns have been read" (the
// loads completed at tcgen05.wait::ld); a release would first wait for the warp's earlier global
// stores to be performed at cluster scope.
__device__ __forceinline__ void mbar_arrive_cluster_relaxed(uint32_t cluster_addr) {
  asm volatile("mbarrier.arrive.relaxed.cluster.shared::cluster.b64 _, [%0];" ::"r"(cluster_addr) : "memory");
}

__device__ __forceinline__ void mbar_arrive_relaxed(uint64_t* bar) {
  asm volatile("mbarrier.arrive.relaxed.cta.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}

// 256-bit global accesses (PTX 8.8, sm_100: LDG/STG.E.ENL2.256): a lane moves one whole 32-byte
// sector, so a "lane = row" store of FP64 columns needs no transposition to fill its sectors.
__device__ __forceinline__ void st_global_v4f64(double* p, double a, double b, double c, double d) {
  asm volatile("st.global.v4.f64 [%0], {%1, %2, %3, %4};" ::"l"(p), "d"(a), "d"(b), "d"(c), "d"(d) : "memory");
}
__device__ __forceinline__ void ld_global_v4f64(const double* p, double& a, double& b, double& c, double& d) {
  asm volatile("ld.global.v4.f64 {%0, %1, %2, %3}, [%4];" : "=d"(a), "=d"(b), "=d"(c), "=d"(d) : "l"(p) : "memory");
}

// 256-bit read-only load: four consecutive doubles, 32-byte aligned (LDG.E.ENL2.256.CONSTANT)
__device__ __forceinline__ void ldg_nc_v4f64(const double* p, double& a, double& b, double& c, double& d) {
  asm volatile("ld.global.nc.v4.f64 {%0, %1, %2, %3}, [%4];" : "=d"(a), "=d"(b), "=d"(c), "=d"(d) : "l"(p));
}

// 16 consecutive 32-bit TMEM columns of this thread's lane (32x32b shape).
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t (&v)[16]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 "
      "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
      : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
        "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
      : "r"(taddr)
      : "memory");
}
// Store 16 consecutive 32-bit TMEM columns of this thread's lane.
__device__ __forceinline__ void tmem_st16(uint32_t taddr, const uint32_t (&v)[16]) {
  asm volatile(
      "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], "
      "{%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16};" ::"r"(taddr),
      "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]), "r"(v[8]), "r"(v[9]),
      "r"(v[10]), "r"(v[11]), "r"(v[12]), "r"(v[13]), "r"(v[14]), "r"(v[15])
      : "memory");
}
__device__ __forceinline__ void tmem_st_wait() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

// Shared-memory matrix descriptor for a K-major INT8 tile whose rows are
// `swz` bytes wide (swz = 32, 64 or 128 = the TMA swizzle span): 8-row groups
// are 8*swz bytes apart (SBO); LBO is unused for swizzled K-major layouts.
// Bit layout (PTX ISA "shared memory matrix descriptor", cross-checked against
// cute/arch/mma_sm100_desc.hpp): addr>>4 [0,14), LBO>>4 [16,30), SBO>>4 [32,46),
// version=1 [46,48), layout type [61,64): 2 = 128B, 4 = 64B, 6 = 32B swizzle.
__device__ __forceinline__ uint64_t make_smem_desc(uint32_t saddr, int swz) {
  const uint64_t layout = (swz == 128) ? 2ull : (swz == 64) ? 4ull : 6ull;
  uint64_t d = 0;
  d |= (uint64_t)((saddr & 0x3FFFFu) >> 4);
  d |= (uint64_t)1 << 16;
  d |= (uint64_t)((8u * (uint32_t)swz) >> 4) << 32;
  d |= (uint64_t)1 << 46;
  d |= layout << 61;
  return d;
}

// Instruction descriptor for kind::i8, signed x signed -> S32, both K-major.
// D format [4,6) = 2 (S32); A format [7,10) = 1, B format [10,13) = 1 (signed
// 8 bit); N>>3 at [17,23); M>>4 at [24,29).
__host__ __device__ __forceinline__ uint32_t make_idesc_i8(int M, int N) {
  return (2u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(N >> 3) << 17) | ((uint32_t)(M >> 4) << 24);
}

}  // namespace dfe
