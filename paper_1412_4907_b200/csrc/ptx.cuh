// ptx.cuh -- hand-written sm_100a PTX wrappers: mbarrier, tcgen05 (alloc / mma / commit / ld), fences.
// Field layouts of the shared-memory matrix descriptor and the instruction descriptor follow the PTX
// ISA "tcgen05" chapter (Matrix Descriptor / Instruction Descriptor tables).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define BF_DEVI __device__ __forceinline__

BF_DEVI uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

// one lane of a fully converged warp; lets the compiler keep the surrounding code warp-uniform
BF_DEVI bool elect_one() {
  uint32_t pred = 0;
  asm volatile(
      "{\n\t.reg .b32 rx;\n\t.reg .pred px;\n\t"
      "elect.sync rx|px, %1;\n\t"
      "@px mov.s32 %0, 1;\n\t}"
      : "+r"(pred)
      : "r"(0xffffffffu));
  return pred != 0;
}

// bf_set_clock_probe: CTA 0 stamps (clock64, globaltimer) at slot 0 = kernel start, 1 = kernel end
BF_DEVI void probe_mark(unsigned long long *probe, int slot) {
  if (probe != nullptr && blockIdx.x == 0 && threadIdx.x == 0) {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    probe[2 * slot] = (unsigned long long)clock64();
    probe[2 * slot + 1] = t;
  }
}

// ---- mbarrier ----------------------------------------------------------------------------------
BF_DEVI void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
BF_DEVI void fence_barrier_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
// generic-proxy writes (st.shared) -> visible to the async proxy (tcgen05.mma operand reads)
BF_DEVI void fence_proxy_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
BF_DEVI void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
BF_DEVI void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
// TMA bulk copy (1-D, contiguous): global -> shared, completion counted in bytes on an mbarrier.
// size and both addresses must be multiples of 16.  SASS: UBLKCP.
BF_DEVI void bulk_g2s(uint32_t dst_smem, const void *src_gmem, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(dst_smem), "l"(src_gmem), "r"(bytes), "r"(bar) : "memory");
}
// TMA tiled tensor copy (3-D): global -> shared through a CUtensorMap; out-of-bounds elements are
// zero-filled, the full box is counted on the mbarrier.  SASS: UTMALDG.
BF_DEVI void tma_load_3d(uint32_t dst_smem, const void *tmap, int x, int y, int z, uint32_t bar) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
      ::"r"(dst_smem), "l"(tmap), "r"(x), "r"(y), "r"(z), "r"(bar) : "memory");
}
// the same in 5-D: the bin-per-lane kernels (bf_umma_i8b.cu, bf_umma_bl.cu) view the voltages as
// {byte in row, 1, bin, row in bin, channel} and fetch one row of 128 consecutive bins per copy
BF_DEVI void tma_load_5d(uint32_t dst_smem, const void *tmap, int x, int y, int z, int w, int v, uint32_t bar) {
  asm volatile(
      "cp.async.bulk.tensor.5d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5, %6}], [%7];"
      ::"r"(dst_smem), "l"(tmap), "r"(x), "r"(y), "r"(z), "r"(w), "r"(v), "r"(bar) : "memory");
}
BF_DEVI void tma_prefetch_desc(const void *tmap) {
  asm volatile("prefetch.tensormap [%0];" ::"l"(tmap) : "memory");
}
BF_DEVI bool mbar_try_wait(uint32_t bar, uint32_t parity) {
  uint32_t ok;
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
      "selp.u32 %0, 1, 0, p;\n\t}"
      : "=r"(ok)
      : "r"(bar), "r"(parity)
      : "memory");
  return ok != 0;
}
// try_wait with a suspend-time hint: the warp sleeps in hardware until the phase completes or the
// hint (ns) expires -- fewer wake-ups, fewer issue slots burnt by waiting roles
BF_DEVI bool mbar_try_wait_hint(uint32_t bar, uint32_t parity, uint32_t ns) {
  uint32_t ok;
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n\t"
      "selp.u32 %0, 1, 0, p;\n\t}"
      : "=r"(ok)
      : "r"(bar), "r"(parity), "r"(ns)
      : "memory");
  return ok != 0;
}
// Test-only jitter build (python -m paper_1412_4907_b200.build --jitter -> libbf_jitter.so, -DBF_JITTER=1): every
// mbarrier wait below first sleeps for a pseudo-random 0-2 us drawn from the SM clock, the CTA and the warp, so that the
// warp-specialised roles meet their barriers in orders and with leads that the undisturbed kernel never shows.  The
// results must not change (tests/test_zy_jitter.py): compute-sanitizer is closed on this pool, and a protocol that only
// holds for the usual timing is exactly what an undisturbed parity test cannot see.  The product library has no trace of it.
#ifdef BF_JITTER
BF_DEVI void bf_jitter() {
  uint32_t x = (uint32_t)clock64() * 2654435761u ^ (threadIdx.x >> 5) * 40503u ^ blockIdx.x * 69069u;
  x ^= x >> 15; x *= 2246822519u; x ^= x >> 13;
  if (x & 0x30000u) return;                    // three waits in four go straight through: leads build up and collapse
  asm volatile("nanosleep.u32 %0;" ::"r"(x & 2047u));
}
#else
BF_DEVI void bf_jitter() {}
#endif

// Waits.  ONE policy for all four flavours below: a wait never spins for ever -- a mis-phased pipeline must fail (trap),
// not hang the GPU -- and its bound is far above anything a healthy run needs (tens of seconds and more: a time-sliced
// or profiled GPU must never trip it), so the exact figure is no part of any contract.  mbar_wait counts SM clocks (it
// looks at clock64 once per 4096 polls, ~20 s at 2 GHz); mbar_wait_backoff / _tight / _hinted count 2^26 polls, each of
// which blocks for the hardware's try_wait time slice (plus the sleep / suspend hint), which comes to the same order.
// They differ only in what a failed poll costs the other warps of the SM.
BF_DEVI void mbar_wait(uint32_t bar, uint32_t parity) {
  bf_jitter();
  if (mbar_try_wait(bar, parity)) return;
  const long long t0 = clock64();
  for (;;) {
#pragma unroll 1
    for (int k = 0; k < 4096; ++k) {
      if (mbar_try_wait(bar, parity)) return;
    }
    if (clock64() - t0 > 40000000000LL) asm volatile("trap;");
  }
}
// Wait for roles that wait LONG (the K-blocked kernel's epilogue sits out a whole K loop): sleep between polls, so
// that the waiting warps stop taking issue slots from the working ones (ncu: 56 % of the streaming kernel's
// instructions were such polls).  Bounded like the others.
BF_DEVI void mbar_wait_backoff(uint32_t bar, uint32_t parity, uint32_t sleep_ns) {
  bf_jitter();
  if (mbar_try_wait(bar, parity)) return;
  for (uint32_t n = 0;; ++n) {
    asm volatile("nanosleep.u32 %0;" ::"r"(sleep_ns));
    if (mbar_try_wait(bar, parity)) return;
    if (n > (1u << 26)) asm volatile("trap;");
  }
}
// Tight bounded wait for roles on the critical chain (the epilogue): two instructions per failed poll, trap after
// 2^26 polls (a try_wait blocks for a hardware-defined slice, so this is seconds, not a hang).
BF_DEVI void mbar_wait_tight(uint32_t bar, uint32_t parity) {
  bf_jitter();
  // four polls per trip of the bounding counter: a failed poll costs two issue slots, and every slot a waiting
  // warp takes is one a working warp of the same sub-partition does not get
  asm volatile(
      "{\n\t.reg .pred p, q;\n\t.reg .u32 n;\n\tmov.u32 n, 0;\n"
      "BFW_%=:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
      "@p bra BFD_%=;\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
      "@p bra BFD_%=;\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
      "@p bra BFD_%=;\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
      "@p bra BFD_%=;\n\t"
      "add.u32 n, n, 1;\n\t"
      "setp.lt.u32 q, n, 0x1000000;\n\t"
      "@q bra BFW_%=;\n\t"
      "trap;\n"
      "BFD_%=:\n\t}" ::"r"(bar), "r"(parity)
      : "memory");
}


// Bounded wait for roles with MANY waiting warps (the bin-per-lane int8-operand kernel's epilogue sets): try_wait with a
// suspend-time hint.  The poll count does not fall (ncu: still ~25 polls per visit), but the waits come out 1-2 %
// faster on sweep-32 and sweep-ci4-16 than the tight spin; in the resident fp16 kernel the same wait is 7 % SLOWER at
// 64 beams (A/B on one box), so that kernel keeps mbar_wait_tight.
BF_DEVI void mbar_wait_hinted(uint32_t bar, uint32_t parity, uint32_t ns) {
  bf_jitter();
  if (mbar_try_wait(bar, parity)) return;
  for (uint32_t n = 0;; ++n) {
    if (mbar_try_wait_hint(bar, parity, ns)) return;
    if (n > (1u << 26)) asm volatile("trap;");
  }
}

// ---- tcgen05 -----------------------------------------------------------------------------------
BF_DEVI void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
BF_DEVI void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
BF_DEVI void tmem_alloc(uint32_t dst_smem, uint32_t ncols) {  // whole warp
  asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(dst_smem), "r"(ncols)
               : "memory");
  asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
BF_DEVI void tmem_dealloc(uint32_t taddr, uint32_t ncols) {  // whole warp
  asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(ncols) : "memory");
}
// arrive on an mbarrier once all previously issued tcgen05.mma of this thread have completed
BF_DEVI void tc_commit(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar)
               : "memory");
}
BF_DEVI void tc_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

// D[tmem] (+)= A[smem] * B[smem], fp16 inputs, fp32 accumulate; one thread issues for the CTA
BF_DEVI void mma_f16_ss(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}" ::"r"(d_tmem),
      "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate)
      : "memory");
}

// The same with the two descriptors given as 32-bit low words plus their common high word: all operand tiles of a
// kernel share the high word (stride, version, swizzle), and advancing along K or to another stage only changes the
// 14-bit address field, so the issuing warp does 32-bit arithmetic instead of 64-bit adds with carries.
BF_DEVI void mma_f16_ss_lo(uint32_t d_tmem, uint32_t adesc_lo, uint32_t bdesc_lo, uint32_t desc_hi, uint32_t idesc,
                           uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t.reg .b64 da, db;\n\t"
      "mov.b64 da, {%1, %5};\n\tmov.b64 db, {%2, %5};\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], da, db, %3, p;\n\t}" ::"r"(d_tmem),
      "r"(adesc_lo), "r"(bdesc_lo), "r"(idesc), "r"(accumulate), "r"(desc_hi)
      : "memory");
}
// low / high word of make_sdesc_k_sw128
BF_DEVI uint32_t sdesc_k_sw128_lo(uint32_t saddr) { return ((saddr >> 4) & 0x3FFFu) | (1u << 16); }
__host__ __device__ constexpr uint32_t sdesc_k_sw128_hi() { return (1024u >> 4) | (1u << 14) | (2u << 29); }

// D[tmem] (+)= A[tmem] * B[smem]: the A operand (M = 128 rows = TMEM lanes, 16 fp16 along K = 8 columns) read from
// tensor memory, B from shared memory
BF_DEVI void mma_f16_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t}" ::"r"(d_tmem),
      "r"(a_tmem), "l"(bdesc), "r"(idesc), "r"(accumulate)
      : "memory");
}
BF_DEVI void tc_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
// 32 lanes x 32 consecutive 32-bit columns, registers -> TMEM: thread l of the warp writes lane (base lane + l)
#define BF_TMEM_ST_32x32b_X32(taddr, r)                                                           \
  asm volatile("tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], "                                     \
               "{%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,"                          \
               "%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31,%32};"                 \
               ::"r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]),     \
                 "r"(r[6]), "r"(r[7]), "r"(r[8]), "r"(r[9]), "r"(r[10]), "r"(r[11]), "r"(r[12]),   \
                 "r"(r[13]), "r"(r[14]), "r"(r[15]), "r"(r[16]), "r"(r[17]), "r"(r[18]),           \
                 "r"(r[19]), "r"(r[20]), "r"(r[21]), "r"(r[22]), "r"(r[23]), "r"(r[24]),           \
                 "r"(r[25]), "r"(r[26]), "r"(r[27]), "r"(r[28]), "r"(r[29]), "r"(r[30]),           \
                 "r"(r[31])                                                                        \
               : "memory")

// Shared-memory matrix descriptor, K-major operand, 128-byte swizzle:
//   bits [0,14) start address >> 4 | [16,30) leading byte offset >> 4 (unused for swizzled K-major,
//   set to 1) | [32,46) stride byte offset >> 4 (distance between 8-row groups = 1024 B) |
//   [46,48) version = 1 on sm_100 | [61,64) layout type: 2 = SWIZZLE_128B
BF_DEVI uint64_t make_sdesc_k_sw128(uint32_t saddr) {
  uint64_t d = 0;
  d |= (uint64_t)((saddr >> 4) & 0x3FFF);
  d |= (uint64_t)1 << 16;
  d |= (uint64_t)(1024 >> 4) << 32;
  d |= (uint64_t)1 << 46;
  d |= (uint64_t)2 << 61;
  return d;
}
// Instruction descriptor for kind::f16: [4,6) D format 1 = f32 | [7,10) A format 0 = f16 | [10,13) B
// format 0 = f16 | bit 15 / 16: A / B major 0 = K | [17,23) N >> 3 | [24,29) M >> 4
__host__ __device__ constexpr uint32_t make_idesc_f16(uint32_t M, uint32_t N) {
  return (1u << 4) | (0u << 7) | (0u << 10) | ((N >> 3) << 17) | ((M >> 4) << 24);
}

// D[tmem] (+)= A[smem] * B[smem], int8 inputs, int32 accumulate (K = 32 per instruction)
BF_DEVI void mma_i8_ss(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::i8 [%0], %1, %2, %3, p;\n\t}" ::"r"(d_tmem),
      "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate)
      : "memory");
}
// the same with the A operand (M = 128 rows = TMEM lanes, 32 int8 along K = 8 columns) read from tensor memory
BF_DEVI void mma_i8_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::i8 [%0], [%1], %2, %3, p;\n\t}" ::"r"(d_tmem),
      "r"(a_tmem), "l"(bdesc), "r"(idesc), "r"(accumulate)
      : "memory");
}
// K-major operand with rows of 64 bytes, 64-byte swizzle (16-byte chunk index ^= (row >> 1) & 3; the
// pattern repeats every 8 rows = 512 bytes = the stride byte offset); layout type 4 = SWIZZLE_64B
BF_DEVI uint64_t make_sdesc_k_sw64(uint32_t saddr) {
  uint64_t d = 0;
  d |= (uint64_t)((saddr >> 4) & 0x3FFF);
  d |= (uint64_t)1 << 16;
  d |= (uint64_t)(512 >> 4) << 32;
  d |= (uint64_t)1 << 46;
  d |= (uint64_t)4 << 61;
  return d;
}
// Instruction descriptor for kind::i8: [4,6) D format 2 = s32 | [7,10) A format 1 = signed 8 bit | [10,13) B
// format 1 = signed 8 bit | bit 15 / 16: A / B major 0 = K | [17,23) N >> 3 | [24,29) M >> 4
__host__ __device__ constexpr uint32_t make_idesc_i8(uint32_t M, uint32_t N) {
  return (2u << 4) | (1u << 7) | (1u << 10) | ((N >> 3) << 17) | ((M >> 4) << 24);
}

// 32 lanes x 32 consecutive 32-bit columns: thread l of the warp gets lane (base lane + l)
#define BF_TMEM_LD_32x32b_X32(taddr, r)                                                           \
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x32.b32 "                                           \
               "{%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,"                           \
               "%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"          \
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]),           \
                 "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]),         \
                 "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]), "=r"(r[17]),     \
                 "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]),     \
                 "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]),     \
                 "=r"(r[30]), "=r"(r[31])                                                          \
               : "r"(taddr))

// packed fp32x2 add
BF_DEVI float2 fadd2(float2 a, float2 b) {
  float2 d;
  asm("add.rn.f32x2 %0, %1, %2;"
      : "=l"(reinterpret_cast<uint64_t &>(d))
      : "l"(reinterpret_cast<uint64_t &>(a)), "l"(reinterpret_cast<uint64_t &>(b)));
  return d;
}
// packed fp32x2 FMA (FFMA2): d = a * b + c on both halves of a 64-bit register pair
BF_DEVI float2 ffma2(float2 a, float2 b, float2 c) {
  float2 d;
  asm("fma.rn.f32x2 %0, %1, %2, %3;"
      : "=l"(reinterpret_cast<uint64_t &>(d))
      : "l"(reinterpret_cast<uint64_t &>(a)), "l"(reinterpret_cast<uint64_t &>(b)),
        "l"(reinterpret_cast<uint64_t &>(c)));
  return d;
}
// the same, but ordered with the surrounding volatile asm (barrier arrives, tcgen05.ld): the compiler must not sink an
// mbarrier.arrive below the squares that follow it
BF_DEVI float2 ffma2v(float2 a, float2 b, float2 c) {
  float2 d;
  asm volatile("fma.rn.f32x2 %0, %1, %2, %3;"
               : "=l"(reinterpret_cast<uint64_t &>(d))
               : "l"(reinterpret_cast<uint64_t &>(a)), "l"(reinterpret_cast<uint64_t &>(b)),
                 "l"(reinterpret_cast<uint64_t &>(c)));
  return d;
}
