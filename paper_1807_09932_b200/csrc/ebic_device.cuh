// ebic_device.cuh -- small device-side building blocks (sm_100a): mbarrier, TMA bulk copy, loads.
// Product code: shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace ebic {

constexpr int kLdAlign = 1024;         // leading dimension (padded rows) is a multiple of this (= one pair-bit tile)
constexpr int kPairTileRows = 1024;    // rows per pair-bit tile: one pair-row of a tile = 32 words = 128 B
constexpr int kRowsPerSlabF32 = 128;   // one warp, 4 float32 rows per lane  (one LDS.128 per column)
constexpr int kRowsPerSlabR8 = 512;    // one warp, 16 uint8 ranks per lane  (one LDS.128 per column)
constexpr unsigned kRankNaN = 0x7Fu;   // rank code of a missing value; real ranks are 0x80 | rank
constexpr int kMaxColsRank8 = 127;     // ranks 0..126 must fit under the 0x80 flag

__device__ __forceinline__ uint32_t smem_u32(const void* p) {
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}

// ---- mbarrier (shared::cta) -------------------------------------------------------------------
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void fence_mbar_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t* bar, uint32_t parity) {
    uint32_t done;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(done)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
    return done != 0;
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    while (!mbar_try_wait(bar, parity)) {
    }
}

// ---- TMA 1-D bulk copy global -> shared, completion counted on an mbarrier (SASS: UBLKCP) ------
// dst / src 16-byte aligned, bytes a multiple of 16.
__device__ __forceinline__ void bulk_copy_g2s(void* smem_dst, const void* gmem_src, uint32_t bytes,
                                              uint64_t* bar) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
            smem_u32(smem_dst)),
        "l"(gmem_src), "r"(bytes), "r"(smem_u32(bar))
        : "memory");
}

// Orders this thread's earlier generic-proxy accesses to shared memory (plain LDS / STS, and those of other threads
// it has synchronised with) before later async-proxy accesses (cp.async.bulk writes into the same bytes).
__device__ __forceinline__ void fence_proxy_async_smem() {
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}

// L2 prefetch of `bytes` (multiple of 16) at a 16-byte aligned global address; no register or shared-memory
// destination, no completion to wait for (SASS: UBLKPF).
__device__ __forceinline__ void bulk_prefetch_l2(const void* gmem_src, uint32_t bytes) {
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(gmem_src), "r"(bytes) : "memory");
}

// 128-bit read-only global load that keeps its place among the other asm statements (SASS: LDG.E.128.CONSTANT).
__device__ __forceinline__ uint4 ldg128_ordered(const void* p) {
    uint4 v;
    asm volatile("ld.global.nc.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p) : "memory");
    return v;
}

// 16-byte asynchronous copy global -> shared that bypasses registers and L1 (SASS: LDGSTS.E.BYPASS.128), and its
// group fence.  A thread that only reads back what it copied itself needs no barrier after the wait.
__device__ __forceinline__ void cp_async16(uint32_t smem_dst, const void* gmem_src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_dst), "l"(gmem_src) : "memory");
}
// The executing thread's earlier cp.async copies, once they have all landed, count as ONE arrival on `bar` (the
// arrival is part of the barrier's initial count: .noinc).
__device__ __forceinline__ void cp_async_arrive_on(uint64_t* bar) {
    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

// 128-bit shared-memory load from a 32-bit shared-window address (SASS: LDS.128 [R+imm]): the address
// comes straight out of one IMAD (id * column stride + lane base), no generic-pointer arithmetic.
__device__ __forceinline__ uint4 lds128(uint32_t addr) {
    uint4 v;
    asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr) : "memory");
    return v;
}

__device__ __forceinline__ uint32_t lds32(uint32_t addr) {
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr));
    return v;
}

// ---- programmatic dependent launch (sm_90+): a kernel launched with the programmatic-stream-serialization
// attribute may start while its predecessor on the stream is still running.  griddep_wait() blocks until every
// prerequisite grid has completed and its memory is visible; griddep_launch_dependents() lets the NEXT kernel's
// CTAs be scheduled once every CTA of this grid has called it (or exited).  Both are no-ops for plain launches.
__device__ __forceinline__ void griddep_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void griddep_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

// Load of something an EARLIER kernel on the stream wrote (meta, records, plans, batch lists).  With programmatic
// dependent launch this kernel is already resident while that kernel writes, and the same addresses are rewritten
// every generation; PTX allows the read-only path (ld.global.nc, __ldg) only for data nobody writes during the
// reading kernel's lifetime.  So: a plain load served by L2 (ld.global.cg), issued after griddep_wait().  __ldg stays
// for what really is immutable while a kernel runs: the matrix, the pair table, the caller's population.
template <class T>
__device__ __forceinline__ T ld_produced(const T* p) { return __ldcg(p); }

__device__ __forceinline__ bool is_nan_bits(float v) {
    return (__float_as_uint(v) & 0x7fffffffu) > 0x7f800000u;
}

}  // namespace ebic
