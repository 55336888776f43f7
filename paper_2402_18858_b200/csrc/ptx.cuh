// ptx.cuh -- thin inline-PTX wrappers for the sm_100a features the tensor path uses:
// mbarrier, TMA (cp.async.bulk.tensor), tcgen05 (alloc / mma / commit / ld / fences), clusters.
// Device-only; included by the .cu files of this library and by nothing else.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace gpuann {
namespace ptx {

__device__ __forceinline__ uint32_t smem_u32(const void *p) {
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}

__device__ __forceinline__ bool elect_one() {
    uint32_t pred;
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "elect.sync _|p, 0xffffffff;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t"
        "}\n"
        : "=r"(pred));
    return pred != 0;
}

// ---------------------------------------------------------------- mbarrier
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}

// makes mbarrier.init visible to the async proxy (TMA, tcgen05.commit) and to the cluster
__device__ __forceinline__ void fence_mbar_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}

__device__ __forceinline__ void mbar_arrive(uint64_t *bar) {
    asm volatile(
        "{\n\t"
        ".reg .b64 st;\n\t"
        "mbarrier.arrive.shared::cta.b64 st, [%0];\n\t"
        "}\n" ::"r"(smem_u32(bar))
        : "memory");
}

__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t *bar, uint32_t bytes) {
    asm volatile(
        "{\n\t"
        ".reg .b64 st;\n\t"
        "mbarrier.arrive.expect_tx.shared::cta.b64 st, [%0], %1;\n\t"
        "}\n" ::"r"(smem_u32(bar)),
        "r"(bytes)
        : "memory");
}

__device__ __forceinline__ bool mbar_try_wait(uint64_t *bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t"
        "}\n"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
    return ok != 0;
}

// Debug build (-DGPUANN_DEBUG_SPIN; `python -m paper_2402_18858_b200.build --debug` -> libgpuann_debug.so, loaded by the
// binding when GPUANN_DEBUG_SPIN=1 is in the environment): a wait that has been polling for more than kSpinLimitNs of
// %globaltimer prints which barrier it is stuck on and traps.  A wrong phase or a missing arrive in a new kernel variant is
// then a failed launch (cudaErrorLaunchFailure at the next synchronisation; the printf line is best effort) instead of a
// GPU that hangs until the lease is killed.  compute-sanitizer is not available on this pool.
// The release build compiles none of this.
#ifdef GPUANN_DEBUG_SPIN
constexpr unsigned long long kSpinLimitNs = 2000000000ull;
__device__ __forceinline__ unsigned long long spin_now_ns() {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}
static __device__ __noinline__ void spin_timeout(uint32_t bar_addr, uint32_t parity, uint32_t bar_addr_b, uint32_t parity_b) {
    printf("gpuann: mbarrier wait > 2 s: block %d thread %d (warp %d) barrier smem 0x%x parity %u%s", (int)blockIdx.x,
           (int)threadIdx.x, (int)(threadIdx.x >> 5), bar_addr, parity, bar_addr_b ? "" : "\n");
    if (bar_addr_b) printf(" / barrier smem 0x%x parity %u\n", bar_addr_b, parity_b);
    __trap();
}
// one poll in 1024 reads the timer
#define GPUANN_SPIN_GUARD(polls, t0, a, pa, b, pb)                                      \
    if (((++(polls)) & 1023u) == 0) {                                                   \
        const unsigned long long now__ = spin_now_ns();                                 \
        if ((t0) == 0) (t0) = now__;                                                    \
        else if (now__ - (t0) > kSpinLimitNs) spin_timeout((a), (pa), (b), (pb));        \
    }
#endif

// Blocks until the phase with the given parity has completed.
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
#ifdef GPUANN_DEBUG_SPIN
    uint32_t polls = 0;
    unsigned long long t0 = 0;
    while (!mbar_try_wait(bar, parity)) {
        GPUANN_SPIN_GUARD(polls, t0, smem_u32(bar), parity, 0u, 0u)
    }
#else
    while (!mbar_try_wait(bar, parity)) {
    }
#endif
}

// Blocks until both phases have completed; the two polls are issued back to back so that their latencies overlap.
__device__ __forceinline__ void mbar_wait2(uint64_t *bar_a, uint32_t parity_a, uint64_t *bar_b, uint32_t parity_b) {
    uint32_t a, b;
#ifdef GPUANN_DEBUG_SPIN
    uint32_t polls = 0;
    unsigned long long t0 = 0;
#endif
    do {
        asm volatile(
            "{\n\t"
            ".reg .pred p, q;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%2], %3;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 q, [%4], %5;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t"
            "selp.u32 %1, 1, 0, q;\n\t"
            "}\n"
            : "=r"(a), "=r"(b)
            : "r"(smem_u32(bar_a)), "r"(parity_a), "r"(smem_u32(bar_b)), "r"(parity_b)
            : "memory");
#ifdef GPUANN_DEBUG_SPIN
        GPUANN_SPIN_GUARD(polls, t0, smem_u32(bar_a), parity_a, smem_u32(bar_b), parity_b)
#endif
    } while (!(a & b));
}

// generic-proxy writes to shared memory (st.shared) -> visible to the async proxy (tcgen05.mma, TMA)
__device__ __forceinline__ void fence_proxy_async_smem() {
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}

// ---------------------------------------------------------------- TMA
__device__ __forceinline__ void prefetch_tensormap(const void *tmap) {
    asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(tmap)) : "memory");
}

// 2-D tile load global -> shared, completion signalled on `bar` (complete_tx::bytes).
// c0 = coordinate along the innermost (contiguous) dimension, c1 = along the outer one.
__device__ __forceinline__ void tma_load_2d(const void *tmap, uint64_t *bar, void *smem_dst, int32_t c0, int32_t c1) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];"
        ::"r"(smem_u32(smem_dst)),
        "l"(reinterpret_cast<uint64_t>(tmap)), "r"(smem_u32(bar)), "r"(c0), "r"(c1)
        : "memory");
}

// ---------------------------------------------------------------- thread-block clusters (pairs of CTAs)
__device__ __forceinline__ uint32_t cluster_ctarank() {
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
// all threads of all CTAs of the cluster
__device__ __forceinline__ void cluster_sync_all() {
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// ---- CTA pairs (cta_group::2): the even CTA of a cluster of two (the "leader") issues every tcgen05.mma for both
// address of `local_smem_addr` (shared::cta window of this CTA) in the shared::cluster window of CTA `cta`
__device__ __forceinline__ uint32_t mapa_u32(uint32_t local_smem_addr, uint32_t cta) {
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(local_smem_addr), "r"(cta));
    return r;
}
// arrive on an mbarrier given by its shared::cluster address (own or peer CTA).  Default semantics (release at CTA scope), as
// CUTLASS's ClusterBarrier::arrive: what the arrivals of this library hand over is tensor memory (ordered by tcgen05.wait /
// tcgen05.fence) or shared memory that only the async proxy reads (ordered by fence.proxy.async), never generic-proxy data
// of the peer.  The .release.cluster / .acquire.cluster forms cost ~1000 clk per arrive behind outstanding global stores and
// a CCTL.IVALL (L1 invalidate) per successful wait.
__device__ __forceinline__ void mbar_arrive_cluster(uint32_t cluster_addr) {
    asm volatile("mbarrier.arrive.shared::cluster.b64 _, [%0];" ::"r"(cluster_addr) : "memory");
}
// wait on an mbarrier of this CTA whose phase may be completed by arrivals / TMA bytes from the peer CTA
__device__ __forceinline__ void mbar_wait_cluster(uint64_t *bar, uint32_t parity) {
    while (!mbar_try_wait(bar, parity)) {
    }
}
// TMA tile load into THIS CTA's shared memory whose completion (complete_tx) is signalled on an mbarrier of either
// CTA of the pair, given by its shared::cluster address (the leader's "full" barrier counts the bytes of both CTAs)
__device__ __forceinline__ void tma_load_2d_cg2(const void *tmap, uint32_t bar_cluster_addr, uint32_t dst_cluster_addr,
                                                int32_t c0, int32_t c1) {
    asm volatile(
        "cp.async.bulk.tensor.2d.cta_group::2.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];"
        ::"r"(dst_cluster_addr), "l"(reinterpret_cast<uint64_t>(tmap)), "r"(bar_cluster_addr), "r"(c0), "r"(c1)
        : "memory");
}
__device__ __forceinline__ void tmem_alloc_cg2(uint32_t *smem_result, uint32_t ncols) {
    asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(smem_result)),
                 "r"(ncols)
                 : "memory");
}
__device__ __forceinline__ void tmem_relinquish_cg2() {
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc_cg2(uint32_t taddr, uint32_t ncols) {
    asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(ncols) : "memory");
}
// D[tmem of both CTAs] (+)= A * B^T over the pair: M = 256 (each CTA supplies its 128 rows of A from its own shared
// memory at desc_a and receives its 128 rows of D), B = N x 16 with rows [0, N/2) in the leader's shared memory at
// desc_b and rows [N/2, N) in the peer's.  Issued by ONE thread of the leader CTA.
__device__ __forceinline__ void umma_bf16_ss_cg2(uint32_t tmem_d, uint64_t desc_a, uint64_t desc_b, uint32_t idesc,
                                                 uint32_t accumulate) {
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::2.kind::f16 [%0], %1, %2, %3, p;\n\t"
        "}\n" ::"r"(tmem_d),
        "l"(desc_a), "l"(desc_b), "r"(idesc), "r"(accumulate)
        : "memory");
}
// the same with the A operand in TENSOR MEMORY (each CTA's 128 rows of A at tmem_a in its own TMEM: lane = row, one 32-bit
// column = two consecutive K elements, 8 columns per K = 16 step) -- no shared-memory read for A
__device__ __forceinline__ void umma_bf16_ts_cg2(uint32_t tmem_d, uint32_t tmem_a, uint64_t desc_b, uint32_t idesc,
                                                 uint32_t accumulate) {
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::2.kind::f16 [%0], [%1], %2, %3, p;\n\t"
        "}\n" ::"r"(tmem_d),
        "r"(tmem_a), "l"(desc_b), "r"(idesc), "r"(accumulate)
        : "memory");
}
// arrives on the mbarrier at the same offset in every CTA of cta_mask when all MMAs issued so far by this thread are done
__device__ __forceinline__ void umma_commit_cg2(uint64_t *bar, uint16_t cta_mask) {
    asm volatile("tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;" ::"r"(
                     smem_u32(bar)),
                 "h"(cta_mask)
                 : "memory");
}

// TMA tile load delivered to the same shared-memory offset of every CTA in cta_mask; each destination CTA's
// mbarrier at the same offset as `bar` receives the complete_tx of the bytes that landed in ITS shared memory
__device__ __forceinline__ void tma_load_2d_multicast(const void *tmap, uint64_t *bar, void *smem_dst, int32_t c0, int32_t c1,
                                                      uint16_t cta_mask) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes.multicast::cluster"
        " [%0], [%1, {%3, %4}], [%2], %5;" ::"r"(smem_u32(smem_dst)),
        "l"(reinterpret_cast<uint64_t>(tmap)), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "h"(cta_mask)
        : "memory");
}
// tcgen05.commit that arrives on the mbarrier at the same offset in every CTA of cta_mask
__device__ __forceinline__ void umma_commit_multicast(uint64_t *bar, uint16_t cta_mask) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;" ::"r"(
                     smem_u32(bar)),
                 "h"(cta_mask)
                 : "memory");
}

// ---------------------------------------------------------------- programmatic dependent launch (the tail kernel behind the fused one)
// griddep_wait: blocks until the grid this one was launched behind (cudaLaunchAttributeProgrammaticStreamSerialization) has
// completed and its memory is visible; a no-op for a normally launched grid.  griddep_launch_dependents: lets the dependent
// grid's CTAs start (their prologue) as soon as every CTA of this grid has executed it or exited.
__device__ __forceinline__ void griddep_wait() {
    asm volatile("griddepcontrol.wait;" ::: "memory");
}
__device__ __forceinline__ void griddep_launch_dependents() {
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
}

// ---------------------------------------------------------------- tcgen05: TMEM allocation
// One full warp executes these (.sync.aligned).  ncols: power of two in [32, 512].
__device__ __forceinline__ void tmem_alloc(uint32_t *smem_result, uint32_t ncols) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(smem_result)),
                 "r"(ncols)
                 : "memory");
}
__device__ __forceinline__ void tmem_relinquish() {
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(uint32_t taddr, uint32_t ncols) {
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(ncols) : "memory");
}

__device__ __forceinline__ void tc_fence_before_sync() {
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
}
__device__ __forceinline__ void tc_fence_after_sync() {
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
}

// ---------------------------------------------------------------- tcgen05: MMA
// Shared-memory matrix descriptor for a K-major operand tile stored with the 128-byte swizzle:
// rows of 64 BF16 (128 B), groups of 8 rows 1024 B apart (SBO), tile base 1024-byte aligned.
// Bits: [0,14) start address >> 4, [16,30) leading byte offset >> 4 (unused for swizzled K-major: 1),
// [32,46) stride byte offset >> 4, [46,48) descriptor version = 1 (sm_100), [61,64) layout = 2 (SWIZZLE_128B).
__device__ __forceinline__ uint64_t umma_desc_sw128_kmajor(uint32_t smem_addr) {
    uint64_t d = 0;
    d |= static_cast<uint64_t>((smem_addr & 0x3FFFFu) >> 4);
    d |= static_cast<uint64_t>(1) << 16;
    d |= static_cast<uint64_t>(1024 >> 4) << 32;
    d |= static_cast<uint64_t>(1) << 46;
    d |= static_cast<uint64_t>(2) << 61;
    return d;
}

// Shared-memory matrix descriptor for a K-major operand tile WITHOUT swizzle (canonical core-matrix order): a core matrix is
// 8 rows x 16 bytes stored as 128 contiguous bytes; `lbo` = byte distance between core matrices adjacent in K, `sbo` =
// between core matrices adjacent in M / N (8-row groups).  Layout field 0, 16-byte aligned base.
__device__ __forceinline__ uint64_t umma_desc_nosw_kmajor(uint32_t smem_addr, uint32_t lbo, uint32_t sbo) {
    uint64_t d = 0;
    d |= static_cast<uint64_t>((smem_addr & 0x3FFFFu) >> 4);
    d |= static_cast<uint64_t>(lbo >> 4) << 16;
    d |= static_cast<uint64_t>(sbo >> 4) << 32;
    d |= static_cast<uint64_t>(1) << 46;
    return d;
}

// Instruction descriptor for kind::f16 with BF16 A and B (both K-major), FP32 accumulate.
// Bits: [4,6) D format (1 = F32), [7,10) A format (1 = BF16), [10,13) B format (1 = BF16),
// 15 / 16 A / B major (0 = K), [17,23) N >> 3, [24,29) M >> 4.
// f16 = true: FP16 A and B (format code 0) instead of BF16 (format code 1) -- same instruction kind, same rate.
__host__ __device__ __forceinline__ uint32_t umma_idesc_bf16_f32(uint32_t M, uint32_t N, bool f16 = false) {
    const uint32_t fmt = f16 ? 0u : 1u;
    return (1u << 4) | (fmt << 7) | (fmt << 10) | ((N >> 3) << 17) | ((M >> 4) << 24);
}

// D[tmem] (+)= A[smem] * B[smem]^T; issued by ONE thread.  accumulate = 0 overwrites D.
__device__ __forceinline__ void umma_bf16_ss(uint32_t tmem_d, uint64_t desc_a, uint64_t desc_b, uint32_t idesc,
                                             uint32_t accumulate) {
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t"
        "}\n" ::"r"(tmem_d),
        "l"(desc_a), "l"(desc_b), "r"(idesc), "r"(accumulate)
        : "memory");
}

// Arrives on `bar` when every tcgen05.mma issued so far by this thread has completed
// (implies tcgen05.fence::before_thread_sync).
__device__ __forceinline__ void umma_commit(uint64_t *bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar))
                 : "memory");
}

// ---------------------------------------------------------------- tcgen05: TMEM -> registers
// 32 lanes x 32 bit, 16 consecutive columns: thread t of the warp receives lane (base_lane + t).
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t (&v)[16]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
          "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
        : "r"(taddr)
        : "memory");
}

// 32 lanes x 32 bit, 8 consecutive columns
__device__ __forceinline__ void tmem_ld8(uint32_t taddr, uint32_t (&v)[8]) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
                 : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7])
                 : "r"(taddr)
                 : "memory");
}

// 32 lanes x 32 bit, 32 consecutive columns
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

// registers -> TMEM: 32 lanes x 32 bit, 16 consecutive columns (thread t of the warp writes lane base_lane + t)
__device__ __forceinline__ void tmem_st16(uint32_t taddr, const uint32_t (&v)[16]) {
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], "
        "{%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16};" ::"r"(taddr),
        "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]), "r"(v[8]), "r"(v[9]),
        "r"(v[10]), "r"(v[11]), "r"(v[12]), "r"(v[13]), "r"(v[14]), "r"(v[15])
        : "memory");
}
__device__ __forceinline__ void tmem_st_wait() {
    asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
}

__device__ __forceinline__ void tmem_ld_wait() {
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}

// ---------------------------------------------------------------- shared-memory vector store
__device__ __forceinline__ void st_shared_v4(uint32_t addr, uint32_t a, uint32_t b, uint32_t c, uint32_t d) {
    asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(a), "r"(b), "r"(c), "r"(d) : "memory");
}

// ---------------------------------------------------------------- register reallocation between warpgroups
// every warp of a warpgroup (4 consecutive warps) executes the same one; inc blocks until other warpgroups released enough
template <int N> __device__ __forceinline__ void setmaxnreg_dec() {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(N));
}
template <int N> __device__ __forceinline__ void setmaxnreg_inc() {
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(N));
}

// ---------------------------------------------------------------- small math helpers
__device__ __forceinline__ float lg2_approx(float x) {
    float y;
    asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float rcp_approx(float x) {
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float ex2_approx(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// two FP32 -> packed BF16x2 (round to nearest even); `lo` lands in the low 16 bits
__device__ __forceinline__ uint32_t pack_bf16x2(float lo, float hi) {
    uint32_t r;
    asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
    return r;
}

// two FP32 -> packed FP16x2 (round to nearest even); `lo` lands in the low 16 bits
__device__ __forceinline__ uint32_t pack_f16x2(float lo, float hi) {
    uint32_t r;
    asm("cvt.rn.f16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
    return r;
}
// operand type of the tensor path chosen at run time (GPUANN_PRECISION_BF16 / _FP16): one select per pair
__device__ __forceinline__ uint32_t pack_half2(float lo, float hi, bool f16) {
    return f16 ? pack_f16x2(lo, hi) : pack_bf16x2(lo, hi);
}

// Two activations at once, packed to BF16x2: returns 2 GELU(v) = v + v tanh(u), u = v (c0 + c1 v^2) (tanh form, R5).
// The factor 1/2 lives in the NEXT layer's weights (exact in BF16; api.cu scales W_l, l >= 2, of the tensor path), and
// the polynomial runs on packed FP32x2 instructions (mul/fma.f32x2): 7 instructions per pair instead of 15.
// f16: pack to FP16x2 instead (the FP16 variant of the tensor path).
__device__ __forceinline__ uint32_t gelu2_pack(float v0, float v1, bool f16 = false) {
    if (f16) {
        float a, b;
        asm("{\n\t"
            ".reg .b64 x, w, t, c0, c1;\n\t"
            "mov.b64 x, {%2, %3};\n\t"
            "mov.b64 c0, {%4, %4};\n\t"
            "mov.b64 c1, {%5, %5};\n\t"
            "mul.f32x2 w, x, x;\n\t"
            "fma.rn.f32x2 t, w, c1, c0;\n\t"
            "mul.f32x2 t, x, t;\n\t"
            "mov.b64 {%0, %1}, t;\n\t"
            "tanh.approx.f32 %0, %0;\n\t"
            "tanh.approx.f32 %1, %1;\n\t"
            "mov.b64 t, {%0, %1};\n\t"
            "fma.rn.f32x2 t, x, t, x;\n\t"
            "mov.b64 {%0, %1}, t;\n\t"
            "}\n"
            : "=&f"(a), "=&f"(b)
            : "f"(v0), "f"(v1), "f"(0.7978845608028654f), "f"(0.0356774081363001f));
        return pack_f16x2(a, b);
    }
    uint32_t out;
    asm("{\n\t"
        ".reg .b64 x, w, t, c0, c1;\n\t"
        ".reg .f32 a, b;\n\t"
        "mov.b64 x, {%1, %2};\n\t"
        "mov.b64 c0, {%3, %3};\n\t"
        "mov.b64 c1, {%4, %4};\n\t"
        "mul.f32x2 w, x, x;\n\t"
        "fma.rn.f32x2 t, w, c1, c0;\n\t"
        "mul.f32x2 t, x, t;\n\t"
        "mov.b64 {a, b}, t;\n\t"
        "tanh.approx.f32 a, a;\n\t"
        "tanh.approx.f32 b, b;\n\t"
        "mov.b64 t, {a, b};\n\t"
        "fma.rn.f32x2 t, x, t, x;\n\t"
        "mov.b64 {a, b}, t;\n\t"
        "cvt.rn.bf16x2.f32 %0, b, a;\n\t"
        "}\n"
        : "=r"(out)
        : "f"(v0), "f"(v1), "f"(0.7978845608028654f), "f"(0.0356774081363001f));
    return out;
}

}  // namespace ptx
}  // namespace gpuann
