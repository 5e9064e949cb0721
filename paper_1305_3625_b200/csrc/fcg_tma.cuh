// fcg_tma.cuh -- sm_100a asynchronous-copy primitives used by the pipelined passes (fcg_async.cuh):
// mbarrier (transaction-count completion), TMA bulk copies global <-> shared (cp.async.bulk, SASS UBLKCP),
// TMA tensor tile loads / stores (cp.async.bulk.tensor.{2,3,4}d, SASS UTMALDG / UTMASTG), proxy fences and L2 cache-policy hints.
// Device-only inline PTX; nothing here computes anything.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace fcg {
namespace tma {

#ifdef __CUDACC__
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
// make the initialised barriers visible to the async proxy (TMA unit) before any copy names them
__device__ __forceinline__ void fence_mbar_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
// one arrival + announce `bytes` of asynchronous traffic that will complete on this barrier
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
// plain arrival (release): everything this thread did before is ordered before the phase completes
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
// Consumer release of a slot that TMA will overwrite: one arrival per warp.  The proxy fence makes every lane's
// earlier ld.shared *complete* first: a load whose result nobody has used yet can still be queued when the arrival
// is seen, and the refill then lands underneath it (measured on sm_100a: row_fwd2 in PLAIN mode, where the strip
// values are only consumed after the loop, read the next strip's data in ~1e-4 of the warps without this fence).
__device__ __forceinline__ void mbar_warp_release(uint64_t* bar) {
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    __syncwarp();
    if ((threadIdx.x & 31) == 0) mbar_arrive(bar);
}
// Release without the proxy fence, for slots whose every loaded value has already been USED by an arithmetic instruction
// of the same thread (in-order issue + scoreboard: the ld.shared has then completed before the arrival is issued).
__device__ __forceinline__ void mbar_warp_release_consumed(uint64_t* bar) {
    __syncwarp();
    if ((threadIdx.x & 31) == 0) mbar_arrive(bar);
}
// one arrival per warp after generic-proxy WRITES that the async proxy will read (the caller fences)
__device__ __forceinline__ void mbar_warp_arrive(uint64_t* bar) {
    __syncwarp();
    if ((threadIdx.x & 31) == 0) mbar_arrive(bar);
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
// Waiting on an mbarrier phase.  Default: the plain spin (each failed try_wait already blocks in hardware for a system-defined
// time).  -DFCG_BOUNDED_WAITS builds the bounded form instead: after WAIT_CAP failed polls (seconds; a legitimate wait is
// microseconds) the thread raises *tmo and gives up, every other waiter that has been polling for a while sees the flag and
// gives up too, the kernel ends with garbage instead of spinning for ever, and the host finds the flag in the scalar block it
// reads back after every solve and returns FCG_CUDA_ERROR.  It is not the default because it costs 3 % of the iteration
// (measured on one B200, same box, interleaved runs: L = 2048 fp64 94.0 -> 97.3 us, L = 8192 fp32 788 -> 810 us; a trap after the
// cap or a non-inlined slow path cost the same: with any bookkeeping in the loop the compiler schedules the phase checks
// differently).  A wait can only fail to complete through a programming error in this file (a wrong
// expect_tx byte count, a lost arrival), which the parity and stress tests at every size would catch as a hang.
constexpr uint32_t WAIT_CAP = 1u << 26, WAIT_LOOK = 1u << 10;
__device__ __forceinline__ void mbar_wait_bounded(uint64_t* bar, uint32_t parity, unsigned int* tmo) {
    uint32_t polls = 0;
    while (!mbar_try_wait(bar, parity)) {
        if ((++polls & (WAIT_LOOK - 1)) == 0) {
            if (*reinterpret_cast<volatile unsigned int*>(tmo) != 0u) return;
            if (polls >= WAIT_CAP) { atomicExch(tmo, 1u); return; }
        }
    }
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity, unsigned int* tmo) {
#ifdef FCG_BOUNDED_WAITS
    if (!mbar_try_wait(bar, parity)) mbar_wait_bounded(bar, parity, tmo);
#else
    (void)tmo;
    while (!mbar_try_wait(bar, parity)) {}
#endif
}

// L2 eviction-priority policies for the cache_hint operand of the copies below
__device__ __forceinline__ uint64_t policy_evict_first() {
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ uint64_t policy_evict_last() {
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
    return p;
}

__device__ __forceinline__ uint64_t policy_evict_normal() {
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_normal.b64 %0, 1.0;" : "=l"(p));
    return p;
}

// contiguous global -> shared, completion counted in bytes on `bar`.  16-byte aligned, size % 16 == 0.
__device__ __forceinline__ void bulk_g2s(void* dst_smem, const void* src_gmem, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst_smem)),
                 "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void bulk_g2s_hint(void* dst_smem, const void* src_gmem, uint32_t bytes, uint64_t* bar, uint64_t policy) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(
                     smem_u32(dst_smem)),
                 "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar)), "l"(policy)
                 : "memory");
}
// 16 bytes global -> shared by the LSU's asynchronous copy (LDGSTS): no register staging, not a TMA request.  Completion: the
// issuing thread calls cp_async_arrive on an mbarrier whose init count includes it (.noinc), which fires once all its copies landed.
__device__ __forceinline__ void cp_async16(void* dst_smem, const void* src_gmem) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(dst_smem)), "l"(src_gmem) : "memory");
}
__device__ __forceinline__ void cp_async_arrive(uint64_t* bar) {
    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
// contiguous shared -> global (bulk async-group completion)
__device__ __forceinline__ void bulk_s2g(void* dst_gmem, const void* src_smem, uint32_t bytes) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst_gmem), "r"(smem_u32(src_smem)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_s2g_hint(void* dst_gmem, const void* src_smem, uint32_t bytes, uint64_t policy) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group.L2::cache_hint [%0], [%1], %2, %3;" ::"l"(dst_gmem), "r"(smem_u32(src_smem)),
                 "r"(bytes), "l"(policy)
                 : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
// wait until the shared-memory source of all committed bulk stores has been read (the CTA may then reuse / exit)
__device__ __forceinline__ void bulk_wait_read0() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }

// 2D tensor tile global -> shared through a CUtensorMap (coordinates in elements: c0 fastest)
__device__ __forceinline__ void tensor_g2s_2d(void* dst_smem, const void* tmap, int c0, int c1, uint64_t* bar) {
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];" ::"r"(
                     smem_u32(dst_smem)),
                 "l"(tmap), "r"(c0), "r"(c1), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void tensor_g2s_2d_hint(void* dst_smem, const void* tmap, int c0, int c1, uint64_t* bar, uint64_t policy) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%2, %3}], [%4], %5;" ::"r"(
            smem_u32(dst_smem)),
        "l"(tmap), "r"(c0), "r"(c1), "r"(smem_u32(bar)), "l"(policy)
        : "memory");
}
__device__ __forceinline__ void tensor_g2s_3d(void* dst_smem, const void* tmap, int c0, int c1, int c2, uint64_t* bar) {
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];" ::"r"(
                     smem_u32(dst_smem)),
                 "l"(tmap), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void tensor_g2s_3d_hint(void* dst_smem, const void* tmap, int c0, int c1, int c2, uint64_t* bar, uint64_t policy) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%2, %3, %4}], [%5], %6;" ::"r"(
            smem_u32(dst_smem)),
        "l"(tmap), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(bar)), "l"(policy)
        : "memory");
}
__device__ __forceinline__ void tensor_g2s_4d(void* dst_smem, const void* tmap, int c0, int c1, int c2, int c3, uint64_t* bar) {
    asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];" ::"r"(
                     smem_u32(dst_smem)),
                 "l"(tmap), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(smem_u32(bar))
                 : "memory");
}
// tensor tile shared -> global (bulk async-group completion), the scatter twin of tensor_g2s_4d
__device__ __forceinline__ void tensor_s2g_4d(const void* tmap, int c0, int c1, int c2, int c3, const void* src_smem) {
    asm volatile("cp.async.bulk.tensor.4d.global.shared::cta.tile.bulk_group [%0, {%1, %2, %3, %4}], [%5];" ::"l"(tmap), "r"(c0), "r"(c1),
                 "r"(c2), "r"(c3), "r"(smem_u32(src_smem))
                 : "memory");
}
// 5-D tiles: the slab decomposition's column pass reads the exchange buffer [source rank][column block][local row pair][column][2 complex] directly
__device__ __forceinline__ void tensor_g2s_5d(void* dst_smem, const void* tmap, int c0, int c1, int c2, int c3, int c4, uint64_t* bar) {
    asm volatile("cp.async.bulk.tensor.5d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5, %6}], [%7];" ::"r"(
                     smem_u32(dst_smem)),
                 "l"(tmap), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void tensor_s2g_5d(const void* tmap, int c0, int c1, int c2, int c3, int c4, const void* src_smem) {
    asm volatile("cp.async.bulk.tensor.5d.global.shared::cta.tile.bulk_group [%0, {%1, %2, %3, %4, %5}], [%6];" ::"l"(tmap), "r"(c0), "r"(c1),
                 "r"(c2), "r"(c3), "r"(c4), "r"(smem_u32(src_smem))
                 : "memory");
}
__device__ __forceinline__ void tensor_s2g_3d(const void* tmap, int c0, int c1, int c2, const void* src_smem) {
    asm volatile("cp.async.bulk.tensor.3d.global.shared::cta.tile.bulk_group [%0, {%1, %2, %3}], [%4];" ::"l"(tmap), "r"(c0), "r"(c1), "r"(c2),
                 "r"(smem_u32(src_smem))
                 : "memory");
}
__device__ __forceinline__ void prefetch_tmap(const void* tmap) {
    asm volatile("prefetch.tensormap [%0];" ::"l"(tmap) : "memory");
}
// Programmatic dependent launch: let the next kernel of the stream start its prologue while this grid drains
// (launch_dependents), and block until the previous grid has completed and its writes are visible (wait).  Both are
// no-ops for a kernel launched without the programmatic-serialization attribute.
__device__ __forceinline__ void grid_dep_launch() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void grid_dep_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
// Start offset between the CTAs that share an SM.  CTAs launched together move through their phases together -- all of them waiting
// for copies, then all of them in the butterflies -- so the copy engine and the arithmetic pipes take turns instead of overlapping.
// A fraction of one work item's time between their starts keeps them out of step for the whole launch (persistent CTAs) or hands the
// offsets on to the CTAs that replace them (one CTA per item).  Cost: the wait itself, at most once per CTA.
__device__ __forceinline__ void stagger_wait(unsigned long long ns) {
    unsigned long long t0, t1;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t0));
    do { __nanosleep(200); asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t1)); } while (t1 - t0 < ns);
}
// generic-proxy writes to shared memory -> visible to the async proxy (before a bulk store reads them)
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// plain global stores with an L2 eviction hint
__device__ __forceinline__ void st_hint(double* p, double v, uint64_t pol) {
    asm volatile("st.global.L2::cache_hint.f64 [%0], %1, %2;" ::"l"(p), "d"(v), "l"(pol) : "memory");
}
__device__ __forceinline__ void st_hint(float* p, float v, uint64_t pol) {
    asm volatile("st.global.L2::cache_hint.f32 [%0], %1, %2;" ::"l"(p), "f"(v), "l"(pol) : "memory");
}
__device__ __forceinline__ void st_hint(double2* p, double2 v, uint64_t pol) {
    asm volatile("st.global.L2::cache_hint.v2.f64 [%0], {%1, %2}, %3;" ::"l"(p), "d"(v.x), "d"(v.y), "l"(pol) : "memory");
}
__device__ __forceinline__ void st_hint(float4* p, float4 v, uint64_t pol) {
    asm volatile("st.global.L2::cache_hint.v4.f32 [%0], {%1, %2, %3, %4}, %5;" ::"l"(p), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w), "l"(pol)
                 : "memory");
}
// plain global loads with an L2 eviction hint
__device__ __forceinline__ double2 ld_hint(const double2* p, uint64_t pol) {
    double2 v;
    asm volatile("ld.global.L2::cache_hint.v2.f64 {%0, %1}, [%2], %3;" : "=d"(v.x), "=d"(v.y) : "l"(p), "l"(pol) : "memory");
    return v;
}
__device__ __forceinline__ float4 ld_hint(const float4* p, uint64_t pol) {
    float4 v;
    asm volatile("ld.global.L2::cache_hint.v4.f32 {%0, %1, %2, %3}, [%4], %5;" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p), "l"(pol) : "memory");
    return v;
}
#endif  // __CUDACC__

}  // namespace tma
}  // namespace fcg
