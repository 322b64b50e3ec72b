// vg_tma.cuh -- mbarrier and TMA bulk-copy (cp.async.bulk, 1-D) helpers shared by the streaming query kernel
// (track tiles: global -> shared ring) and the navigator (daughter table: global -> shared, once per CTA).
// SASS: UBLKCP (bulk copy), SYNCS (mbarrier).
#pragma once
#include "vg_math.cuh"

namespace vg {

VG_DEV uint32_t smem_u32(const void *p) { return static_cast<uint32_t>(__cvta_generic_to_shared(p)); }

VG_DEV void mbar_init(uint64_t *bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}

// makes the initialised barriers visible to the async proxy (the bulk-copy engine)
VG_DEV void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }

VG_DEV void mbar_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}

VG_DEV void mbar_arrive(uint64_t *bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}

// try_wait suspends the thread in hardware for a bounded time; loop until the phase with this parity completes
VG_DEV void mbar_wait(uint64_t *bar, uint32_t parity)
{
    uint32_t b = smem_u32(bar), done = 0;
    while (!done) {
        asm volatile("{\n"
                     ".reg .pred p;\n"
                     "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
                     "selp.u32 %0, 1, 0, p;\n"
                     "}\n"
                     : "=r"(done)
                     : "r"(b), "r"(parity)
                     : "memory");
    }
}

// one bulk copy global -> shared of `bytes` (multiple of 16; both addresses 16-byte aligned), completion counted
// on `bar` in bytes
VG_DEV void bulk_g2s(void *dst_smem, const void *src_gmem, uint32_t bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst_smem)),
                 "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

// same with an L2 eviction-priority hint (evict_first: every track byte is read exactly once)
VG_DEV void bulk_g2s_hint(void *dst_smem, const void *src_gmem, uint32_t bytes, uint64_t *bar, uint64_t policy)
{
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(
            smem_u32(dst_smem)),
        "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar)), "l"(policy)
        : "memory");
}

VG_DEV uint64_t policy_evict_first()
{
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    return p;
}

// ---- cluster launch control (sm_100): a running CTA asks the hardware scheduler to cancel a CTA of the same grid
// that has not been launched yet and takes over its block index -- dynamic load balancing for persistent CTAs
// without any global counter.  The 16-byte response lands in shared memory asynchronously (async proxy) and
// completes 16 bytes on `bar`.  After the first failed request a CTA must not ask again.
VG_DEV void clc_try_cancel(void *resp_smem16, uint64_t *bar)
{
    asm volatile("clusterlaunchcontrol.try_cancel.async.shared::cta.mbarrier::complete_tx::bytes.b128 [%0], [%1];" ::"r"(
                     smem_u32(resp_smem16)),
                 "r"(smem_u32(bar))
                 : "memory");
}

// decode a response: returns the stolen blockIdx.x, or -1 if nothing was left to cancel
VG_DEV int clc_decode_x(const void *resp_smem16)
{
    uint32_t ok, bx;
    asm volatile("{\n"
                 ".reg .b128 r;\n"
                 ".reg .pred p;\n"
                 "ld.shared.b128 r, [%2];\n"
                 "clusterlaunchcontrol.query_cancel.is_canceled.pred.b128 p, r;\n"
                 "selp.u32 %0, 1, 0, p;\n"
                 "@p clusterlaunchcontrol.query_cancel.get_first_ctaid::x.b32.b128 %1, r;\n"
                 "@!p mov.u32 %1, 0;\n"
                 "}\n"
                 : "=r"(ok), "=r"(bx)
                 : "r"(smem_u32(resp_smem16))
                 : "memory");
    return ok ? int(bx) : -1;
}

// ---- programmatic dependent launch: a kernel launched with cudaLaunchAttributeProgrammaticStreamSerialization may be
// scheduled while its predecessor in the stream is still draining; pdl_wait() blocks until the predecessor grid has
// completed and its memory operations are visible, so everything before it (barrier set-up, index arithmetic, the
// launch latency itself) overlaps the predecessor's tail.  Both are no-ops in a kernel launched without the attribute.
VG_DEV void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
VG_DEV void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

// orders this thread's generic-proxy accesses to shared memory before later async-proxy writes to it
VG_DEV void fence_proxy_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

} // namespace vg
