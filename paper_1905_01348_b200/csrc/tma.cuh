// tma.cuh -- mbarrier and 1-D bulk asynchronous copy (TMA, cp.async.bulk) helpers used by the slab passes.
// SASS: UBLKCP (bulk copy), SYNCS.* (mbarrier).  No tensor maps: every transfer here is a contiguous run of
// 16-byte elements, so the 1-D form is enough and needs no driver-API descriptor.
#pragma once
#include "codelets.cuh"

namespace ptfock {

// ---- mbarrier + 1-D bulk async copy (TMA) helpers: global -> shared, completion counted in bytes ----
PTF_DEV unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
PTF_DEV void mbar_init(unsigned long long *bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
PTF_DEV void mbar_expect_tx(unsigned long long *bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
PTF_DEV void mbar_wait(unsigned long long *bar, unsigned parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
PTF_DEV void bulk_g2s(void *dst_smem, const void *src_gmem, unsigned bytes, unsigned long long *bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst_smem)),
                 "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
PTF_DEV void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

}  // namespace ptfock
