// slab3.cuh -- warp-specialised versions of the 3-stage slab passes (slab2.cuh).
//
// ncu on slab2 (profiles/r01_*): with one 8-warp CTA per SM every stage is "all warps load shared
// memory -> all warps do FP64 -> all warps store", so the L1/shared pipe (~60 % busy) and the FP64 pipe
// (~35 % busy) take turns instead of overlapping.  Here a CTA has two groups of NT threads that work on
// DIFFERENT stages of consecutive orbitals at the same time, handing tiles over through two shared-memory
// buffers guarded by named barriers (bar.sync / bar.arrive):
//   pass A:  group P = global phi -> x psi_j -> stage 1 -> tile[b]      group Q = stage 2, stage 3 -> global
//   pass C:  group X = global W -> stage 1' -> stage 2' -> tile[b]      group Y = stage 3' -> x phi_i -> sum_i
// Register budget 128 per thread (512 threads): P holds psi_j plus a two-deep register prefetch of phi,
// Y holds the accumulators plus a one-deep prefetch of phi, X a one-deep prefetch of the pair density.
#pragma once
#include "slab2.cuh"

#ifndef PTF_REGS_X
#define PTF_REGS_X 144      // setmaxnreg split of pass C: X prefetches the pair density in registers,
#define PTF_REGS_Y 112      // Y keeps the accumulators; 256 * (144 + 112) = 64 Ki registers
#endif

namespace ptfock {

PTF_DEV void named_sync(int id, int count) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(count) : "memory"); }
PTF_DEV void named_arrive(int id, int count) { asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(count) : "memory"); }

template <int R> PTF_DEV void reg_dealloc() { asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(R)); }
template <int R> PTF_DEV void reg_alloc() { asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(R)); }

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

enum { BAR_FULL0 = 1, BAR_FULL1 = 2, BAR_EMPTY0 = 3, BAR_EMPTY1 = 4, BAR_GROUP = 5, BAR_GROUP2 = 6 };

template <class S> struct Slab3 {
    static constexpr int NT2 = 2 * S::NT;
    static constexpr int TILE = S::N1 * S::P;                 // elements per tile buffer
    static constexpr int SMEM_BYTES = 2 * TILE * (int)sizeof(cd);
    // pass C adds a padded staging tile for phi_i (filled by bulk async copies) and one mbarrier
    static constexpr int SMEM_BYTES_INV = 3 * TILE * (int)sizeof(cd) + 16;
    static_assert(S::S2 <= S::NT, "stage 2 must fit one group");
    static_assert(S::A2 == 16, "group Y interleaves the second half of the radix-16 codelet with the accumulation");
};

// ---- pass A ---------------------------------------------------------------------------------------
template <class S>
__global__ void __launch_bounds__(2 * S::NT, 1) slab3_fwd(const SlabArgs g) {
    constexpr int N2 = S::N2, B1 = S::B1, A2 = S::A2, B2 = S::B2, P = S::P, NT = S::NT;
    constexpr int NT2 = Slab3<S>::NT2, TILE = Slab3<S>::TILE;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cd *tile = reinterpret_cast<cd *>(smem_raw);
    const int x0 = blockIdx.y, jj = blockIdx.x;
    const long long slab_off = (long long)x0 * S::NPTS;
    const int per = (g.na + gridDim.z - 1) / gridDim.z;
    const int ii_beg = blockIdx.z * per, ii_end = min(g.na, ii_beg + per);
    const int n_it = ii_end - ii_beg;
    if (n_it <= 0) return;
    if (threadIdx.x < NT) {
        // ---------------- group P: product + stage 1 ----------------
        const int tid = threadIdx.x;
        const int b2 = tid % B2, x1 = stage1_row<S>(tid / B2);
        const int goff = x1 * N2 + b2;
        const cd *psi = g.b + (long long)(g.b0 + jj) * g.grid_pts + slab_off + goff;
        const cd *phi0 = g.a + (long long)(g.a0 + ii_beg) * g.grid_pts + slab_off + goff;
        cd pj[A2], v[A2];
#pragma unroll
        for (int a2 = 0; a2 < A2; ++a2) pj[a2] = psi[a2 * B2];
#pragma unroll
        for (int a2 = 0; a2 < A2; ++a2) v[a2] = __ldg(reinterpret_cast<const double2 *>(phi0 + a2 * B2));
        for (int it = 0; it < n_it; ++it) {
            const int b = it & 1;
            cd *d = tile + b * TILE + x1 * P + b2;
            // the tile was handed to Q two iterations ago; Q is the longer stage, so the phi loads issued
            // at the end of the previous iteration have had a whole Q iteration to land
            if (it >= 2) named_sync(BAR_EMPTY0 + b, NT2);
#pragma unroll
            for (int a2 = 0; a2 < A2; ++a2) v[a2] = cmulc(pj[a2], v[a2]);
            DFT<A2, false>::run(v);
#pragma unroll
            for (int k = 0; k < A2; ++k) d[k * B2] = v[k];
            if (it + 1 < n_it) {
                const cd *phi = phi0 + (long long)(it + 1) * g.grid_pts;
#pragma unroll
                for (int a2 = 0; a2 < A2; ++a2) v[a2] = __ldg(reinterpret_cast<const double2 *>(phi + a2 * B2));
            }
            named_arrive(BAR_FULL0 + b, NT2);
        }
    } else {
        // ---------------- group Q: stage 2 + stage 3 + store ----------------
        const int tid = threadIdx.x - NT;
        const int pos2 = tid % N2, k1a = tid / N2;
        cd tw2r[B2 > 1 ? B2 - 1 : 1], tw1r[S::A1 > 1 ? S::A1 - 1 : 1];
        load_stage2_twiddles<S>(g.tw1, g.tw2, tid < S::S2 ? tid : 0, tw2r, tw1r);
        for (int it = 0; it < n_it; ++it) {
            const int b = it & 1;
            cd *s = tile + b * TILE;
            named_sync(BAR_FULL0 + b, NT2);
            if (tid < S::S2) stage2<S, false>(s, tid, tw2r, tw1r);
            named_sync(BAR_GROUP, NT);
            cd w[B1];
#pragma unroll
            for (int q = 0; q < B1; ++q) w[q] = s[(k1a * B1 + q) * P + pos2];
            if (it + 2 < n_it) named_arrive(BAR_EMPTY0 + b, NT2);
            DFT<B1, false>::run(w);
            cd *dst = g.scratch + ((long long)((ii_beg + it) * g.stride_loop + jj * g.stride_cta) * g.n0 + x0) * S::NPTS +
                      k1a * B1 * N2 + pos2;
#pragma unroll
            for (int q = 0; q < B1; ++q) dst[q * N2] = w[q];
        }
    }
}

// ---- pass C ---------------------------------------------------------------------------------------
template <class S>
__global__ void __launch_bounds__(2 * S::NT, 1) slab3_inv_acc(const SlabArgs g) {
    constexpr int N2 = S::N2, B1 = S::B1, A2 = S::A2, B2 = S::B2, P = S::P, NT = S::NT;
    constexpr int NT2 = Slab3<S>::NT2, TILE = Slab3<S>::TILE;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cd *tile = reinterpret_cast<cd *>(smem_raw);
    const int x0 = blockIdx.y, tt = blockIdx.x;
    const long long slab_off = (long long)x0 * S::NPTS;
    const int n_it = g.na;
    if (n_it <= 0) return;
    if (threadIdx.x < NT) {
        // ---------------- group X: load pair density, stage 1', stage 2' ----------------
        reg_alloc<PTF_REGS_X>();
        const int tid = threadIdx.x;
        const int pos2 = tid % N2, k1a = tid / N2;
        cd tw2r[B2 > 1 ? B2 - 1 : 1], tw1r[S::A1 > 1 ? S::A1 - 1 : 1];
        load_stage2_twiddles<S>(g.tw1, g.tw2, tid < S::S2 ? tid : 0, tw2r, tw1r);
        const long long pair_stride = (long long)g.stride_loop * g.n0 * S::NPTS;
        const cd *src0 = g.scratch + ((long long)(tt * g.stride_cta) * g.n0 + x0) * S::NPTS + k1a * B1 * N2 + pos2;
        cd w[B1];
#pragma unroll
        for (int q = 0; q < B1; ++q) w[q] = src0[q * N2];
        for (int it = 0; it < n_it; ++it) {
            const int b = it & 1;
            cd *s = tile + b * TILE;
            if (it >= 2) named_sync(BAR_EMPTY0 + b, NT2);
            DFT<B1, true>::run(w);
#pragma unroll
            for (int q = 0; q < B1; ++q) s[(k1a * B1 + q) * P + pos2] = w[q];
            if (it + 1 < n_it) {
                const cd *src = src0 + (long long)(it + 1) * pair_stride;
#pragma unroll
                for (int q = 0; q < B1; ++q) w[q] = src[q * N2];
            }
            named_sync(BAR_GROUP, NT);
            if (tid < S::S2) stage2<S, true>(s, tid, tw2r, tw1r);
            named_arrive(BAR_FULL0 + b, NT2);
        }
    } else {
        // ---------------- group Y: stage 3', x phi, accumulate ----------------
        reg_dealloc<PTF_REGS_Y>();
        const int tid = threadIdx.x - NT;
        const int b2 = tid % B2, x1 = stage1_row<S>(tid / B2);
        const int goff = x1 * N2 + b2;
        cd *fbuf = tile + 2 * TILE;                                           // phi_i slab, same padded layout as a tile
        unsigned long long *fbar = reinterpret_cast<unsigned long long *>(fbuf + TILE);
        const cd *phi_slab0 = g.a + (long long)g.a0 * g.grid_pts + slab_off;  // contiguous N1*N2 slab of orbital a0
        constexpr unsigned ROW_BYTES = N2 * sizeof(cd);
        if (tid == 0) {
            mbar_init(fbar, 1);
            fence_proxy_async();
            mbar_expect_tx(fbar, S::N1 * ROW_BYTES);
            for (int r = 0; r < S::N1; ++r) bulk_g2s(fbuf + r * P, phi_slab0 + r * N2, ROW_BYTES, fbar);
        }
        cd acc[A2];
#pragma unroll
        for (int a2 = 0; a2 < A2; ++a2) acc[a2] = make_double2(0.0, 0.0);
        const cd *fs = fbuf + x1 * P + b2;
        for (int it = 0; it < n_it; ++it) {
            const int b = it & 1;
            const cd *s = tile + b * TILE + x1 * P + b2;
            named_sync(BAR_FULL0 + b, NT2);
            cd v[A2];
#pragma unroll
            for (int k = 0; k < A2; ++k) v[k] = s[k * B2];
            if (it + 2 < n_it) named_arrive(BAR_EMPTY0 + b, NT2);
            DFT<A2, true>::first_half(v);
            mbar_wait(fbar, it & 1);                                          // phi_i slab has landed
#pragma unroll
            for (int k1 = 0; k1 < 4; ++k1) {
                DFT<A2, true>::second_half(v, k1);                            // v[4 k1 + k2] = W(a2 = k1 + 4 k2)
#pragma unroll
                for (int k2 = 0; k2 < 4; ++k2) {
                    const int a2 = k1 + 4 * k2;
                    const cd f = fs[a2 * B2];
                    const cd pr = g.conj_w ? cmulc(f, v[4 * k1 + k2]) : cmul(f, v[4 * k1 + k2]);
                    acc[a2].x += pr.x;
                    acc[a2].y += pr.y;
                }
            }
            named_sync(BAR_GROUP2, NT);                                       // every Y thread is done with fbuf
            if (tid == 0 && it + 1 < n_it) {
                const cd *src = phi_slab0 + (long long)(it + 1) * g.grid_pts;
                fence_proxy_async();
                mbar_expect_tx(fbar, S::N1 * ROW_BYTES);
                for (int r = 0; r < S::N1; ++r) bulk_g2s(fbuf + r * P, src + r * N2, ROW_BYTES, fbar);
            }
        }
        cd *o = g.out + (long long)(g.b0 + tt) * g.grid_pts + slab_off + goff;
#pragma unroll
        for (int a2 = 0; a2 < A2; ++a2) {
            cd cur = o[a2 * B2];
            cur.x += acc[a2].x;
            cur.y += acc[a2].y;
            o[a2 * B2] = cur;
        }
    }
}

}  // namespace ptfock
