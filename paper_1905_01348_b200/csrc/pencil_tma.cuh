// pencil_tma.cuh -- pass B with tensor-map TMA: the [N0 rows] x [CW contiguous slab positions] tile of one pair is
// fetched by ONE cp.async.bulk.tensor.2d load (rows are slab_pts*16 bytes apart in the pair scratch), transformed
// IN PLACE in shared memory (forward DFT along x0, x v'(G), inverse DFT along x0; Alg. 2 line 7, the
// "Poisson-like equation"), and written back by one tensor store.  All global traffic is asynchronous and needs no
// address registers; several CTAs per SM run out of phase.  SASS: UTMALDG / UTMASTG.
#pragma once
#include <cuda.h>
#include "kernels.cuh"
#include "tma.cuh"

namespace ptfock {

PTF_DEV void tensor_g2s_2d(void *dst_smem, const CUtensorMap *map, int c0, int c1, unsigned long long *bar) {
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
                 ::"r"(smem_u32(dst_smem)), "l"(map), "r"(c0), "r"(c1), "r"(smem_u32(bar)) : "memory");
}
PTF_DEV void tensor_s2g_2d(const CUtensorMap *map, int c0, int c1, const void *src_smem) {
    asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.bulk_group [%0, {%1, %2}], [%3];"
                 ::"l"(map), "r"(c0), "r"(c1), "r"(smem_u32(src_smem)) : "memory");
}

template <int N0> struct PencilTma {
    static constexpr int R1 = Split<N0>::R1, R2 = Split<N0>::R2;
    // measured on B200: small tiles and MANY co-resident CTAs (each is load -> 3 stages -> store, so the SM needs
    // several in different phases to keep HBM busy): 16-wide tiles, 128 threads; 8 CTAs/SM (64 registers) at n0 = 64
    // reach 97 % of the measured copy bandwidth, 6 CTAs/SM (80 registers) at n0 = 128 / 120 reach 93 % / 91 %
    static constexpr int CW = 16;
    static constexpr int NT = CW * 8;
    static constexpr int TILE_BYTES = N0 * CW * 16;
    static constexpr int SMEM_BYTES = TILE_BYTES + N0 * 16 + 16;      // tile, twiddles, mbarrier
    static constexpr int MINB = (N0 >= 120) ? 6 : (N0 == 64 ? 8 : 4);
    static_assert(R2 > 1, "single-stage pencils use pencil_mid");
};

struct PencilTmaArgs {
    const double *v;     // [N0 positions][slab_pts], digit-permuted, -alpha/N folded in
    const cd *tw0;
    int slab_pts;
    int tri_nj;          // see PencilArgs
    int pair0;           // pair index (in the scratch the tensor map covers) of the wave's first pair
};

// grid = (ceil(slab_pts / CW), pairs); the tensor map views the scratch as [pairs*N0 rows][2*slab_pts doubles]
template <int N0>
__global__ void __launch_bounds__(PencilTma<N0>::NT, PencilTma<N0>::MINB)
pencil_tma(const __grid_constant__ CUtensorMap map, const PencilTmaArgs g) {
    using S = PencilTma<N0>;
    constexpr int R1 = S::R1, R2 = S::R2, CW = S::CW, NT = S::NT;
    extern __shared__ __align__(128) unsigned char smem_pt[];
    cd *s = reinterpret_cast<cd *>(smem_pt);
    cd *tw = reinterpret_cast<cd *>(smem_pt + S::TILE_BYTES);
    unsigned long long *bar = reinterpret_cast<unsigned long long *>(smem_pt + S::TILE_BYTES + N0 * 16);
    const int tid = threadIdx.x;
    const long long sp = g.slab_pts;
    if (g.tri_nj > 0 && (int)blockIdx.y / g.tri_nj > (int)blockIdx.y % g.tri_nj) return;
    const int p0 = blockIdx.x * CW;
    const int row0 = (g.pair0 + blockIdx.y) * N0;
    if (tid == 0) {
        mbar_init(bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        fence_proxy_async();
        mbar_expect_tx(bar, S::TILE_BYTES);
        tensor_g2s_2d(s, &map, 2 * p0, row0, bar);
    }
    for (int t = tid; t < N0; t += NT) tw[t] = g.tw0[t];
    const int cvalid = (sp - p0 < CW) ? (int)(sp - p0) : CW;          // ragged last tile: the load zero-fills, the store clips
    __syncthreads();
    mbar_wait(bar, 0);
    // stage 1: DFT over a (x0 = a R2 + b), twiddle w^(b k1), in place at rows k1 R2 + b
    for (int t = tid; t < CW * R2; t += NT) {
        const int c = t % CW, b = t / CW;
        cd v[R1];
#pragma unroll
        for (int a = 0; a < R1; ++a) v[a] = s[(a * R2 + b) * CW + c];
        DFT<R1, false>::run(v);
#pragma unroll
        for (int k1 = 1; k1 < R1; ++k1) v[k1] = cmul(v[k1], tw[b * k1]);
#pragma unroll
        for (int k1 = 0; k1 < R1; ++k1) s[(k1 * R2 + b) * CW + c] = v[k1];
    }
    __syncthreads();
    // middle: forward DFT over b, x v', inverse DFT over k2
    for (int t = tid; t < CW * R1; t += NT) {
        const int c = t % CW, k1 = t / CW;
        cd v[R2];
#pragma unroll
        for (int b = 0; b < R2; ++b) v[b] = s[(k1 * R2 + b) * CW + c];
        DFT<R2, false>::run(v);
#pragma unroll
        for (int k2 = 0; k2 < R2; ++k2)
            v[k2] = cscale(v[k2], c < cvalid ? __ldg(g.v + (long long)(k1 * R2 + k2) * sp + p0 + c) : 0.0);
        DFT<R2, true>::run(v);
#pragma unroll
        for (int b = 0; b < R2; ++b) s[(k1 * R2 + b) * CW + c] = v[b];
    }
    __syncthreads();
    // last: conj twiddle, inverse DFT over k1, in place
    for (int t = tid; t < CW * R2; t += NT) {
        const int c = t % CW, b = t / CW;
        cd v[R1];
#pragma unroll
        for (int k1 = 0; k1 < R1; ++k1) v[k1] = s[(k1 * R2 + b) * CW + c];
#pragma unroll
        for (int k1 = 1; k1 < R1; ++k1) v[k1] = cmulc(v[k1], tw[b * k1]);
        DFT<R1, true>::run(v);
#pragma unroll
        for (int a = 0; a < R1; ++a) s[(a * R2 + b) * CW + c] = v[a];
    }
    fence_proxy_async();
    __syncthreads();
    if (tid == 0) {
        tensor_s2g_2d(&map, 2 * p0, row0, s);
        asm volatile("cp.async.bulk.commit_group;" ::: "memory");
        asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");     // shared memory must outlive the store's reads
    }
}

}  // namespace ptfock
