// pass8.cuh -- the two-stage split of the pair-solve ("8 + 10 + 8 bits" at 64^3; Alg. 2 lines 6-10, Eq. (3)).
//
// The three passes of kernels.cuh / slabx.cuh give the slab passes three butterfly stages (six shared-memory crossings
// per point) and the pencil pass one or two; ncu showed the slab passes bound by the L1 / shared-memory data pipe, not
// by HBM (profiles/r01_ncu_full_si512.md).  Here the slab passes keep only TWO stages and hand the low digit b1 of x1
// to the pencil pass, which has the slack:
//
//   x0 = a0*B0 + b0,  x1 = a1*B1 + b1,  x2 = a2*B2 + b2,  b1 = q*RQ + r  (RQ = 4)
//   pass A  p8_fwd     : rho = conj(phi_i) psi_j;  2-D DFT over (a1, a2) + both twiddles | DFT over b2
//                        one CTA = one (target, x0, q); phi_i's rows (A1 runs of RQ*N2 elements) arrive by bulk async
//                        copies (TMA) in a ring of shared-memory buffers, both stages work in place in the landed
//                        buffer through an XOR swizzle, results leave from registers in runs of NT2 elements.
//   pass B  p8_mid     : 2-D DFT over (x0, b1): stage (a0, b1) + twiddle | DFT over b0, x v'(G), and back;
//                        tile = [q][x0][P positions x RQ r] (128-byte rows) by ONE swizzled tensor-map TMA load / store.
//   pass C  p8_inv_acc : mirror of A; x phi_i and the sum over i in registers.
//
// Instantiated for 64^3 (A1 = A2 = 4, A0 = 2: 16-point slab stages, 32 x 32 pencil stages; 64-thread CTAs / groups),
// 48^3 (A1 = A2 = 3, A0 = 2: 9 | 16 and 32 | 24) and 32^3 (A1 = 4, A2 = 2, A0 = 2: 8 | 16 and 16 | 16).  The stages' task counts may differ (NT1 != NT2, NTB1 != NTB2):
// threads without a task only keep the barriers.
//
// Pair scratch: [pair][q][x0][k2b][k1a][k2a][r] (16-byte elements): a pass A / C CTA owns one contiguous row
// (pair, q, x0) of QPTS elements; pass B sees the NQ*N0 rows (q, x0) of one pair, 128 contiguous bytes of each.
// Frequencies: k0 = k0a + A0*k0b, k1 = k1a + A1*k1b, k2 = k2a + A2*k2b; nothing is ever un-permuted (the v' table is
// stored in pass B's register order, build_vtable).
#pragma once
#include <cuda.h>
#include "kernels.cuh"
#include "tma.cuh"

namespace ptfock {

template <int N0_, int N1_, int N2_, int A1_, int A2_, int A0_, int MAXREG_A_ = 168, int MAXREG_C_ = 255, int NBUF_C_ = 3>
struct P8 {
    static constexpr int N0 = N0_, N1 = N1_, N2 = N2_, A1 = A1_, A2 = A2_, A0 = A0_;
    static constexpr int B1 = N1 / A1, B2 = N2 / A2, B0 = N0 / A0;
    static_assert(A1 * B1 == N1 && A2 * B2 == N2 && A0 * B0 == N0, "bad split");
    static_assert(B0 % 8 == 0 && B2 % 8 == 0, "the XOR swizzles work on groups of 8");
    static constexpr int RQ = 4, NQ = B1 / RQ;              // b1 = q*RQ + r
    static_assert(NQ * RQ == B1, "B1 must be a multiple of 4");
    // slab passes: stage-1 tasks (r, b2), A1*A2 points each; stage-2 tasks (k1a, k2a, r), B2 points each
    static constexpr int NT1 = RQ * B2, NT2 = A1 * A2 * RQ;
    static constexpr int NT = ((NT1 > NT2 ? NT1 : NT2) + 31) / 32 * 32;
    static constexpr int QPTS = A1 * RQ * N2;               // points of one (slab, q) row of the scratch
    static_assert(QPTS == NT1 * A1 * A2 && QPTS == NT2 * B2, "task counts");
    static constexpr int NT2P = (NT2 + 7) / 8 * 8;          // pass C's in-place exchange swizzles task indices in groups of 8
    static constexpr int RING = B2 * NT2P;                  // elements of one ring buffer (>= QPTS)
    static constexpr int NPOS = A1 * A2 * B2;               // slab positions (k2b, k1a, k2a) per row
    static constexpr int NBUF_A = 2;                        // pass A: ring of landed phi_i quarter slabs
    static constexpr int SMEM_A = NBUF_A * RING * 16 + 64;
    static constexpr int NBUF_C = NBUF_C_;                  // pass C: ring of landed pair-density rows
    static constexpr int SMEM_C = NBUF_C * RING * 16 + 64;
    static constexpr int MAXREG_A = MAXREG_A_, MAXREG_C = MAXREG_C_;
    // pass B: tile = [q][x0][P positions x RQ r] (128-byte rows); stage-1 / 3 tasks (b0, p): the A0 x B1 points
    // (a0, b1) at x0 = a0*B0 + b0; middle tasks (k0a, k1b, p): the B0 points b0
    static constexpr int P = 2;                             // slab positions per tile: rows of P*RQ*16 = 128 bytes
    static constexpr int ROWS = NQ * N0;                    // tile rows (q, x0)
    static_assert(ROWS <= 256 && ROWS % 8 == 0, "TMA box limit; 1 KB swizzle period");
    static constexpr int TILE_B = ROWS * P * RQ * 16;
    static constexpr int NTB1 = B0 * P, NTB2 = A0 * B1 * P;
    static constexpr int NTB = ((NTB1 > NTB2 ? NTB1 : NTB2) + 31) / 32 * 32;    // threads of one tile's group
    static_assert(NTB1 * A0 * B1 == ROWS * P * RQ && NTB2 * B0 == ROWS * P * RQ, "pass B task counts");
    static constexpr int GB = 3;                            // tiles (groups) per CTA, sharing one copy of v'
    static constexpr int V_BYTES = ROWS * P * RQ * 8;       // = NTB2 * B0 doubles
    static constexpr int SMEM_B = GB * TILE_B + V_BYTES + 64;   // + mbarriers
    static constexpr int MAXREG_B = 168;
    static constexpr int NGRP = NPOS / P;                   // tiles per pair
    static_assert(NPOS % P == 0, "positions per tile");
};

// ---- DFT32 = 4 x 8 (register resident, natural order in and out) -----------------------------------------------
__host__ __device__ constexpr double c32(int m) {          // cos(2 pi m / 32), m in [0, 32)
    m &= 31;
    if (m > 16) m = 32 - m;
    const bool neg = m > 8;
    if (neg) m = 16 - m;
    double v = 0.0;
    switch (m) {
        case 0: v = 1.0; break;
        case 1: v = 0.98078528040323044912618223613423904; break;
        case 2: v = 0.92387953251128675612818318939678829; break;
        case 3: v = 0.83146961230254523707878837761790576; break;
        case 4: v = 0.70710678118654752440084436210484904; break;
        case 5: v = 0.55557023301960222474283081394853287; break;
        case 6: v = 0.38268343236508977172845998403039887; break;
        case 7: v = 0.19509032201612826784828486847702224; break;
        default: v = 0.0; break;
    }
    return neg ? -v : v;
}
__host__ __device__ constexpr double s32(int m) { return c32(m - 8); }     // sin(2 pi m / 32)

template <bool INV> struct DFT<32, INV> {
    static PTF_DEV void run(cd (&v)[32]) {
        // n = 8a + b (a < 4, b < 8): DFT4 over a, twiddle w32^(b k1), DFT8 over b -> X[k1 + 4 k2]
#pragma unroll
        for (int b = 0; b < 8; ++b) DFT<4, INV>::run(v[b], v[8 + b], v[16 + b], v[24 + b]);
#pragma unroll
        for (int k1 = 1; k1 < 4; ++k1)
#pragma unroll
            for (int b = 1; b < 8; ++b) {
                const int m = b * k1;
                if (m == 8) v[8 * k1 + b] = mul_mi<INV>(v[8 * k1 + b]);
                else v[8 * k1 + b] = twmul<INV>(v[8 * k1 + b], make_double2(c32(m), -s32(m)));
            }
        cd o[32];
#pragma unroll
        for (int k1 = 0; k1 < 4; ++k1) {
            cd t[8];
#pragma unroll
            for (int b = 0; b < 8; ++b) t[b] = v[8 * k1 + b];
            DFT<8, INV>::run(t);
#pragma unroll
            for (int k2 = 0; k2 < 8; ++k2) o[k1 + 4 * k2] = t[k2];
        }
#pragma unroll
        for (int k = 0; k < 32; ++k) v[k] = o[k];
    }
};

// rows of R: DFT over the R index of u[r*C + c] for every c; cols likewise (u is an R x C register tile)
template <int R, int C, bool INV> PTF_DEV void dft_rows(cd (&u)[R * C]) {
    if constexpr (R > 1) {
#pragma unroll
        for (int c = 0; c < C; ++c) {
            cd t[R];
#pragma unroll
            for (int r = 0; r < R; ++r) t[r] = u[r * C + c];
            DFT<R, INV>::run(t);
#pragma unroll
            for (int r = 0; r < R; ++r) u[r * C + c] = t[r];
        }
    }
}
template <int R, int C, bool INV> PTF_DEV void dft_cols(cd (&u)[R * C]) {
    if constexpr (C > 1) {
#pragma unroll
        for (int r = 0; r < R; ++r) {
            cd t[C];
#pragma unroll
            for (int c = 0; c < C; ++c) t[c] = u[r * C + c];
            DFT<C, INV>::run(t);
#pragma unroll
            for (int c = 0; c < C; ++c) u[r * C + c] = t[c];
        }
    }
}

// ---- pass A ---------------------------------------------------------------------------------------------------
// 128-bit global load past L1, kept where it is written (the register budget below depends on loads not being hoisted)
PTF_DEV cd ldcg_v(const cd *p) {
    cd v;
    asm volatile("ld.global.cg.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p));
    return v;
}

// grid = (targets in the wave, N0 * NQ, chunks of the i loop); 64 threads.  Registers: psi_j (16 points = 64 registers)
// + the working tile (64) + twiddles.  phi_i's quarter slab (RQ rows of every a1 chunk: A1 runs of 4 KB) arrives by
// 1-D bulk async copies (TMA) in a ring of NBUF_A shared-memory buffers, one iteration ahead and without holding
// registers; both stages work IN PLACE in the landed buffer, exchanging through an XOR swizzle (slot (t2, b2) at
// t2*B2 + (b2 ^ (t2 & 7))), conflict free both ways; results leave from registers in 1 KB runs.
template <class S>
__global__ void __maxnreg__(S::MAXREG_A) p8_fwd(const SlabArgs g) {
    constexpr int N1 = S::N1, N2 = S::N2, A1 = S::A1, A2 = S::A2, B1 = S::B1, B2 = S::B2, RQ = S::RQ;
    constexpr int NBUF = S::NBUF_A, CH = RQ * N2;        // one a1 chunk: RQ contiguous rows
    constexpr bool ALL1 = S::NT1 == S::NT, ALL2 = S::NT2 == S::NT;     // every thread owns a stage-1 / stage-2 task
    extern __shared__ __align__(128) unsigned char smem_raw[];
    cd *ring = reinterpret_cast<cd *>(smem_raw);
    unsigned long long *bars = reinterpret_cast<unsigned long long *>(smem_raw + (size_t)NBUF * S::RING * 16);
    const int tid = threadIdx.x;
    const int jj = blockIdx.x, x0 = blockIdx.y / S::NQ, q = blockIdx.y % S::NQ;
    const int per = (g.na + gridDim.z - 1) / gridDim.z;
    int ii_beg, ii_end;
    tri_range(g.tri, jj, blockIdx.z * per, min(g.na, blockIdx.z * per + per), ii_beg, ii_end);
    const int n_it = ii_end - ii_beg;
    if (n_it <= 0) return;
    // stage-1 task (r, b2): the A1 x A2 points (a1, a2) at x1 = a1*B1 + b1, x2 = a2*B2 + b2
    const bool act1 = ALL1 || tid < S::NT1, act2 = ALL2 || tid < S::NT2;
    const int t1 = act1 ? tid : 0;
    const int b2 = t1 % B2, r = t1 / B2, b1 = q * RQ + r;
    const long long off1 = (long long)x0 * (N1 * N2) + b1 * N2 + b2;
    // chunk a1 of the quarter slab of orbital it: phi0 + it*grid_pts + a1*B1*N2
    const cd *phi0 = g.a + (long long)(g.a0 + ii_beg) * g.grid_pts + (long long)x0 * (N1 * N2) + (q * RQ) * N2;
    auto issue = [&](int it) {          // warp 0: lanes 0 .. A1-1 copy one chunk each
        const int buf = it % NBUF;
        if (tid == 0) mbar_expect_tx(&bars[buf], S::QPTS * 16u);
        __syncwarp();
        if (tid < A1)
            bulk_g2s(ring + buf * S::RING + tid * CH, phi0 + (long long)it * g.grid_pts + (long long)tid * (B1 * N2), CH * 16u, &bars[buf]);
    };
    if (tid == 0) {
#pragma unroll
        for (int k = 0; k < NBUF; ++k) mbar_init(&bars[k], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        fence_proxy_async();
    }
    __syncthreads();
    if (tid < 32) {
#pragma unroll
        for (int k = 0; k < NBUF - 1; ++k)
            if (k < n_it) issue(k);
    }
    cd pj[A1 * A2];
    if (act1) {
        const cd *psi = g.b + (long long)(g.b0 + jj) * g.grid_pts + off1;
#pragma unroll
        for (int a1 = 0; a1 < A1; ++a1)
#pragma unroll
            for (int a2 = 0; a2 < A2; ++a2) pj[a1 * A2 + a2] = psi[a1 * (B1 * N2) + a2 * B2];
    }
    cd tw1[A1 - 1], tw2[A2 - 1];
#pragma unroll
    for (int k = 1; k < A1; ++k) tw1[k - 1] = g.tw1[b1 * k];          // w_N1^(b1 k1a)
#pragma unroll
    for (int k = 1; k < A2; ++k) tw2[k - 1] = g.tw2[b2 * k];          // w_N2^(b2 k2a)
    const int ld1 = r * N2 + b2;                                       // + a1*CH + a2*B2
    const long long pair0 = (long long)ii_beg * g.stride_loop + (long long)jj * g.stride_cta;
    cd *dst = g.scratch + ((pair0 * S::NQ + q) * S::N0 + x0) * (long long)S::QPTS + (act2 ? tid : 0);
    const long long dst_step = (long long)g.stride_loop * S::NQ * S::N0 * S::QPTS;
#pragma unroll 1
    for (int it = 0; it < n_it; ++it) {
        cd *T = ring + (it % NBUF) * S::RING;
        mbar_wait(&bars[it % NBUF], (it / NBUF) & 1);
        cd u[A1 * A2];
        if (act1) {
#pragma unroll
            for (int a1 = 0; a1 < A1; ++a1)
#pragma unroll
                for (int a2 = 0; a2 < A2; ++a2) u[a1 * A2 + a2] = T[ld1 + a1 * CH + a2 * B2];
        }
        fence_proxy_async();
        __syncthreads();                                // phi_i read; the buffer of iteration it - 1 is free
        if (tid < 32 && it + NBUF - 1 < n_it) issue(it + NBUF - 1);
        if (act1) {
#pragma unroll
            for (int k = 0; k < A1 * A2; ++k) u[k] = cmulc(pj[k], u[k]);  // psi_j conj(phi_i)
            dft_rows<A1, A2, false>(u);
#pragma unroll
            for (int k1 = 1; k1 < A1; ++k1)
#pragma unroll
                for (int a2 = 0; a2 < A2; ++a2) u[k1 * A2 + a2] = cmul(u[k1 * A2 + a2], tw1[k1 - 1]);
            dft_cols<A1, A2, false>(u);
#pragma unroll
            for (int k2 = 1; k2 < A2; ++k2)
#pragma unroll
                for (int k1 = 0; k1 < A1; ++k1) u[k1 * A2 + k2] = cmul(u[k1 * A2 + k2], tw2[k2 - 1]);
            // value (k1a, k2a) of this thread belongs to stage-2 task t2 = (k1a*A2 + k2a)*RQ + r, index b2
#pragma unroll
            for (int k = 0; k < A1 * A2; ++k) T[(k * RQ + r) * B2 + (b2 ^ ((k * RQ + r) & 7))] = u[k];
        }
        __syncthreads();
        // stage 2: task tid, DFT over b2; output k2b at k2b*NT2 + tid of the scratch row
        if (act2) {
            cd w[B2];
#pragma unroll
            for (int b = 0; b < B2; ++b) w[b] = T[tid * B2 + (b ^ (tid & 7))];
            DFT<B2, false>::run(w);
#pragma unroll
            for (int m = 0; m < B2; ++m) dst[m * S::NT2] = w[m];
        }
        dst += dst_step;
    }
}

// ---- pass C ---------------------------------------------------------------------------------------------------
// grid = (targets, N0 * NQ): out[b0+tt] += sum_ss a[a0+ss] * W[ss*stride_loop + tt*stride_cta]   (W or conj(W)).
// The pair-density rows (16 KB, contiguous) arrive by 1-D bulk async copies (TMA) in a ring of NBUF_C shared-memory
// buffers, two iterations ahead and without holding registers: under load a global load takes several microseconds,
// so an SM needs ~100 KB of reads in flight to keep HBM busy.  Both stages work IN PLACE in the landed buffer; the
// exchange between them is an XOR swizzle (slot (b2, t2) at b2*NT2 + (t2 ^ (b2 & 7))), conflict free both ways.
// phi_i is prefetched one iteration ahead through registers (16 points), accumulators in registers (16 points).
template <class S>
__global__ void __maxnreg__(S::MAXREG_C) p8_inv_acc(const SlabArgs g) {
    constexpr int N1 = S::N1, N2 = S::N2, A1 = S::A1, A2 = S::A2, B1 = S::B1, B2 = S::B2, RQ = S::RQ;
    constexpr int NBUF = S::NBUF_C, NT2 = S::NT2, NT2P = S::NT2P;
    constexpr bool ALL1 = S::NT1 == S::NT, ALL2 = S::NT2 == S::NT;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    cd *ring = reinterpret_cast<cd *>(smem_raw);
    unsigned long long *bars = reinterpret_cast<unsigned long long *>(smem_raw + (size_t)NBUF * S::RING * 16);
    const int tid = threadIdx.x;
    const int tt = blockIdx.x, x0 = blockIdx.y / S::NQ, q = blockIdx.y % S::NQ;
    int it_lo, it_hi;
    tri_range(g.tri, tt, 0, g.na, it_lo, it_hi);
    const int n_it = it_hi - it_lo;
    if (n_it <= 0) return;
    const bool act1 = ALL1 || tid < S::NT1, act2 = ALL2 || tid < S::NT2;    // owner of a last-stage / first-stage task
    const int t1 = act1 ? tid : 0;
    const int b2 = t1 % B2, r = t1 / B2, b1 = q * RQ + r;
    const long long off1 = (long long)x0 * (N1 * N2) + b1 * N2 + b2;
    const long long pair_stride = (long long)g.stride_loop * S::NQ * S::N0 * S::QPTS;
    const cd *src = g.scratch + (((long long)tt * g.stride_cta * S::NQ + q) * S::N0 + x0) * (long long)S::QPTS
                    + (long long)it_lo * pair_stride;
    if (tid == 0) {
#pragma unroll
        for (int k = 0; k < NBUF; ++k) mbar_init(&bars[k], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        fence_proxy_async();
#pragma unroll
        for (int k = 0; k < NBUF - 1; ++k)
            if (k < n_it) {
                mbar_expect_tx(&bars[k], S::QPTS * 16u);
                bulk_g2s(ring + k * S::RING, src + (long long)k * pair_stride, S::QPTS * 16u, &bars[k]);
            }
    }
    cd tw1[A1 - 1], tw2[A2 - 1];
#pragma unroll
    for (int k = 1; k < A1; ++k) tw1[k - 1] = g.tw1[b1 * k];
#pragma unroll
    for (int k = 1; k < A2; ++k) tw2[k - 1] = g.tw2[b2 * k];
    cd acc[A1 * A2];
#pragma unroll
    for (int k = 0; k < A1 * A2; ++k) acc[k] = make_double2(0.0, 0.0);
    const cd *phi = g.a + (long long)(g.a0 + it_lo) * g.grid_pts + off1;
    cd f[A1 * A2];
    if (act1) {
#pragma unroll
        for (int a1 = 0; a1 < A1; ++a1)
#pragma unroll
            for (int a2 = 0; a2 < A2; ++a2) f[a1 * A2 + a2] = ldcg_v(phi + a1 * (B1 * N2) + a2 * B2);
    }
    const bool cw = g.conj_w != 0;
    __syncthreads();                                    // mbarrier inits visible
#pragma unroll 1
    for (int it = 0; it < n_it; ++it) {
        cd *T = ring + (it % NBUF) * S::RING;
        mbar_wait(&bars[it % NBUF], (it / NBUF) & 1);
        cd w[B2];
        if (act2) {
#pragma unroll
            for (int m = 0; m < B2; ++m) w[m] = T[m * NT2 + tid];
        }
        fence_proxy_async();
        __syncthreads();                                // row read; the buffer of iteration it - 1 is free
        if (tid == 0 && it + NBUF - 1 < n_it) {
            const int nx = it + NBUF - 1;
            mbar_expect_tx(&bars[nx % NBUF], S::QPTS * 16u);
            bulk_g2s(ring + (nx % NBUF) * S::RING, src + (long long)nx * pair_stride, S::QPTS * 16u, &bars[nx % NBUF]);
        }
        // stage 1': inverse DFT over k2b of task tid = (k1a*A2 + k2a)*RQ + r, back in place (swizzled)
        if (act2) {
            DFT<B2, true>::run(w);
#pragma unroll
            for (int b = 0; b < B2; ++b) T[b * NT2P + (tid ^ (b & 7))] = w[b];      // pitch NT2P: the XOR stays in range
        }
        __syncthreads();
        if (act1) {
            cd u[A1 * A2];
#pragma unroll
            for (int k = 0; k < A1 * A2; ++k) u[k] = T[b2 * NT2P + ((k * RQ + r) ^ (b2 & 7))];
#pragma unroll
            for (int k2 = 1; k2 < A2; ++k2)
#pragma unroll
                for (int k1 = 0; k1 < A1; ++k1) u[k1 * A2 + k2] = cmulc(u[k1 * A2 + k2], tw2[k2 - 1]);
            dft_cols<A1, A2, true>(u);
#pragma unroll
            for (int k1 = 1; k1 < A1; ++k1)
#pragma unroll
                for (int a2 = 0; a2 < A2; ++a2) u[k1 * A2 + a2] = cmulc(u[k1 * A2 + a2], tw1[k1 - 1]);
            dft_rows<A1, A2, true>(u);
            if (cw) {
#pragma unroll
                for (int k = 0; k < A1 * A2; ++k) {
                    const cd pr = cmulc(f[k], u[k]);
                    acc[k].x += pr.x; acc[k].y += pr.y;
                }
            } else {
#pragma unroll
                for (int k = 0; k < A1 * A2; ++k) {
                    const cd pr = cmul(f[k], u[k]);
                    acc[k].x += pr.x; acc[k].y += pr.y;
                }
            }
            phi += g.grid_pts;
            if (it + 1 < n_it) {                        // next phi_i: on its way during the next iteration's first half
#pragma unroll
                for (int a1 = 0; a1 < A1; ++a1)
#pragma unroll
                    for (int a2 = 0; a2 < A2; ++a2) f[a1 * A2 + a2] = ldcg_v(phi + a1 * (B1 * N2) + a2 * B2);
            }
        }
    }
    if (!act1) return;
    cd *o = g.out + (long long)(g.b0 + tt) * g.grid_pts + off1;
#pragma unroll
    for (int a1 = 0; a1 < A1; ++a1)
#pragma unroll
        for (int a2 = 0; a2 < A2; ++a2) {
            cd cur = o[a1 * (B1 * N2) + a2 * B2];
            cur.x += acc[a1 * A2 + a2].x;
            cur.y += acc[a1 * A2 + a2].y;
            o[a1 * (B1 * N2) + a2 * B2] = cur;
        }
}

// ---- pass B ---------------------------------------------------------------------------------------------------
struct P8MidArgs {
    const double2 *v;    // [tile group][B0 / 2][NTB2 middle tasks]: the middle-stage thread's v' values (k0b = 2m, 2m + 1)
    const cd *tw0;       // exp(-2 pi i t / N0)
    int n_pairs;         // pairs in the wave
    int tri_nj;          // > 0: diagonal block of the symmetric schedule, pair = i*tri_nj + j exists only for i <= j
    int pair0;           // pair index (in the scratch the tensor map covers) of the wave's first pair
};

PTF_DEV void tensor_g2s_2d_sw(void *dst_smem, const CUtensorMap *map, int c0, int c1, unsigned long long *bar) {
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
                 ::"r"(smem_u32(dst_smem)), "l"(map), "r"(c0), "r"(c1), "r"(smem_u32(bar)) : "memory");
}
PTF_DEV void tensor_s2g_2d_sw(const CUtensorMap *map, int c0, int c1, const void *src_smem) {
    asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.bulk_group [%0, {%1, %2}], [%3];"
                 ::"l"(map), "r"(c0), "r"(c1), "r"(smem_u32(src_smem)) : "memory");
}

// grid = (NGRP tile positions, ceil(pairs / GB)); a CTA is GB independent groups of 64 threads, one tile each (the same
// tile position grp of GB consecutive pairs), sharing ONE copy of the position's v' values in shared memory, brought
// in by a bulk async copy next to the tiles.  Why not a global load in the middle stage: an L2 hit issued while the
// SM has tile loads outstanding queues behind them and costs a DRAM round trip (measured: 0.76 of the HBM peak with
// the loads, 0.98 with the same arithmetic and no loads); why not registers: 64 more live registers halve the
// CTAs per SM (0.83).  Groups synchronise among themselves with named barriers only.
// The tensor map views the scratch as [pairs*NQ*N0 rows][2*QPTS doubles] with the 128-byte swizzle: element e of row R
// sits at (R*8 + (e ^ (R & 7))) * 16 bytes of the tile.
template <class S>
__global__ void __maxnreg__(S::MAXREG_B) p8_mid(const __grid_constant__ CUtensorMap map, const P8MidArgs g) {
    constexpr int N0 = S::N0, A0 = S::A0, B0 = S::B0, B1 = S::B1, RQ = S::RQ, NQ = S::NQ, P = S::P, GB = S::GB;
    // the 128-byte swizzle pattern repeats every 1 KB: the tiles must start on 1 KB boundaries of the shared window
    extern __shared__ __align__(1024) unsigned char smem_b[];
    const double2 *vs = reinterpret_cast<const double2 *>(smem_b + GB * S::TILE_B);
    unsigned long long *bars = reinterpret_cast<unsigned long long *>(smem_b + GB * S::TILE_B + S::V_BYTES);
    if (smem_u32(smem_b) & 1023u) __trap();
    const int grp_pos = blockIdx.x;
    const int gi = threadIdx.x / S::NTB, tid = threadIdx.x % S::NTB;       // group, thread in group
    const int pair = blockIdx.y * GB + gi;
    cd *s = reinterpret_cast<cd *>(smem_b + gi * S::TILE_B);
    // pair pr of the wave is solved unless it lies past the wave's end or above the diagonal of a triangular block
    auto live = [&](int pr) { return pr < g.n_pairs && !(g.tri_nj > 0 && pr / g.tri_nj > pr % g.tri_nj); };
    if (threadIdx.x == 0) {
#pragma unroll
        for (int k = 0; k <= GB; ++k) mbar_init(&bars[k], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        fence_proxy_async();
        bool any = false;
#pragma unroll
        for (int k = 0; k < GB; ++k) any |= live(blockIdx.y * GB + k);
        // a CTA whose GB pairs are all skipped (e.g. pairs (3,0) (3,1) (3,2) of a triangular block) returns below without
        // waiting on anything: it must not leave a bulk copy and its complete_tx in flight into shared memory that the
        // SM's next CTA may already own.  With one live group, that group waits for v' before the CTA can exit.
        if (any) {
            mbar_expect_tx(&bars[GB], S::V_BYTES);
            bulk_g2s(smem_b + GB * S::TILE_B, g.v + (long long)grp_pos * (S::V_BYTES / 16), S::V_BYTES, &bars[GB]);
        }
#pragma unroll
        for (int k = 0; k < GB; ++k)
            if (live(blockIdx.y * GB + k)) {
                mbar_expect_tx(&bars[k], S::TILE_B);
                tensor_g2s_2d_sw(smem_b + k * S::TILE_B, &map, grp_pos * (P * RQ * 2), (g.pair0 + blockIdx.y * GB + k) * S::ROWS, &bars[k]);
            }
    }
    // stage 1 / 3 task (b0, p): element (a0, q, r) at row q*N0 + a0*B0 + b0, chunk (p*RQ + r) ^ (b0 & 7)
    const bool act1 = S::NTB1 == S::NTB || tid < S::NTB1, act2 = S::NTB2 == S::NTB || tid < S::NTB2;
    const int t1 = act1 ? tid : 0, t2 = act2 ? tid : 0;
    const int b0 = t1 % B0, p = t1 / B0;
    cd tw[A0 - 1];
#pragma unroll
    for (int k = 1; k < A0; ++k) tw[k - 1] = g.tw0[b0 * k];           // w_N0^(b0 k0a)
    // middle task: t2 = ((k0a*NQ + q)*P + p)*RQ + r; element b0' at row q*N0 + k0a*B0 + b0', chunk (p*RQ + r) ^ (b0' & 7)
    const int mr = t2 % RQ, mp = (t2 / RQ) % P, mq = (t2 / (RQ * P)) % NQ, mk = t2 / (RQ * P * NQ);
    const int rb = (mq * N0 + mk * B0) * 8, mc = mp * RQ + mr;
    __syncthreads();                                    // mbarrier inits visible; from here on the groups are independent
    if (!live(pair)) return;
    auto group_sync = [&]() {                           // named barrier 1 + gi over the group's threads
        if (gi == 0) asm volatile("bar.sync 1, %0;" ::"n"(S::NTB) : "memory");
        else if (gi == 1) asm volatile("bar.sync 2, %0;" ::"n"(S::NTB) : "memory");
        else asm volatile("bar.sync 3, %0;" ::"n"(S::NTB) : "memory");
    };
    static_assert(GB <= 3, "one named barrier per group");
    mbar_wait(&bars[gi], 0);
    if (act1) {
        cd u[A0 * B1];                                                  // u[a0*B1 + b1], b1 = q*RQ + r
#pragma unroll
        for (int a0 = 0; a0 < A0; ++a0)
#pragma unroll
            for (int q = 0; q < NQ; ++q)
#pragma unroll
                for (int r = 0; r < RQ; ++r)
                    u[a0 * B1 + q * RQ + r] = s[(q * N0 + a0 * B0 + b0) * 8 + ((p * RQ + r) ^ (b0 & 7))];
        dft_rows<A0, B1, false>(u);
#pragma unroll
        for (int k = 1; k < A0; ++k)
#pragma unroll
            for (int c = 0; c < B1; ++c) u[k * B1 + c] = cmul(u[k * B1 + c], tw[k - 1]);
        dft_cols<A0, B1, false>(u);
#pragma unroll
        for (int a0 = 0; a0 < A0; ++a0)
#pragma unroll
            for (int q = 0; q < NQ; ++q)
#pragma unroll
                for (int r = 0; r < RQ; ++r)
                    s[(q * N0 + a0 * B0 + b0) * 8 + ((p * RQ + r) ^ (b0 & 7))] = u[a0 * B1 + q * RQ + r];
    }
    group_sync();
    mbar_wait(&bars[GB], 0);                            // v' landed (requested before the tiles)
    if (act2) {
        cd u[B0];
#pragma unroll
        for (int b = 0; b < B0; ++b) u[b] = s[rb + b * 8 + (mc ^ (b & 7))];
        DFT<B0, false>::run(u);
#pragma unroll
        for (int m = 0; m < B0 / 2; ++m) {
            const double2 vv = vs[m * S::NTB2 + tid];
            u[2 * m] = cscale(u[2 * m], vv.x);
            u[2 * m + 1] = cscale(u[2 * m + 1], vv.y);
        }
        DFT<B0, true>::run(u);
#pragma unroll
        for (int b = 0; b < B0; ++b) s[rb + b * 8 + (mc ^ (b & 7))] = u[b];
    }
    group_sync();
    if (act1) {
        cd u[A0 * B1];
#pragma unroll
        for (int a0 = 0; a0 < A0; ++a0)
#pragma unroll
            for (int q = 0; q < NQ; ++q)
#pragma unroll
                for (int r = 0; r < RQ; ++r)
                    u[a0 * B1 + q * RQ + r] = s[(q * N0 + a0 * B0 + b0) * 8 + ((p * RQ + r) ^ (b0 & 7))];
        dft_cols<A0, B1, true>(u);
#pragma unroll
        for (int k = 1; k < A0; ++k)
#pragma unroll
            for (int c = 0; c < B1; ++c) u[k * B1 + c] = cmulc(u[k * B1 + c], tw[k - 1]);
        dft_rows<A0, B1, true>(u);
#pragma unroll
        for (int a0 = 0; a0 < A0; ++a0)
#pragma unroll
            for (int q = 0; q < NQ; ++q)
#pragma unroll
                for (int r = 0; r < RQ; ++r)
                    s[(q * N0 + a0 * B0 + b0) * 8 + ((p * RQ + r) ^ (b0 & 7))] = u[a0 * B1 + q * RQ + r];
    }
    fence_proxy_async();
    group_sync();
    if (tid == 0) {
        tensor_s2g_2d_sw(&map, grp_pos * (P * RQ * 2), (g.pair0 + pair) * S::ROWS, s);
        asm volatile("cp.async.bulk.commit_group;" ::: "memory");
        asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");     // shared memory must outlive the store's reads
    }
}

}  // namespace ptfock
