// pass8.cuh -- the "8 + 10 + 8 bit" split of the pair-solve for 64^3 grids (Alg. 2 lines 6-10, Eq. (3)).
//
// The three passes of kernels.cuh / slabx.cuh give the slab passes 12 index bits (three butterfly stages, six
// shared-memory crossings per point) and the pencil pass 6; ncu showed the slab passes bound by the L1/shared-memory
// data pipe, not by HBM (profiles/r01_ncu_full_si512.md).  Here the slab passes keep only TWO stages and hand the low
// digit b1 of x1 to the pencil pass, which has the slack:
//
//   x1 = a1*B1 + b1,  x2 = a2*B2 + b2          (64^3: A1 = 4, B1 = 16, A2 = 4, B2 = 16)
//   pass A  p8_fwd     : rho = conj(phi_i) psi_j;  2-D DFT over (a1, a2) + both twiddles | DFT over b2
//                        one CTA = 64 threads = one (target, x0, quarter q of b1 = 4q + r); phi_i comes straight from
//                        global memory into registers (128-bit, 256-byte runs), one padded exchange through shared
//                        memory, results leave from registers in 1 KB runs: 4 crossings of the LSU pipe per point.
//   pass B  p8_mid     : 2-D DFT over (x0, b1) = 64 x 16 = 32 x 32 points per slab position, x v'(G), inverse;
//                        tile = [q][x0][2 positions x 4 r] (32 KB) by ONE swizzled tensor-map TMA load / store.
//   pass C  p8_inv_acc : mirror of A; x phi_i and the sum over i in registers.
//
// Pair scratch: [pair][q][x0][k2b][k1a][k2a][r] (16-byte elements): a pass A / C CTA owns one contiguous 16 KB
// row (pair, q, x0); pass B sees 256 rows (q, x0) of one pair, 128 contiguous bytes of each.
// Frequencies: k0 = k0a + A0*k0b, k1 = k1a + A1*k1b, k2 = k2a + A2*k2b; nothing is ever un-permuted (the v' table is
// stored in pass B's register order, build_vtable8).
#pragma once
#include <cuda.h>
#include "kernels.cuh"
#include "tma.cuh"

#ifndef P8_VMODE
#define P8_VMODE 2
#endif
#ifndef P8_A_PREF
#define P8_A_PREF 0          // 1: pass A prefetches the next phi_i through registers (255 registers, 4 CTAs per SM)
#endif
#ifndef P8_C_PREF
#define P8_C_PREF 0          // 1: pass C prefetches the next pair density through registers (255 registers)
#endif
#ifndef P8_C_L2PF
#define P8_C_L2PF 2          // pass C: L2 prefetch distance (iterations) for the pair-density rows, 0 = off
#endif
#ifndef P8_SKEL_B
#define P8_SKEL_B 0          // timing experiments only: 1 = butterflies compiled out, 2 = tile load + store only
#endif
#ifndef P8_MAXREG_B
#define P8_MAXREG_B 168
#endif

namespace ptfock {

template <int N0_, int N1_, int N2_, int A1_, int A2_, int A0_>
struct P8 {
    static constexpr int N0 = N0_, N1 = N1_, N2 = N2_, A1 = A1_, A2 = A2_, A0 = A0_;
    static constexpr int B1 = N1 / A1, B2 = N2 / A2, B0 = N0 / A0;
    static_assert(A1 * B1 == N1 && A2 * B2 == N2 && A0 * B0 == N0, "bad split");
    static_assert(B0 == 32 && A0 * B1 == 32, "pass B works on 32 x 32 points per slab position");
    static constexpr int RQ = 4, NQ = B1 / RQ;              // b1 = q*RQ + r
    static_assert(NQ * RQ == B1, "B1 must be a multiple of 4");
    static constexpr int NT = RQ * B2;                      // slab passes: stage-1 tasks (r, b2)
    static constexpr int NT2 = A1 * A2 * RQ;                // stage-2 tasks (k1a, k2a, r)
    static_assert(NT == NT2 && NT == 64, "one task per thread in both stages");
    static constexpr int PW = B2 + 1;                       // exchange tile pitch (elements): conflict free both ways
    static constexpr int WORK = NT2 * PW;
    static constexpr int SMEM_A = 2 * WORK * 16;            // two exchange tiles: one CTA barrier per orbital
    static constexpr int SMEM_C = SMEM_A + (A1 - 1 + A2 - 1) * NT * 16;       // + per-thread twiddles
    static constexpr int QPTS = A1 * RQ * N2;               // points of one (slab, q) row of the scratch
    static constexpr int NPOS = A1 * A2 * B2;               // slab positions (k2b, k1a, k2a) per row
    static constexpr int MAXREG_A = P8_A_PREF ? 255 : 168, MAXREG_C = P8_C_PREF ? 255 : 192;    // 6 / 4 CTAs per SM
    // pass B
    static constexpr int P = 2;                             // slab positions per tile: rows of P*RQ*16 = 128 bytes
    static constexpr int ROWS = NQ * N0;                    // tile rows (q, x0)
    static_assert(ROWS <= 256, "TMA box limit");
    static constexpr int TILE_B = ROWS * P * RQ * 16;       // 32 KB
    static constexpr int NTB = 32 * P;                      // 64 threads
    static_assert(A0 * NQ * P * RQ == NTB, "middle-stage tasks");
    static constexpr int SMEM_B = TILE_B + 16;              // + mbarrier
    static constexpr int MINB_B = 6;
    static constexpr int NGRP = NPOS / P;                   // tiles per pair
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

PTF_DEV void l2_prefetch_bulk(const void *p, unsigned bytes) {
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p), "r"(bytes) : "memory");
}

// ---- pass A ---------------------------------------------------------------------------------------------------
// 128-bit global load past L1, kept where it is written (the register budget below depends on loads not being hoisted)
PTF_DEV cd ldcg_v(const cd *p) {
    cd v;
    asm volatile("ld.global.cg.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p));
    return v;
}

// grid = (targets in the wave, N0 * NQ, chunks of the i loop); 64 threads.  Registers: psi_j (16 points = 64 registers)
// + the working tile (64) + twiddles; phi_i is NOT prefetched through registers -- the other CTAs of the SM (MINB_A of
// them, out of phase) cover its latency.
template <class S>
__global__ void __maxnreg__(S::MAXREG_A) p8_fwd(const SlabArgs g) {
    constexpr int N1 = S::N1, N2 = S::N2, A1 = S::A1, A2 = S::A2, B1 = S::B1, B2 = S::B2, RQ = S::RQ, PW = S::PW;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cd *work = reinterpret_cast<cd *>(smem_raw);
    const int tid = threadIdx.x;
    const int jj = blockIdx.x, x0 = blockIdx.y / S::NQ, q = blockIdx.y % S::NQ;
    const int per = (g.na + gridDim.z - 1) / gridDim.z;
    const int ii_beg = blockIdx.z * per, ii_end = min(g.na, ii_beg + per);
    const int n_it = ii_end - ii_beg;
    if (n_it <= 0) return;
    // stage-1 task (r, b2): the 4 x 4 points (a1, a2) at x1 = a1*B1 + b1, x2 = a2*B2 + b2
    const int b2 = tid % B2, r = tid / B2, b1 = q * RQ + r;
    const long long off1 = (long long)x0 * (N1 * N2) + b1 * N2 + b2;
    cd pj[A1 * A2];
    {
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
    const cd *phi = g.a + (long long)(g.a0 + ii_beg) * g.grid_pts + off1;
    const int st1 = r * PW + b2;                                       // + (k1a*A2 + k2a) * RQ * PW
    const long long pair0 = (long long)ii_beg * g.stride_loop + (long long)jj * g.stride_cta;
    cd *dst = g.scratch + ((pair0 * S::NQ + q) * S::N0 + x0) * (long long)S::QPTS + tid;
    const long long dst_step = (long long)g.stride_loop * S::NQ * S::N0 * S::QPTS;
#if P8_A_PREF
    cd f[A1 * A2];
#pragma unroll
    for (int a1 = 0; a1 < A1; ++a1)
#pragma unroll
        for (int a2 = 0; a2 < A2; ++a2) f[a1 * A2 + a2] = ldcg_v(phi + a1 * (B1 * N2) + a2 * B2);
#endif
#pragma unroll 1
    for (int it = 0; it < n_it; ++it) {
        cd u[A1 * A2];
#if P8_A_PREF
#pragma unroll
        for (int k = 0; k < A1 * A2; ++k) u[k] = cmulc(pj[k], f[k]);  // psi_j conj(phi_i)
        phi += g.grid_pts;
        if (it + 1 < n_it) {
#pragma unroll
            for (int a1 = 0; a1 < A1; ++a1)
#pragma unroll
                for (int a2 = 0; a2 < A2; ++a2) f[a1 * A2 + a2] = ldcg_v(phi + a1 * (B1 * N2) + a2 * B2);
        }
#else
#pragma unroll
        for (int a1 = 0; a1 < A1; ++a1)
#pragma unroll
            for (int a2 = 0; a2 < A2; ++a2) u[a1 * A2 + a2] = ldcg_v(phi + a1 * (B1 * N2) + a2 * B2);
        phi += g.grid_pts;
#pragma unroll
        for (int k = 0; k < A1 * A2; ++k) u[k] = cmulc(pj[k], u[k]);  // psi_j conj(phi_i)
#endif
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
        cd *W = work + (it & 1) * S::WORK;
#pragma unroll
        for (int k = 0; k < A1 * A2; ++k) W[st1 + k * (RQ * PW)] = u[k];
        __syncthreads();
        // stage 2: task tid = (k1a*A2 + k2a)*RQ + r, DFT over b2; output k2b at k2b*NT2 + tid of the scratch row
        cd w[B2];
#pragma unroll
        for (int b = 0; b < B2; ++b) w[b] = W[tid * PW + b];
        DFT<B2, false>::run(w);
#pragma unroll
        for (int m = 0; m < B2; ++m) dst[m * S::NT2] = w[m];
        dst += dst_step;
    }
}

// ---- pass C ---------------------------------------------------------------------------------------------------
// grid = (targets, N0 * NQ): out[b0+tt] += sum_ss a[a0+ss] * W[ss*stride_loop + tt*stride_cta]   (W or conj(W)).
// Registers: the accumulators (64) + the working tile (64) + phi_i two columns at a time (32); the twiddles are re-read
// from shared memory every iteration.
template <class S>
__global__ void __maxnreg__(S::MAXREG_C) p8_inv_acc(const SlabArgs g) {
    constexpr int N1 = S::N1, N2 = S::N2, A1 = S::A1, A2 = S::A2, B1 = S::B1, B2 = S::B2, RQ = S::RQ, PW = S::PW;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cd *work = reinterpret_cast<cd *>(smem_raw);
    cd *tws = work + 2 * S::WORK;                  // [k-1][tid]: w_N1^(b1 k) for k < A1, then w_N2^(b2 k) for k < A2
    const int tid = threadIdx.x;
    const int tt = blockIdx.x, x0 = blockIdx.y / S::NQ, q = blockIdx.y % S::NQ;
    const int n_it = g.na;
    if (n_it <= 0) return;
    const int b2 = tid % B2, r = tid / B2, b1 = q * RQ + r;
    const long long off1 = (long long)x0 * (N1 * N2) + b1 * N2 + b2;
#pragma unroll
    for (int k = 1; k < A1; ++k) tws[(k - 1) * S::NT + tid] = g.tw1[b1 * k];
#pragma unroll
    for (int k = 1; k < A2; ++k) tws[(A1 - 1 + k - 1) * S::NT + tid] = g.tw2[b2 * k];
    cd acc[A1 * A2];
#pragma unroll
    for (int k = 0; k < A1 * A2; ++k) acc[k] = make_double2(0.0, 0.0);
    const long long pair_stride = (long long)g.stride_loop * S::NQ * S::N0 * S::QPTS;
    const cd *src = g.scratch + (((long long)tt * g.stride_cta * S::NQ + q) * S::N0 + x0) * (long long)S::QPTS + tid;
    const cd *phi = g.a + (long long)g.a0 * g.grid_pts + off1;
    const int st1 = r * PW + b2;
    const bool cw = g.conj_w != 0;
#if P8_C_L2PF
    if (tid == 0) {
#pragma unroll
        for (int d = 1; d < P8_C_L2PF; ++d)
            if (d < n_it) l2_prefetch_bulk(src - tid + (long long)d * pair_stride, S::QPTS * 16u);
    }
#endif
#if P8_C_PREF
    cd w[B2];
#pragma unroll
    for (int m = 0; m < B2; ++m) w[m] = ldcg_v(src + m * S::NT2);
#endif
#pragma unroll 1
    for (int it = 0; it < n_it; ++it) {
        cd *W = work + (it & 1) * S::WORK;
#if P8_C_L2PF
        if (tid == 0 && it + P8_C_L2PF < n_it) l2_prefetch_bulk(src + (long long)P8_C_L2PF * pair_stride, S::QPTS * 16u);
#endif
        {
            // stage 1': inverse DFT over k2b of task tid = (k1a*A2 + k2a)*RQ + r
#if !P8_C_PREF
            cd w[B2];
#pragma unroll
            for (int m = 0; m < B2; ++m) w[m] = ldcg_v(src + m * S::NT2);
#endif
            src += pair_stride;
            DFT<B2, true>::run(w);
#pragma unroll
            for (int b = 0; b < B2; ++b) W[tid * PW + b] = w[b];
#if P8_C_PREF
            if (it + 1 < n_it) {
#pragma unroll
                for (int m = 0; m < B2; ++m) w[m] = ldcg_v(src + m * S::NT2);
            }
#endif
        }
        __syncthreads();
        cd u[A1 * A2];
#pragma unroll
        for (int k = 0; k < A1 * A2; ++k) u[k] = W[st1 + k * (RQ * PW)];
        cd f[2][A1];                                    // phi_i, columns a2 and a2 + 1 in flight
#pragma unroll
        for (int c = 0; c < 2 && c < A2; ++c)
#pragma unroll
            for (int a1 = 0; a1 < A1; ++a1) f[c][a1] = ldcg_v(phi + a1 * (B1 * N2) + c * B2);
#pragma unroll
        for (int k2 = 1; k2 < A2; ++k2) {
            const cd t2 = tws[(A1 - 1 + k2 - 1) * S::NT + tid];
#pragma unroll
            for (int k1 = 0; k1 < A1; ++k1) u[k1 * A2 + k2] = cmulc(u[k1 * A2 + k2], t2);
        }
        dft_cols<A1, A2, true>(u);
#pragma unroll
        for (int k1 = 1; k1 < A1; ++k1) {
            const cd t1 = tws[(k1 - 1) * S::NT + tid];
#pragma unroll
            for (int a2 = 0; a2 < A2; ++a2) u[k1 * A2 + a2] = cmulc(u[k1 * A2 + a2], t1);
        }
#pragma unroll
        for (int a2 = 0; a2 < A2; ++a2) {
            cd t[A1];
#pragma unroll
            for (int k1 = 0; k1 < A1; ++k1) t[k1] = u[k1 * A2 + a2];
            DFT<A1, true>::run(t);
#pragma unroll
            for (int a1 = 0; a1 < A1; ++a1) {
                const cd fv = f[a2 & 1][a1];
                const cd pr = cw ? cmulc(fv, t[a1]) : cmul(fv, t[a1]);
                acc[a1 * A2 + a2].x += pr.x;
                acc[a1 * A2 + a2].y += pr.y;
            }
            if (a2 + 2 < A2) {
#pragma unroll
                for (int a1 = 0; a1 < A1; ++a1) f[a2 & 1][a1] = ldcg_v(phi + a1 * (B1 * N2) + (a2 + 2) * B2);
            }
        }
        phi += g.grid_pts;
    }
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
    const double2 *v;    // [tile group][16][64 threads]: the middle-stage thread's v' values (k0b = 2m, 2m + 1)
    const cd *tw0;       // exp(-2 pi i t / N0)
};

PTF_DEV void tensor_g2s_2d_sw(void *dst_smem, const CUtensorMap *map, int c0, int c1, unsigned long long *bar) {
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
                 ::"r"(smem_u32(dst_smem)), "l"(map), "r"(c0), "r"(c1), "r"(smem_u32(bar)) : "memory");
}
PTF_DEV void tensor_s2g_2d_sw(const CUtensorMap *map, int c0, int c1, const void *src_smem) {
    asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.bulk_group [%0, {%1, %2}], [%3];"
                 ::"l"(map), "r"(c0), "r"(c1), "r"(smem_u32(src_smem)) : "memory");
}

// grid = (NGRP tiles per pair, pairs); the tensor map views the scratch as [pairs*NQ*N0 rows][2*QPTS doubles] with
// the 128-byte swizzle: element e of row R sits at (R*8 + (e ^ (R & 7))) * 16 bytes of the tile.
template <class S>
__global__ void __maxnreg__(P8_MAXREG_B) p8_mid(const __grid_constant__ CUtensorMap map, const P8MidArgs g) {
    constexpr int N0 = S::N0, A0 = S::A0, B1 = S::B1, RQ = S::RQ, NQ = S::NQ, P = S::P;
    // the 128-byte swizzle pattern repeats every 1 KB: the tile must start on a 1 KB boundary of the shared window
    extern __shared__ __align__(1024) unsigned char smem_b[];
    cd *s = reinterpret_cast<cd *>(smem_b);
    unsigned long long *bar = reinterpret_cast<unsigned long long *>(smem_b + S::TILE_B);
    if (smem_u32(smem_b) & 1023u) __trap();
    const int tid = threadIdx.x;
    const int grp = blockIdx.x, row0 = blockIdx.y * S::ROWS;
    if (tid == 0) {
        mbar_init(bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        fence_proxy_async();
        mbar_expect_tx(bar, S::TILE_B);
        tensor_g2s_2d_sw(s, &map, grp * (P * RQ * 2), row0, bar);
    }
    const double2 *vt = g.v + ((long long)grp * 16) * S::NTB + tid;
#if P8_VMODE == 3
    // the middle stage's v' values are requested together with the tile: an L2 hit issued later queues behind the
    // tile loads of the SM's other CTAs and costs a DRAM round trip (measured: 0.76 -> 0.83 of the HBM peak)
    double2 vv[16];
#pragma unroll
    for (int m = 0; m < 16; ++m)
        asm volatile("ld.global.nc.v2.f64 {%0, %1}, [%2];" : "=d"(vv[m].x), "=d"(vv[m].y) : "l"(vt + m * S::NTB));
#endif
    __syncthreads();
    mbar_wait(bar, 0);
#if P8_VMODE == 4
    double2 vv[16];
#pragma unroll
    for (int m = 0; m < 16; ++m)
        asm volatile("ld.global.nc.v2.f64 {%0, %1}, [%2];" : "=d"(vv[m].x), "=d"(vv[m].y) : "l"(vt + m * S::NTB));
#endif
    // stage 1 / 3 task: (b0 = x0 mod 32, p); element (a0, q, r) at row q*N0 + a0*32 + b0, chunk (p*RQ + r) ^ (b0 & 7)
    const int b0 = tid % 32, p = tid / 32;
    cd tw[A0 - 1];
#pragma unroll
    for (int k = 1; k < A0; ++k) tw[k - 1] = g.tw0[b0 * k];           // w_N0^(b0 k0a)
    // middle task: tid = ((k0a*NQ + q)*P + p)*RQ + r; element b0' at row q*N0 + k0a*32 + b0', chunk (p*RQ + r) ^ (b0' & 7)
    const int mr = tid % RQ, mp = (tid / RQ) % P, mq = (tid / (RQ * P)) % NQ, mk = tid / (RQ * P * NQ);
    if (P8_SKEL_B != 2) {
    {
        cd u[A0 * B1];                                                  // u[a0*B1 + b1], b1 = q*RQ + r
#pragma unroll
        for (int a0 = 0; a0 < A0; ++a0)
#pragma unroll
            for (int q = 0; q < NQ; ++q)
#pragma unroll
                for (int r = 0; r < RQ; ++r)
                    u[a0 * B1 + q * RQ + r] = s[(q * N0 + a0 * 32 + b0) * 8 + ((p * RQ + r) ^ (b0 & 7))];
        if (P8_SKEL_B != 1 && P8_SKEL_B != 4) dft_rows<A0, B1, false>(u);
#pragma unroll
        for (int k = 1; k < A0; ++k)
#pragma unroll
            for (int c = 0; c < B1; ++c) u[k * B1 + c] = cmul(u[k * B1 + c], tw[k - 1]);
        if (P8_SKEL_B != 1 && P8_SKEL_B != 4) dft_cols<A0, B1, false>(u);
#pragma unroll
        for (int a0 = 0; a0 < A0; ++a0)
#pragma unroll
            for (int q = 0; q < NQ; ++q)
#pragma unroll
                for (int r = 0; r < RQ; ++r)
                    s[(q * N0 + a0 * 32 + b0) * 8 + ((p * RQ + r) ^ (b0 & 7))] = u[a0 * B1 + q * RQ + r];
    }
    __syncthreads();
    {
        cd u[32];
        const int rb = (mq * N0 + mk * 32) * 8, c = mp * RQ + mr;
#pragma unroll
        for (int b = 0; b < 32; ++b) u[b] = s[rb + b * 8 + (c ^ (b & 7))];
#if P8_VMODE == 2
        double2 vv[16];
#pragma unroll
        for (int m = 0; m < 16; ++m) {
            if (P8_SKEL_B >= 3) vv[m] = make_double2(1.0 + tid, 2.0);
            else asm volatile("ld.global.nc.v2.f64 {%0, %1}, [%2];" : "=d"(vv[m].x), "=d"(vv[m].y) : "l"(vt + m * S::NTB));
        }
#endif
        if (P8_SKEL_B != 1 && P8_SKEL_B != 4) DFT<32, false>::run(u);
#if P8_VMODE == 0
        double2 vv[16];
#pragma unroll
        for (int m = 0; m < 16; ++m) vv[m] = __ldg(vt + m * S::NTB);
#endif
#pragma unroll
        for (int m = 0; m < 16; ++m) {
            u[2 * m] = cscale(u[2 * m], vv[m].x);
            u[2 * m + 1] = cscale(u[2 * m + 1], vv[m].y);
        }
        if (P8_SKEL_B != 1 && P8_SKEL_B != 4) DFT<32, true>::run(u);
#pragma unroll
        for (int b = 0; b < 32; ++b) s[rb + b * 8 + (c ^ (b & 7))] = u[b];
    }
    __syncthreads();
    {
        cd u[A0 * B1];
#pragma unroll
        for (int a0 = 0; a0 < A0; ++a0)
#pragma unroll
            for (int q = 0; q < NQ; ++q)
#pragma unroll
                for (int r = 0; r < RQ; ++r)
                    u[a0 * B1 + q * RQ + r] = s[(q * N0 + a0 * 32 + b0) * 8 + ((p * RQ + r) ^ (b0 & 7))];
        if (P8_SKEL_B != 1 && P8_SKEL_B != 4) dft_cols<A0, B1, true>(u);
#pragma unroll
        for (int k = 1; k < A0; ++k)
#pragma unroll
            for (int c = 0; c < B1; ++c) u[k * B1 + c] = cmulc(u[k * B1 + c], tw[k - 1]);
        if (P8_SKEL_B != 1 && P8_SKEL_B != 4) dft_rows<A0, B1, true>(u);
#pragma unroll
        for (int a0 = 0; a0 < A0; ++a0)
#pragma unroll
            for (int q = 0; q < NQ; ++q)
#pragma unroll
                for (int r = 0; r < RQ; ++r)
                    s[(q * N0 + a0 * 32 + b0) * 8 + ((p * RQ + r) ^ (b0 & 7))] = u[a0 * B1 + q * RQ + r];
    }
    }
    fence_proxy_async();
    __syncthreads();
    if (tid == 0) {
        tensor_s2g_2d_sw(&map, grp * (P * RQ * 2), row0, s);
        asm volatile("cp.async.bulk.commit_group;" ::: "memory");
        asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");     // shared memory must outlive the store's reads
    }
}

}  // namespace ptfock
