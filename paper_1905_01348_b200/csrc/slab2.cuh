// slab2.cuh -- register-resident 3-stage slab passes (the fast path of pass A and pass C).
//
// A (x1, x2) slab of N1 x N2 points is transformed in THREE butterfly stages instead of four:
//     x2 = a2*B2 + b2   (N2 = A2*B2),      x1 = a1*B1 + b1   (N1 = A1*B1)
//   stage 1 : radix-A2 DFT over a2          thread <-> (x1, b2)       data straight from global memory
//   stage 2 : 2-D radix (A1 x B2) butterfly  thread <-> (b1, k2a)      both inter-stage twiddles applied here,
//             over (a1, b2)                                            held in registers across the orbital loop
//   stage 3 : radix-B1 DFT over b1           thread <-> (k1a, pos2)    results straight to global, 16 B x 32 lanes
// so shared memory is crossed twice per transform (64 B per point) and global memory is touched only from
// registers.  Frequencies are left at position pos2 = k2a*B2 + k2b (k = k2a + A2*k2b) and
// pos1 = k1a*B1 + k1b (k = k1a + A1*k1b); pass C is the exact mirror (decimation in time).
// The x phi_i product (pass A) and the x phi_i multiply + sum over i (pass C) happen in registers
// (BASELINE.json north_star (2); Alg. 2 line 8).
#pragma once
#include "kernels.cuh"

namespace ptfock {

template <int N1_, int N2_, int A1_, int B1_, int A2_, int B2_, int MINB_>
struct Slab2 {
    static constexpr int N1 = N1_, N2 = N2_, A1 = A1_, B1 = B1_, A2 = A2_, B2 = B2_, MINB = MINB_;
    static_assert(A1 * B1 == N1 && A2 * B2 == N2, "bad split");
    static_assert(N1 * B2 == A1 * N2, "stage 1 and stage 3 must use the same number of threads");
    static constexpr int NT = N1 * B2;          // threads per CTA
    static constexpr int S2 = B1 * A2;          // stage-2 butterflies
    static constexpr int P = N2 + 1;            // odd pitch
    static constexpr int NPTS = N1 * N2;
    static constexpr int SMEM_BYTES = N1 * P * (int)sizeof(cd);
};

// stage 2, forward: twiddle(b2 k2a) -> DFT over b2 -> DFT over a1 -> twiddle(b1 k1a)
template <class S, bool INV>
PTF_DEV void stage2(cd *s, int t, const cd (&tw2r)[S::B2 > 1 ? S::B2 - 1 : 1], const cd (&tw1r)[S::A1 > 1 ? S::A1 - 1 : 1]) {
    constexpr int A1 = S::A1, B1 = S::B1, B2 = S::B2, P = S::P;
    const int b1 = t % B1, k2a = t / B1;
    cd *p = s + b1 * P + k2a * B2;
    cd u[A1][B2];
#pragma unroll
    for (int a1 = 0; a1 < A1; ++a1)
#pragma unroll
        for (int b2 = 0; b2 < B2; ++b2) u[a1][b2] = p[a1 * B1 * P + b2];
    if (!INV) {
#pragma unroll
        for (int a1 = 0; a1 < A1; ++a1) {
#pragma unroll
            for (int b2 = 1; b2 < B2; ++b2) u[a1][b2] = cmul(u[a1][b2], tw2r[b2 - 1]);
            DFT<B2, false>::run(u[a1]);
        }
#pragma unroll
        for (int k2b = 0; k2b < B2; ++k2b) {
            cd c[A1];
#pragma unroll
            for (int a1 = 0; a1 < A1; ++a1) c[a1] = u[a1][k2b];
            DFT<A1, false>::run(c);
#pragma unroll
            for (int k1a = 0; k1a < A1; ++k1a) u[k1a][k2b] = (k1a == 0) ? c[0] : cmul(c[k1a], tw1r[k1a - 1]);
        }
    } else {
#pragma unroll
        for (int k2b = 0; k2b < B2; ++k2b) {
            cd c[A1];
#pragma unroll
            for (int k1a = 0; k1a < A1; ++k1a) c[k1a] = (k1a == 0) ? u[0][k2b] : cmulc(u[k1a][k2b], tw1r[k1a - 1]);
            DFT<A1, true>::run(c);
#pragma unroll
            for (int a1 = 0; a1 < A1; ++a1) u[a1][k2b] = c[a1];
        }
#pragma unroll
        for (int a1 = 0; a1 < A1; ++a1) {
            DFT<B2, true>::run(u[a1]);
#pragma unroll
            for (int b2 = 1; b2 < B2; ++b2) u[a1][b2] = cmulc(u[a1][b2], tw2r[b2 - 1]);
        }
    }
#pragma unroll
    for (int a1 = 0; a1 < A1; ++a1)
#pragma unroll
        for (int b2 = 0; b2 < B2; ++b2) p[a1 * B1 * P + b2] = u[a1][b2];
}

// Row handled by stage-1 thread group q (q = tid / B2).  Rows are dealt out so that the 8 lanes of a
// quarter-warp hit 8 different 16-byte bank groups of the odd-pitch tile: bank = (x1 + b2) mod 8 = lane mod 8.
template <class S>
PTF_DEV int stage1_row(int q) {
    if (S::N1 % S::B2 == 0) return S::B2 * (q % (S::N1 / S::B2)) + q / (S::N1 / S::B2);
    return (S::B2 * q) % S::N1;        // gcd(B2, N1) = 1
}

template <class S>
PTF_DEV void load_stage2_twiddles(const cd *tw1, const cd *tw2, int t, cd (&tw2r)[S::B2 > 1 ? S::B2 - 1 : 1],
                                  cd (&tw1r)[S::A1 > 1 ? S::A1 - 1 : 1]) {
    const int sb1 = t % S::B1, sk2a = t / S::B1;
#pragma unroll
    for (int q = 1; q < S::B2; ++q) tw2r[q - 1] = tw2[q * sk2a];
#pragma unroll
    for (int q = 1; q < S::A1; ++q) tw1r[q - 1] = tw1[q * sb1];
}

// ---- pass A ---------------------------------------------------------------------------------------
template <class S>
__global__ void __launch_bounds__(S::NT, S::MINB) slab2_fwd(const SlabArgs g) {
    constexpr int N2 = S::N2, A1 = S::A1, B1 = S::B1, A2 = S::A2, B2 = S::B2, P = S::P, NT = S::NT;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cd *s = reinterpret_cast<cd *>(smem_raw);
    const int tid = threadIdx.x;
    const int b2 = tid % B2, x1 = stage1_row<S>(tid / B2);             // stage 1
    const int pos2 = tid % N2, k1a = tid / N2;          // stage 3
    cd tw2r[B2 > 1 ? B2 - 1 : 1], tw1r[A1 > 1 ? A1 - 1 : 1];
    load_stage2_twiddles<S>(g.tw1, g.tw2, tid < S::S2 ? tid : 0, tw2r, tw1r);
    const int x0 = blockIdx.y, jj = blockIdx.x;     // CTAs that share the phi slabs run together (L2 reuse)
    const long long slab_off = (long long)x0 * S::NPTS;
    const int goff = x1 * N2 + b2;                        // + a2 * B2
    const cd *psi = g.b + (long long)(g.b0 + jj) * g.grid_pts + slab_off + goff;
    cd pj[A2];
#pragma unroll
    for (int a2 = 0; a2 < A2; ++a2) pj[a2] = psi[a2 * B2];
    const int per = (g.na + gridDim.z - 1) / gridDim.z;
    const int ii_beg = blockIdx.z * per, ii_end = min(g.na, ii_beg + per);
    cd v[A2];
    if (ii_beg < ii_end) {
        const cd *phi = g.a + (long long)(g.a0 + ii_beg) * g.grid_pts + slab_off + goff;
#pragma unroll
        for (int a2 = 0; a2 < A2; ++a2) v[a2] = __ldg(reinterpret_cast<const double2 *>(phi + a2 * B2));
    }
    for (int ii = ii_beg; ii < ii_end; ++ii) {
#pragma unroll
        for (int a2 = 0; a2 < A2; ++a2) v[a2] = cmulc(pj[a2], v[a2]);       // psi_j conj(phi_i)
        DFT<A2, false>::run(v);
#pragma unroll
        for (int k = 0; k < A2; ++k) s[x1 * P + k * B2 + b2] = v[k];
        if (ii + 1 < ii_end) {      // prefetch the next orbital's slab while stages 2 and 3 run
            const cd *phi = g.a + (long long)(g.a0 + ii + 1) * g.grid_pts + slab_off + goff;
#pragma unroll
            for (int a2 = 0; a2 < A2; ++a2) v[a2] = __ldg(reinterpret_cast<const double2 *>(phi + a2 * B2));
        }
        __syncthreads();
        if (S::S2 <= NT) {
            if (tid < S::S2) stage2<S, false>(s, tid, tw2r, tw1r);
        } else {
            for (int t = tid; t < S::S2; t += NT) {
                load_stage2_twiddles<S>(g.tw1, g.tw2, t, tw2r, tw1r);
                stage2<S, false>(s, t, tw2r, tw1r);
            }
        }
        __syncthreads();
        cd w[B1];
#pragma unroll
        for (int q = 0; q < B1; ++q) w[q] = s[(k1a * B1 + q) * P + pos2];
        DFT<B1, false>::run(w);
        cd *dst = g.scratch + ((long long)(ii * g.stride_loop + jj * g.stride_cta) * g.n0 + x0) * S::NPTS + k1a * B1 * N2 + pos2;
#pragma unroll
        for (int q = 0; q < B1; ++q) dst[q * N2] = w[q];
        __syncthreads();
    }
}

// ---- pass C ---------------------------------------------------------------------------------------
template <class S>
__global__ void __launch_bounds__(S::NT, S::MINB) slab2_inv_acc(const SlabArgs g) {
    constexpr int N2 = S::N2, A1 = S::A1, B1 = S::B1, A2 = S::A2, B2 = S::B2, P = S::P, NT = S::NT;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cd *s = reinterpret_cast<cd *>(smem_raw);
    const int tid = threadIdx.x;
    const int b2 = tid % B2, x1 = stage1_row<S>(tid / B2);             // last stage (mirror of forward stage 1)
    const int pos2 = tid % N2, k1a = tid / N2;          // first stage (mirror of forward stage 3)
    cd tw2r[B2 > 1 ? B2 - 1 : 1], tw1r[A1 > 1 ? A1 - 1 : 1];
    load_stage2_twiddles<S>(g.tw1, g.tw2, tid < S::S2 ? tid : 0, tw2r, tw1r);
    const int x0 = blockIdx.y, tt = blockIdx.x;
    const long long slab_off = (long long)x0 * S::NPTS;
    const int goff = x1 * N2 + b2;
    cd acc[A2];
#pragma unroll
    for (int a2 = 0; a2 < A2; ++a2) acc[a2] = make_double2(0.0, 0.0);
    cd w[B1];
    if (g.na > 0) {
        const cd *src = g.scratch + ((long long)(tt * g.stride_cta) * g.n0 + x0) * S::NPTS + k1a * B1 * N2 + pos2;
#pragma unroll
        for (int q = 0; q < B1; ++q) w[q] = src[q * N2];
    }
    for (int ss = 0; ss < g.na; ++ss) {
        DFT<B1, true>::run(w);
#pragma unroll
        for (int q = 0; q < B1; ++q) s[(k1a * B1 + q) * P + pos2] = w[q];
        // this iteration's orbital slab and the next iteration's pair density: in flight during stage 2
        const cd *phi = g.a + (long long)(g.a0 + ss) * g.grid_pts + slab_off + goff;
        cd f[A2];
#pragma unroll
        for (int a2 = 0; a2 < A2; ++a2) f[a2] = __ldg(reinterpret_cast<const double2 *>(phi + a2 * B2));
        if (ss + 1 < g.na) {
            const cd *src = g.scratch + ((long long)((ss + 1) * g.stride_loop + tt * g.stride_cta) * g.n0 + x0) * S::NPTS + k1a * B1 * N2 + pos2;
#pragma unroll
            for (int q = 0; q < B1; ++q) w[q] = src[q * N2];
        }
        __syncthreads();
        if (S::S2 <= NT) {
            if (tid < S::S2) stage2<S, true>(s, tid, tw2r, tw1r);
        } else {
            for (int t = tid; t < S::S2; t += NT) {
                load_stage2_twiddles<S>(g.tw1, g.tw2, t, tw2r, tw1r);
                stage2<S, true>(s, t, tw2r, tw1r);
            }
        }
        __syncthreads();
        cd v[A2];
#pragma unroll
        for (int k = 0; k < A2; ++k) v[k] = s[x1 * P + k * B2 + b2];
        DFT<A2, true>::run(v);
        if (g.conj_w) {
#pragma unroll
            for (int a2 = 0; a2 < A2; ++a2) {
                const cd pr = cmulc(f[a2], v[a2]);
                acc[a2].x += pr.x; acc[a2].y += pr.y;
            }
        } else {
#pragma unroll
            for (int a2 = 0; a2 < A2; ++a2) {
                const cd pr = cmul(f[a2], v[a2]);
                acc[a2].x += pr.x; acc[a2].y += pr.y;
            }
        }
        __syncthreads();
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

}  // namespace ptfock
