// kernels.cuh -- the three fused passes of one wave of pair-solves (Alg. 2 lines 6-10).
//
//   pass A  slab_fwd<N1,N2>   : rho = conj(phi_i) psi_j formed on load (K1 of SURVEY.md Sec. 2), forward DFT
//                                along x2 and x1 of one contiguous (x1,x2) slab in shared memory, slab
//                                written to the pair scratch in digit-permuted frequency order.
//   pass B  pencil_mid<N0>    : forward DFT along x0, multiply by v'(G) = -alpha/N v(G) (K3), inverse DFT
//                                along x0, in place in the scratch; 512-byte coalesced rows.
//   pass C  slab_inv_acc<N1,N2>: inverse DFT along x1 and x2 of one slab, x phi_s and the sum over the
//                                wave's orbitals accumulated in registers (K5), one read-modify-write of out.
//
// Forward transforms are decimation-in-frequency and leave each axis in digit-permuted order
// (position q = k1*R2 + k2 holds frequency k = k1 + R1*k2); the v' table is stored in that order and
// the inverse transforms are the exact mirror (decimation in time), so no reordering pass exists.
#pragma once
#include "codelets.cuh"

namespace ptfock {

// radix split per supported edge: n = R1 * R2 (R2 == 1: single stage)
template <int N> struct Split;
template <> struct Split<16> { static constexpr int R1 = 16, R2 = 1; };
template <> struct Split<32> { static constexpr int R1 = 8, R2 = 4; };
template <> struct Split<48> { static constexpr int R1 = 16, R2 = 3; };
template <> struct Split<64> { static constexpr int R1 = 8, R2 = 8; };
template <> struct Split<128> { static constexpr int R1 = 16, R2 = 8; };
template <> struct Split<120> { static constexpr int R1 = 15, R2 = 8; };   // paper grid (NEXT-2): pencil axis only

constexpr int kSlabThreads = 256;

// ---- one axis of a shared-memory tile -------------------------------------------------------------
// element (batch, x) of the axis lives at s[batch * SB + x * SA].  NB batches.  Lanes run over the
// batch index first (SB is 1 or an odd pitch => 16-byte bank groups are conflict free).
template <int N, int NB, int SA, int SB, int NT>
PTF_DEV void axis_forward(cd *s, const cd *tw, int tid) {
    constexpr int R1 = Split<N>::R1, R2 = Split<N>::R2;
    // stage 1: DFT over a (x = a R2 + b), twiddle w_N^(b k1), stored at k1 R2 + b
    for (int t = tid; t < NB * R2; t += NT) {
        const int batch = t % NB, b = t / NB;
        cd *p = s + batch * SB + b * SA;
        cd v[R1];
#pragma unroll
        for (int a = 0; a < R1; ++a) v[a] = p[a * R2 * SA];
        DFT<R1, false>::run(v);
        if (R2 > 1) {
#pragma unroll
            for (int k1 = 1; k1 < R1; ++k1) v[k1] = cmul(v[k1], tw[b * k1]);
        }
#pragma unroll
        for (int k1 = 0; k1 < R1; ++k1) p[k1 * R2 * SA] = v[k1];
    }
    __syncthreads();
    if (R2 > 1) {
        // stage 2: DFT over b, result k2 stored at k1 R2 + k2
        for (int t = tid; t < NB * R1; t += NT) {
            const int batch = t % NB, k1 = t / NB;
            cd *p = s + batch * SB + k1 * R2 * SA;
            cd v[R2];
#pragma unroll
            for (int b = 0; b < R2; ++b) v[b] = p[b * SA];
            DFT<R2, false>::run(v);
#pragma unroll
            for (int b = 0; b < R2; ++b) p[b * SA] = v[b];
        }
        __syncthreads();
    }
}

template <int N, int NB, int SA, int SB, int NT>
PTF_DEV void axis_inverse(cd *s, const cd *tw, int tid) {
    constexpr int R1 = Split<N>::R1, R2 = Split<N>::R2;
    if (R2 > 1) {
        for (int t = tid; t < NB * R1; t += NT) {
            const int batch = t % NB, k1 = t / NB;
            cd *p = s + batch * SB + k1 * R2 * SA;
            cd v[R2];
#pragma unroll
            for (int b = 0; b < R2; ++b) v[b] = p[b * SA];
            DFT<R2, true>::run(v);
#pragma unroll
            for (int b = 0; b < R2; ++b) p[b * SA] = v[b];
        }
        __syncthreads();
    }
    for (int t = tid; t < NB * R2; t += NT) {
        const int batch = t % NB, b = t / NB;
        cd *p = s + batch * SB + b * SA;
        cd v[R1];
#pragma unroll
        for (int k1 = 0; k1 < R1; ++k1) v[k1] = p[k1 * R2 * SA];
        if (R2 > 1) {
#pragma unroll
            for (int k1 = 1; k1 < R1; ++k1) v[k1] = cmulc(v[k1], tw[b * k1]);
        }
        DFT<R1, true>::run(v);
#pragma unroll
        for (int a = 0; a < R1; ++a) p[a * R2 * SA] = v[a];
    }
    __syncthreads();
}

template <int N1, int N2> struct SlabShape {
    static constexpr int P = N2 + 1;                       // odd row pitch (elements)
    static constexpr int NPTS = N1 * N2;
    static constexpr int SMEM_BYTES = (N1 * P + N1 + N2) * (int)sizeof(cd);
    static constexpr int PER_THREAD = NPTS / kSlabThreads;
    static_assert(NPTS % kSlabThreads == 0, "slab must be a multiple of the CTA size");
};

struct SlabArgs {
    const cd *a;        // pass A: phi (conjugated factor)   pass C: summed orbitals (multiplied in)
    const cd *b;        // pass A: psi (targets)             pass C: unused
    cd *scratch;        // [pair][x0][slab]
    cd *out;            // pass C: targets' output (read-modify-write)
    const cd *tw1, *tw2;
    long long grid_pts; // N = n0 * N1 * N2
    int n0;
    int a0, na;         // first index / count along the looped orbital set
    int b0;             // first index of the per-CTA (blockIdx.y) set
    int stride_loop;    // scratch pair index = loop_local * stride_loop + cta_local * stride_cta
    int stride_cta;
    int conj_w;         // pass C: use conj(W) (pair symmetry W_ji = conj(W_ij))
    int tri;            // diagonal block of the pair-symmetric schedule: 1 = loop index <= CTA index only (pairs i <= j),
                        // 2 = loop index > CTA index only (the conj(W) accumulate of the same block); 0 = whole range
};

// loop range [lo, hi) of a slab pass for CTA index `cta` out of [beg, end)
PTF_DEV void tri_range(int tri, int cta, int beg, int end, int &lo, int &hi) {
    lo = beg; hi = end;
    if (tri == 1) hi = min(end, cta + 1);
    else if (tri == 2) lo = max(beg, cta + 1);
}

// ---- pass A ---------------------------------------------------------------------------------------
// grid = (number of targets in the wave, n0, chunks of the i loop); CTA (jj, x0, z) loops over its share of
// the wave's orbitals i.
template <int N1, int N2>
__global__ void __launch_bounds__(kSlabThreads) slab_fwd(const SlabArgs g) {
    using S = SlabShape<N1, N2>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cd *s = reinterpret_cast<cd *>(smem_raw);
    cd *tw1 = s + N1 * S::P, *tw2 = tw1 + N1;
    const int tid = threadIdx.x;
    for (int t = tid; t < N1; t += kSlabThreads) tw1[t] = g.tw1[t];
    for (int t = tid; t < N2; t += kSlabThreads) tw2[t] = g.tw2[t];
    const int x0 = blockIdx.y, jj = blockIdx.x;
    const long long slab_off = (long long)x0 * S::NPTS;
    const cd *psi = g.b + (long long)(g.b0 + jj) * g.grid_pts + slab_off;
    cd pj[S::PER_THREAD];
#pragma unroll
    for (int k = 0; k < S::PER_THREAD; ++k) pj[k] = psi[tid + k * kSlabThreads];
    const int per = (g.na + gridDim.z - 1) / gridDim.z;
    int ii_beg, ii_end;
    tri_range(g.tri, jj, blockIdx.z * per, min(g.na, blockIdx.z * per + per), ii_beg, ii_end);
    for (int ii = ii_beg; ii < ii_end; ++ii) {
        const cd *phi = g.a + (long long)(g.a0 + ii) * g.grid_pts + slab_off;
#pragma unroll
        for (int k = 0; k < S::PER_THREAD; ++k) {
            const int p = tid + k * kSlabThreads;
            const cd f = __ldg(reinterpret_cast<const double2 *>(phi + p));
            s[(p / N2) * S::P + (p % N2)] = cmulc(pj[k], f);          // psi_j * conj(phi_i)
        }
        __syncthreads();
        axis_forward<N2, N1, 1, S::P, kSlabThreads>(s, tw2, tid);
        axis_forward<N1, N2, S::P, 1, kSlabThreads>(s, tw1, tid);
        cd *dst = g.scratch + ((long long)(ii * g.stride_loop + jj * g.stride_cta) * g.n0 + x0) * S::NPTS;
#pragma unroll
        for (int k = 0; k < S::PER_THREAD; ++k) {
            const int p = tid + k * kSlabThreads;
            dst[p] = s[(p / N2) * S::P + (p % N2)];
        }
        __syncthreads();
    }
}

// ---- pass C ---------------------------------------------------------------------------------------
// grid = (number of targets, n0); CTA (tt, x0) sums over the looped orbitals s:
//   out[b0+tt] += sum_s a[a0+s] * W[s*stride_loop + tt*stride_cta]   (W or conj(W))
template <int N1, int N2>
__global__ void __launch_bounds__(kSlabThreads) slab_inv_acc(const SlabArgs g) {
    using S = SlabShape<N1, N2>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cd *s = reinterpret_cast<cd *>(smem_raw);
    cd *tw1 = s + N1 * S::P, *tw2 = tw1 + N1;
    const int tid = threadIdx.x;
    for (int t = tid; t < N1; t += kSlabThreads) tw1[t] = g.tw1[t];
    for (int t = tid; t < N2; t += kSlabThreads) tw2[t] = g.tw2[t];
    const int x0 = blockIdx.y, tt = blockIdx.x;
    const long long slab_off = (long long)x0 * S::NPTS;
    cd acc[S::PER_THREAD];
#pragma unroll
    for (int k = 0; k < S::PER_THREAD; ++k) acc[k] = make_double2(0.0, 0.0);
    int ss_beg, ss_end;
    tri_range(g.tri, tt, 0, g.na, ss_beg, ss_end);
    for (int ss = ss_beg; ss < ss_end; ++ss) {
        const cd *src = g.scratch + ((long long)(ss * g.stride_loop + tt * g.stride_cta) * g.n0 + x0) * S::NPTS;
#pragma unroll
        for (int k = 0; k < S::PER_THREAD; ++k) {
            const int p = tid + k * kSlabThreads;
            s[(p / N2) * S::P + (p % N2)] = src[p];
        }
        __syncthreads();
        axis_inverse<N1, N2, S::P, 1, kSlabThreads>(s, tw1, tid);
        axis_inverse<N2, N1, 1, S::P, kSlabThreads>(s, tw2, tid);
        const cd *phi = g.a + (long long)(g.a0 + ss) * g.grid_pts + slab_off;
#pragma unroll
        for (int k = 0; k < S::PER_THREAD; ++k) {
            const int p = tid + k * kSlabThreads;
            const cd f = __ldg(reinterpret_cast<const double2 *>(phi + p));
            const cd w = s[(p / N2) * S::P + (p % N2)];
            const cd pr = g.conj_w ? cmulc(f, w) : cmul(f, w);
            acc[k].x += pr.x;
            acc[k].y += pr.y;
        }
        __syncthreads();
    }
    cd *o = g.out + (long long)(g.b0 + tt) * g.grid_pts + slab_off;
#pragma unroll
    for (int k = 0; k < S::PER_THREAD; ++k) {
        const int p = tid + k * kSlabThreads;
        cd cur = o[p];
        cur.x += acc[k].x;
        cur.y += acc[k].y;
        o[p] = cur;
    }
}

// ---- pass B (n0 <= 48; longer pencils: pencil_tma.cuh, 64^3: pass8.cuh) ------------------------------------------
// grid = (slab_pts / CW, pairs).  A CTA owns CW contiguous slab positions for all x0 of one pair.
template <int N0> struct PencilShape {
    static constexpr int CW = 32;                                  // contiguous slab positions per CTA
    static constexpr int R1 = Split<N0>::R1, R2 = Split<N0>::R2;
    static constexpr int NT = (R2 == 1) ? 128 : 256;
    static constexpr int SMEM_BYTES = (R2 == 1) ? 0 : (N0 * CW + N0) * (int)sizeof(cd);
    static constexpr int MINB = (R2 == 1) ? 1 : 3;
};

struct PencilArgs {
    cd *scratch;
    const double *v;     // [N0 positions][slab_pts], digit-permuted, -alpha/N folded in
    const cd *tw0;
    int slab_pts;
    int tri_nj;          // > 0: diagonal block of the symmetric schedule, pair = i*tri_nj + j exists only for i <= j
};

template <int N0>
__global__ void __launch_bounds__(PencilShape<N0>::NT, PencilShape<N0>::MINB) pencil_mid(const PencilArgs g) {
    using S = PencilShape<N0>;
    constexpr int R1 = S::R1, R2 = S::R2, CW = S::CW, NT = S::NT;
    const int tid = threadIdx.x;
    const long long sp = g.slab_pts;
    if (g.tri_nj > 0 && (int)blockIdx.y / g.tri_nj > (int)blockIdx.y % g.tri_nj) return;
    cd *base = g.scratch + (long long)blockIdx.y * N0 * sp;
    if (R2 == 1) {
        // whole pencil in one thread's registers: no shared memory at all
        const long long p = (long long)blockIdx.x * NT + tid;
        if (p >= sp) return;
        cd v[R1];
#pragma unroll
        for (int a = 0; a < R1; ++a) v[a] = base[a * sp + p];
        DFT<R1, false>::run(v);
#pragma unroll
        for (int k = 0; k < R1; ++k) v[k] = cscale(v[k], __ldg(g.v + k * sp + p));
        DFT<R1, true>::run(v);
#pragma unroll
        for (int a = 0; a < R1; ++a) base[a * sp + p] = v[a];
        return;
    } else {
        extern __shared__ __align__(16) unsigned char smem_raw[];
        cd *s = reinterpret_cast<cd *>(smem_raw);
        cd *tw = s + N0 * CW;
        for (int t = tid; t < N0; t += NT) tw[t] = g.tw0[t];
        __syncthreads();
        const long long p0 = (long long)blockIdx.x * CW;
        const int cvalid = (sp - p0 < CW) ? (int)(sp - p0) : CW;      // ragged last tile (slab_pts % CW != 0)
        // stage 1: global -> registers -> DFT over a -> twiddle -> shared
        for (int t = tid; t < CW * R2; t += NT) {
            const int c = t % CW, b = t / CW;
            cd v[R1];
#pragma unroll
            for (int a = 0; a < R1; ++a)
                v[a] = c < cvalid ? base[(long long)(a * R2 + b) * sp + p0 + c] : make_double2(0.0, 0.0);
            DFT<R1, false>::run(v);
#pragma unroll
            for (int k1 = 1; k1 < R1; ++k1) v[k1] = cmul(v[k1], tw[b * k1]);
#pragma unroll
            for (int k1 = 0; k1 < R1; ++k1) s[(k1 * R2 + b) * CW + c] = v[k1];
        }
        __syncthreads();
        // middle: forward DFT over b, x v', inverse DFT over k2, all in registers
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
        // last: shared -> registers -> conj twiddle -> inverse DFT over k1 -> global
        for (int t = tid; t < CW * R2; t += NT) {
            const int c = t % CW, b = t / CW;
            cd v[R1];
#pragma unroll
            for (int k1 = 0; k1 < R1; ++k1) v[k1] = s[(k1 * R2 + b) * CW + c];
#pragma unroll
            for (int k1 = 1; k1 < R1; ++k1) v[k1] = cmulc(v[k1], tw[b * k1]);
            DFT<R1, true>::run(v);
            if (c < cvalid) {
#pragma unroll
                for (int a = 0; a < R1; ++a) base[(long long)(a * R2 + b) * sp + p0 + c] = v[a];
            }
        }
    }
}

// ---- FP64 pipe peak (measurement aid for bench.py: the second roof of SURVEY.md 8(d)) ---------------------------
// 8 independent register-resident DFMA chains per thread; 2 * 8 * iters flops per thread.
__global__ void __launch_bounds__(256) fp64_peak_kernel(double *sink, int iters, double a, double b) {
    double x0 = threadIdx.x, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5, x6 = x0 + 6, x7 = x0 + 7;
    for (int k = 0; k < iters; ++k) {
        x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
        x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
    }
    const double r = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
    if (r == 123.456) sink[0] = r;          // never true: keeps the loop alive
}

// ---- copy bandwidth (measurement aid: L2-resident vs HBM-resident working sets) ------------------
// dst[k] = src[k] over n 16-byte elements, grid-stride, 4 independent 128-bit loads in flight per thread.
__global__ void __launch_bounds__(256) copy_bw_kernel(const double2 *__restrict__ src, double2 *__restrict__ dst, long long n) {
    const long long stride = (long long)gridDim.x * blockDim.x;
    long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    for (; k + 3 * stride < n; k += 4 * stride) {
        const double2 a = src[k], b = src[k + stride], c = src[k + 2 * stride], d = src[k + 3 * stride];
        dst[k] = a; dst[k + stride] = b; dst[k + 2 * stride] = c; dst[k + 3 * stride] = d;
    }
    for (; k < n; k += stride) dst[k] = src[k];
}

// ---- helpers --------------------------------------------------------------------------------------
// partial[b] = sum over the block's share of conj(psi) * vx
__global__ void __launch_bounds__(256) dot_partial(const cd *psi, const cd *vx, long long n, double2 *partial) {
    __shared__ double2 red[256];
    double sr = 0.0, si = 0.0;
    for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (long long)gridDim.x * blockDim.x) {
        const cd a = psi[k], b = vx[k];
        sr += a.x * b.x + a.y * b.y;
        si += a.x * b.y - a.y * b.x;
    }
    red[threadIdx.x] = make_double2(sr, si);
    __syncthreads();
    for (int h = 128; h > 0; h >>= 1) {
        if (threadIdx.x < h) {
            red[threadIdx.x].x += red[threadIdx.x + h].x;
            red[threadIdx.x].y += red[threadIdx.x + h].y;
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) partial[blockIdx.x] = red[0];
}

__global__ void __launch_bounds__(256) dot_final(const double2 *partial, int n, double scale, double2 *result) {
    __shared__ double2 red[256];
    double sr = 0.0, si = 0.0;
    for (int k = threadIdx.x; k < n; k += 256) { sr += partial[k].x; si += partial[k].y; }
    red[threadIdx.x] = make_double2(sr, si);
    __syncthreads();
    for (int h = 128; h > 0; h >>= 1) {
        if (threadIdx.x < h) {
            red[threadIdx.x].x += red[threadIdx.x + h].x;
            red[threadIdx.x].y += red[threadIdx.x + h].y;
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) *result = make_double2(red[0].x * scale, red[0].y * scale);
}

}  // namespace ptfock
