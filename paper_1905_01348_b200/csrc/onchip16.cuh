// onchip16.cuh -- single-pass, zero-scratch pair-solves for 16^3 grids (SURVEY.md 8(f) NEXT-1, 8(a) "16^3 fits a
// single CTA"; Eq. (3), Alg. 2 lines 6-10).
//
// One pair density (4096 points = 64 KB) lives in ONE CTA's shared memory from the product conj(phi_i) psi_j to the
// accumulation into (V_X psi)_j: nothing but the orbitals and the result ever touches global memory, and one
// application is two launches (this kernel + the fixed-order reduction of the i-chunks) instead of three per wave.
//
//   CTA (target j, chunk c of the i loop), 256 threads, psi_j and the running sum in registers (16 points each):
//     1  thread (x1, x2): u = psi_j conj(phi_i) for x0 = 0..15, DFT16 over x0                         -> tile
//     2  thread (k0, x2): DFT16 over x1, in place
//     3  thread (k0, k1): DFT16 over x2, x v'(k0, k1, k2), inverse DFT16 over k2, in place
//     4  thread (k0, x2): inverse DFT16 over k1, in place
//     5  thread (x1, x2): inverse DFT16 over k0, x phi_i, += accumulators
//   tile element (k0, a, b) sits at k0*256 + a*16 + (b ^ (a & 7)): every access of every step is conflict free, and
//   each thread of steps 2-4 reads and writes the same 16 slots, so four CTA barriers per pair are enough.
// All codelets leave their output in natural order, so v' is the natural-order table, stored [k2][k0][k1].
// The chunks' partial sums are written to partial[c][j] and added in chunk order by onchip_reduce (deterministic).
#pragma once
#include "kernels.cuh"

namespace ptfock {

struct OnchipArgs {
    const cd *phi;          // orbitals of the sum (conjugated in the product)
    const cd *mul;          // orbitals multiplied in at the end (= phi; a grid of ones for ptfock_debug_pair)
    const cd *psi;          // targets
    cd *partial;            // [chunk][target][4096]
    const double *vt;       // v'[k2*256 + k0*16 + k1] = -alpha/N v(G(k0, k1, k2))
    int phi0, n_i;          // first orbital / count of the sum
    int mul_stride;         // grids between consecutive `mul` orbitals (0: the same grid for every i)
    int psi0;               // first target
    int i_per_cta;
};

constexpr int kOnchipThreads = 256;
constexpr int kOnchipSmem = 4096 * (int)sizeof(cd);

__global__ void __launch_bounds__(kOnchipThreads, 1) onchip16_apply(const OnchipArgs g) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cd *T = reinterpret_cast<cd *>(smem_raw);
    const int tid = threadIdx.x;
    const int jj = blockIdx.x, chunk = blockIdx.y;
    const int hi = tid >> 4, lo = tid & 15;               // (x1, x2) in steps 1 / 5, (k0, x2) in 2 / 4, (k0, k1) in 3
    const int i_beg = chunk * g.i_per_cta, i_end = min(g.n_i, i_beg + g.i_per_cta);
    cd pj[16], acc[16];
    {
        const cd *psi = g.psi + (long long)(g.psi0 + jj) * 4096 + tid;
#pragma unroll
        for (int x0 = 0; x0 < 16; ++x0) { pj[x0] = psi[x0 * 256]; acc[x0] = make_double2(0.0, 0.0); }
    }
    const int s15 = hi * 16 + (lo ^ (hi & 7));            // steps 1 / 5: + k0*256
    const int s24 = hi * 256;                             // steps 2 / 4: + a*16 + (lo ^ (a & 7))
    const int s3 = hi * 256 + lo * 16;                    // step 3:      + (b ^ (lo & 7))
#pragma unroll 1
    for (int i = i_beg; i < i_end; ++i) {
        const cd *phi = g.phi + (long long)(g.phi0 + i) * 4096 + tid;
        cd u[16];
#pragma unroll
        for (int x0 = 0; x0 < 16; ++x0) u[x0] = cmulc(pj[x0], __ldg(reinterpret_cast<const double2 *>(phi + x0 * 256)));
        DFT<16, false>::run(u);
#pragma unroll
        for (int k0 = 0; k0 < 16; ++k0) T[k0 * 256 + s15] = u[k0];
        __syncthreads();
#pragma unroll
        for (int a = 0; a < 16; ++a) u[a] = T[s24 + a * 16 + (lo ^ (a & 7))];
        DFT<16, false>::run(u);
#pragma unroll
        for (int a = 0; a < 16; ++a) T[s24 + a * 16 + (lo ^ (a & 7))] = u[a];
        __syncthreads();
#pragma unroll
        for (int b = 0; b < 16; ++b) u[b] = T[s3 + (b ^ (lo & 7))];
        DFT<16, false>::run(u);
#pragma unroll
        for (int k2 = 0; k2 < 16; ++k2) u[k2] = cscale(u[k2], __ldg(g.vt + k2 * 256 + tid));
        DFT<16, true>::run(u);
#pragma unroll
        for (int b = 0; b < 16; ++b) T[s3 + (b ^ (lo & 7))] = u[b];
        __syncthreads();
#pragma unroll
        for (int a = 0; a < 16; ++a) u[a] = T[s24 + a * 16 + (lo ^ (a & 7))];
        DFT<16, true>::run(u);
#pragma unroll
        for (int a = 0; a < 16; ++a) T[s24 + a * 16 + (lo ^ (a & 7))] = u[a];
        __syncthreads();
#pragma unroll
        for (int k0 = 0; k0 < 16; ++k0) u[k0] = T[k0 * 256 + s15];
        DFT<16, true>::run(u);
        const cd *mul = g.mul + ((long long)g.phi0 * (g.mul_stride != 0) + (long long)i * g.mul_stride) * 4096 + tid;
#pragma unroll
        for (int x0 = 0; x0 < 16; ++x0) {
            const cd pr = cmul(__ldg(reinterpret_cast<const double2 *>(mul + x0 * 256)), u[x0]);
            acc[x0].x += pr.x; acc[x0].y += pr.y;
        }
        __syncthreads();                                  // the tile is read: the next product may overwrite it
    }
    cd *dst = g.partial + ((long long)chunk * gridDim.x + jj) * 4096 + tid;
#pragma unroll
    for (int x0 = 0; x0 < 16; ++x0) dst[x0 * 256] = acc[x0];
}

// out[j][p] = sum over chunks c (in order) of partial[c][j][p]; overwrites out (Alg. 2 line 1 needs no separate memset)
__global__ void __launch_bounds__(256) onchip_reduce(const cd *partial, int n_chunks, long long per_chunk, cd *out) {
    const long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= per_chunk) return;
    cd s = partial[k];
    for (int c = 1; c < n_chunks; ++c) {
        const cd t = partial[(long long)c * per_chunk + k];
        s.x += t.x; s.y += t.y;
    }
    out[k] = s;
}

}  // namespace ptfock
