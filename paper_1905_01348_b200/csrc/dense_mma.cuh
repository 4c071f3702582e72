// dense_mma.cuh -- the two GEMM-shaped dense-algebra neighbours on the FP64 tensor cores (mma.sync m8n8k4, SASS DMMA.8x8x4):
// the overlap matrix S = w A^H B (Alg. 3 line 2; "Psi^* Psi") and the rotation
// out = A S with the fused BLAS-1 epilogues (Alg. 3 lines 4-5; Alg. 1 line 1).  These ARE dense contractions, so they
// belong on the tensor pipe: a warp-level DMMA needs two 8-byte operands per lane for 256 FMAs where the register-tiled
// DFMA kernels of dense.cuh need 128 bytes of shared-memory reads per thread for 64 (they sit at half the FP64 peak,
// bound by the shared-memory pipe).  Measured DMMA peak on B200: 37.1 TFLOP/s (DFMA loop: 34.1).
//
// Complex products on a real MMA: orbitals are interleaved (re, im), i.e. a row of K complex points IS a row of 2K
// reals.  With a' = (ar, ai, ...), b' = (br, bi, ...), b'' = (bi, -br, ...):
//     Re sum conj(a) b = a' . b'        Im sum conj(a) b = a' . b''
// so the A fragment is read as stored and the two B fragments (b', b'') come from ONE 16-byte read of the complex
// element (the lane picks x / y and a sign).  Everything is deterministic (fixed split-K order, no atomics).
#pragma once
#include "dense.cuh"
#include "tma.cuh"

namespace ptfock {

PTF_DEV void dmma884(double &d0, double &d1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}
PTF_DEV void cp_async16(void *dst_smem, const void *src, bool valid) {
    const unsigned sz = valid ? 16u : 0u;                 // src-size 0: the 16 bytes are zero-filled
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(smem_u32(dst_smem)), "l"(src), "r"(sz) : "memory");
}
PTF_DEV void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> PTF_DEV void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// FP64 tensor-pipe peak (measurement aid: the roof of the two kernels below): 8 independent accumulator tiles per warp
__global__ void __launch_bounds__(256) dmma_peak_kernel(double *sink, int iters, double a, double b) {
    double c[8][2];
#pragma unroll
    for (int i = 0; i < 8; ++i) { c[i][0] = threadIdx.x + i; c[i][1] = 0.0; }
    for (int k = 0; k < iters; ++k)
#pragma unroll
        for (int i = 0; i < 8; ++i) dmma884(c[i][0], c[i][1], a, b);
    double r = 0.0;
#pragma unroll
    for (int i = 0; i < 8; ++i) r += c[i][0] + c[i][1];
    if (r == 123.456) sink[0] = r;          // never true: keeps the loop alive
}

// ---- overlap: part[ks][m][n] = sum over this split's points of conj(a[m][r]) b[n][r] ------------------------------------
// grid = (ceil(n_a / 64), ceil(n_b / 64), k_splits), or (T (T + 1) / 2, 1, k_splits) lower-triangle tiles for a Hermitian
// product (OverlapArgs::lower); 128 threads = 2 x 2 warps, warp tile 32 x 32 = 4 x 4 DMMA tiles for
// the real and 4 x 4 for the imaginary part (128 accumulator registers).  K advances 16 points per stage through a
// 3-stage cp.async ring; a tile row is 16 points = 256 bytes + 32 bytes of padding: the fragment reads (8 rows x 32
// bytes for A, 8 rows x 2 complex elements for B) then touch every bank exactly once per 128-byte wavefront.
constexpr int kMK = 16;                                   // points per stage
constexpr int kMPitch = kMK + 2;                          // row pitch in complex elements (288 bytes)
constexpr int kMStages = 3;                                // 108 KB per CTA: two CTAs per SM
constexpr int kMStageElems = 2 * 64 * kMPitch;            // A tile + B tile
constexpr int kOverlapMmaSmem = kMStages * kMStageElems * (int)sizeof(cd);

__global__ void __launch_bounds__(128, 2) overlap_mma(const OverlapArgs g) {
    extern __shared__ __align__(16) unsigned char dense_smem[];
    cd *ring = reinterpret_cast<cd *>(dense_smem);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int wm = (warp >> 1) * 32, wn = (warp & 1) * 32;
    int tm = blockIdx.x, tn = blockIdx.y;
    if (g.lower) {                                         // blockIdx.x = tm (tm + 1) / 2 + tn with tn <= tm
        tm = (int)((sqrt(8.0 * (double)blockIdx.x + 1.0) - 1.0) * 0.5);
        while ((tm + 1) * (tm + 2) / 2 <= (int)blockIdx.x) ++tm;
        while (tm * (tm + 1) / 2 > (int)blockIdx.x) --tm;
        tn = (int)blockIdx.x - tm * (tm + 1) / 2;
    }
    const int m0 = tm * 64, n0 = tn * 64;
    const long long r_beg = (long long)blockIdx.z * g.pts_per_split;
    const long long r_end = min(g.n_pts, r_beg + g.pts_per_split);
    const int n_steps = (int)((r_end - r_beg + kMK - 1) / kMK);
    // loader: chunk c = tid + 128 i (i < 8) of a 64 x 16 tile: row c / 16, point c % 16
    auto load_stage = [&](int step) {
        cd *As = ring + (step % kMStages) * kMStageElems, *Bs = As + 64 * kMPitch;
        const long long r = r_beg + (long long)step * kMK;
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            const int c = tid + 128 * i, row = c >> 4, e = c & 15;
            const bool in = r + e < r_end;
            const bool a_ok = in && m0 + row < g.n_a, b_ok = in && n0 + row < g.n_b;
            cp_async16(As + row * kMPitch + e, g.a + (a_ok ? (long long)(m0 + row) * g.n_pts + r + e : 0), a_ok);
            cp_async16(Bs + row * kMPitch + e, g.b + (b_ok ? (long long)(n0 + row) * g.n_pts + r + e : 0), b_ok);
        }
    };
    double re[4][4][2], im[4][4][2];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) { re[i][j][0] = re[i][j][1] = im[i][j][0] = im[i][j][1] = 0.0; }
#pragma unroll
    for (int s = 0; s < kMStages - 1; ++s) {
        if (s < n_steps) load_stage(s);
        cp_async_commit();
    }
    const int fr = lane >> 2, fk = lane & 3;              // fragment row (m or n within the 8 x 8 tile), real k index
    const bool odd = fk & 1;
    for (int step = 0; step < n_steps; ++step) {
        cp_async_wait<kMStages - 2>();
        __syncthreads();                                  // stage `step` landed for everyone; stage step - 1 is free
        if (step + kMStages - 1 < n_steps) load_stage(step + kMStages - 1);
        cp_async_commit();
        const cd *As = ring + (step % kMStages) * kMStageElems, *Bs = As + 64 * kMPitch;
        const double *Ad = reinterpret_cast<const double *>(As);
#pragma unroll
        for (int kk = 0; kk < kMK / 2; ++kk) {            // 2 points = 4 real k per DMMA
            double af[4], b1[4], b2[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) af[i] = Ad[(wm + 8 * i + fr) * (2 * kMPitch) + 4 * kk + fk];
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const cd z = Bs[(wn + 8 * j + fr) * kMPitch + 2 * kk + (fk >> 1)];
                b1[j] = odd ? z.y : z.x;
                b2[j] = odd ? -z.x : z.y;
            }
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    dmma884(re[i][j][0], re[i][j][1], af[i], b1[j]);
                    dmma884(im[i][j][0], im[i][j][1], af[i], b2[j]);
                }
        }
    }
    cd *out = g.part + (long long)blockIdx.z * g.n_a * g.ld;
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j)
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int m = m0 + wm + 8 * i + fr, n = n0 + wn + 8 * j + 2 * fk + h;
                if (m < g.n_a && n < g.n_b) out[(long long)m * g.ld + n] = make_double2(re[i][j][h], im[i][j][h]);
            }
}

// ---- rotation with the fused epilogues of rotate_kernel (dense.cuh): acc_n(r) = sum_m a_m(r) c(m, n) --------------------
// grid = (ceil(n_out / 64), ceil(n_pts / 64)): the column tiles of one point tile are neighbours in launch order, so
// the a tile they share is read from HBM once.  128 threads = 2 x 2 warps, warp tile 32 columns x 32 points.
// Real form: with c = (cr, ci), a = (ar, ai):  Re = sum cr ar - ci ai,  Im = sum ci ar + cr ai, i.e. the MMA "A" operand is
// (cr, -ci, ...) for the real and (ci, cr, ...) for the imaginary part (both from one 16-byte read of c), the "B"
// operand is the component (k parity) of a[m][r].  Tiles: Cs[64 n][16 m] (pitch 18; transposed on the way in, one
// 16-byte cp.async per element), As[16 m][64 r] (pitch 68: the two rows a fragment read touches sit in different banks).
constexpr int kRK = 16;                                   // orbitals m per stage
constexpr int kRPitchC = kRK + 2, kRPitchA = 64 + 4;
constexpr int kRStageElems = 64 * kRPitchC + kRK * kRPitchA;
constexpr int kRStages = 3;
constexpr int kRotateMmaSmem = kRStages * kRStageElems * (int)sizeof(cd);

__global__ void __launch_bounds__(128, 2) rotate_mma(const RotateArgs g) {
    extern __shared__ __align__(16) unsigned char dense_smem[];
    cd *ring = reinterpret_cast<cd *>(dense_smem);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int wn = (warp >> 1) * 32, wr = (warp & 1) * 32;
    const long long r0 = (long long)blockIdx.y * 64;
    const int n0 = g.n_first + blockIdx.x * 64, n_end = g.n_first + g.n_out;
    const int n_steps = (g.n_a + kRK - 1) / kRK;
    auto load_stage = [&](int step) {
        cd *Cs = ring + (step % kRStages) * kRStageElems, *As = Cs + 64 * kRPitchC;
        const int mb = step * kRK;
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            const int c = tid + 128 * i;
            {   // a tile: row m = c / 64, point c % 64 (coalesced 1 KB rows)
                const int m = c >> 6, e = c & 63;
                const bool ok = mb + m < g.n_a && r0 + e < g.n_pts;
                cp_async16(As + m * kRPitchA + e, g.a + (ok ? (long long)(mb + m) * g.n_pts + r0 + e : 0), ok);
            }
            if (g.conj_t) {     // c(m, n) = conj(S[n][m]): rows n, m contiguous
                const int n = c >> 4, m = c & 15;
                const bool ok = mb + m < g.n_a && n0 + n < n_end;
                cp_async16(Cs + n * kRPitchC + m, g.s + (ok ? (long long)(n0 + n) * g.ld + mb + m : 0), ok);
            } else {            // c(m, n) = S[m][n]: rows m, n contiguous -> transposed element by element
                const int m = c >> 6, n = c & 63;
                const bool ok = mb + m < g.n_a && n0 + n < n_end;
                cp_async16(Cs + n * kRPitchC + m, g.s + (ok ? (long long)(mb + m) * g.ld + n0 + n : 0), ok);
            }
        }
    };
    double re[4][4][2], im[4][4][2];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) { re[i][j][0] = re[i][j][1] = im[i][j][0] = im[i][j][1] = 0.0; }
#pragma unroll
    for (int s = 0; s < kRStages - 1; ++s) {
        if (s < n_steps) load_stage(s);
        cp_async_commit();
    }
    const int fr = lane >> 2, fk = lane & 3;
    const bool odd = fk & 1;
    const double sgn = g.conj_t ? -1.0 : 1.0;             // conj(S): ci -> -ci
    for (int step = 0; step < n_steps; ++step) {
        cp_async_wait<kRStages - 2>();
        __syncthreads();
        if (step + kRStages - 1 < n_steps) load_stage(step + kRStages - 1);
        cp_async_commit();
        const cd *Cs = ring + (step % kRStages) * kRStageElems, *As = Cs + 64 * kRPitchC;
        const double *Ad = reinterpret_cast<const double *>(As);
#pragma unroll
        for (int kk = 0; kk < kRK / 2; ++kk) {
            double a1[4], a2[4], bf[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const cd z = Cs[(wn + 8 * i + fr) * kRPitchC + 2 * kk + (fk >> 1)];
                const double ci = sgn * z.y;
                a1[i] = odd ? -ci : z.x;
                a2[i] = odd ? z.x : ci;
            }
#pragma unroll
            for (int j = 0; j < 4; ++j) bf[j] = Ad[((2 * kk + (fk >> 1)) * kRPitchA + wr + 8 * j + fr) * 2 + (fk & 1)];
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    dmma884(re[i][j][0], re[i][j][1], a1[i], bf[j]);
                    dmma884(im[i][j][0], im[i][j][1], a2[i], bf[j]);
                }
        }
    }
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j)
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int n = n0 + wn + 8 * i + fr;
                const long long r = r0 + wr + 8 * j + 2 * fk + h;
                if (n >= n_end || r >= g.n_pts) continue;
                const long long k = (long long)n * g.n_pts + r;
                cd v = make_double2(re[i][j][h], im[i][j][h]);
                if (g.mode == 1) {
                    v = csub(g.h[k], v);
                } else if (g.mode == 2) {
                    const cd d = csub(g.h[k], v), pv = g.p[k], qv = g.q[k];
                    v = make_double2(pv.x + g.fx * d.x - g.fy * d.y - qv.x, pv.y + g.fx * d.y + g.fy * d.x - qv.y);
                } else if (g.mode == 3) {
                    v = csub(g.out[k], v);
                }
                g.out[k] = v;
            }
}

}  // namespace ptfock
