// dense.cuh -- the dense-algebra neighbours of the Fock exchange path on one GPU:
// overlap matrices, rotations, the PT-CN residuals, the density, Cholesky + triangular solve orthonormalisation
// (Sec. 3.3 Alg. 3; Sec. 3.4).  The paper calls cuBLAS / cuSOLVER for these; here they
// are hand-written fp64 kernels, all deterministic (split-K partial sums are added in a fixed order, no atomics).
// This file: argument structs, reductions, the density, the blocked Cholesky and the triangular-solve blocks (plain
// FP64 pipe); the two big contractions (overlap, rotation) run on the FP64 tensor cores: dense_mma.cuh.
//
// Orbitals are [orbital][grid point] complex fp64, the inner product is (a, b) = w sum_r conj(a(r)) b(r), w = Omega/N.
#pragma once
#include "codelets.cuh"

namespace ptfock {

constexpr int kDT = 64;         // output tile edge of the GEMM-like kernels
constexpr int kDK = 16;         // contraction step staged through shared memory
constexpr int kDP = kDK + 1;    // pitch of a [64][16] tile (elements)

// ---- overlap: part[ks][m][n] = sum over this split's points of conj(a[m][r]) b[n][r]   (kernel: overlap_mma) ----------
struct OverlapArgs {
    const cd *a, *b;
    cd *part;               // [k_splits][n_a][ld]
    long long n_pts, pts_per_split;
    int n_a, n_b, ld;       // ld = row pitch of part / S (>= n_b)
    int lower;              // 1: a == b (Hermitian product): gridDim.x counts the 64 x 64 tiles tm >= tn only, the tiles above
                            //    the diagonal are never computed (overlap_reduce mirrors them)
};

// s[m][n] = w * sum_ks part[ks][m][n] (fixed order); herm: entries of the tiles above the diagonal are the conjugates of
// their mirror images (those tiles hold no partial sums)
__global__ void __launch_bounds__(256) overlap_reduce(const cd *part, int k_splits, int n_a, int n_b, int ld_part, double w,
                                                      cd *s, int ld_s, int herm) {
    const long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= (long long)n_a * n_b) return;
    const int m = (int)(k / n_b), n = (int)(k % n_b);
    const bool mirror = herm && (m >> 6) < (n >> 6);
    const int row = mirror ? n : m, col = mirror ? m : n;
    cd t = part[(long long)row * ld_part + col];
    for (int q = 1; q < k_splits; ++q) {
        const cd u = part[((long long)q * n_a + row) * ld_part + col];
        t.x += u.x; t.y += u.y;
    }
    s[(long long)m * ld_s + n] = make_double2(t.x * w, mirror ? -t.y * w : t.y * w);
}

// ---- rotation with fused epilogues: acc_n(r) = sum_m a_m(r) c(m, n) ---------------------------------------------------
// c(m, n) = S[m*ld + n]  or, for the triangular solve, conj(S[n*ld + m]);
// mode 0: out = acc                      (Alg. 3 line 4, Psi_temp = Psi_f S)
// mode 1: out = h - acc                  (Alg. 1 line 1, R_n = H Psi - Psi S)
// mode 2: out = p + f (h - acc) - q      (Alg. 3 line 5, R_f; f = i dt / 2)
// mode 3: out = out - acc                (blocked triangular solve: block column minus the finished columns' part)
// (kernel: rotate_mma)
struct RotateArgs {
    const cd *a;            // [n_a][n_pts]
    const cd *s;            // coefficients
    const cd *h, *p, *q;    // epilogue operands, [n_out][n_pts]
    cd *out;                // [n_out][n_pts]
    long long n_pts;
    int n_a, n_out, ld, conj_t, mode;
    int n_first;            // first output column (offset into h, p, q, out and into S's column index)
    double fx, fy;          // f
};

// ---- density: part[s][r] = sum over this split's orbitals of |psi_i(r)|^2; rho = sum_s part (fixed order) -----------------
__global__ void __launch_bounds__(256) density_partial(const cd *psi, long long n_pts, int n, int per_split, double *part) {
    const long long r = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= n_pts) return;
    const int i_beg = blockIdx.y * per_split, i_end = min(n, i_beg + per_split);
    double s = 0.0;
    for (int i = i_beg; i < i_end; ++i) {
        const cd z = psi[(long long)i * n_pts + r];
        s = fma(z.x, z.x, fma(z.y, z.y, s));
    }
    part[(long long)blockIdx.y * n_pts + r] = s;
}
__global__ void __launch_bounds__(256) density_reduce(const double *part, long long n_pts, int splits, double *rho) {
    const long long r = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= n_pts) return;
    double s = part[r];
    for (int q = 1; q < splits; ++q) s += part[(long long)q * n_pts + r];
    rho[r] = s;
}

// ---- blocked Cholesky of S (np x np, np a multiple of 64, row major, lower triangle) -----------------------------------
// panel k: chol_diag factors the 64 x 64 diagonal block in shared memory; tri_solve_block solves the rows below against
// it (L21 = A21 L11^{-H}); chol_update subtracts L21 L21^H from the trailing lower triangle.
constexpr int kBlkSmem = 64 * 65 * (int)sizeof(cd);       // one padded 64 x 64 block (dynamic shared memory)

// diag0[k] = S[k][k] before the factorisation: the scale a pivot is judged against
__global__ void __launch_bounds__(256) save_diag(const cd *s, int ld, int np, double *diag0) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k < np) diag0[k] = s[(long long)k * ld + k].x;
}

// a pivot below 1e-12 of the column's original diagonal means a numerically dependent column: flagged in *info
__global__ void __launch_bounds__(64) chol_diag(cd *s, int ld, int k0, const double *diag0, int *info) {
    extern __shared__ __align__(16) unsigned char dense_smem[];
    cd *L = reinterpret_cast<cd *>(dense_smem);
    const int t = threadIdx.x;                            // row
    for (int c = 0; c < 64; ++c) L[t * 65 + c] = s[(long long)(k0 + t) * ld + k0 + c];
    __syncthreads();
    for (int c = 0; c < 64; ++c) {
        // column c: d = sqrt(L[c][c] - sum_{k<c} |L[c][k]|^2); rows t > c: (L[t][c] - sum_k L[t][k] conj(L[c][k])) / d
        cd v = L[t * 65 + c];
        for (int k = 0; k < c; ++k) {
            const cd x = L[t * 65 + k], y = L[c * 65 + k];
            v.x -= x.x * y.x + x.y * y.y;
            v.y -= x.y * y.x - x.x * y.y;
        }
        __syncthreads();
        if (t == c) {
            if (!(v.x > 1e-12 * diag0[k0 + c])) { atomicCAS(info, 0, k0 + c + 1); v.x = 1.0; }
            L[c * 65 + c] = make_double2(sqrt(v.x), 0.0);
        }
        __syncthreads();
        if (t > c) {
            const double d = 1.0 / L[c * 65 + c].x;
            L[t * 65 + c] = make_double2(v.x * d, v.y * d);
        } else if (t < c) {
            L[t * 65 + c] = make_double2(0.0, 0.0);
        }
        __syncthreads();
    }
    for (int c = 0; c < 64; ++c) s[(long long)(k0 + t) * ld + k0 + c] = L[t * 65 + c];
}

// trailing update: tile (bi >= bj) of A22 -= L21(bi) L21(bj)^H, K = 64.  grid.x = lower-triangular tile index.
__global__ void __launch_bounds__(256) chol_update(cd *s, int ld, int k0, int np) {
    __shared__ cd Ri[kDT * kDP], Rj[kDT * kDP];
    int bi = 0, idx = blockIdx.x;
    while (idx > bi) { idx -= bi + 1; ++bi; }             // blockIdx.x = bi (bi + 1) / 2 + bj
    const int bj = idx;
    const int tid = threadIdx.x, tx = tid & 15, ty = tid >> 4;
    const int i0 = k0 + 64 + bi * 64, j0 = k0 + 64 + bj * 64;
    const int lrow = tid >> 2, lk = (tid & 3) * 4;
    cd acc[4][4];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = make_double2(0.0, 0.0);
    for (int kc = 0; kc < 64; kc += kDK) {
        __syncthreads();
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            Ri[lrow * kDP + lk + q] = s[(long long)(i0 + lrow) * ld + k0 + kc + lk + q];
            Rj[lrow * kDP + lk + q] = s[(long long)(j0 + lrow) * ld + k0 + kc + lk + q];
        }
        __syncthreads();
#pragma unroll
        for (int kk = 0; kk < kDK; ++kk) {
            cd x[4], y[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) x[i] = Ri[(ty + 16 * i) * kDP + kk];
#pragma unroll
            for (int j = 0; j < 4; ++j) y[j] = Rj[(tx + 16 * j) * kDP + kk];
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) {           // acc += x conj(y)
                    acc[i][j].x = fma(x[i].x, y[j].x, fma(x[i].y, y[j].y, acc[i][j].x));
                    acc[i][j].y = fma(x[i].y, y[j].x, fma(-x[i].x, y[j].y, acc[i][j].y));
                }
        }
    }
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int r = i0 + ty + 16 * i, c = j0 + tx + 16 * j;
            if (c > r) continue;
            cd *p = s + (long long)r * ld + c;
            *p = csub(*p, acc[i][j]);
        }
}

// identity on the padding (rows / columns n .. np - 1) so that the padded matrix factors as blockdiag(L, I)
__global__ void __launch_bounds__(256) pad_identity(cd *s, int ld, int n, int np) {
    const long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= (long long)np * np) return;
    const int r = (int)(k / np), c = (int)(k % np);
    if (r >= n || c >= n) s[(long long)r * ld + c] = make_double2(r == c ? 1.0 : 0.0, 0.0);
}

// ---- triangular solve against one 64 x 64 diagonal block: X L^H = Y in place, one thread per vector --------------------
// vector v, column c lives at x[v * v_stride + c * c_stride]: orbitals (v = grid point: v_stride 1, c_stride n_pts) for
// Psi <- Psi L^{-H} ("Trsm"), rows of S (v = row: v_stride ld, c_stride 1) for the Cholesky panel
// L21 = A21 L11^{-H}.  16 columns at a time in registers: x_c = (y_c - sum_{k<c} x_k conj(L[c][k])) / L[c][c].
__global__ void __launch_bounds__(128) tri_solve_block(cd *x, long long n_vec, long long v_stride, long long c_stride,
                                                       const cd *l, int ld, int c0, int nc) {
    extern __shared__ __align__(16) unsigned char dense_smem[];
    cd *L = reinterpret_cast<cd *>(dense_smem);
    for (int e = threadIdx.x; e < 64 * 64; e += blockDim.x) {
        const int rr = e >> 6, c = e & 63;
        L[rr * 65 + c] = (rr < nc && c < nc) ? l[(long long)(c0 + rr) * ld + c0 + c] : make_double2(rr == c ? 1.0 : 0.0, 0.0);
    }
    __syncthreads();
    const long long v = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (v >= n_vec) return;
    cd *xv = x + v * v_stride;
    for (int sb = 0; sb < nc; sb += 16) {
        cd t[16];
#pragma unroll
        for (int c = 0; c < 16; ++c) t[c] = (sb + c < nc) ? xv[(long long)(sb + c) * c_stride] : make_double2(0.0, 0.0);
        for (int m = 0; m < sb; ++m) {                    // this block's finished columns (read back: final values)
            const cd xm = xv[(long long)m * c_stride];
#pragma unroll
            for (int c = 0; c < 16; ++c) {
                const cd y = L[(sb + c) * 65 + m];
                t[c].x -= xm.x * y.x + xm.y * y.y;
                t[c].y -= xm.y * y.x - xm.x * y.y;
            }
        }
#pragma unroll
        for (int c = 0; c < 16; ++c) {
            cd u = t[c];
#pragma unroll
            for (int k = 0; k < c; ++k) {
                const cd y = L[(sb + c) * 65 + sb + k];
                u.x -= t[k].x * y.x + t[k].y * y.y;
                u.y -= t[k].y * y.x - t[k].x * y.y;
            }
            const double d = 1.0 / L[(sb + c) * 65 + sb + c].x;
            t[c] = make_double2(u.x * d, u.y * d);
        }
#pragma unroll
        for (int c = 0; c < 16; ++c)
            if (sb + c < nc) xv[(long long)(sb + c) * c_stride] = t[c];
    }
}

}  // namespace ptfock
