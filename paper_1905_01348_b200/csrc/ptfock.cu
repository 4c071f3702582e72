// ptfock.cu -- host side of libptfock.so: the C ABI of include/ptfock.h, plan construction
// (v' table, twiddles, scratch) and the pair scheduler (Alg. 2 loops i x j, batched as in
// PAPER.md:149 "Batched implementation"; i <= j pair symmetry when Psi = Phi).
#include "../../include/ptfock.h"
#include "kernels.cuh"
#include "slabx.cuh"
#include "pencil_tma.cuh"
#include "pass8.cuh"
#include "onchip16.cuh"
#include "dense.cuh"
#include "dense_mma.cuh"

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <initializer_list>
#include <mutex>
#include <new>
#include <vector>

using namespace ptfock;

namespace {

thread_local int g_last_cuda = 0;

#define CU(call)                                              \
    do {                                                      \
        cudaError_t e__ = (call);                             \
        if (e__ != cudaSuccess) {                             \
            g_last_cuda = (int)e__;                           \
            return PTFOCK_ERR_CUDA;                           \
        }                                                     \
    } while (0)

// makes `device` current for the duration of a call and restores the caller's device afterwards
struct DeviceGuard {
    int prev;
    cudaError_t err;
    explicit DeviceGuard(int device) : prev(-1), err(cudaSuccess) {
        err = cudaGetDevice(&prev);
        if (err == cudaSuccess && prev != device) err = cudaSetDevice(device);
        else if (err == cudaSuccess) prev = -1;
    }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};
#define GUARD(dev) DeviceGuard guard__(dev); CU(guard__.err)

typedef void (*slab_launch_fn)(const SlabArgs &, dim3, cudaStream_t);
typedef void (*pencil_launch_fn)(const PencilArgs &, int pairs, cudaStream_t);

template <int N1, int N2> void launch_slab_fwd(const SlabArgs &a, dim3 grid, cudaStream_t st) {
    slab_fwd<N1, N2><<<grid, kSlabThreads, SlabShape<N1, N2>::SMEM_BYTES, st>>>(a);
}
template <int N1, int N2> void launch_slab_inv(const SlabArgs &a, dim3 grid, cudaStream_t st) {
    slab_inv_acc<N1, N2><<<grid, kSlabThreads, SlabShape<N1, N2>::SMEM_BYTES, st>>>(a);
}
template <int N0> void launch_pencil(const PencilArgs &a, int pairs, cudaStream_t st) {
    using S = PencilShape<N0>;
    const int gx = (S::R2 == 1) ? (a.slab_pts + S::NT - 1) / S::NT : (a.slab_pts + S::CW - 1) / S::CW;
    pencil_mid<N0><<<dim3(gx, pairs), S::NT, S::SMEM_BYTES, st>>>(a);
}

struct SlabEntry {
    int n1, n2;
    slab_launch_fn fwd, inv;
    cudaError_t (*prepare)();
    int ax1_r1, ax1_r2, ax2_r1, ax2_r2;     // digit split per axis: position k1*r2 + k2 holds frequency k1 + r1*k2
    int nt3;                                // 0: scratch slab is [pos1][pos2]; else slabx's free layout
                                            //    s = m*nt3 + k2a*n1 + k1  (k1 natural), k2 = k2a + ax2_r1*m
};

template <int N1, int N2> cudaError_t prepare_slab() {
    cudaError_t e = cudaFuncSetAttribute(slab_fwd<N1, N2>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         SlabShape<N1, N2>::SMEM_BYTES);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(slab_inv_acc<N1, N2>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                SlabShape<N1, N2>::SMEM_BYTES);
}

// TMA-fed in-place kernels (slabx.cuh)
template <class S> void launch_slabx_fwd(const SlabArgs &a, dim3 grid, cudaStream_t st) {
    slabx_fwd<S><<<grid, S::NT, S::SMEM_A, st>>>(a);
}
template <class S> void launch_slabx_inv(const SlabArgs &a, dim3 grid, cudaStream_t st) {
    slabx_inv_acc<S><<<grid, S::NT, S::SMEM_C, st>>>(a);
}
template <class S> cudaError_t prepare_slabx() {
    cudaError_t e = cudaFuncSetAttribute(slabx_fwd<S>, cudaFuncAttributeMaxDynamicSharedMemorySize, S::SMEM_A);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(slabx_inv_acc<S>, cudaFuncAttributeMaxDynamicSharedMemorySize, S::SMEM_C);
}
//          N1   N2  A1  B1  A2  B2  kind Q  bulk stores  CTAs/SM
typedef SX<64, 64, 16, 4, 4, 16, false, true> SX_64x64;
typedef SX<128, 48, 8, 16, 3, 16, true, false> SX_128x48;     // kind Q: 256 threads, 24-point first stage
typedef SX<48, 48, 3, 16, 3, 16, true, false, 2> SX_48x48;    // kind Q: 9-point first stage, 144-task DFT16 stages; 36 KB tiles, 128 registers
typedef SX<32, 32, 2, 16, 2, 16, true, false, 2> SX_32x32;
typedef SX<90, 60, 6, 15, 4, 15, true, false> SX_90x60;        // paper grid 120 x 90 x 60: 24-point first stage, DFT15 stages
#define SLABX(S) { S::N1, S::N2, launch_slabx_fwd<S>, launch_slabx_inv<S>, prepare_slabx<S>, S::A1, S::B1, S::A2, S::B2, S::TS ? 0 : S::NT3 }
#define SLAB(N1, N2) { N1, N2, launch_slab_fwd<N1, N2>, launch_slab_inv<N1, N2>, prepare_slab<N1, N2>, \
                       Split<N1>::R1, Split<N1>::R2, Split<N2>::R1, Split<N2>::R2, 0 }
// the TMA-fed 3-stage kernels serve the BASELINE slab shapes, the generic 4-stage ones the small / mixed ones
const SlabEntry kSlabs[] = {
    SLABX(SX_64x64), SLABX(SX_128x48), SLABX(SX_48x48), SLABX(SX_32x32), SLABX(SX_90x60),
    SLAB(16, 16), SLAB(16, 32), SLAB(32, 16), SLAB(16, 48), SLAB(48, 32), SLAB(32, 64),
    // the rest of {16, 32, 48, 64, 128}^2 (north_star (1): "grid edges 16/32/48/64/128") on the generic passes; only the
    // 128 x 128 slab is missing: 256 KB of complex fp64 do not fit one CTA's shared memory
    SLAB(16, 64), SLAB(16, 128), SLAB(32, 48), SLAB(32, 128), SLAB(48, 16), SLAB(48, 64), SLAB(48, 128),
    SLAB(64, 16), SLAB(64, 32), SLAB(64, 48), SLAB(64, 128), SLAB(128, 16), SLAB(128, 32), SLAB(128, 64),
};
#undef SLAB
#undef SLABX

typedef void (*pencil_tma_launch_fn)(const CUtensorMap &, const PencilTmaArgs &, int pairs, cudaStream_t);
struct PencilEntry {
    int n0;
    pencil_launch_fn run;
    cudaError_t (*prepare)();
    pencil_tma_launch_fn run_tma;       // tensor-map TMA variant (pencil_tma.cuh); null for single-stage pencils
    cudaError_t (*prepare_tma)();
    int tma_cw;
};
template <int N0> void launch_pencil_tma(const CUtensorMap &m, const PencilTmaArgs &a, int pairs, cudaStream_t st) {
    using S = PencilTma<N0>;
    pencil_tma<N0><<<dim3((a.slab_pts + S::CW - 1) / S::CW, pairs), S::NT, S::SMEM_BYTES, st>>>(m, a);
}
template <int N0> cudaError_t prepare_pencil_tma() {
    return cudaFuncSetAttribute(pencil_tma<N0>, cudaFuncAttributeMaxDynamicSharedMemorySize, PencilTma<N0>::SMEM_BYTES);
}
template <int N0> cudaError_t prepare_pencil() {
    if (PencilShape<N0>::SMEM_BYTES <= 48 * 1024) return cudaSuccess;
    return cudaFuncSetAttribute(pencil_mid<N0>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                PencilShape<N0>::SMEM_BYTES);
}
#define PENCIL(N0) { N0, nullptr, nullptr, launch_pencil_tma<N0>, prepare_pencil_tma<N0>, PencilTma<N0>::CW }
#define PENCIL_REG(N0) { N0, launch_pencil<N0>, prepare_pencil<N0>, nullptr, nullptr, 0 }
// the tensor-map variant serves the long pencils; at n0 <= 48 its 16-wide tiles leave most threads idle (measured slower)
const PencilEntry kPencils[] = { PENCIL_REG(16), PENCIL_REG(32), PENCIL_REG(48), PENCIL(64), PENCIL(128), PENCIL(120) };
#undef PENCIL_REG
#undef PENCIL

// ---- 8 + 10 + 8 bit split (pass8.cuh) ---------------------------------------------------------------------------
struct P8Entry {
    int n0, n1, n2, a0, a1, a2;                 // k0 = k0a + a0*k0b, k1 = k1a + a1*k1b, k2 = k2a + a2*k2b
    int nq, rq, p, rows, qpts, npos, ntb2, b0;    // ntb2 = middle-stage tasks of a pass B tile, b0 = their points
    void (*fwd)(const SlabArgs &, dim3, cudaStream_t);
    void (*inv)(const SlabArgs &, dim3, cudaStream_t);
    void (*mid)(const CUtensorMap &, const P8MidArgs &, int pairs, cudaStream_t);
    cudaError_t (*prepare)();
};
template <class S> void launch_p8_fwd(const SlabArgs &a, dim3 grid, cudaStream_t st) { p8_fwd<S><<<grid, S::NT, S::SMEM_A, st>>>(a); }
template <class S> void launch_p8_inv(const SlabArgs &a, dim3 grid, cudaStream_t st) { p8_inv_acc<S><<<grid, S::NT, S::SMEM_C, st>>>(a); }
template <class S> void launch_p8_mid(const CUtensorMap &m, const P8MidArgs &a, int pairs, cudaStream_t st) {
    p8_mid<S><<<dim3(S::NGRP, (pairs + S::GB - 1) / S::GB), S::NTB * S::GB, S::SMEM_B, st>>>(m, a);
}
template <class S> cudaError_t prepare_p8() {
    cudaError_t e = cudaFuncSetAttribute(p8_fwd<S>, cudaFuncAttributeMaxDynamicSharedMemorySize, S::SMEM_A);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(p8_inv_acc<S>, cudaFuncAttributeMaxDynamicSharedMemorySize, S::SMEM_C);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(p8_mid<S>, cudaFuncAttributeMaxDynamicSharedMemorySize, S::SMEM_B);
    // several small CTAs per SM: ask for the largest shared-memory carve-out
    if (e == cudaSuccess) e = cudaFuncSetAttribute(p8_fwd<S>, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(p8_inv_acc<S>, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(p8_mid<S>, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
    return e;
}
//         N0  N1  N2  A1 A2 A0  regs A / C  ring C
typedef P8<64, 64, 64, 4, 4, 2> P8_64;                     // 16-point stages: 64 threads, 6 / 4 CTAs per SM
typedef P8<32, 32, 32, 4, 2, 2, 128, 200, 3> P8_32;        // 8-point first stage (4 x 2): 64 threads; pass B 2 x 8 | 16
typedef P8<48, 48, 48, 3, 3, 2, 152, 232, 3> P8_48;        // 9-point first stage (3 x 3), DFT16; pass B 2 x 16 | DFT24 (x0 = 24 a0 + b0)
// (48^3 as P8<48, 48, 48, 6, 3, 3>, 18-point first stages at 224 / 255 registers and 12 KB pass B tiles, measured slower
//  than the three-stage kernels: Si216 315 vs 246 ms, profiles/r02_rejected_variants.md #17)
#define P8E(S) { S::N0, S::N1, S::N2, S::A0, S::A1, S::A2, S::NQ, S::RQ, S::P, S::ROWS, S::QPTS, S::NPOS, S::NTB2, S::B0, \
                 launch_p8_fwd<S>, launch_p8_inv<S>, launch_p8_mid<S>, prepare_p8<S> }
const P8Entry kP8[] = { P8E(P8_64), P8E(P8_48), P8E(P8_32) };
#undef P8E

// position -> frequency index of the digit-permuted order the forward passes leave an axis in
int freq_of_pos(int r1, int r2, int pos) {
    const int k1 = pos / r2, k2 = pos % r2;
    return k1 + r1 * k2;
}
void pencil_split(int n, int &r1, int &r2) {
    switch (n) {
        case 16: r1 = Split<16>::R1; r2 = Split<16>::R2; break;
        case 32: r1 = Split<32>::R1; r2 = Split<32>::R2; break;
        case 48: r1 = Split<48>::R1; r2 = Split<48>::R2; break;
        case 64: r1 = Split<64>::R1; r2 = Split<64>::R2; break;
        case 120: r1 = Split<120>::R1; r2 = Split<120>::R2; break;
        default: r1 = Split<128>::R1; r2 = Split<128>::R2; break;
    }
}

double det3(const double *a) {
    return a[0] * (a[4] * a[8] - a[5] * a[7]) - a[1] * (a[3] * a[8] - a[5] * a[6]) + a[2] * (a[3] * a[7] - a[4] * a[6]);
}

__global__ void fill_ones(cd *p, long long n) {
    long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (k < n) p[k] = make_double2(1.0, 0.0);
}

}  // namespace

struct ptfock_plan {
    ptfock_desc d;
    long long N;
    int slab_pts;
    double volume;
    double *v_dev;
    cd *tw_dev[3];
    cd *scratch;
    size_t scratch_bytes;
    int Ib, Jb;
    // two waves in flight (general schedule): the scratch holds `slots` waves of Ib * Jb pair densities; waves of
    // j-blocks with an odd index run on aux_stream in the second slot, so one wave's passes fill the SMs while the
    // other wave's kernel drains (the tail of a launch is one CTA lifetime long, ~20 % of pass A)
    int slots;
    cudaStream_t aux_stream;
    cudaEvent_t fork_ev, join_ev;
    bool v_even;
    const SlabEntry *slab;
    const PencilEntry *pencil;
    // exchange energy
    double2 *partials, *result_dev, *result_host;
    cd *energy_buf;
    // host path staging
    cd *st_phi, *st_psi, *st_out;
    cudaStream_t copy_stream;           // host path: copies run here, chunk by chunk, overlapped with the waves
    std::vector<cudaEvent_t> *copy_ev;
    int sm_count;
    cd *ones;                           // ptfock_debug_pair: a grid of ones (lazily allocated)
    int *chol_info;                     // ptfock_orthonormalize: first non-positive pivot (device), and its pinned host copy
    int *chol_info_host;
    // cross-stream ordering: the plan's scratch is shared by consecutive calls, so a call on another stream first
    // waits for the event the previous call recorded at its end
    cudaEvent_t busy_ev;
    cudaStream_t last_stream;
    int has_last;
    // statistics
    long long last_launches, last_pairs, total_launches;
    int last_symmetric;
    CUtensorMap tmap;                   // pair scratch as [pairs*n0 rows][2*slab_pts doubles] (pass B, TMA variant)
    int use_tma;
    // 8 + 10 + 8 bit split (pass8.cuh): own tensor map (128-byte swizzle) and v' table in pass B's register order
    const struct P8Entry *p8;
    CUtensorMap tmap8;
    double2 *v8_dev;
    int onchip;                         // 16^3: single-pass on-chip kernel (onchip16.cuh); v_dev then holds v'[k2][k0][k1]
    // optional per-pass device timing (ptfock_set_profiling): events bracket every launch
    int profiling;
    std::vector<cudaEvent_t> *ev_pool;
    size_t ev_used;
    std::vector<int> *ev_tags;         // tag of the interval that ENDS at event k (0/1/2 = pass A/B/C, -1 = none)
};

// ================================================================================================
// plan
// ================================================================================================
namespace {

const int kEdges[] = { 16, 32, 48, 64, 128, 60, 90, 120 };     // 60/90/120: only as the paper grid's roles (slab 90x60, pencil 120)
bool edge_ok(int n) {
    for (int e : kEdges) if (e == n) return true;
    return false;
}

void free_plan(ptfock_plan *p) {
    if (!p) return;
    cudaFree(p->v_dev);
    cudaFree(p->v8_dev);
    for (int d = 0; d < 3; ++d) cudaFree(p->tw_dev[d]);
    cudaFree(p->scratch);
    cudaFree(p->partials);
    cudaFree(p->result_dev);
    if (p->result_host) cudaFreeHost(p->result_host);
    cudaFree(p->energy_buf);
    cudaFree(p->st_phi);
    cudaFree(p->st_psi);
    cudaFree(p->st_out);
    cudaFree(p->ones);
    cudaFree(p->chol_info);
    if (p->chol_info_host) cudaFreeHost(p->chol_info_host);
    if (p->busy_ev) cudaEventDestroy(p->busy_ev);
    if (p->fork_ev) cudaEventDestroy(p->fork_ev);
    if (p->join_ev) cudaEventDestroy(p->join_ev);
    if (p->aux_stream) cudaStreamDestroy(p->aux_stream);
    if (p->ev_pool) { for (cudaEvent_t e : *p->ev_pool) cudaEventDestroy(e); delete p->ev_pool; }
    if (p->copy_ev) { for (cudaEvent_t e : *p->copy_ev) cudaEventDestroy(e); delete p->copy_ev; }
    if (p->copy_stream) cudaStreamDestroy(p->copy_stream);
    delete p->ev_tags;
    delete p;
}

// v'(pos0, pos1, pos2) = -alpha/N * v(|G|^2) in the permuted order; also reports whether v(-G) = v(G)
// holds on the grid (needed by the pair-symmetric schedule; fails for skew cells at Nyquist planes).
int build_vtable(const ptfock_desc &d, const SlabEntry &se, const P8Entry *p8, bool onchip, std::vector<double> &vperm, bool &even) {
    const int n0 = d.n[0], n1 = d.n[1], n2 = d.n[2];
    const long long N = (long long)n0 * n1 * n2;
    const double *a = d.cell;
    const double vol = det3(a);
    if (vol == 0.0 || !std::isfinite(vol)) return PTFOCK_ERR_INVALID_ARG;
    const double two_pi = 6.283185307179586476925286766559;
    const double f = two_pi / vol;
    // reciprocal rows b_d = 2 pi (a_e x a_f) / vol
    double b[9];
    b[0] = f * (a[4] * a[8] - a[5] * a[7]); b[1] = f * (a[5] * a[6] - a[3] * a[8]); b[2] = f * (a[3] * a[7] - a[4] * a[6]);
    b[3] = f * (a[7] * a[2] - a[8] * a[1]); b[4] = f * (a[8] * a[0] - a[6] * a[2]); b[5] = f * (a[6] * a[1] - a[7] * a[0]);
    b[6] = f * (a[1] * a[5] - a[2] * a[4]); b[7] = f * (a[2] * a[3] - a[0] * a[5]); b[8] = f * (a[0] * a[4] - a[1] * a[3]);
    std::vector<double> vnat((size_t)N);
    const double four_pi = 2.0 * two_pi;
    const double inv4w2 = (d.kernel == PTFOCK_KERNEL_HSE) ? 1.0 / (4.0 * d.omega * d.omega) : 0.0;
    for (int k0 = 0; k0 < n0; ++k0) {
        const int m0 = (k0 < n0 / 2) ? k0 : k0 - n0;
        for (int k1 = 0; k1 < n1; ++k1) {
            const int m1 = (k1 < n1 / 2) ? k1 : k1 - n1;
            for (int k2 = 0; k2 < n2; ++k2) {
                const int m2 = (k2 < n2 / 2) ? k2 : k2 - n2;
                const double gx = m0 * b[0] + m1 * b[3] + m2 * b[6];
                const double gy = m0 * b[1] + m1 * b[4] + m2 * b[7];
                const double gz = m0 * b[2] + m1 * b[5] + m2 * b[8];
                const double g2 = gx * gx + gy * gy + gz * gz;
                double val;
                if ((m0 | m1 | m2) == 0)
                    val = (d.kernel == PTFOCK_KERNEL_HSE) ? 0.5 * two_pi / (d.omega * d.omega) : 0.0;
                else if (d.kernel == PTFOCK_KERNEL_KINETIC)
                    val = 0.5 * g2;
                else if (d.kernel == PTFOCK_KERNEL_HSE)
                    val = four_pi / g2 * (-std::expm1(-g2 * inv4w2));
                else
                    val = four_pi / g2;
                vnat[((size_t)k0 * n1 + k1) * n2 + k2] = val;
            }
        }
    }
    even = true;
    for (int k0 = 0; k0 < n0 && even; ++k0)
        for (int k1 = 0; k1 < n1 && even; ++k1)
            for (int k2 = 0; k2 < n2; ++k2) {
                const double x = vnat[((size_t)k0 * n1 + k1) * n2 + k2];
                const double y = vnat[((size_t)((n0 - k0) % n0) * n1 + (n1 - k1) % n1) * n2 + (n2 - k2) % n2];
                if (std::fabs(x - y) > 1e-14 * (std::fabs(x) + std::fabs(y))) { even = false; break; }
            }
    // exchange kernels: -alpha/N folded in; the kinetic 'kernel' of the model Hamiltonian (ptfock_hloc_apply): +1/N
    const double scale = (d.kernel == PTFOCK_KERNEL_KINETIC ? 1.0 : -d.alpha) / (double)N;
    vperm.resize((size_t)N);
    if (onchip) {
        // onchip16.cuh: natural frequency order, stored [k2][k0][k1]
        for (int k0 = 0; k0 < n0; ++k0)
            for (int k1 = 0; k1 < n1; ++k1)
                for (int k2 = 0; k2 < n2; ++k2)
                    vperm[((size_t)k2 * n0 + k0) * n1 + k1] = scale * vnat[((size_t)k0 * n1 + k1) * n2 + k2];
        return PTFOCK_OK;
    }
    if (p8) {
        // pass8.cuh order: [tile group][m < b0 / 2][middle-stage task t < ntb2] pairs (k0b = 2m, 2m + 1), where
        // t = ((k0a*nq + q)*p + pp)*rq + r, k1b = q*rq + r, slab position = group*p + pp = (k2b*a1 + k1a)*a2 + k2a
        const int ngrp = p8->npos / p8->p, hm = p8->b0 / 2;
        for (int grp = 0; grp < ngrp; ++grp)
            for (int m = 0; m < hm; ++m)
                for (int t = 0; t < p8->ntb2; ++t) {
                    const int r = t % p8->rq, pp = (t / p8->rq) % p8->p, q = (t / (p8->rq * p8->p)) % p8->nq;
                    const int k0a = t / (p8->rq * p8->p * p8->nq);
                    const int pos = grp * p8->p + pp;
                    const int k2a = pos % p8->a2, k1a = (pos / p8->a2) % p8->a1, k2b = pos / (p8->a2 * p8->a1);
                    const int k1 = k1a + p8->a1 * (q * p8->rq + r), k2 = k2a + p8->a2 * k2b;
                    for (int h = 0; h < 2; ++h) {
                        const int k0 = k0a + p8->a0 * (2 * m + h);
                        vperm[(((size_t)grp * hm + m) * p8->ntb2 + t) * 2 + h] = scale * vnat[((size_t)k0 * n1 + k1) * n2 + k2];
                    }
                }
        return PTFOCK_OK;
    }
    int p_r1, p_r2;
    pencil_split(n0, p_r1, p_r2);
    for (int p0 = 0; p0 < n0; ++p0) {
        const int k0 = freq_of_pos(p_r1, p_r2, p0);
        for (int s = 0; s < n1 * n2; ++s) {
            int k1, k2;
            if (se.nt3) {
                const int m = s / se.nt3, t = s % se.nt3;
                k1 = t % n1;
                k2 = (t / n1) + se.ax2_r1 * m;
            } else {
                k1 = freq_of_pos(se.ax1_r1, se.ax1_r2, s / n2);
                k2 = freq_of_pos(se.ax2_r1, se.ax2_r2, s % n2);
            }
            vperm[(size_t)p0 * n1 * n2 + s] = scale * vnat[((size_t)k0 * n1 + k1) * n2 + k2];
        }
    }
    return PTFOCK_OK;
}

}  // namespace

extern "C" int ptfock_create(const ptfock_desc *desc, ptfock_plan **out) {
    if (!desc || !out) return PTFOCK_ERR_INVALID_ARG;
    const ptfock_desc &d = *desc;
    if (d.n_occ < 1 || d.max_targets < 1 || d.block_i < 0 || d.block_j < 0) return PTFOCK_ERR_INVALID_ARG;
    if (d.kernel != PTFOCK_KERNEL_COULOMB && d.kernel != PTFOCK_KERNEL_HSE && d.kernel != PTFOCK_KERNEL_KINETIC)
        return PTFOCK_ERR_INVALID_ARG;
    if (d.kernel == PTFOCK_KERNEL_KINETIC && d.n_occ != 1) return PTFOCK_ERR_INVALID_ARG;   // its one "orbital" is the constant 1
    if (d.kernel == PTFOCK_KERNEL_HSE && !(d.omega > 0.0)) return PTFOCK_ERR_INVALID_ARG;
    if (!std::isfinite(d.alpha)) return PTFOCK_ERR_INVALID_ARG;
    for (int k = 0; k < 3; ++k) if (!edge_ok(d.n[k])) return PTFOCK_ERR_UNSUPPORTED_GRID;
    const SlabEntry *slab = nullptr;
    for (const SlabEntry &e : kSlabs)
        if (!slab && e.n1 == d.n[1] && e.n2 == d.n[2]) slab = &e;
    const PencilEntry *pencil = nullptr;
    for (const PencilEntry &e : kPencils) if (e.n0 == d.n[0]) pencil = &e;
    if (!slab || !pencil) return PTFOCK_ERR_UNSUPPORTED_GRID;
    if (det3(d.cell) == 0.0) return PTFOCK_ERR_INVALID_ARG;
    const P8Entry *p8 = nullptr;
    if (!(d.flags & PTFOCK_FLAG_THREE_STAGE_SLABS))
        for (const P8Entry &e : kP8) if (e.n0 == d.n[0] && e.n1 == d.n[1] && e.n2 == d.n[2]) p8 = &e;

    int ndev = 0;
    CU(cudaGetDeviceCount(&ndev));
    if (d.device < 0 || d.device >= ndev) return PTFOCK_ERR_UNSUPPORTED_DEVICE;
    cudaDeviceProp prop;
    CU(cudaGetDeviceProperties(&prop, d.device));
    if (prop.major != 10) return PTFOCK_ERR_UNSUPPORTED_DEVICE;     // sm_100a code only, no fallback
    GUARD(d.device);

    ptfock_plan *p = new (std::nothrow) ptfock_plan();
    if (!p) return PTFOCK_ERR_ALLOC;
    std::memset(p, 0, sizeof(*p));
    p->d = d;
    p->N = (long long)d.n[0] * d.n[1] * d.n[2];
    p->slab_pts = d.n[1] * d.n[2];
    p->volume = std::fabs(det3(d.cell));
    p->slab = slab;
    p->pencil = pencil;
    p->p8 = p8;
    p->onchip = (d.n[0] == 16 && d.n[1] == 16 && d.n[2] == 16 && !(d.flags & PTFOCK_FLAG_THREE_STAGE_SLABS)) ? 1 : 0;
    p->sm_count = prop.multiProcessorCount;

    std::vector<double> vperm;
    bool even = false;
    int rc = build_vtable(d, *slab, p8, p->onchip != 0, vperm, even);
    if (rc != PTFOCK_OK) { free_plan(p); return rc; }
    p->v_even = even;

#define CUP(call) do { cudaError_t e__ = (call); if (e__ != cudaSuccess) { g_last_cuda = (int)e__; free_plan(p); \
        return (e__ == cudaErrorMemoryAllocation) ? PTFOCK_ERR_ALLOC : PTFOCK_ERR_CUDA; } } while (0)

    if (p->onchip) {
        CUP(cudaFuncSetAttribute(onchip16_apply, cudaFuncAttributeMaxDynamicSharedMemorySize, kOnchipSmem));
        CUP(cudaMalloc(&p->v_dev, sizeof(double) * p->N));
        CUP(cudaMemcpy(p->v_dev, vperm.data(), sizeof(double) * p->N, cudaMemcpyHostToDevice));
    } else if (p8) {
        CUP(p8->prepare());
        CUP(cudaMalloc(&p->v8_dev, sizeof(double) * p->N));
        CUP(cudaMemcpy(p->v8_dev, vperm.data(), sizeof(double) * p->N, cudaMemcpyHostToDevice));
    } else {
        CUP(slab->prepare());
        if (pencil->prepare) CUP(pencil->prepare());
        CUP(cudaMalloc(&p->v_dev, sizeof(double) * p->N));
        CUP(cudaMemcpy(p->v_dev, vperm.data(), sizeof(double) * p->N, cudaMemcpyHostToDevice));
    }
    for (int k = 0; k < 3; ++k) {
        const int n = d.n[k];
        std::vector<cd> tw((size_t)n);
        for (int t = 0; t < n; ++t) {
            const long double ang = 2.0L * 3.14159265358979323846264338327950288L * (long double)t / (long double)n;
            tw[t] = make_double2((double)cosl(ang), (double)(-sinl(ang)));     // exp(-2 pi i t / n)
        }
        CUP(cudaMalloc(&p->tw_dev[k], sizeof(cd) * n));
        CUP(cudaMemcpy(p->tw_dev[k], tw.data(), sizeof(cd) * n, cudaMemcpyHostToDevice));
    }
    // pair-scheduler tile
    int Ib = d.block_i > 0 ? d.block_i : 64;
    // targets per wave: passes A and C launch Jb * n0 one-per-SM CTAs; aim at ~7 rounds of the SMs and, if the last
    // round would be badly filled (n0 = 120: 960 CTAs = 6.5 rounds), take the next Jb (a divisor of max_targets if
    // there is one) that fills whole rounds
    int Jb = d.block_j;
    if (Jb <= 0) {
        const int sms = prop.multiProcessorCount, base = (1024 / d.n[0] > 8 ? 1024 / d.n[0] : 8);
        auto eff = [&](int c) {
            const long long ctas = (long long)c * d.n[0], rounds = (ctas + sms - 1) / sms;
            return (double)ctas / (double)(rounds * sms);
        };
        Jb = base;
        for (int pass = 0; pass < 2 && Jb == base; ++pass) {
            double best = eff(base) + 0.02;
            for (int c = base + 1; c <= 2 * base && c <= d.max_targets; ++c) {
                if (pass == 0 && d.max_targets % c) continue;
                if (eff(c) > best) { best = eff(c); Jb = c; }
            }
        }
    }
    if (Ib > d.n_occ) Ib = d.n_occ;
    if (Jb > d.max_targets) Jb = d.max_targets;
    const size_t pair_bytes = sizeof(cd) * (size_t)p->N;
    // default scratch: at most 12 GiB and at most 60 % of what is free now (Phi of Si1536 alone is 39 GB)
    size_t limit = d.workspace_bytes ? (size_t)d.workspace_bytes : ((size_t)12 << 30);
    if (!d.workspace_bytes) {
        size_t free_b = 0, total_b = 0;
        if (cudaMemGetInfo(&free_b, &total_b) == cudaSuccess && free_b / 10 * 6 < limit) limit = free_b / 10 * 6;
        if (limit < pair_bytes) limit = pair_bytes;
    }
    while ((long long)Ib * Jb > 65535 && Ib > 1) Ib = (Ib + 1) / 2;     // pass B puts the wave's pairs on gridDim.y
    while ((long long)Ib * Jb > 65535 && Jb > 1) Jb = (Jb + 1) / 2;
    while ((size_t)Ib * Jb * pair_bytes > limit && Ib > 1) Ib = (Ib + 1) / 2;
    while ((size_t)Ib * Jb * pair_bytes > limit && Jb > 1) Jb = (Jb + 1) / 2;
    if ((size_t)Ib * Jb * pair_bytes > limit) { free_plan(p); return PTFOCK_ERR_ALLOC; }
    // the dense-algebra calls keep an n x n matrix (padded to the 64-wide blocks) and a few split-K partial sums in the
    // same scratch: never size it below that
    size_t dense_min = 0;
    {
        const size_t nmax = (size_t)std::max(d.n_occ, d.max_targets), npad = (nmax + 63) / 64 * 64;
        const size_t ks = 8;                                 // overlap_into picks 1 .. 8 splits
        dense_min = sizeof(cd) * (npad * npad + npad + ks * nmax * nmax);
    }
    // a failing allocation (fragmentation, another allocator holding the memory) shrinks the wave instead of failing
    // a second slot (two waves in flight) if it fits the bound
    int slots = (!(d.flags & PTFOCK_FLAG_SINGLE_STREAM) && !p->onchip && 2 * (size_t)Ib * Jb * pair_bytes <= limit &&
                 2LL * Ib * Jb <= 65535) ? 2 : 1;
    for (;;) {
        // with a caller's bound the dense-algebra minimum is clipped to it (those calls return PTFOCK_ERR_ALLOC when the
        // scratch is too small for them); without one the scratch is never sized below it
        p->scratch_bytes = std::max((size_t)slots * Ib * Jb * pair_bytes,
                                    d.workspace_bytes ? std::min(dense_min, (size_t)d.workspace_bytes) : dense_min);
        cudaError_t e = cudaMalloc(&p->scratch, p->scratch_bytes);
        if (e == cudaSuccess) break;
        cudaGetLastError();
        p->scratch = nullptr;
        if (e != cudaErrorMemoryAllocation || (slots == 1 && (d.workspace_bytes || (Ib == 1 && Jb == 1)))) {
            g_last_cuda = (int)e; free_plan(p); return PTFOCK_ERR_ALLOC;
        }
        if (slots == 2) slots = 1;
        else if (Ib > 1) Ib = (Ib + 1) / 2;
        else Jb = (Jb + 1) / 2;
    }
    p->Ib = Ib;
    p->Jb = Jb;
    p->slots = slots;
    CUP(cudaEventCreateWithFlags(&p->busy_ev, cudaEventDisableTiming));
    if (slots == 2) {
        CUP(cudaStreamCreateWithFlags(&p->aux_stream, cudaStreamNonBlocking));
        CUP(cudaEventCreateWithFlags(&p->fork_ev, cudaEventDisableTiming));
        CUP(cudaEventCreateWithFlags(&p->join_ev, cudaEventDisableTiming));
    }
    p->use_tma = 0;
    {
        typedef CUresult (*encode_fn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                      const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                      CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
        void *fn = nullptr;
        cudaDriverEntryPointQueryResult qres;
        CUP(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres));
        const bool have = fn && qres == cudaDriverEntryPointSuccess;
        const cuuint32_t estr[2] = { 1, 1 };
        if (p8) {
            // scratch as [pairs * nq * n0 rows][2 * qpts doubles]; box = 128 bytes x all (q, x0) rows of one pair
            if (!have) { free_plan(p); return PTFOCK_ERR_CUDA; }
            const cuuint64_t dims[2] = { (cuuint64_t)2 * p8->qpts, (cuuint64_t)slots * Ib * Jb * p8->rows };
            const cuuint64_t strides[1] = { (cuuint64_t)p8->qpts * sizeof(cd) };
            const cuuint32_t box[2] = { (cuuint32_t)(2 * p8->p * p8->rq), (cuuint32_t)p8->rows };
            CUresult r = ((encode_fn)fn)(&p->tmap8, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, p->scratch, dims, strides, box, estr,
                                         CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                                         CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
            if (r != CUDA_SUCCESS) { g_last_cuda = (int)r; free_plan(p); return PTFOCK_ERR_CUDA; }
        } else if (pencil->run_tma) {
            if (!have) { free_plan(p); return PTFOCK_ERR_CUDA; }
            const cuuint64_t dims[2] = { (cuuint64_t)2 * p->slab_pts, (cuuint64_t)slots * Ib * Jb * d.n[0] };
            const cuuint64_t strides[1] = { (cuuint64_t)p->slab_pts * sizeof(cd) };
            const cuuint32_t box[2] = { (cuuint32_t)(2 * pencil->tma_cw), (cuuint32_t)d.n[0] };
            CUresult r = ((encode_fn)fn)(&p->tmap, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, p->scratch, dims, strides, box, estr,
                                         CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                         CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
            if (r != CUDA_SUCCESS) { g_last_cuda = (int)r; free_plan(p); return PTFOCK_ERR_CUDA; }
            CUP(pencil->prepare_tma());
            p->use_tma = 1;
        }
    }
    CUP(cudaFuncSetAttribute(overlap_mma, cudaFuncAttributeMaxDynamicSharedMemorySize, kOverlapMmaSmem));
    CUP(cudaFuncSetAttribute(rotate_mma, cudaFuncAttributeMaxDynamicSharedMemorySize, kRotateMmaSmem));
    CUP(cudaMalloc(&p->partials, sizeof(double2) * 1024));
    CUP(cudaMalloc(&p->result_dev, sizeof(double2)));
    CUP(cudaMallocHost(&p->result_host, sizeof(double2)));
#undef CUP
    *out = p;
    return PTFOCK_OK;
}

extern "C" int ptfock_destroy(ptfock_plan *plan) {
    if (!plan) return PTFOCK_OK;
    DeviceGuard guard(plan->d.device);
    cudaDeviceSynchronize();
    free_plan(plan);
    return PTFOCK_OK;
}

extern "C" const char *ptfock_strerror(int code) {
    switch (code) {
        case PTFOCK_OK: return "ok";
        case PTFOCK_ERR_INVALID_ARG: return "invalid argument";
        case PTFOCK_ERR_UNSUPPORTED_GRID: return "unsupported grid (n0 in {16,32,48,64,120,128}; built slab shapes (n1,n2): {16,32,48,64,128}^2 except (128,128), and (90,60); see ptfock.h)";
        case PTFOCK_ERR_UNSUPPORTED_DEVICE: return "unsupported device (needs compute capability 10.x; there is no CPU fallback)";
        case PTFOCK_ERR_ALIGNMENT: return "pointer not 16-byte aligned";
        case PTFOCK_ERR_ALLOC: return "allocation failed or workspace too small";
        case PTFOCK_ERR_CUDA: return "CUDA runtime error (see ptfock_last_cuda_error)";
        case PTFOCK_ERR_ALIAS: return "out overlaps an input";
        case PTFOCK_ERR_NOT_POSITIVE: return "overlap matrix is not positive definite (linearly dependent orbitals)";
        case PTFOCK_ERR_TOO_LARGE: return "too many bands for the built-in scratch (ptfock_banddot_static: n <= PTFOCK_STATIC_MAX_BANDS = 4096; split the call)";
        default: return "unknown error";
    }
}

extern "C" int ptfock_last_cuda_error(void) { return g_last_cuda; }

extern "C" int ptfock_plan_info(const ptfock_plan *plan, int64_t info[8]) {
    if (!plan || !info) return PTFOCK_ERR_INVALID_ARG;
    info[0] = plan->Ib;
    info[1] = plan->Jb;
    info[2] = (int64_t)plan->scratch_bytes;
    info[3] = plan->last_launches;
    info[4] = plan->last_pairs;
    info[5] = plan->last_symmetric;
    info[6] = plan->total_launches;
    info[7] = (plan->onchip ? 2 : (plan->p8 ? 1 : 0)) | (plan->slots == 2 ? 16 : 0);
    return PTFOCK_OK;
}

// ================================================================================================
// pair scheduler
// ================================================================================================
namespace {

struct Wave {
    ptfock_plan *p;
    cudaStream_t st;                    // the stream the next wave's launches go to (the caller's, or the plan's aux stream)
    long long launches, pairs;
    cudaError_t err;                    // first failure of an event / wait / launch in this call
    cudaStream_t st0 = nullptr;         // the caller's stream
    int slot = 0;                       // scratch slot of the next wave
    void note(cudaError_t e) { if (e != cudaSuccess && err == cudaSuccess) err = e; }
    void use(int s) { slot = s; st = s ? p->aux_stream : st0; }
    long long pair0() const { return (long long)slot * p->Ib * p->Jb; }
    cd *scratch() const { return p->scratch + (size_t)pair0() * (size_t)p->N; }
};

// every call that touches the plan's buffers starts with begin_call and ends with end_call: a call on another stream
// than the previous one waits for the previous call's end (the scratch, the energy buffer and the staging buffers
// are shared by consecutive calls)
cudaError_t begin_call(ptfock_plan *p, cudaStream_t st) {
    if (p->has_last && p->last_stream != st) return cudaStreamWaitEvent(st, p->busy_ev, 0);
    return cudaSuccess;
}
cudaError_t end_call(ptfock_plan *p, cudaStream_t st) {
    cudaError_t e = cudaEventRecord(p->busy_ev, st);
    if (e == cudaSuccess) { p->last_stream = st; p->has_last = 1; }
    return e;
}
// an error return after begin_call may already have queued work on `st` (a first-use fill, part of a wave): the busy
// event is recorded on EVERY way out, so that the next call on another stream is still ordered behind it
struct CallScope {
    ptfock_plan *p;
    cudaStream_t st;
    bool closed;
    cudaError_t close() { closed = true; return end_call(p, st); }
    ~CallScope() { if (!closed) end_call(p, st); }
};
#define BEGIN_CALL(plan_, st_) CU(begin_call(plan_, st_)); CallScope call_scope__{ plan_, st_, false }
#define END_CALL() CU(call_scope__.close())

// profiling: record an event that closes an interval of kind `tag` (-1: opens a new run of intervals)
void mark(Wave &w, int tag) {
    ptfock_plan *p = w.p;
    if (!p->profiling) return;
    if (!p->ev_pool) { p->ev_pool = new std::vector<cudaEvent_t>(); p->ev_tags = new std::vector<int>(); }
    if (p->ev_used == p->ev_pool->size()) {
        cudaEvent_t e;
        const cudaError_t ce = cudaEventCreate(&e);
        if (ce != cudaSuccess) { w.note(ce); return; }
        p->ev_pool->push_back(e);
        p->ev_tags->push_back(-1);
    }
    w.note(cudaEventRecord((*p->ev_pool)[p->ev_used], w.st));
    (*p->ev_tags)[p->ev_used] = tag;
    p->ev_used++;
}

// A + B for the block of pairs (i in [i0, i0+ni)) x (j in [j0, j0+nj)); pair index = ii * nj + jj.
void wave_forward_mid(Wave &w, const cd *phi, const cd *psi, int i0, int ni, int j0, int nj, int tri = 0) {
    ptfock_plan *p = w.p;
    SlabArgs a;
    a.a = phi; a.b = psi; a.scratch = w.scratch(); a.out = nullptr;
    a.tw1 = p->tw_dev[1]; a.tw2 = p->tw_dev[2];
    a.grid_pts = p->N; a.n0 = p->d.n[0];
    a.a0 = i0; a.na = ni; a.b0 = j0;
    a.stride_loop = nj; a.stride_cta = 1; a.conj_w = 0; a.tri = tri;
    // split the i loop over blockIdx.z until the grid has a few CTAs per SM
    int z = 1;
    const long long base = (long long)p->d.n[0] * nj;
    while (z < ni && base * z * (p->p8 ? p->p8->nq : 1) < (long long)p->sm_count * (p->p8 ? 12 : 6)) z *= 2;
    if (z > ni) z = ni;
    mark(w, -1);
    if (p->p8) {
        p->p8->fwd(a, dim3(nj, p->d.n[0] * p->p8->nq, z), w.st);
        mark(w, 0);
        P8MidArgs b;
        b.v = p->v8_dev; b.tw0 = p->tw_dev[0];
        b.n_pairs = ni * nj; b.tri_nj = tri ? nj : 0; b.pair0 = (int)w.pair0();
        p->p8->mid(p->tmap8, b, ni * nj, w.st);
        mark(w, 1);
        w.launches += 2;
        w.pairs += tri ? (long long)nj * (nj + 1) / 2 : (long long)ni * nj;
        return;
    }
    p->slab->fwd(a, dim3(nj, p->d.n[0], z), w.st);
    mark(w, 0);
    if (p->use_tma) {
        PencilTmaArgs b;
        b.v = p->v_dev; b.tw0 = p->tw_dev[0]; b.slab_pts = p->slab_pts; b.tri_nj = tri ? nj : 0; b.pair0 = (int)w.pair0();
        p->pencil->run_tma(p->tmap, b, ni * nj, w.st);
    } else {
        PencilArgs b;
        b.scratch = w.scratch(); b.v = p->v_dev; b.tw0 = p->tw_dev[0]; b.slab_pts = p->slab_pts; b.tri_nj = tri ? nj : 0;
        p->pencil->run(b, ni * nj, w.st);
    }
    mark(w, 1);
    w.launches += 2;
    w.pairs += tri ? (long long)nj * (nj + 1) / 2 : (long long)ni * nj;
}

// C: out[t0 + tt] += sum_ss orb[s0 + ss] * W(ss, tt)
void wave_accumulate(Wave &w, const cd *orb, int s0, int ns, cd *out, int t0, int nt, int stride_loop, int stride_cta,
                     int conj_w, int tri = 0) {
    ptfock_plan *p = w.p;
    SlabArgs a;
    a.a = orb; a.b = nullptr; a.scratch = w.scratch(); a.out = out;
    a.tw1 = p->tw_dev[1]; a.tw2 = p->tw_dev[2];
    a.grid_pts = p->N; a.n0 = p->d.n[0];
    a.a0 = s0; a.na = ns; a.b0 = t0;
    a.stride_loop = stride_loop; a.stride_cta = stride_cta; a.conj_w = conj_w; a.tri = tri;
    if (p->p8) p->p8->inv(a, dim3(nt, p->d.n[0] * p->p8->nq, 1), w.st);
    else p->slab->inv(a, dim3(nt, p->d.n[0], 1), w.st);
    mark(w, 2);
    w.launches += 1;
    w.note(cudaPeekAtLastError());
}

bool overlaps(const void *a, size_t na, const void *b, size_t nb) {
    const uintptr_t x = (uintptr_t)a, y = (uintptr_t)b;
    return x < y + nb && y < x + na;
}

int check_apply_args(const ptfock_plan *p, const void *phi, const void *psi, int self_offset, int n_targets,
                     const void *out) {
    if (!p || !phi || n_targets < 0) return PTFOCK_ERR_INVALID_ARG;
    if (!out && n_targets > 0) return PTFOCK_ERR_INVALID_ARG;
    if (!psi && (self_offset < 0 || (long long)self_offset + n_targets > p->d.n_occ)) return PTFOCK_ERR_INVALID_ARG;
    if (((uintptr_t)phi | (uintptr_t)psi | (uintptr_t)out) & 15) return PTFOCK_ERR_ALIGNMENT;
    // device pointers on the plan's device (managed memory is accepted)
    const void *ptrs[3] = { phi, psi, out };
    for (const void *q : ptrs) {
        if (!q) continue;
        cudaPointerAttributes at;
        if (cudaPointerGetAttributes(&at, q) != cudaSuccess) { cudaGetLastError(); return PTFOCK_ERR_INVALID_ARG; }
        if (at.type == cudaMemoryTypeManaged) continue;
        if (at.type != cudaMemoryTypeDevice || at.device != p->d.device) return PTFOCK_ERR_INVALID_ARG;
    }
    return PTFOCK_OK;
}

// Host path (ptfock_apply_host): Phi is copied in chunks of `chunk` orbitals and Psi in chunks of `jchunk` targets on
// the plan's copy stream, one event per chunk; a wave waits only for the chunks it reads, so the copy of the rest
// overlaps the first waves.  The result goes back the same way: when the last i block has accumulated into a j-block
// of `out`, that block is final and its device-to-host copy is queued on the copy stream behind an event, so it
// overlaps the remaining waves (only the last block's copy is exposed).
struct HostPipe {
    cudaStream_t cs;
    std::vector<cudaEvent_t> *ev;       // [0, n_chunks): Phi chunk landed; [n_chunks]: fork event;
                                        // [psi_base, psi_base + n_jchunks): Psi chunk landed; [out_base, ...): out block final
    int chunk, n_chunks;
    int jchunk, n_jchunks, psi_base, out_base;
    std::vector<char> waited[2], waited_psi[2];      // per stream (slot) of the two-wave schedule
    cd *out_host;                       // host destination of the result (streamed back block by block)
    size_t gbytes;
    bool out_streamed;                  // apply_device queued every block of `out`
    cudaError_t err = cudaSuccess;
    void note(cudaError_t e) { if (e != cudaSuccess && err == cudaSuccess) err = e; }
    void need(cudaStream_t st, int slot, int lo, int hi) {        // orbitals [lo, hi) of Phi, for the waves of `slot` on `st`
        for (int c = lo / chunk; c <= (hi - 1) / chunk && c < n_chunks; ++c)
            if (!waited[slot][c]) {
                note(cudaStreamWaitEvent(st, (*ev)[c], 0));
                waited[slot][c] = 1;
            }
    }
    void need_psi(cudaStream_t st, int slot, int lo, int hi) {    // targets [lo, hi) of Psi
        for (int c = lo / jchunk; c <= (hi - 1) / jchunk && c < n_jchunks; ++c)
            if (!waited_psi[slot][c]) {
                note(cudaStreamWaitEvent(st, (*ev)[psi_base + c], 0));
                waited_psi[slot][c] = 1;
            }
    }
    void emit_out(cudaStream_t st, const cd *out_dev, int j0, int nj) {   // out[j0, j0 + nj) is final on `st`
        cudaEvent_t e = (*ev)[out_base + j0 / jchunk];
        note(cudaEventRecord(e, st));
        note(cudaStreamWaitEvent(cs, e, 0));
        note(cudaMemcpyAsync(out_host + (size_t)j0 * (gbytes / sizeof(cd)), out_dev + (size_t)j0 * (gbytes / sizeof(cd)),
                             gbytes * nj, cudaMemcpyDeviceToHost, cs));
    }
};

// 16^3: out[j] = sum_i mul_i * W_ij with the whole pair-solve inside one CTA (onchip16.cuh); the i loop is split into
// chunks so that the grid fills the SMs, the chunks' partial sums go through the plan's scratch and are added in order
int apply_onchip(ptfock_plan *p, const cd *phi, const cd *mul, int mul_stride, int phi0, int n_i, const cd *tgt, int n_targets,
                 cd *out, cudaStream_t st, Wave &w) {
    const size_t gbytes = sizeof(cd) * (size_t)p->N;
    const int max_batch = (int)std::min<size_t>(p->scratch_bytes / gbytes, 65535);
    for (int t0 = 0; t0 < n_targets; t0 += max_batch) {
        const int nt = std::min(max_batch, n_targets - t0);
        int n_chunks = (2 * p->sm_count + nt - 1) / nt;
        n_chunks = std::max(1, std::min(n_chunks, n_i));
        n_chunks = (int)std::min<size_t>((size_t)n_chunks, p->scratch_bytes / (gbytes * nt));
        n_chunks = std::min(n_chunks, 65535);
        const int per = (n_i + n_chunks - 1) / n_chunks;
        n_chunks = (n_i + per - 1) / per;
        OnchipArgs a;
        a.phi = phi; a.mul = mul; a.psi = tgt; a.partial = p->scratch; a.vt = p->v_dev;
        a.phi0 = phi0; a.n_i = n_i; a.mul_stride = mul_stride; a.psi0 = t0; a.i_per_cta = per;
        mark(w, -1);
        onchip16_apply<<<dim3(nt, n_chunks), kOnchipThreads, kOnchipSmem, st>>>(a);
        mark(w, 0);
        const long long per_chunk = (long long)nt * p->N;
        onchip_reduce<<<(unsigned)((per_chunk + 255) / 256), 256, 0, st>>>(p->scratch, n_chunks, per_chunk, out + (size_t)t0 * p->N);
        mark(w, 2);
        w.launches += 2;
        w.pairs += (long long)n_i * nt;
        w.note(cudaPeekAtLastError());
    }
    return PTFOCK_OK;
}

int apply_device(ptfock_plan *p, const cd *phi, const cd *psi, int self_offset, int n_targets, cd *out,
                 cudaStream_t st, HostPipe *hp = nullptr) {
    const size_t gbytes = sizeof(cd) * (size_t)p->N;
    if (n_targets == 0) { p->last_launches = 0; p->last_pairs = 0; p->last_symmetric = 0; return PTFOCK_OK; }
    if (overlaps(out, gbytes * n_targets, phi, gbytes * p->d.n_occ)) return PTFOCK_ERR_ALIAS;
    if (psi && overlaps(out, gbytes * n_targets, psi, gbytes * n_targets)) return PTFOCK_ERR_ALIAS;
    Wave w{ p, st, 0, 0, cudaSuccess };
    w.st0 = st;
    const int n_occ = p->d.n_occ;
    const bool symmetric = (!psi) && self_offset == 0 && n_targets == n_occ && p->v_even && n_occ > 1 && !p->onchip;
    if (p->onchip) {
        if (hp) { hp->need(st, 0, 0, n_occ); if (psi) hp->need_psi(st, 0, 0, n_targets); }
        apply_onchip(p, phi, phi, 1, 0, n_occ, psi ? psi : phi + (size_t)self_offset * p->N, n_targets, out, st, w);
        if (hp) w.note(hp->err);
        w.note(cudaGetLastError());
        if (w.err != cudaSuccess) { g_last_cuda = (int)w.err; return PTFOCK_ERR_CUDA; }
        p->last_launches = w.launches;
        p->last_pairs = w.pairs;
        p->last_symmetric = 0;
        p->total_launches += w.launches;
        return PTFOCK_OK;
    }
    CU(cudaMemsetAsync(out, 0, gbytes * n_targets, st));             // Alg. 2 line 1
    if (symmetric) {
        // square blocks; block pair (bi <= bj): W_ij for i in bi, j in bj serves out_j (as is) and, off the
        // diagonal, out_i through W_ji = conj(W_ij) (v real and even).
        int bs = p->Ib < p->Jb ? p->Ib : p->Jb;
        while ((size_t)(bs * 2) * (bs * 2) * gbytes <= p->scratch_bytes && bs * 2 <= n_occ && (bs * 2) * (bs * 2) <= 65535 &&
               (long long)(bs * 2) * (bs * 2) <= (long long)p->slots * p->Ib * p->Jb) bs *= 2;      // (the tensor maps cover slots*Ib*Jb pairs)
        for (int j0 = 0; j0 < n_occ; j0 += bs) {
            const int nj = (n_occ - j0 < bs) ? n_occ - j0 : bs;
            for (int i0 = 0; i0 <= j0; i0 += bs) {
                const int ni = (n_occ - i0 < bs) ? n_occ - i0 : bs;
                if (hp) { hp->need(st, 0, i0, i0 + ni); hp->need(st, 0, j0, j0 + nj); }
                // diagonal blocks (i0 == j0): only the pairs i <= j are solved; W_ij then serves out_j (loop i <= j) and,
                // through conj, out_i (loop j > i)
                const int tri = (i0 == j0) ? 1 : 0;
                wave_forward_mid(w, phi, phi, i0, ni, j0, nj, tri);
                wave_accumulate(w, phi, i0, ni, out, j0, nj, nj, 1, 0, tri);
                if (nj > 1 || !tri) wave_accumulate(w, phi, j0, nj, out, i0, ni, 1, nj, 1, tri ? 2 : 0);
            }
        }
    } else {
        const cd *tgt = psi ? psi : phi + (size_t)self_offset * p->N;
        // two waves in flight: j-blocks with an odd index run on the plan's aux stream in the second scratch slot.  A
        // j-block always runs on the same stream, so the read-modify-writes of its `out` stay ordered; the two streams
        // never touch the same targets.  (Per-pass profiling keeps everything on the caller's stream.)
        const bool dual = p->slots == 2 && !p->profiling && n_targets > p->Jb;
        if (dual) {
            w.note(cudaEventRecord(p->fork_ev, st));
            w.note(cudaStreamWaitEvent(p->aux_stream, p->fork_ev, 0));
        }
        if (hp) {
            // host path: i blocks outermost, so every chunk of Phi is used by all j-blocks as soon as it has landed
            // and the rest of the copy hides behind those waves (out_j accumulates over the waves in any order);
            // during the last i block every finished j-block of `out` starts its way back to the host
            for (int i0 = 0; i0 < n_occ; i0 += p->Ib) {
                const int ni = (n_occ - i0 < p->Ib) ? n_occ - i0 : p->Ib;
                const bool last = i0 + ni >= n_occ;
                for (int j0 = 0; j0 < n_targets; j0 += p->Jb) {
                    const int nj = (n_targets - j0 < p->Jb) ? n_targets - j0 : p->Jb;
                    w.use(dual ? (j0 / p->Jb) & 1 : 0);
                    hp->need(w.st, w.slot, i0, i0 + ni);
                    if (psi) hp->need_psi(w.st, w.slot, j0, j0 + nj);
                    else hp->need(w.st, w.slot, self_offset + j0, self_offset + j0 + nj);
                    wave_forward_mid(w, phi, tgt, i0, ni, j0, nj);
                    wave_accumulate(w, phi, i0, ni, out, j0, nj, nj, 1, 0);
                    if (last) hp->emit_out(w.st, out, j0, nj);
                }
            }
            hp->out_streamed = true;
        } else {
            for (int j0 = 0; j0 < n_targets; j0 += p->Jb) {
                const int nj = (n_targets - j0 < p->Jb) ? n_targets - j0 : p->Jb;
                w.use(dual ? (j0 / p->Jb) & 1 : 0);
                for (int i0 = 0; i0 < n_occ; i0 += p->Ib) {
                    const int ni = (n_occ - i0 < p->Ib) ? n_occ - i0 : p->Ib;
                    wave_forward_mid(w, phi, tgt, i0, ni, j0, nj);
                    wave_accumulate(w, phi, i0, ni, out, j0, nj, nj, 1, 0);
                }
            }
        }
        w.use(0);
        if (dual) {
            w.note(cudaEventRecord(p->join_ev, p->aux_stream));
            w.note(cudaStreamWaitEvent(st, p->join_ev, 0));
        }
    }
    if (hp) w.note(hp->err);
    w.note(cudaGetLastError());
    if (w.err != cudaSuccess) { g_last_cuda = (int)w.err; return PTFOCK_ERR_CUDA; }
    p->last_launches = w.launches;
    p->last_pairs = w.pairs;
    p->last_symmetric = symmetric ? 1 : 0;
    p->total_launches += w.launches;
    return PTFOCK_OK;
}

}  // namespace

extern "C" int ptfock_apply(ptfock_plan *plan, const void *phi, const void *psi, int32_t self_offset,
                            int32_t n_targets, void *out, void *stream) {
    int rc = check_apply_args(plan, phi, psi, self_offset, n_targets, out);
    if (rc != PTFOCK_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    GUARD(plan->d.device);
    BEGIN_CALL(plan, st);
    rc = apply_device(plan, (const cd *)phi, (const cd *)psi, self_offset, n_targets, (cd *)out, st);
    END_CALL();
    return rc;
}

extern "C" int ptfock_exchange_energy(ptfock_plan *plan, const void *phi, const void *psi, int32_t self_offset,
                                      int32_t n_targets, const void *vx_psi, double *e_host, void *stream) {
    if (!plan || !phi || !e_host || n_targets < 0) return PTFOCK_ERR_INVALID_ARG;
    if (!psi && (self_offset < 0 || (long long)self_offset + n_targets > plan->d.n_occ)) return PTFOCK_ERR_INVALID_ARG;
    if (((uintptr_t)phi | (uintptr_t)psi | (uintptr_t)vx_psi) & 15) return PTFOCK_ERR_ALIGNMENT;
    cudaStream_t st = (cudaStream_t)stream;
    GUARD(plan->d.device);
    if (n_targets == 0) { *e_host = 0.0; return PTFOCK_OK; }
    BEGIN_CALL(plan, st);
    const cd *vx = (const cd *)vx_psi;
    if (!vx) {
        if (n_targets > plan->d.max_targets) return PTFOCK_ERR_INVALID_ARG;
        if (!plan->energy_buf) {
            cudaError_t e = cudaMalloc(&plan->energy_buf, sizeof(cd) * (size_t)plan->N * plan->d.max_targets);
            if (e != cudaSuccess) { g_last_cuda = (int)e; return PTFOCK_ERR_ALLOC; }
        }
        int rc = apply_device(plan, (const cd *)phi, (const cd *)psi, self_offset, n_targets, plan->energy_buf, st);
        if (rc != PTFOCK_OK) return rc;
        vx = plan->energy_buf;
    }
    const cd *tgt = psi ? (const cd *)psi : (const cd *)phi + (size_t)self_offset * plan->N;
    const long long n = plan->N * (long long)n_targets;
    int blocks = (int)((n + 255) / 256);
    if (blocks > 1024) blocks = 1024;
    dot_partial<<<blocks, 256, 0, st>>>(tgt, vx, n, plan->partials);
    dot_final<<<1, 256, 0, st>>>(plan->partials, blocks, 0.5 * plan->volume / (double)plan->N, plan->result_dev);
    plan->total_launches += 2;
    CU(cudaGetLastError());
    CU(cudaMemcpyAsync(plan->result_host, plan->result_dev, sizeof(double2), cudaMemcpyDeviceToHost, st));
    END_CALL();
    CU(cudaStreamSynchronize(st));
    *e_host = plan->result_host->x;
    return PTFOCK_OK;
}

extern "C" int ptfock_apply_host(ptfock_plan *plan, const void *phi_host, const void *psi_host, int32_t self_offset,
                                 int32_t n_targets, void *out_host, void *stream) {
    if (!plan || !phi_host || !out_host || n_targets < 0 || n_targets > plan->d.max_targets) return PTFOCK_ERR_INVALID_ARG;
    if (!psi_host && (self_offset < 0 || (long long)self_offset + n_targets > plan->d.n_occ)) return PTFOCK_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    GUARD(plan->d.device);
    const size_t gbytes = sizeof(cd) * (size_t)plan->N;
    auto ensure = [&](cd **buf, size_t bytes) -> int {
        if (*buf) return PTFOCK_OK;
        cudaError_t e = cudaMalloc(buf, bytes);
        if (e != cudaSuccess) { g_last_cuda = (int)e; return PTFOCK_ERR_ALLOC; }
        return PTFOCK_OK;
    };
    int rc = ensure(&plan->st_phi, gbytes * plan->d.n_occ);
    if (rc == PTFOCK_OK) rc = ensure(&plan->st_out, gbytes * plan->d.max_targets);
    if (rc == PTFOCK_OK && psi_host) rc = ensure(&plan->st_psi, gbytes * plan->d.max_targets);
    if (rc != PTFOCK_OK) return rc;
    if (n_targets == 0) return PTFOCK_OK;
    if (!plan->copy_stream) CU(cudaStreamCreateWithFlags(&plan->copy_stream, cudaStreamNonBlocking));
    HostPipe hp;
    hp.cs = plan->copy_stream;
    hp.chunk = plan->Ib;
    hp.n_chunks = (plan->d.n_occ + hp.chunk - 1) / hp.chunk;
    hp.jchunk = plan->Jb;
    hp.n_jchunks = (n_targets + hp.jchunk - 1) / hp.jchunk;
    hp.psi_base = hp.n_chunks + 1;
    hp.out_base = hp.psi_base + hp.n_jchunks;
    hp.out_host = (cd *)out_host;
    hp.gbytes = gbytes;
    hp.out_streamed = false;
    if (!plan->copy_ev) plan->copy_ev = new std::vector<cudaEvent_t>();
    while ((int)plan->copy_ev->size() < hp.out_base + hp.n_jchunks) {
        cudaEvent_t e;
        CU(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
        plan->copy_ev->push_back(e);
    }
    hp.ev = plan->copy_ev;
    for (int k = 0; k < 2; ++k) { hp.waited[k].assign(hp.n_chunks, 0); hp.waited_psi[k].assign(hp.n_jchunks, 0); }
    BEGIN_CALL(plan, st);
    // the copy stream starts after whatever the caller queued on `stream`
    CU(cudaEventRecord((*hp.ev)[hp.n_chunks], st));
    CU(cudaStreamWaitEvent(hp.cs, (*hp.ev)[hp.n_chunks], 0));
    // from here on async copies out of the caller's host buffers may be in flight: every exit drains the copy stream
#define CUH(call) do { cudaError_t e__ = (call); if (e__ != cudaSuccess) { g_last_cuda = (int)e__; cudaStreamSynchronize(hp.cs); \
        cudaStreamSynchronize(st); return PTFOCK_ERR_CUDA; } } while (0)
    auto copy_psi = [&](int c) -> cudaError_t {
        const int lo = c * hp.jchunk, cnt = (n_targets - lo < hp.jchunk) ? n_targets - lo : hp.jchunk;
        cudaError_t e = cudaMemcpyAsync(plan->st_psi + (size_t)lo * plan->N, (const cd *)psi_host + (size_t)lo * plan->N, gbytes * cnt,
                                        cudaMemcpyHostToDevice, hp.cs);
        return e != cudaSuccess ? e : cudaEventRecord((*hp.ev)[hp.psi_base + c], hp.cs);
    };
    auto copy_phi = [&](int c) -> cudaError_t {
        const int lo = c * hp.chunk, cnt = (plan->d.n_occ - lo < hp.chunk) ? plan->d.n_occ - lo : hp.chunk;
        cudaError_t e = cudaMemcpyAsync(plan->st_phi + (size_t)lo * plan->N, (const cd *)phi_host + (size_t)lo * plan->N, gbytes * cnt,
                                        cudaMemcpyHostToDevice, hp.cs);
        return e != cudaSuccess ? e : cudaEventRecord((*hp.ev)[c], hp.cs);
    };
    // copy order = the order the waves read: the first j-block of Psi and the first chunk of Phi, the rest of Psi (the
    // first i block sweeps all j-blocks), then the rest of Phi.  Psi = Phi[self_offset ...]: the chunks that hold the
    // targets go first.
    std::vector<int> order;
    const int t_lo = psi_host ? 0 : self_offset / hp.chunk, t_hi = psi_host ? -1 : (self_offset + n_targets - 1) / hp.chunk;
    for (int c = t_lo; c <= t_hi; ++c) order.push_back(c);
    for (int c = 0; c < hp.n_chunks; ++c) if (c < t_lo || c > t_hi) order.push_back(c);
    if (psi_host) CUH(copy_psi(0));
    size_t first = 0;
    if (psi_host && !order.empty()) { CUH(copy_phi(order[0])); first = 1; }
    if (psi_host) for (int c = 1; c < hp.n_jchunks; ++c) CUH(copy_psi(c));
    for (size_t k = first; k < order.size(); ++k) CUH(copy_phi(order[k]));
    rc = apply_device(plan, plan->st_phi, psi_host ? plan->st_psi : nullptr, self_offset, n_targets, plan->st_out, st, &hp);
    if (rc != PTFOCK_OK) { cudaStreamSynchronize(hp.cs); cudaStreamSynchronize(st); return rc; }
    if (!hp.out_streamed) CUH(cudaMemcpyAsync(out_host, plan->st_out, gbytes * n_targets, cudaMemcpyDeviceToHost, st));
    CUH(call_scope__.close());
    CUH(cudaStreamSynchronize(st));
    CUH(cudaStreamSynchronize(hp.cs));
    return PTFOCK_OK;
#undef CUH
}

extern "C" int ptfock_debug_pair(ptfock_plan *plan, const void *phi_i, const void *psi_j, void *w_out, void *stream) {
    if (!plan || !phi_i || !psi_j || !w_out) return PTFOCK_ERR_INVALID_ARG;
    if (((uintptr_t)phi_i | (uintptr_t)psi_j | (uintptr_t)w_out) & 15) return PTFOCK_ERR_ALIGNMENT;
    cudaStream_t st = (cudaStream_t)stream;
    GUARD(plan->d.device);
    const size_t gbytes = sizeof(cd) * (size_t)plan->N;
    BEGIN_CALL(plan, st);
    if (!plan->ones) {
        cudaError_t e = cudaMalloc(&plan->ones, gbytes);
        if (e != cudaSuccess) { g_last_cuda = (int)e; return PTFOCK_ERR_ALLOC; }
        fill_ones<<<(unsigned)((plan->N + 255) / 256), 256, 0, st>>>(plan->ones, plan->N);
    }
    Wave w{ plan, st, 0, 0, cudaSuccess };
    w.st0 = st;
    if (plan->onchip) {
        apply_onchip(plan, (const cd *)phi_i, plan->ones, 0, 0, 1, (const cd *)psi_j, 1, (cd *)w_out, st, w);
    } else {
        CU(cudaMemsetAsync(w_out, 0, gbytes, st));
        wave_forward_mid(w, (const cd *)phi_i, (const cd *)psi_j, 0, 1, 0, 1);
        wave_accumulate(w, plan->ones, 0, 1, (cd *)w_out, 0, 1, 1, 1, 0);
    }
    plan->total_launches += w.launches + 1;
    w.note(cudaGetLastError());
    if (w.err != cudaSuccess) { g_last_cuda = (int)w.err; return PTFOCK_ERR_CUDA; }
    END_CALL();
    return PTFOCK_OK;
}

// ================================================================================================
// dense-algebra neighbours (dense.cuh): PAPER.md Alg. 3 (Sec. 3.3), Sec. 3.4
// ================================================================================================
namespace {

int check_dev_ptrs(const ptfock_plan *p, std::initializer_list<const void *> ptrs) {
    for (const void *q : ptrs) {
        if (!q) continue;
        if ((uintptr_t)q & 15) return PTFOCK_ERR_ALIGNMENT;
        cudaPointerAttributes at;
        if (cudaPointerGetAttributes(&at, q) != cudaSuccess) { cudaGetLastError(); return PTFOCK_ERR_INVALID_ARG; }
        if (at.type == cudaMemoryTypeManaged) continue;
        if (at.type != cudaMemoryTypeDevice || at.device != p->d.device) return PTFOCK_ERR_INVALID_ARG;
    }
    return PTFOCK_OK;
}

// the same for an array of doubles (rho, vloc): 8-byte alignment
int check_dev_doubles(const ptfock_plan *p, const double *q) {
    if (!q) return PTFOCK_OK;
    if ((uintptr_t)q & 7) return PTFOCK_ERR_ALIGNMENT;
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, q) != cudaSuccess) { cudaGetLastError(); return PTFOCK_ERR_INVALID_ARG; }
    if (at.type == cudaMemoryTypeManaged) return PTFOCK_OK;
    return (at.type == cudaMemoryTypeDevice && at.device == p->d.device) ? PTFOCK_OK : PTFOCK_ERR_INVALID_ARG;
}

// S (n_a x n_b, row pitch ld_s) = w * A^H B; split-K partial sums go to `work` (bytes available: work_bytes).
// A Hermitian product (same orbitals on both sides, "Psi^* Psi") computes the 64 x 64 tiles on and below the
// diagonal only -- half of the 8 N n^2 flops -- and mirrors the rest.
int overlap_into(ptfock_plan *p, const cd *a, int n_a, const cd *b, int n_b, cd *s, int ld_s, cd *work, size_t work_bytes,
                 cudaStream_t st) {
    const bool herm = a == b && n_a == n_b;
    const int ta = (n_a + kDT - 1) / kDT, tb = (n_b + kDT - 1) / kDT;
    const int tiles = herm ? ta * (ta + 1) / 2 : ta * tb;
    // split K so that the CTAs fill whole rounds of the 2 x sm_count resident CTAs: the split with the least
    // (rounds / splits) wins, the smaller one on a tie (1024 orbitals: 256 tiles x 8 splits = 6.9 rounds)
    const size_t per = sizeof(cd) * (size_t)n_a * n_b;
    long long ks_max = std::min<long long>(8, p->N / 1024 > 0 ? p->N / 1024 : 1LL);
    ks_max = std::min<long long>(ks_max, (long long)(work_bytes / per));
    if (ks_max < 1) return PTFOCK_ERR_ALLOC;
    long long ks = 1;
    {
        const long long slots = 2LL * p->sm_count;
        double best = 1e300;
        for (long long c = 1; c <= ks_max; ++c) {
            const double cost = (double)((tiles * c + slots - 1) / slots) / (double)c;
            if (cost < best * (1.0 - 1e-9)) { best = cost; ks = c; }
        }
    }
    long long pps = (p->N + ks - 1) / ks;
    pps = (pps + kDK - 1) / kDK * kDK;
    ks = (p->N + pps - 1) / pps;
    OverlapArgs g;
    g.a = a; g.b = b; g.part = work; g.n_pts = p->N; g.pts_per_split = pps; g.n_a = n_a; g.n_b = n_b; g.ld = n_b; g.lower = herm ? 1 : 0;
    overlap_mma<<<herm ? dim3(tiles, 1, (unsigned)ks) : dim3(ta, tb, (unsigned)ks), 128, kOverlapMmaSmem, st>>>(g);
    const long long cnt = (long long)n_a * n_b;
    overlap_reduce<<<(unsigned)((cnt + 255) / 256), 256, 0, st>>>(work, (int)ks, n_a, n_b, n_b, p->volume / (double)p->N, s, ld_s, herm ? 1 : 0);
    p->total_launches += 2;
    return PTFOCK_OK;
}

void rotate_launch(ptfock_plan *p, const RotateArgs &g, cudaStream_t st) {
    rotate_mma<<<dim3((g.n_out + kDT - 1) / kDT, (unsigned)((g.n_pts + kDT - 1) / kDT)), 128, kRotateMmaSmem, st>>>(g);
    p->total_launches += 1;
}

}  // namespace

extern "C" int ptfock_overlap(ptfock_plan *plan, const void *a, int32_t n_a, const void *b, int32_t n_b, void *s, void *stream) {
    if (!plan || !a || !b || !s || n_a < 1 || n_b < 1) return PTFOCK_ERR_INVALID_ARG;
    int rc = check_dev_ptrs(plan, { a, b, s });
    if (rc != PTFOCK_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    GUARD(plan->d.device);
    BEGIN_CALL(plan, st);
    rc = overlap_into(plan, (const cd *)a, n_a, (const cd *)b, n_b, (cd *)s, n_b, plan->scratch, plan->scratch_bytes, st);
    if (rc != PTFOCK_OK) return rc;
    CU(cudaGetLastError());
    END_CALL();
    return PTFOCK_OK;
}

extern "C" int ptfock_rotate(ptfock_plan *plan, const void *a, int32_t n_a, const void *s, int32_t n_out, void *out, void *stream) {
    if (!plan || !a || !s || !out || n_a < 1 || n_out < 1) return PTFOCK_ERR_INVALID_ARG;
    int rc = check_dev_ptrs(plan, { a, s, out });
    if (rc != PTFOCK_OK) return rc;
    const size_t gbytes = sizeof(cd) * (size_t)plan->N;
    if (overlaps(out, gbytes * n_out, a, gbytes * n_a)) return PTFOCK_ERR_ALIAS;
    cudaStream_t st = (cudaStream_t)stream;
    GUARD(plan->d.device);
    RotateArgs g = {};
    g.a = (const cd *)a; g.s = (const cd *)s; g.out = (cd *)out; g.n_pts = plan->N; g.n_a = n_a; g.n_out = n_out; g.ld = n_out;
    rotate_launch(plan, g, st);
    CU(cudaGetLastError());
    return PTFOCK_OK;
}

extern "C" int ptfock_residual(ptfock_plan *plan, const void *psi, const void *hpsi, const void *psi_half, int32_t n, double dt,
                               void *r_out, void *stream) {
    if (!plan || !psi || !hpsi || !r_out || n < 1 || !std::isfinite(dt)) return PTFOCK_ERR_INVALID_ARG;
    int rc = check_dev_ptrs(plan, { psi, hpsi, psi_half, r_out });
    if (rc != PTFOCK_OK) return rc;
    const size_t gbytes = sizeof(cd) * (size_t)plan->N;
    if (overlaps(r_out, gbytes * n, psi, gbytes * n)) return PTFOCK_ERR_ALIAS;      // every CTA reads all of Psi
    const size_t s_bytes = sizeof(cd) * (size_t)n * n;
    if (s_bytes * 2 > plan->scratch_bytes) return PTFOCK_ERR_ALLOC;
    cudaStream_t st = (cudaStream_t)stream;
    GUARD(plan->d.device);
    BEGIN_CALL(plan, st);
    cd *S = plan->scratch;
    rc = overlap_into(plan, (const cd *)psi, n, (const cd *)hpsi, n, S, n, plan->scratch + (size_t)n * n,
                      plan->scratch_bytes - s_bytes, st);                          // Alg. 3 lines 2-3
    if (rc != PTFOCK_OK) return rc;
    RotateArgs g = {};
    g.a = (const cd *)psi; g.s = S; g.h = (const cd *)hpsi; g.p = (const cd *)psi; g.q = (const cd *)psi_half; g.out = (cd *)r_out;
    g.n_pts = plan->N; g.n_a = n; g.n_out = n; g.ld = n;
    g.mode = psi_half ? 2 : 1;
    g.fx = 0.0; g.fy = 0.5 * dt;                                                   // f = i dt / 2
    rotate_launch(plan, g, st);                                                    // Alg. 3 lines 4-5 fused
    CU(cudaGetLastError());
    END_CALL();
    return PTFOCK_OK;
}

extern "C" int ptfock_density(ptfock_plan *plan, const void *psi, int32_t n, double *rho, void *stream) {
    if (!plan || !psi || !rho || n < 1) return PTFOCK_ERR_INVALID_ARG;
    int rc = check_dev_ptrs(plan, { psi });
    if (rc != PTFOCK_OK) return rc;
    rc = check_dev_doubles(plan, rho);
    if (rc != PTFOCK_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    GUARD(plan->d.device);
    BEGIN_CALL(plan, st);
    const long long blocks = (plan->N + 255) / 256;
    int splits = (int)std::max<long long>(1, std::min<long long>(n, (8LL * plan->sm_count + blocks - 1) / blocks));
    splits = (int)std::min<size_t>((size_t)splits, plan->scratch_bytes / (sizeof(double) * (size_t)plan->N));
    if (splits < 1) return PTFOCK_ERR_ALLOC;
    const int per = (n + splits - 1) / splits;
    splits = (n + per - 1) / per;
    double *part = reinterpret_cast<double *>(plan->scratch);
    density_partial<<<dim3((unsigned)blocks, splits), 256, 0, st>>>((const cd *)psi, plan->N, n, per, part);
    density_reduce<<<(unsigned)blocks, 256, 0, st>>>(part, plan->N, splits, rho);
    plan->total_launches += 2;
    CU(cudaGetLastError());
    END_CALL();
    return PTFOCK_OK;
}

extern "C" int ptfock_orthonormalize(ptfock_plan *plan, void *psi, int32_t n, void *stream) {
    if (!plan || !psi || n < 1) return PTFOCK_ERR_INVALID_ARG;
    int rc = check_dev_ptrs(plan, { psi });
    if (rc != PTFOCK_OK) return rc;
    const int np = (n + 63) / 64 * 64;
    const size_t s_bytes = sizeof(cd) * ((size_t)np * np + np);        // S, then the saved diagonal
    if (s_bytes + sizeof(cd) * (size_t)n * n > plan->scratch_bytes) return PTFOCK_ERR_ALLOC;
    cudaStream_t st = (cudaStream_t)stream;
    GUARD(plan->d.device);
    if (!plan->chol_info || !plan->chol_info_host) {                    // either allocation may have failed in an earlier call
        CU(cudaFuncSetAttribute(chol_diag, cudaFuncAttributeMaxDynamicSharedMemorySize, kBlkSmem));
        CU(cudaFuncSetAttribute(tri_solve_block, cudaFuncAttributeMaxDynamicSharedMemorySize, kBlkSmem));
        if (!plan->chol_info && cudaMalloc(&plan->chol_info, sizeof(int)) != cudaSuccess) {
            plan->chol_info = nullptr; cudaGetLastError(); return PTFOCK_ERR_ALLOC;
        }
        if (!plan->chol_info_host && cudaMallocHost(&plan->chol_info_host, sizeof(int)) != cudaSuccess) {
            plan->chol_info_host = nullptr; cudaGetLastError(); return PTFOCK_ERR_ALLOC;
        }
    }
    BEGIN_CALL(plan, st);
    cd *S = plan->scratch, *X = (cd *)psi;
    CU(cudaMemsetAsync(plan->chol_info, 0, sizeof(int), st));
    // S = Psi^* Psi, padded with the identity to a multiple of the block size
    double *diag0 = reinterpret_cast<double *>(plan->scratch + (size_t)np * np);
    rc = overlap_into(plan, X, n, X, n, S, np, plan->scratch + (size_t)np * np + np, plan->scratch_bytes - s_bytes, st);
    if (rc != PTFOCK_OK) return rc;
    if (np != n) pad_identity<<<(unsigned)(((long long)np * np + 255) / 256), 256, 0, st>>>(S, np, n, np);
    save_diag<<<(np + 255) / 256, 256, 0, st>>>(S, np, np, diag0);
    // blocked right-looking Cholesky S = L L^H (lower triangle, in place)
    for (int k0 = 0; k0 < np; k0 += 64) {
        chol_diag<<<1, 64, kBlkSmem, st>>>(S, np, k0, diag0, plan->chol_info);
        const int below = np - k0 - 64;
        if (below > 0) {
            tri_solve_block<<<(below + 127) / 128, 128, kBlkSmem, st>>>(S + (size_t)(k0 + 64) * np + k0, below, np, 1, S, np, k0, 64);
            const int t = below / 64;
            chol_update<<<t * (t + 1) / 2, 256, 0, st>>>(S, np, k0, np);
            plan->total_launches += 2;
        }
        plan->total_launches += 1;
    }
    // Psi <- Psi L^{-H}, 64 columns at a time: subtract the finished columns' part, then solve against the diagonal block
    for (int c0 = 0; c0 < n; c0 += 64) {
        const int nc = std::min(64, n - c0);
        if (c0 > 0) {
            RotateArgs g = {};
            g.a = X; g.s = S; g.out = X; g.n_pts = plan->N; g.n_a = c0; g.n_out = nc; g.ld = np; g.conj_t = 1; g.mode = 3; g.n_first = c0;
            rotate_launch(plan, g, st);
        }
        tri_solve_block<<<(unsigned)((plan->N + 127) / 128), 128, kBlkSmem, st>>>(X + (size_t)c0 * plan->N, plan->N, 1, plan->N, S, np, c0, nc);
        plan->total_launches += 1;
    }
    CU(cudaGetLastError());
    CU(cudaMemcpyAsync(plan->chol_info_host, plan->chol_info, sizeof(int), cudaMemcpyDeviceToHost, st));
    END_CALL();
    CU(cudaStreamSynchronize(st));
    return *plan->chol_info_host ? PTFOCK_ERR_NOT_POSITIVE : PTFOCK_OK;
}

// ================================================================================================
// PT-CN step helpers (Alg. 1, PAPER.md:194-198 Anderson mixing)
// ================================================================================================
namespace {
__global__ void __launch_bounds__(256) add_vloc_kernel(const double *vloc, const cd *psi, cd *out, long long n_pts, long long total) {
    const long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= total) return;
    const double v = vloc[k % n_pts];
    const cd z = psi[k];
    cd o = out[k];
    o.x = fma(v, z.x, o.x);
    o.y = fma(v, z.y, o.y);
    out[k] = o;
}
// out_j = a_j x_j + b_j y_j (y may be null) for the kAxpbyChunk orbitals from j0 on; the coefficients travel by value in the
// kernel's parameter space, so the caller's host arrays are free again when the launch returns (pinned or pageable)
constexpr int kAxpbyChunk = 64;
struct AxpbyCoef { cd a[kAxpbyChunk], b[kAxpbyChunk]; };
__global__ void __launch_bounds__(256) axpby_kernel(const __grid_constant__ AxpbyCoef coef, int j0, const cd *x, const cd *y, cd *out, long long n_pts) {
    const long long r = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const int c = blockIdx.y;
    if (r >= n_pts) return;
    const long long k = (long long)(j0 + c) * n_pts + r;
    cd v = cmul(coef.a[c], x[k]);
    if (y) v = cadd(v, cmul(coef.b[c], y[k]));
    out[k] = v;
}
// v_out = v_ext + g rho (v_ext may be null = 0)
__global__ void __launch_bounds__(256) vloc_update_kernel(const double *v_ext, double g, const double *rho, double *v_out, long long n_pts) {
    const long long r = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= n_pts) return;
    v_out[r] = fma(g, rho[r], v_ext ? v_ext[r] : 0.0);
}
// partial[b] = (sum over block b's grid-stride points of |a - b|, 0)
__global__ void __launch_bounds__(256) absdiff_partial(const double *a, const double *b, long long n, double2 *partial) {
    __shared__ double red[256];
    double sacc = 0.0;
    for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (long long)gridDim.x * blockDim.x) sacc += fabs(a[k] - b[k]);
    red[threadIdx.x] = sacc;
    __syncthreads();
    for (int h = 128; h > 0; h >>= 1) {
        if (threadIdx.x < h) red[threadIdx.x] += red[threadIdx.x + h];
        __syncthreads();
    }
    if (threadIdx.x == 0) partial[blockIdx.x] = make_double2(red[0], 0.0);
}
// part[j][b] = sum over block b's points of conj(a_j) b_j; out[j] = w * sum_b part[j][b] (fixed order)
__global__ void __launch_bounds__(256) banddot_partial(const cd *a, const cd *b, long long n_pts, int blocks_per, double2 *part) {
    __shared__ double2 red[256];
    const int j = blockIdx.y;
    double sr = 0.0, si = 0.0;
    for (long long r = (long long)blockIdx.x * 256 + threadIdx.x; r < n_pts; r += (long long)blocks_per * 256) {
        const cd x = a[(long long)j * n_pts + r], y = b[(long long)j * n_pts + r];
        sr += x.x * y.x + x.y * y.y;
        si += x.x * y.y - x.y * y.x;
    }
    red[threadIdx.x] = make_double2(sr, si);
    __syncthreads();
    for (int h = 128; h > 0; h >>= 1) {
        if (threadIdx.x < h) { red[threadIdx.x].x += red[threadIdx.x + h].x; red[threadIdx.x].y += red[threadIdx.x + h].y; }
        __syncthreads();
    }
    if (threadIdx.x == 0) part[(long long)j * blocks_per + blockIdx.x] = red[0];
}
__global__ void __launch_bounds__(64) banddot_final(const double2 *part, int blocks_per, int n, double w, double2 *out) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n) return;
    double sr = 0.0, si = 0.0;
    for (int b = 0; b < blocks_per; ++b) { sr += part[(long long)j * blocks_per + b].x; si += part[(long long)j * blocks_per + b].y; }
    out[j] = make_double2(sr * w, si * w);
}
}  // namespace

extern "C" int ptfock_hloc_apply(ptfock_plan *plan, const double *vloc, const void *psi, int32_t n, void *out, void *stream) {
    if (!plan || !psi || !out || n < 1 || plan->d.kernel != PTFOCK_KERNEL_KINETIC) return PTFOCK_ERR_INVALID_ARG;
    int rc = check_dev_ptrs(plan, { psi, out });
    if (rc != PTFOCK_OK) return rc;
    rc = check_dev_doubles(plan, vloc);
    if (rc != PTFOCK_OK) return rc;
    const size_t gbytes = sizeof(cd) * (size_t)plan->N;
    if (overlaps(out, gbytes * n, psi, gbytes * n)) return PTFOCK_ERR_ALIAS;
    cudaStream_t st = (cudaStream_t)stream;
    GUARD(plan->d.device);
    BEGIN_CALL(plan, st);
    if (!plan->ones) {
        cudaError_t e = cudaMalloc(&plan->ones, gbytes);
        if (e != cudaSuccess) { g_last_cuda = (int)e; return PTFOCK_ERR_ALLOC; }
        fill_ones<<<(unsigned)((plan->N + 255) / 256), 256, 0, st>>>(plan->ones, plan->N);
    }
    // T psi_j = IFFT[ |G|^2/2 FFT(conj(1) psi_j) ] * 1: the exchange passes with the constant orbital and the kinetic table
    rc = apply_device(plan, plan->ones, (const cd *)psi, 0, n, (cd *)out, st);
    if (rc != PTFOCK_OK) return rc;
    if (vloc) {
        const long long total = plan->N * (long long)n;
        add_vloc_kernel<<<(unsigned)((total + 255) / 256), 256, 0, st>>>(vloc, (const cd *)psi, (cd *)out, plan->N, total);
        plan->total_launches += 1;
    }
    CU(cudaGetLastError());
    END_CALL();
    return PTFOCK_OK;
}

extern "C" int ptfock_axpby(ptfock_plan *plan, int32_t n, const double *a_host, const void *x, const double *b_host, const void *y,
                            void *out, void *stream) {
    if (!plan || !a_host || !x || !out || n < 1 || (y && !b_host)) return PTFOCK_ERR_INVALID_ARG;
    int rc = check_dev_ptrs(plan, { x, y, out });
    if (rc != PTFOCK_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    GUARD(plan->d.device);
    BEGIN_CALL(plan, st);
    for (int j0 = 0; j0 < n; j0 += kAxpbyChunk) {
        const int nc = std::min(kAxpbyChunk, n - j0);
        AxpbyCoef coef;
        std::memset(&coef, 0, sizeof(coef));
        std::memcpy(coef.a, a_host + 2 * (size_t)j0, sizeof(cd) * nc);
        if (y) std::memcpy(coef.b, b_host + 2 * (size_t)j0, sizeof(cd) * nc);
        axpby_kernel<<<dim3((unsigned)((plan->N + 255) / 256), nc), 256, 0, st>>>(coef, j0, (const cd *)x, (const cd *)y, (cd *)out, plan->N);
        plan->total_launches += 1;
    }
    CU(cudaGetLastError());
    END_CALL();
    return PTFOCK_OK;
}

extern "C" int ptfock_banddot(ptfock_plan *plan, const void *a, const void *b, int32_t n, double *out_host, void *stream) {
    if (!plan || !a || !b || !out_host || n < 1) return PTFOCK_ERR_INVALID_ARG;
    int rc = check_dev_ptrs(plan, { a, b });
    if (rc != PTFOCK_OK) return rc;
    const int blocks_per = (int)std::max<long long>(1, std::min<long long>(64, plan->N / 2048));
    if (sizeof(double2) * (size_t)n * (blocks_per + 1) > plan->scratch_bytes) return PTFOCK_ERR_ALLOC;
    cudaStream_t st = (cudaStream_t)stream;
    GUARD(plan->d.device);
    BEGIN_CALL(plan, st);
    double2 *part = reinterpret_cast<double2 *>(plan->scratch), *res = part + (size_t)n * blocks_per;
    banddot_partial<<<dim3(blocks_per, n), 256, 0, st>>>((const cd *)a, (const cd *)b, plan->N, blocks_per, part);
    banddot_final<<<(n + 63) / 64, 64, 0, st>>>(part, blocks_per, n, plan->volume / (double)plan->N, res);
    plan->total_launches += 2;
    CU(cudaGetLastError());
    CU(cudaMemcpyAsync(out_host, res, sizeof(double2) * n, cudaMemcpyDeviceToHost, st));
    END_CALL();
    CU(cudaStreamSynchronize(st));
    return PTFOCK_OK;
}

extern "C" int ptfock_vloc_update(ptfock_plan *plan, const double *v_ext, double g, const double *rho, double *v_out, void *stream) {
    if (!plan || !rho || !v_out) return PTFOCK_ERR_INVALID_ARG;
    for (const double *q : { v_ext, rho, (const double *)v_out }) {
        int rc = check_dev_doubles(plan, q);
        if (rc != PTFOCK_OK) return rc;
    }
    cudaStream_t st = (cudaStream_t)stream;
    GUARD(plan->d.device);
    vloc_update_kernel<<<(unsigned)((plan->N + 255) / 256), 256, 0, st>>>(v_ext, g, rho, v_out, plan->N);
    plan->total_launches += 1;
    CU(cudaGetLastError());
    return PTFOCK_OK;
}

extern "C" int ptfock_density_change(ptfock_plan *plan, const double *rho_a, const double *rho_b, double *change_host, void *stream) {
    if (!plan || !rho_a || !rho_b || !change_host) return PTFOCK_ERR_INVALID_ARG;
    for (const double *q : { rho_a, rho_b }) {
        int rc = check_dev_doubles(plan, q);
        if (rc != PTFOCK_OK) return rc;
    }
    cudaStream_t st = (cudaStream_t)stream;
    GUARD(plan->d.device);
    BEGIN_CALL(plan, st);                                                // plan->partials / result buffers are shared by consecutive calls
    const int blocks = (int)std::min<long long>(1024, (plan->N + 255) / 256);
    absdiff_partial<<<blocks, 256, 0, st>>>(rho_a, rho_b, plan->N, plan->partials);
    dot_final<<<1, 256, 0, st>>>(plan->partials, blocks, plan->volume / (double)plan->N, plan->result_dev);
    plan->total_launches += 2;
    CU(cudaGetLastError());
    CU(cudaMemcpyAsync(plan->result_host, plan->result_dev, sizeof(double2), cudaMemcpyDeviceToHost, st));
    END_CALL();
    CU(cudaStreamSynchronize(st));
    *change_host = plan->result_host->x;
    return PTFOCK_OK;
}

// out_host[(k * n + j)] = (a_j, b^k_j) for k < n_sets: the inner products of one orbital set with n_sets others in ONE call
// (one synchronisation): a new row of the Anderson Gram matrices and their right-hand sides
extern "C" int ptfock_banddot_many(ptfock_plan *plan, const void *a, const void *const *b_sets_host, int32_t n_sets, int32_t n,
                                   double *out_host, void *stream) {
    if (!plan || !a || !b_sets_host || !out_host || n < 1 || n_sets < 1) return PTFOCK_ERR_INVALID_ARG;
    int rc = check_dev_ptrs(plan, { a });
    if (rc != PTFOCK_OK) return rc;
    for (int k = 0; k < n_sets; ++k) {
        if (!b_sets_host[k]) return PTFOCK_ERR_INVALID_ARG;
        rc = check_dev_ptrs(plan, { b_sets_host[k] });
        if (rc != PTFOCK_OK) return rc;
    }
    const int blocks_per = (int)std::max<long long>(1, std::min<long long>(64, plan->N / 2048));
    const size_t per_set = (size_t)n * (blocks_per + 1);                 // partial sums + results of one set
    if (sizeof(double2) * per_set * (size_t)n_sets > plan->scratch_bytes) return PTFOCK_ERR_ALLOC;
    cudaStream_t st = (cudaStream_t)stream;
    GUARD(plan->d.device);
    BEGIN_CALL(plan, st);
    double2 *part = reinterpret_cast<double2 *>(plan->scratch), *res = part + (size_t)n_sets * n * blocks_per;
    for (int k = 0; k < n_sets; ++k) {
        banddot_partial<<<dim3(blocks_per, n), 256, 0, st>>>((const cd *)a, (const cd *)b_sets_host[k], plan->N, blocks_per,
                                                             part + (size_t)k * n * blocks_per);
        banddot_final<<<(n + 63) / 64, 64, 0, st>>>(part + (size_t)k * n * blocks_per, blocks_per, n, plan->volume / (double)plan->N,
                                                     res + (size_t)k * n);
    }
    plan->total_launches += 2 * n_sets;
    CU(cudaGetLastError());
    CU(cudaMemcpyAsync(out_host, res, sizeof(double2) * (size_t)n * n_sets, cudaMemcpyDeviceToHost, st));
    END_CALL();
    CU(cudaStreamSynchronize(st));
    return PTFOCK_OK;
}

// ---- ptfock_banddot_static: the same two kernels with their partial sums in a built-in array (no allocation) ----------
// For callers that must not trigger a cudaMalloc (all HBM owned by their own pool, or a loop whose other streams a
// device-wide synchronising allocation would stall); see include/ptfock.h.
namespace {
constexpr int kStaticBlocksPer = 64;                                    // the most blocks per band banddot_partial is launched with
constexpr int kStaticMaxDevices = 64;
// Per-block partial sums of one call: [band][block].  One copy per GPU that loads the library (4 MiB), alive until exit.
// Host code must NOT hand this name to a kernel: on the host it is only a handle for cudaGetSymbolAddress.
static __device__ __align__(256) double2 g_banddot_static_part[(size_t)PTFOCK_STATIC_MAX_BANDS * kStaticBlocksPer];
double2 *g_static_part_addr[kStaticMaxDevices] = {};                    // device address of the array, per ordinal (0 = not looked up yet)
std::mutex g_static_mu;

// `device` is current.  Looks the array's device address up once per device; no allocation.
int static_part_address(int device, double2 **out) {
    std::lock_guard<std::mutex> lk(g_static_mu);
    if (!g_static_part_addr[device]) {
        void *p = nullptr;
        CU(cudaGetSymbolAddress(&p, g_banddot_static_part));
        if (!p) return PTFOCK_ERR_CUDA;
        g_static_part_addr[device] = static_cast<double2 *>(p);
    }
    *out = g_static_part_addr[device];
    return PTFOCK_OK;
}
}  // namespace

extern "C" int ptfock_banddot_static(int32_t device, int64_t n_points, double weight, const void *a, const void *b, int32_t n,
                                     void *out, void *stream) {
    if (!a || !b || !out || n < 1 || n_points < 1 || device < 0 || device >= kStaticMaxDevices) return PTFOCK_ERR_INVALID_ARG;
    if (n > PTFOCK_STATIC_MAX_BANDS) return PTFOCK_ERR_TOO_LARGE;
    int count = 0;
    CU(cudaGetDeviceCount(&count));
    if (device >= count) return PTFOCK_ERR_INVALID_ARG;
    for (const void *q : { a, b, (const void *)out }) {
        if ((uintptr_t)q & 15) return PTFOCK_ERR_ALIGNMENT;
        cudaPointerAttributes at;
        if (cudaPointerGetAttributes(&at, q) != cudaSuccess) { cudaGetLastError(); return PTFOCK_ERR_INVALID_ARG; }
        if (at.type == cudaMemoryTypeManaged) continue;
        if (at.type != cudaMemoryTypeDevice || at.device != device) return PTFOCK_ERR_INVALID_ARG;
    }
    cudaStream_t st = (cudaStream_t)stream;
    GUARD(device);
    double2 *part = nullptr;
    int rc = static_part_address(device, &part);                        // first call on this device: cudaGetSymbolAddress
    if (rc != PTFOCK_OK) return rc;
    // same launch shape as ptfock_banddot, so the sums are taken in the same order; every part[j][0 .. blocks_per) that
    // banddot_final reads is written by banddot_partial first, so what an earlier call left in the array does not matter
    const int blocks_per = (int)std::max<long long>(1, std::min<long long>(kStaticBlocksPer, n_points / 2048));
    banddot_partial<<<dim3(blocks_per, n), 256, 0, st>>>((const cd *)a, (const cd *)b, n_points, blocks_per, part);
    banddot_final<<<(n + 63) / 64, 64, 0, st>>>(part, blocks_per, n, weight, (double2 *)out);
    CU(cudaGetLastError());
    return PTFOCK_OK;
}

namespace {
int measure_fp64_peak(int32_t device, bool tensor, double *tflops_host);
}
extern "C" int ptfock_measure_dfma_peak(int32_t device, double *tflops_host) { return measure_fp64_peak(device, false, tflops_host); }
extern "C" int ptfock_measure_dmma_peak(int32_t device, double *tflops_host) { return measure_fp64_peak(device, true, tflops_host); }
namespace {
int measure_fp64_peak(int32_t device, bool tensor, double *tflops_host) {
    if (!tflops_host) return PTFOCK_ERR_INVALID_ARG;
    GUARD(device);
    cudaDeviceProp prop;
    CU(cudaGetDeviceProperties(&prop, device));
    if (prop.major != 10) return PTFOCK_ERR_UNSUPPORTED_DEVICE;
    double *sink = nullptr;
    CU(cudaMalloc(&sink, sizeof(double)));
    cudaEvent_t e0, e1;
    CU(cudaEventCreate(&e0));
    CU(cudaEventCreate(&e1));
    const int blocks = prop.multiProcessorCount * 8, iters = 1 << 16;
    double best = 0.0;
    for (int rep = 0; rep < 6; ++rep) {             // first repetitions warm the clocks up
        cudaEventRecord(e0, 0);
        if (tensor) dmma_peak_kernel<<<blocks, 256>>>(sink, iters, 1e-3, 1e-3);
        else fp64_peak_kernel<<<blocks, 256>>>(sink, iters, 1.0000001, 1e-9);
        cudaEventRecord(e1, 0);
        cudaError_t e = cudaEventSynchronize(e1);
        if (e != cudaSuccess) { g_last_cuda = (int)e; cudaFree(sink); return PTFOCK_ERR_CUDA; }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        // per thread and iteration: 8 DFMAs, or 8 warp-wide 8 x 8 x 4 MMAs (256 FMAs shared by 32 lanes = 8 per lane)
        const double tf = (tensor ? 8.0 : 1.0) * 2.0 * 8.0 * (double)iters * 256.0 * blocks / (ms * 1e-3) / 1e12;
        if (rep >= 2 && tf > best) best = tf;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(sink);
    *tflops_host = best;
    return PTFOCK_OK;
}
}  // namespace

extern "C" int ptfock_measure_copy_bandwidth(int32_t device, uint64_t bytes, int32_t reps, double *gbs_host) {
    if (!gbs_host || bytes < 4096 || reps < 1) return PTFOCK_ERR_INVALID_ARG;
    GUARD(device);
    cudaDeviceProp prop;
    CU(cudaGetDeviceProperties(&prop, device));
    if (prop.major != 10) return PTFOCK_ERR_UNSUPPORTED_DEVICE;
    const long long n = (long long)(bytes / sizeof(double2));
    double2 *src = nullptr, *dst = nullptr;
    if (cudaMalloc(&src, n * sizeof(double2)) != cudaSuccess) return PTFOCK_ERR_ALLOC;
    if (cudaMalloc(&dst, n * sizeof(double2)) != cudaSuccess) { cudaFree(src); return PTFOCK_ERR_ALLOC; }
    cudaMemset(src, 0, n * sizeof(double2));
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    const int blocks = prop.multiProcessorCount * 8;
    double best = 0.0;
    int rc = PTFOCK_OK;
    for (int rep = 0; rep < 5 && rc == PTFOCK_OK; ++rep) {          // the working set stays where the previous pass left it
        cudaEventRecord(e0, 0);
        for (int r = 0; r < reps; ++r) copy_bw_kernel<<<blocks, 256>>>(src, dst, n);
        cudaEventRecord(e1, 0);
        cudaError_t e = cudaEventSynchronize(e1);
        if (e != cudaSuccess) { g_last_cuda = (int)e; rc = PTFOCK_ERR_CUDA; break; }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        const double gbs = 2.0 * (double)n * sizeof(double2) * reps / (ms * 1e-3) / 1e9;
        if (rep >= 1 && gbs > best) best = gbs;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(src);
    cudaFree(dst);
    *gbs_host = best;
    return rc;
}

extern "C" int ptfock_set_profiling(ptfock_plan *plan, int32_t on) {
    if (!plan) return PTFOCK_ERR_INVALID_ARG;
    plan->profiling = on ? 1 : 0;
    return PTFOCK_OK;
}

extern "C" int ptfock_get_profile(ptfock_plan *plan, double ms[3], int64_t launches[3], int32_t reset) {
    if (!plan || !ms || !launches) return PTFOCK_ERR_INVALID_ARG;
    for (int k = 0; k < 3; ++k) { ms[k] = 0.0; launches[k] = 0; }
    if (plan->ev_pool && plan->ev_used > 0) {
        GUARD(plan->d.device);
        CU(cudaEventSynchronize((*plan->ev_pool)[plan->ev_used - 1]));
        for (size_t k = 1; k < plan->ev_used; ++k) {
            const int tag = (*plan->ev_tags)[k];
            if (tag < 0) continue;
            float t = 0.f;
            CU(cudaEventElapsedTime(&t, (*plan->ev_pool)[k - 1], (*plan->ev_pool)[k]));
            ms[tag] += (double)t;
            launches[tag] += 1;
        }
    }
    if (reset) plan->ev_used = 0;
    return PTFOCK_OK;
}
