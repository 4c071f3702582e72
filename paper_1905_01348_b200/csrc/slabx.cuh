// slabx.cuh -- TMA-fed, in-place slab passes (pass A and pass C of the BASELINE shapes 64x64 and 128x48).
//
// Same three butterfly stages per (x1, x2) slab as the generic slab passes of kernels.cuh, ordered so that every byte
// that crosses the L1/shared-memory pipe is useful (ncu on a round-1 predecessor of these kernels: the LSU data pipe
// was the busiest unit, and its orbital loads touched only half of every 128-byte line):
//
//   * x1 is transformed FIRST and x2 LAST.  Stage 1 threads own points that are consecutive in x2, so the
//     psi_j / phi_i / out accesses of Eq. (3)'s products (Alg. 2 lines 7-9,
//     PAPER.md:135-138) are full 128-byte lines.
//   * The slab order inside the pair scratch is free (pass B only needs "same order as the v' table"):
//     stage-3 thread t writes its m-th output at  m*NT3 + t, so scratch stores (pass A) and scratch loads
//     (pass C) are perfectly coalesced as well.  Position s = m*NT3 + k2a*N1 + k1 holds the frequencies
//     k1 (natural order) and k2 = k2a + A2*m.
//   * phi_i slabs (pass A) and pair-density slabs (pass C) are brought in by 1-D bulk async copies (TMA,
//     cp.async.bulk + mbarrier) straight into the padded tile the butterflies then work on IN PLACE, two
//     or three tiles rotating; nothing is prefetched through registers, so 256 threads x <= 255 registers
//     hold psi_j (pass A) or the sum over i (pass C) without spills, also for the 24-point stage of 128x48.
//
// Digit structure (decimation in frequency, mirrored in pass C):  x1 = a1*B1 + b1,  x2 = a2*B2 + b2
//   kind P (64x64 : A1=16 B1=4 A2=4 B2=16):  S1 = DFT over a1 | S2 = 2-D DFT over (b1, a2) | S3 = DFT over b2
//   kind Q (128x48: A1=8 B1=16 A2=3 B2=16):  S1 = 2-D DFT over (a1, a2) | S2 = DFT over b1  | S3 = DFT over b2
// S1 has exactly 256 tasks (one per thread: psi_j / the accumulators live in its registers).
#pragma once
#include "kernels.cuh"
#include "tma.cuh"

namespace ptfock {

// TS_: pass A hands its finished tile to bulk async STORES (the scratch slab is then the tile's own order,
// [pos1][pos2], and pass C works in the pass A layout); otherwise stage 3 stores from registers in the free
// layout above.  Needs three rotating tiles (the store has to drain before the tile is refilled).
template <int N1_, int N2_, int A1_, int B1_, int A2_, int B2_, bool Q_, bool TS_, int MINB_ = 1>
struct SX {
    static constexpr int MINB = MINB_;                      // CTAs per SM the register budget is capped for
    static constexpr int N1 = N1_, N2 = N2_, A1 = A1_, B1 = B1_, A2 = A2_, B2 = B2_;
    static constexpr bool Q = Q_, TS = TS_, CLAYOUT = !TS_;
    static_assert(A1 * B1 == N1 && A2 * B2 == N2, "bad split");
    static constexpr int NPTS = N1 * N2;
    static constexpr int R1 = A1, C1 = Q ? A2 : 1;          // stage-1 butterfly: R1 x C1 points
    static constexpr int R2 = B1, C2 = Q ? 1 : A2;          // stage-2 butterfly
    static constexpr int CB1 = Q ? B2 : N2;                 // stage-1 tasks: (b1, cb)
    static constexpr int CB2 = Q ? N2 : B2;                 // stage-2 tasks: (k1a, cb)
    static constexpr int NT1 = B1 * CB1, NT2 = A1 * CB2, NT3 = N1 * A2;
    static constexpr int NT = (NT1 + 31) / 32 * 32;         // stage 1: one task per thread (threads >= NT1 sit it out)
    static_assert(NT <= 512 && (Q || NT2 <= NT), "bad thread count");
    static constexpr int PM = NT3 + 1;                      // pass C tile (free layout): [m][k2a][k1], odd pitch
    static constexpr int TILE_A = A1 * (B1 * N2 + 1), TILE_C = TS ? TILE_A : B2 * PM;   // elements (Addr below)
    static constexpr int MAXSM = 232448 - 64;
    static constexpr int NBUF_A = (3 * TILE_A * 16 <= MAXSM) ? 3 : 2;
    static constexpr int NBUF_C = (3 * TILE_C * 16 <= MAXSM) ? 3 : 2;
    static constexpr int SMEM_A = NBUF_A * TILE_A * 16 + 64;
    static constexpr int SMEM_C = NBUF_C * TILE_C * 16 + 64 + (Q ? (N1 + N2) * 16 : 0);   // + twiddle tables (Q)
    static_assert(!TS || NBUF_A == 3, "bulk stores need three tiles");
    static constexpr bool FUSE = NBUF_A == 3 && NBUF_C == 3;     // stage 3 of one orbital next to stage 1 of the next
    static constexpr int NTWR = (Q ? A1 : B1) > 1 ? (Q ? A1 : B1) - 1 : 1;
    static constexpr int NTWC = A2 > 1 ? A2 - 1 : 1;
};

// u[r*C + c] <-> p[r*SR + c*SC]
template <int R, int C, int SR, int SC>
PTF_DEV void tile_load(cd (&u)[R * C], const cd *p) {
#pragma unroll
    for (int r = 0; r < R; ++r)
#pragma unroll
        for (int c = 0; c < C; ++c) u[r * C + c] = p[r * SR + c * SC];
}
// same, from global memory past L1 (streamed once: keep the L1/shared SRAM for the tiles)
template <int R, int C, int SR, int SC>
PTF_DEV void tile_load_cg(cd (&u)[R * C], const cd *p) {
#pragma unroll
    for (int r = 0; r < R; ++r)
#pragma unroll
        for (int c = 0; c < C; ++c) u[r * C + c] = __ldcg(reinterpret_cast<const double2 *>(p + r * SR + c * SC));
}
template <int R, int C, int SR, int SC>
PTF_DEV void tile_store(const cd (&u)[R * C], cd *p) {
#pragma unroll
    for (int r = 0; r < R; ++r)
#pragma unroll
        for (int c = 0; c < C; ++c) p[r * SR + c * SC] = u[r * C + c];
}
template <int R, int C, bool INV>
PTF_DEV void dft_over_r(cd (&u)[R * C]) {
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
template <int R, int C, bool INV>
PTF_DEV void dft_over_c(cd (&u)[R * C]) {
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
template <int R, int C, bool CONJ>
PTF_DEV void tw_rows(cd (&u)[R * C], const cd *tw) {        // u[r][.] *= tw[r-1]
#pragma unroll
    for (int r = 1; r < R; ++r)
#pragma unroll
        for (int c = 0; c < C; ++c) u[r * C + c] = CONJ ? cmulc(u[r * C + c], tw[r - 1]) : cmul(u[r * C + c], tw[r - 1]);
}
template <int R, int C, bool CONJ>
PTF_DEV void tw_cols(cd (&u)[R * C], const cd *tw) {        // u[.][c] *= tw[c-1]
#pragma unroll
    for (int c = 1; c < C; ++c)
#pragma unroll
        for (int r = 0; r < R; ++r) u[r * C + c] = CONJ ? cmulc(u[r * C + c], tw[c - 1]) : cmul(u[r * C + c], tw[c - 1]);
}

// The twiddled stage (P: stage 2, Q: stage 1) of thread `t`:  twr = w_N1^(b1*k1a) (P: over b1, task k1a;
// Q: over k1a, task b1), twc = w_N2^(b2*k2a) over k2a for the task's b2.
template <class S>
PTF_DEV void load_twiddles(const cd *tw1, const cd *tw2, int t, cd (&twr)[S::NTWR], cd (&twc)[S::NTWC]) {
    const int cb = t % (S::Q ? S::CB1 : S::CB2), rb = t / (S::Q ? S::CB1 : S::CB2);   // Q: (b2, b1)   P: (b2, k1a)
#pragma unroll
    for (int q = 1; q <= (S::Q ? S::A1 : S::B1) - 1; ++q) twr[q - 1] = tw1[q * rb];
#pragma unroll
    for (int q = 1; q < S::A2; ++q) twc[q - 1] = tw2[q * cb];
}

// ---- tile addressing -------------------------------------------------------------------------------
// A row is named by its digits (k1a, b1): row = k1a*B1 + b1.
// pass A layout: A1 chunks of B1 dense rows, one element of padding per chunk (one bulk copy per chunk):
//                (k1a, b1, col) -> k1a*CH + b1*N2 + col,  CH = B1*N2 + 1.
// pass C layout: (k1a, b1, col) -> (col % B2)*PM + (col / B2)*N1 + (k1a + A1*b1)      [m][k2a][k1].
template <class S, bool CL> struct Addr {
    static constexpr int CH = S::B1 * S::N2 + 1;
    static constexpr int RA = CL ? 1 : CH;                           // stride of +1 in k1a / a1 (row += B1)
    static constexpr int RB = CL ? S::A1 : S::N2;                    // stride of +1 in b1 / k1b (row += 1)
    static constexpr int COLB = CL ? S::N1 : S::B2;                  // stride of +B2 columns (next a2 / k2a)
    static constexpr int COL1 = CL ? S::PM : 1;                      // stride of +1 column inside a B2 block
    static PTF_DEV int at(int k1a, int b1, int col) {
        return CL ? (col % S::B2) * S::PM + (col / S::B2) * S::N1 + k1a + S::A1 * b1 : k1a * CH + b1 * S::N2 + col;
    }
};

template <class S, bool CL> PTF_DEV int s1_base(int t) {             // element (a1, a2) at base + a1*RA + a2*COLB
    const int cb = t % S::CB1, b1 = t / S::CB1;
    return Addr<S, CL>::at(0, b1, cb);
}
template <class S, bool CL> PTF_DEV int s2_base(int t) {             // element (b1, a2) at base + b1*RB + a2*COLB
    const int cb = t % S::CB2, k1a = t / S::CB2;
    return Addr<S, CL>::at(k1a, 0, cb);
}
// stage-3 task t = k2a*N1 + k1 with k1 = k1a + A1*k1b: consecutive lanes sit in different chunks of the pass A
// tile (conflict-free), and k1 is the natural x1 frequency.
template <class S, bool CL> PTF_DEV int s3_base(int t) {             // element b2 at base + b2*COL1
    const int k1 = t % S::N1, k2a = t / S::N1;
    return Addr<S, CL>::at(k1 % S::A1, k1 / S::A1, k2a * S::B2);
}

// ---- bulk-copy issue (warp 0) -------------------------------------------------------------------------
PTF_DEV void l2_prefetch(const void *p, unsigned bytes) {
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p), "r"(bytes) : "memory");
}

// pass A: A1 chunks of B1 rows -> padded chunks
template <class S>
PTF_DEV void issue_rows(cd *tile, const cd *src, unsigned long long *bar, int lane) {
    if (lane == 0) mbar_expect_tx(bar, S::NPTS * 16u);
    __syncwarp();
    if (lane < S::A1) bulk_g2s(tile + lane * (S::B1 * S::N2 + 1), src + lane * (S::B1 * S::N2), S::B1 * S::N2 * 16u, bar);
}
// pass A with bulk stores: padded chunks -> A1 chunks of B1 rows of the scratch slab (one bulk group per lane)
PTF_DEV void bulk_s2g(void *dst_gmem, const void *src_smem, unsigned bytes) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst_gmem), "r"(smem_u32(src_smem)), "r"(bytes)
                 : "memory");
}
PTF_DEV void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
PTF_DEV void bulk_wait_read_all() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
template <class S>
PTF_DEV void store_rows(const cd *tile, cd *dst, int lane) {
    if (lane < S::A1) {
        bulk_s2g(dst + lane * (S::B1 * S::N2), tile + lane * (S::B1 * S::N2 + 1), S::B1 * S::N2 * 16u);
        bulk_commit();
    }
}
// pass C: B2 blocks of NT3 elements -> padded blocks
template <class S>
PTF_DEV void issue_blocks(cd *tile, const cd *src, unsigned long long *bar, int lane) {
    if (lane == 0) mbar_expect_tx(bar, S::NPTS * 16u);
    __syncwarp();
    if (lane < S::B2) bulk_g2s(tile + lane * S::PM, src + lane * S::NT3, S::NT3 * 16u, bar);
}

// ---- pass A ---------------------------------------------------------------------------------------
// grid = (targets in the wave, n0, chunks of the i loop)
template <class S>
__global__ void __launch_bounds__(S::NT, S::MINB) slabx_fwd(const SlabArgs g) {
    constexpr int N2 = S::N2, B1 = S::B1, B2 = S::B2, R1 = S::R1, C1 = S::C1, R2 = S::R2, C2 = S::C2;
    constexpr int NT = S::NT, NBUF = S::NBUF_A, TILE = S::TILE_A;
    using A = Addr<S, false>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cd *tiles = reinterpret_cast<cd *>(smem_raw);
    unsigned long long *bars = reinterpret_cast<unsigned long long *>(smem_raw + (size_t)NBUF * TILE * 16);
    const int tid = threadIdx.x, lane = tid & 31;
    const int x0 = blockIdx.y, jj = blockIdx.x;
    const long long slab_off = (long long)x0 * S::NPTS;
    const int per = (g.na + gridDim.z - 1) / gridDim.z;
    int ii_beg, ii_end;
    tri_range(g.tri, jj, blockIdx.z * per, min(g.na, blockIdx.z * per + per), ii_beg, ii_end);
    const int n_it = ii_end - ii_beg;
    if (n_it <= 0) return;
    const cd *phi0 = g.a + (long long)(g.a0 + ii_beg) * g.grid_pts + slab_off;      // slab of the first orbital
    if (tid == 0) {
#pragma unroll
        for (int b = 0; b < NBUF; ++b) mbar_init(&bars[b], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        fence_proxy_async();
    }
    __syncthreads();
    if (tid < 32) {
        for (int it = 0; it < NBUF - 1 && it < n_it; ++it)
            issue_rows<S>(tiles + it * TILE, phi0 + (long long)it * g.grid_pts, &bars[it], lane);
    }
    // stage-1 task of this thread: psi_j values in registers for the whole loop
    const int cb = tid % S::CB1, b1 = tid / S::CB1;
    const int base1 = s1_base<S, false>(tid);
    const bool act1 = S::NT1 == NT || tid < S::NT1;      // this thread owns a stage-1 task
    cd pj[R1 * C1];
    if (act1) {
        const cd *psi = g.b + (long long)(g.b0 + jj) * g.grid_pts + slab_off + b1 * N2 + cb;
        tile_load<R1, C1, B1 * N2, B2>(pj, psi);
    }
    cd twr[S::NTWR], twc[S::NTWC];
    load_twiddles<S>(g.tw1, g.tw2, (S::Q ? act1 : tid < S::NT2) ? tid : 0, twr, twc);
    const int base2 = s2_base<S, false>(tid);            // P: the twiddled stage-2 task of this thread

    // ---- stage 1: rho = psi_j conj(phi_i), DFT over a1 (Q: and a2, with both twiddles), in place
    auto stage1 = [&](cd *T) {
        if (!act1) return;
        cd u[R1 * C1];
        tile_load<R1, C1, A::RA, A::COLB>(u, T + base1);
#pragma unroll
        for (int k = 0; k < R1 * C1; ++k) u[k] = cmulc(pj[k], u[k]);
        dft_over_r<R1, C1, false>(u);
        if (S::Q) {
            tw_rows<R1, C1, false>(u, twr);
            dft_over_c<R1, C1, false>(u);
            tw_cols<R1, C1, false>(u, twc);
        }
        tile_store<R1, C1, A::RA, A::COLB>(u, T + base1);
    };
    auto stage2 = [&](cd *T) {
        if (S::Q) {
            for (int t = tid; t < S::NT2; t += NT) {
                cd u[R2 * C2];
                cd *p = T + s2_base<S, false>(t);
                tile_load<R2, C2, A::RB, A::COLB>(u, p);
                dft_over_r<R2, C2, false>(u);
                tile_store<R2, C2, A::RB, A::COLB>(u, p);
            }
        } else if (S::NT2 == NT || tid < S::NT2) {
            cd u[R2 * C2];
            tile_load<R2, C2, A::RB, A::COLB>(u, T + base2);
            tw_rows<R2, C2, false>(u, twr);
            dft_over_r<R2, C2, false>(u);
            dft_over_c<R2, C2, false>(u);
            tw_cols<R2, C2, false>(u, twc);
            tile_store<R2, C2, A::RB, A::COLB>(u, T + base2);
        }
    };
    // ---- stage 3: DFT over b2; TS: in place (the tile leaves by bulk stores), else registers -> scratch (m*NT3 + t)
    auto stage3 = [&](cd *T, int it) {
        cd *dst = g.scratch + ((long long)((ii_beg + it) * g.stride_loop + jj * g.stride_cta) * g.n0 + x0) * S::NPTS;
        for (int t = tid; t < S::NT3; t += NT) {
            cd w[B2];
            cd *p = T + s3_base<S, false>(t);
            tile_load<1, B2, 0, A::COL1>(w, p);
            DFT<B2, false>::run(w);
            if (S::TS) {
                tile_store<1, B2, 0, A::COL1>(w, p);
            } else {
#pragma unroll
                for (int m = 0; m < B2; ++m) dst[m * S::NT3 + t] = w[m];
            }
        }
    };
    auto refill = [&](int nx) {     // warp 0: tile nx % NBUF <- phi slab of loop index nx
        issue_rows<S>(tiles + (nx % NBUF) * TILE, phi0 + (long long)nx * g.grid_pts, &bars[nx % NBUF], lane);
    };

    mbar_wait(&bars[0], 0);
    stage1(tiles);
    for (int it = 0; it < n_it; ++it) {
        cd *T = tiles + (it % NBUF) * TILE;
        // here: stage 1 of orbital it and stage 3 of orbital it-1 are done by this thread
        fence_proxy_async();
        __syncthreads();
        if (S::TS) {
            if (tid < 32 && it >= 1)    // the previous orbital's finished tile goes out as bulk stores
                store_rows<S>(tiles + ((it - 1) % NBUF) * TILE,
                              g.scratch + ((long long)((ii_beg + it - 1) * g.stride_loop + jj * g.stride_cta) * g.n0 + x0) * S::NPTS, lane);
        } else if (tid < 32 && it + NBUF - 1 < n_it) {
            refill(it + NBUF - 1);      // the tile stage 3 of the previous orbital drained
        }
        stage2(T);
        __syncthreads();
        if (S::TS && tid < 32 && it + NBUF - 1 < n_it) {
            bulk_wait_read_all();       // the stores issued one barrier ago by these lanes have read their tile
            __syncwarp();
            refill(it + NBUF - 1);
        }
        if (it + 1 < n_it) {
            cd *Tn = tiles + ((it + 1) % NBUF) * TILE;
            if (S::FUSE) {
                // the next tile landed long ago (three tiles): stage 3 of this orbital and stage 1 of the next one
                // share a basic block, so one's shared-memory latency hides behind the other's arithmetic
                mbar_wait(&bars[(it + 1) % NBUF], ((it + 1) / NBUF) & 1);
                if (S::TS && S::NT3 == NT) {
                    // both stages' shared-memory loads are issued before either stage's stores (the compiler
                    // cannot prove the tiles distinct, so the order is spelled out here)
                    cd w[B2], u[R1 * C1];
                    cd *p3 = T + s3_base<S, false>(tid);
                    tile_load<1, B2, 0, A::COL1>(w, p3);
                    tile_load<R1, C1, A::RA, A::COLB>(u, Tn + base1);
                    DFT<B2, false>::run(w);
                    tile_store<1, B2, 0, A::COL1>(w, p3);
#pragma unroll
                    for (int k = 0; k < R1 * C1; ++k) u[k] = cmulc(pj[k], u[k]);
                    dft_over_r<R1, C1, false>(u);
                    if (S::Q) {
                        tw_rows<R1, C1, false>(u, twr);
                        dft_over_c<R1, C1, false>(u);
                        tw_cols<R1, C1, false>(u, twc);
                    }
                    tile_store<R1, C1, A::RA, A::COLB>(u, Tn + base1);
                } else {
                    stage3(T, it);
                    stage1(Tn);
                }
            } else {
                stage3(T, it);
                mbar_wait(&bars[(it + 1) % NBUF], ((it + 1) / NBUF) & 1);
                stage1(Tn);
            }
        } else {
            stage3(T, it);
        }
    }
    if (S::TS) {
        fence_proxy_async();
        __syncthreads();
        if (tid < 32) {
            store_rows<S>(tiles + ((n_it - 1) % NBUF) * TILE,
                          g.scratch + ((long long)((ii_end - 1) * g.stride_loop + jj * g.stride_cta) * g.n0 + x0) * S::NPTS, lane);
            bulk_wait_read_all();       // shared memory must outlive the reads
        }
    }
}

// ---- pass C ---------------------------------------------------------------------------------------
// grid = (targets, n0): out[b0+tt] += sum_ss a[a0+ss] * W[ss*stride_loop + tt*stride_cta]   (W or conj(W))
template <class S>
__global__ void __launch_bounds__(S::NT, S::MINB) slabx_inv_acc(const SlabArgs g) {
    constexpr int N2 = S::N2, B1 = S::B1, B2 = S::B2, R1 = S::R1, C1 = S::C1, R2 = S::R2, C2 = S::C2;
    constexpr int NT = S::NT, NBUF = S::NBUF_C, TILE = S::TILE_C;
    constexpr bool CL = S::CLAYOUT;
    using A = Addr<S, CL>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cd *tiles = reinterpret_cast<cd *>(smem_raw);
    unsigned long long *bars = reinterpret_cast<unsigned long long *>(smem_raw + (size_t)NBUF * TILE * 16);
    const int tid = threadIdx.x, lane = tid & 31;
    const int x0 = blockIdx.y, tt = blockIdx.x;
    const long long slab_off = (long long)x0 * S::NPTS;
    int it_lo, it_hi;
    tri_range(g.tri, tt, 0, g.na, it_lo, it_hi);
    const int n_it = it_hi - it_lo;
    if (n_it <= 0) return;
    const long long pair_stride = (long long)g.stride_loop * g.n0 * S::NPTS;
    const cd *src0 = g.scratch + ((long long)(tt * g.stride_cta) * g.n0 + x0) * S::NPTS + (long long)it_lo * pair_stride;
    if (tid == 0) {
#pragma unroll
        for (int b = 0; b < NBUF; ++b) mbar_init(&bars[b], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        fence_proxy_async();
    }
    __syncthreads();
    if (tid < 32) {
        for (int it = 0; it < NBUF - 1 && it < n_it; ++it)
            {
            if (CL) issue_blocks<S>(tiles + it * TILE, src0 + (long long)it * pair_stride, &bars[it], lane);
            else issue_rows<S>(tiles + it * TILE, src0 + (long long)it * pair_stride, &bars[it], lane);
        }
    }
    const int cb = tid % S::CB1, b1 = tid / S::CB1;
    const int base1 = s1_base<S, CL>(tid);
    const cd *phi0 = g.a + (long long)(g.a0 + it_lo) * g.grid_pts + slab_off + b1 * N2 + cb;
    const bool act1 = S::NT1 == NT || tid < S::NT1;      // this thread owns a last-stage task (and its accumulators)
    cd acc[R1 * C1];
#pragma unroll
    for (int k = 0; k < R1 * C1; ++k) acc[k] = make_double2(0.0, 0.0);
    // P: the twiddled stage's factors live in registers; Q (24-point last stage, 96 accumulator registers): they
    // are re-read from a shared-memory copy of the two tables in every iteration instead
    cd twr[S::Q ? 1 : S::NTWR], twc[S::Q ? 1 : S::NTWC];
    cd *tws1 = reinterpret_cast<cd *>(smem_raw + (size_t)NBUF * TILE * 16 + 64), *tws2 = tws1 + S::N1;
    if (S::Q) {
        for (int t = tid; t < S::N1; t += NT) tws1[t] = g.tw1[t];
        for (int t = tid; t < S::N2; t += NT) tws2[t] = g.tw2[t];
        __syncthreads();
    } else {
        load_twiddles<S>(g.tw1, g.tw2, tid < S::NT2 ? tid : 0, *reinterpret_cast<cd (*)[S::NTWR]>(twr),
                         *reinterpret_cast<cd (*)[S::NTWC]>(twc));
    }
    const int base2 = s2_base<S, CL>(tid);

    // ---- stage 1': inverse DFT over k2b (mirror of forward stage 3), in place
    auto stage1i = [&](cd *T) {
#pragma unroll 1
        for (int t = tid; t < S::NT3; t += NT) {
            cd w[B2];
            cd *p = T + s3_base<S, CL>(t);
            tile_load<1, B2, 0, A::COL1>(w, p);
            DFT<B2, true>::run(w);
            tile_store<1, B2, 0, A::COL1>(w, p);
        }
    };
    auto stage2i = [&](cd *T) {
        if (S::Q) {
#pragma unroll 1
            for (int t = tid; t < S::NT2; t += NT) {
                cd u[R2 * C2];
                cd *p = T + s2_base<S, CL>(t);
                tile_load<R2, C2, A::RB, A::COLB>(u, p);
                dft_over_r<R2, C2, true>(u);
                tile_store<R2, C2, A::RB, A::COLB>(u, p);
            }
        } else if (S::NT2 == NT || tid < S::NT2) {
            cd u[R2 * C2];
            tile_load<R2, C2, A::RB, A::COLB>(u, T + base2);
            tw_cols<R2, C2, true>(u, twc);
            dft_over_c<R2, C2, true>(u);
            dft_over_r<R2, C2, true>(u);
            tw_rows<R2, C2, true>(u, twr);
            tile_store<R2, C2, A::RB, A::COLB>(u, T + base2);
        }
    };
    // ---- stage 3' (P): inverse DFT over k1a, x phi_i (already in f), sum over i
    auto stage3i_p = [&](cd *T, const cd (&f)[R1 * C1]) {
        cd u[R1 * C1];
        tile_load<R1, C1, A::RA, A::COLB>(u, T + base1);
        dft_over_r<R1, C1, true>(u);
        if (g.conj_w) {
#pragma unroll
            for (int k = 0; k < R1 * C1; ++k) {
                const cd pr = cmulc(f[k], u[k]);
                acc[k].x += pr.x; acc[k].y += pr.y;
            }
        } else {
#pragma unroll
            for (int k = 0; k < R1 * C1; ++k) {
                const cd pr = cmul(f[k], u[k]);
                acc[k].x += pr.x; acc[k].y += pr.y;
            }
        }
    };
    // ---- stage 3' (Q): 2-D inverse over (k1a, k2a); phi_i is fetched column block by column block
    auto stage3i_q = [&](cd *T, const cd *phi, cd (&f)[R1]) {
        if (!act1) return;
        cd u[R1 * C1];
        tile_load<R1, C1, A::RA, A::COLB>(u, T + base1);
#pragma unroll
        for (int c = 1; c < C1; ++c) {                         // conj(w_N2^(b2 k2a))
            const cd w = tws2[c * cb];
#pragma unroll
            for (int r = 0; r < R1; ++r) u[r * C1 + c] = cmulc(u[r * C1 + c], w);
        }
        dft_over_c<R1, C1, true>(u);
#pragma unroll
        for (int r = 1; r < R1; ++r) {                         // conj(w_N1^(b1 k1a))
            const cd w = tws1[r * b1];
#pragma unroll
            for (int c = 0; c < C1; ++c) u[r * C1 + c] = cmulc(u[r * C1 + c], w);
        }
#pragma unroll
        for (int c = 0; c < C1; ++c) {
            cd t[R1];
#pragma unroll
            for (int r = 0; r < R1; ++r) t[r] = u[r * C1 + c];
            DFT<R1, true>::run(t);
#pragma unroll
            for (int r = 0; r < R1; ++r) {
                const cd pr = g.conj_w ? cmulc(f[r], t[r]) : cmul(f[r], t[r]);
                acc[r * C1 + c].x += pr.x; acc[r * C1 + c].y += pr.y;
            }
            if (c + 1 < C1) {
#pragma unroll
                for (int r = 0; r < R1; ++r)
                    f[r] = __ldcg(reinterpret_cast<const double2 *>(phi + r * B1 * N2 + (c + 1) * B2));
            }
        }
    };
    auto refill = [&](int nx) {     // warp 0: tile nx % NBUF <- pair density of loop index nx
        if (CL) issue_blocks<S>(tiles + (nx % NBUF) * TILE, src0 + (long long)nx * pair_stride, &bars[nx % NBUF], lane);
        else issue_rows<S>(tiles + (nx % NBUF) * TILE, src0 + (long long)nx * pair_stride, &bars[nx % NBUF], lane);
    };

    mbar_wait(&bars[0], 0);
    stage1i(tiles);
    for (int it = 0; it < n_it; ++it) {
        cd *T = tiles + (it % NBUF) * TILE;
        const cd *phi = phi0 + (long long)it * g.grid_pts;
        if (tid == 0 && it + 1 < n_it)      // next orbital's slab into L2 while this one is transformed
            l2_prefetch(g.a + (long long)(g.a0 + it_lo + it + 1) * g.grid_pts + slab_off, S::NPTS * 16u);
        // here: stage 1' of pair it and stage 3' of pair it-1 are done by this thread
        fence_proxy_async();
        __syncthreads();
        if (tid < 32 && it + NBUF - 1 < n_it) refill(it + NBUF - 1);
        cd fq[S::Q ? R1 : 1];
        if (S::Q && act1) {     // first column block of phi_i: in flight during stage 2'
#pragma unroll
            for (int r = 0; r < R1; ++r) fq[r] = __ldcg(reinterpret_cast<const double2 *>(phi + r * B1 * N2));
        }
        stage2i(T);
        __syncthreads();
        const bool more = it + 1 < n_it;
        cd *Tn = tiles + ((it + 1) % NBUF) * TILE;
        if (!S::Q) {
            if (more && S::FUSE && S::NT3 == NT) {
                // stage 1' of the next pair and stage 3' of this one, loads first (see pass A)
                mbar_wait(&bars[(it + 1) % NBUF], ((it + 1) / NBUF) & 1);
                cd w[B2], u[R1 * C1], f[R1 * C1];
                cd *p3 = Tn + s3_base<S, CL>(tid);
                tile_load<1, B2, 0, A::COL1>(w, p3);
                tile_load<R1, C1, A::RA, A::COLB>(u, T + base1);
                DFT<B2, true>::run(w);
                tile_store<1, B2, 0, A::COL1>(w, p3);
                tile_load_cg<R1, C1, B1 * N2, B2>(f, phi);      // phi_i (L2-prefetched): lands during the next DFT
                dft_over_r<R1, C1, true>(u);
                if (g.conj_w) {
#pragma unroll
                    for (int k = 0; k < R1 * C1; ++k) {
                        const cd pr = cmulc(f[k], u[k]);
                        acc[k].x += pr.x; acc[k].y += pr.y;
                    }
                } else {
#pragma unroll
                    for (int k = 0; k < R1 * C1; ++k) {
                        const cd pr = cmul(f[k], u[k]);
                        acc[k].x += pr.x; acc[k].y += pr.y;
                    }
                }
            } else {
                cd f[R1 * C1];
                tile_load_cg<R1, C1, B1 * N2, B2>(f, phi);
                stage3i_p(T, f);
                if (more) {
                    mbar_wait(&bars[(it + 1) % NBUF], ((it + 1) / NBUF) & 1);
                    stage1i(Tn);
                }
            }
        } else {
            stage3i_q(T, phi, *reinterpret_cast<cd (*)[R1]>(fq));
            if (more) {
                mbar_wait(&bars[(it + 1) % NBUF], ((it + 1) / NBUF) & 1);
                stage1i(Tn);
            }
        }
    }
    if (!act1) return;
    cd *o = g.out + (long long)(g.b0 + tt) * g.grid_pts + slab_off + b1 * N2 + cb;
#pragma unroll
    for (int r = 0; r < R1; ++r)
#pragma unroll
        for (int c = 0; c < C1; ++c) {
            cd cur = o[r * B1 * N2 + c * B2];
            cur.x += acc[r * C1 + c].x;
            cur.y += acc[r * C1 + c].y;
            o[r * B1 * N2 + c * B2] = cur;
        }
}

}  // namespace ptfock
