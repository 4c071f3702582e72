/*
 * ptfock.h -- C ABI of the B200-native plane-wave Fock exchange library (libptfock.so).
 *
 * The operation (Sec. 2, Eq. (3); Sec. 3.2, Alg. 2 lines 6-10):
 *
 *     (V_X[Phi] psi_j)(r) = - alpha * sum_i phi_i(r) * IFFT[ v(G) * FFT( conj(phi_i) psi_j ) ](r)
 *
 * on a periodic cell with a regular real-space grid n = (n0, n1, n2), N = n0 n1 n2 points.
 * Forward DFT exp(-i), unnormalised; inverse exp(+i) with 1/N (any consistent pair gives the same
 * result).  v(G) is evaluated on every grid frequency m_d in [-n_d/2, n_d/2):
 *     PTFOCK_KERNEL_COULOMB : 4 pi / |G|^2,                              v(0) = 0
 *     PTFOCK_KERNEL_HSE     : 4 pi / |G|^2 * (1 - exp(-|G|^2/(4 omega^2))), v(0) = pi / omega^2
 * ("kernel for the (possibly screened) electron-electron interaction"; the formulas are
 * BASELINE.json north_star's; the paper prints none -- DESIGN.md readings Q1-Q3).
 *
 * Array layout: C order [orbital][x0][x1][x2], x2 contiguous, interleaved (re, im) IEEE fp64,
 * i.e. one grid = 16 N bytes, orbital k starts at byte 16 N k.  All orbital pointers must be
 * 16-byte aligned.  Unless a function says HOST, pointers are DEVICE pointers on the plan's device.
 *
 * Everything runs in hand-written sm_100a kernels (no cuFFT / cuBLAS / cuSOLVER); there is no CPU fallback: on a machine without
 * such a device ptfock_create returns PTFOCK_ERR_UNSUPPORTED_DEVICE (or PTFOCK_ERR_CUDA).
 *
 * Error behaviour: every function returns 0 (PTFOCK_OK) or a negative code below; nothing throws
 * or aborts across the ABI.  A plan is not thread-safe (one host thread at a time); distinct plans are
 * independent.  Calls on one plan may use different streams: the plan's scratch is shared by
 * consecutive calls, so a call on another stream than the previous one first waits (on the device,
 * cudaStreamWaitEvent) for the previous call to finish.  The caller's current device is left as it was.
 *
 * Supported grids: n0 in {16, 32, 48, 64, 120, 128}; (n1, n2) one of the built slab shapes
 *   (64,64) (128,48) (48,48) (32,32) (90,60)            -- TMA-fed three-stage slab passes
 *   every other pair from {16, 32, 48, 64, 128}^2 except (128,128)   -- generic slab passes
 * (all BASELINE.json configs, the paper's own 60 x 90 x 120 grid stored as 120 x 90 x 60, and 120 of the 125 grids with
 * edges from {16, 32, 48, 64, 128}; a 128 x 128 slab, 256 KB of complex fp64, does not fit one CTA's shared memory and
 * has no kernel yet: n0 x 128 x 128 returns PTFOCK_ERR_UNSUPPORTED_GRID -- store such a cell with a shorter axis last
 * two, e.g. 128 x 128 x 64 instead of 64 x 128 x 128).
 * 64 x 64 x 64, 48 x 48 x 48 and 32 x 32 x 32 additionally have the two-stage slab passes + two-stage pencil pass, and 16 x 16 x 16
 * the single-pass on-chip kernel (whole pair-solve in one CTA, no scratch); these are the default for their grids.
 * The dense-algebra contractions (ptfock_overlap / rotate / residual / orthonormalize) run on the FP64 tensor cores.
 */
#ifndef PTFOCK_H
#define PTFOCK_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ptfock_plan ptfock_plan; /* opaque, owned by the library */

enum {
    PTFOCK_KERNEL_COULOMB = 0,
    PTFOCK_KERNEL_HSE = 1,
    PTFOCK_KERNEL_KINETIC = 2           /* not an interaction: |G|^2 / 2, for ptfock_hloc_apply's plan (n_occ must be 1) */
};

enum {
    PTFOCK_OK = 0,
    PTFOCK_ERR_INVALID_ARG = -1,        /* null pointer, negative count, bad enum, pointer not on the plan's device,
                                           n_targets > max_targets where a call says so ...                    */
    PTFOCK_ERR_UNSUPPORTED_GRID = -2,   /* n0 or the slab shape (n1, n2) has no kernel (list above)             */
    PTFOCK_ERR_UNSUPPORTED_DEVICE = -3, /* device is not compute capability 10.x */
    PTFOCK_ERR_ALIGNMENT = -4,          /* an orbital pointer is not 16-byte aligned */
    PTFOCK_ERR_ALLOC = -5,              /* device or host allocation failed (workspace too small included) */
    PTFOCK_ERR_CUDA = -6,               /* a CUDA runtime call failed; see ptfock_last_cuda_error */
    PTFOCK_ERR_ALIAS = -7,              /* out overlaps phi or psi */
    PTFOCK_ERR_NOT_POSITIVE = -8,       /* ptfock_orthonormalize: the overlap matrix is not positive definite */
    PTFOCK_ERR_TOO_LARGE = -9           /* ptfock_banddot_static: n exceeds PTFOCK_STATIC_MAX_BANDS (fixed built-in scratch) */
};

typedef struct {
    double cell[9];           /* rows = lattice vectors a0, a1, a2 in bohr                                  */
    int32_t n[3];             /* grid (supported shapes: see above); index = (x0*n1 + x1)*n2 + x2           */
    int32_t n_occ;            /* number of Phi orbitals (N_i of Eq. 3's sum), >= 1                         */
    int32_t max_targets;      /* largest n_targets of ptfock_apply_host and of ptfock_exchange_energy with
                                 vx_psi == NULL (sizes their buffers) and the default wave; ptfock_apply
                                 itself accepts any n_targets                                                */
    int32_t kernel;           /* PTFOCK_KERNEL_*                                                            */
    double omega;             /* bohr^-1; HSE only                                                          */
    double alpha;             /* mixing fraction multiplying V_X; 1.0 in all BASELINE configs */
    int32_t device;           /* CUDA ordinal                                                               */
    int32_t block_i;          /* pair-scheduler tile: orbitals i per wave (0 = library chooses)            */
    int32_t block_j;          /* pair-scheduler tile: targets j per wave  (0 = library chooses)            */
    uint64_t workspace_bytes; /* upper bound for the scratch (0 = library chooses, and never below what the
                                 dense-algebra calls need for max(n_occ, max_targets) orbitals); with a bound
                                 the scratch never exceeds it and a dense-algebra call that needs more returns
                                 PTFOCK_ERR_ALLOC                                                            */
    uint32_t flags;           /* PTFOCK_FLAG_* (0 = library chooses the kernels)                            */
} ptfock_desc;

enum {
    /* use the three-pass path (slab passes + pencil pass through the pair scratch) even where a grid has a faster
     * dedicated path (64^3: pass8.cuh, 16^3: onchip16.cuh): same results, kept for A/B timing and as a second
     * implementation the tests compare with the oracle */
    PTFOCK_FLAG_THREE_STAGE_SLABS = 1u,
    /* keep every wave on the caller's stream.  By default, when the scratch bound allows two waves, the general
     * (non-symmetric) schedule runs the j-blocks with an odd index on a stream of the plan's, in a second scratch slot,
     * forked from and joined to `stream` inside the call: one wave's kernels fill the SMs while the other's drain.
     * Same results bit for bit; kept for A/B timing. */
    PTFOCK_FLAG_SINGLE_STREAM = 2u
};

/* Builds the plan: v(G) table (with -alpha/N folded in, stored in the kernels' digit-permuted
 * frequency order), twiddle tables, scratch for one wave of pair densities.  *out is written only
 * on success.  Synchronous. */
int ptfock_create(const ptfock_desc *desc, ptfock_plan **out);

/* out[j] = V_X[Phi] psi_j for j = 0 .. n_targets-1 (overwritten; Alg. 2 line 1 zero-initialises).
 *   phi : n_occ grids.
 *   psi : n_targets grids, or NULL meaning Psi = Phi[self_offset : self_offset + n_targets]
 *         (when that range is all of Phi the scheduler uses the rho_ji = conj(rho_ij) pair symmetry).
 *   out : n_targets grids; must not overlap phi or psi.
 * The caller owns all three and keeps them alive until `stream` has passed the call.
 * Asynchronous on `stream` (a cudaStream_t passed as void*; NULL = the legacy default stream). */
int ptfock_apply(ptfock_plan *plan, const void *phi, const void *psi, int32_t self_offset,
                 int32_t n_targets, void *out, void *stream);

/* E_x = 1/2 * (Omega/N) * Re sum_j sum_r conj(psi_j(r)) (V_X[Phi] psi_j)(r)   ("total energy
 * evaluation"; reading Q11).  vx_psi: a previous ptfock_apply result for the same arguments, or
 * NULL (the library applies into its own buffer first).  Writes one double to HOST memory *e_host and
 * synchronises `stream`. */
int ptfock_exchange_energy(ptfock_plan *plan, const void *phi, const void *psi, int32_t self_offset,
                           int32_t n_targets, const void *vx_psi, double *e_host, void *stream);

/* Same as ptfock_apply but phi, psi, out are HOST pointers (pinned memory gives full PCIe speed;
 * pageable works).  The library copies Phi (and Psi) to device buffers it owns, applies, copies the
 * result back, and synchronises `stream`.  The copies run on a stream of the plan's: Phi in chunks of block_i
 * orbitals, Psi in chunks of block_j targets, each wave waiting only for the chunks it reads; every block_j
 * targets of the result start their way back as soon as the last block of orbitals has been accumulated into
 * them, so nearly all of the transfer overlaps the kernels.  n_targets <= max_targets. */
int ptfock_apply_host(ptfock_plan *plan, const void *phi_host, const void *psi_host, int32_t self_offset,
                      int32_t n_targets, void *out_host, void *stream);

/* ---- dense-algebra neighbours of the exchange operator ------------------------------------
 * The steps either side of H Psi in one PT-CN step (Alg. 1): the residuals of PAPER.md:171-188
 * (Sec. 3.3, Alg. 3), the density of PAPER.md:192 and the re-orthogonalisation of PAPER.md:200 (Sec. 3.4), on ONE GPU
 * (the paper's Alltoallv / Allreduce steps, Alg. 3 lines 1, 3, 6, have nothing to do here).  Orbital sets are
 * [orbital][x0][x1][x2] complex fp64 DEVICE arrays on the plan's grid; (a, b) = (Omega/N) sum_r conj(a(r)) b(r).
 * Matrices are row-major complex fp64 DEVICE arrays.  All calls are asynchronous on `stream` except where stated,
 * use the plan's scratch (PTFOCK_ERR_ALLOC if it is too small) and are deterministic (no atomics). */

/* S[m][n] = (a_m, b_n), m < n_a, n < n_b (Alg. 3 line 2: "S = Psi_f^* H_f Psi_f"; "Psi^* Psi"). */
int ptfock_overlap(ptfock_plan *plan, const void *a, int32_t n_a, const void *b, int32_t n_b, void *s, void *stream);

/* out_n(r) = sum_m a_m(r) S[m][n], n < n_out; S is n_a x n_out (Alg. 3 line 4: "Psi_temp = Psi_f S").  out must not
 * overlap a. */
int ptfock_rotate(ptfock_plan *plan, const void *a, int32_t n_a, const void *s, int32_t n_out, void *out, void *stream);

/* psi_half == NULL:  R = H Psi - Psi (Psi^* H Psi)                                   (Alg. 1 line 1, R_n)
 * else:              R = Psi + (i dt/2) (H Psi - Psi (Psi^* H Psi)) - Psi_half       (Alg. 3 line 5, R_f; the minus signs
 *                    the extraction of PAPER.md dropped are those of Eq. (5))
 * psi, hpsi, psi_half, r_out: n orbitals each; r_out must not overlap psi. */
int ptfock_residual(ptfock_plan *plan, const void *psi, const void *hpsi, const void *psi_half, int32_t n, double dt,
                    void *r_out, void *stream);

/* rho(r) = sum_{i<n} |psi_i(r)|^2; rho: N doubles, DEVICE. */
int ptfock_density(ptfock_plan *plan, const void *psi, int32_t n, double *rho, void *stream);

/* Psi <- Psi L^{-H} with L L^H = Psi^* Psi (overlap, Cholesky, triangular solve), IN PLACE; afterwards
 * (psi_m, psi_n) = delta_mn.  Synchronises `stream`; PTFOCK_ERR_NOT_POSITIVE if a pivot is not positive (psi is then
 * left modified). */
int ptfock_orthonormalize(ptfock_plan *plan, void *psi, int32_t n, void *stream);

/* ---- pieces of one PT-CN time step with a MODEL Hamiltonian (Alg. 1) -----------
 * H[Psi] psi = -1/2 Laplacian psi + v_loc psi + V_X[Psi] psi: a real Hamiltonian needs the pseudopotentials the paper
 * uses, which are not available; the model keeps the structure of Alg. 1 (residuals, fixed point with
 * Anderson mixing over per-wavefunction least squares PAPER.md:194-198, density, re-orthogonalisation).  The step itself
 * is sequenced by paper_1905_01348_b200/ptcn.py; every operation on grids goes through the calls of this header. */

/* out_j = -1/2 Laplacian psi_j + vloc psi_j, j < n, on a plan created with kernel = PTFOCK_KERNEL_KINETIC, n_occ = 1
 * (the kinetic operator runs through the same three passes as the exchange operator: a pair-solve with the constant
 * orbital and the table |G|^2 / 2).  vloc: N doubles (DEVICE) or NULL.  out must not overlap psi.  Asynchronous. */
int ptfock_hloc_apply(ptfock_plan *plan, const double *vloc, const void *psi, int32_t n, void *out, void *stream);

/* out_j = a_j x_j + b_j y_j, j < n, with per-orbital complex coefficients from HOST arrays of n (re, im) pairs (the mixing
 * coefficients of PAPER.md:194 are per wavefunction); y and b_host may be NULL.  out may be x or y.  Asynchronous, with
 * no copy and no synchronisation: the coefficients are passed to the kernels by value (64 orbitals per launch), so the
 * host arrays, pinned or pageable, may be reused when the call returns. */
int ptfock_axpby(ptfock_plan *plan, int32_t n, const double *a_host, const void *x, const double *b_host, const void *y,
                 void *out, void *stream);

/* out_host[j] = (a_j, b_j) = (Omega/N) sum_r conj(a_j(r)) b_j(r), j < n (n (re, im) pairs, HOST): the entries of the
 * per-wavefunction least-squares problems of the Anderson mixing.  Synchronises `stream`. */
int ptfock_banddot(ptfock_plan *plan, const void *a, const void *b, int32_t n, double *out_host, void *stream);

/* out_host[k * n + j] = (a_j, b^k_j), k < n_sets, j < n: ptfock_banddot of one orbital set `a` against n_sets others in one
 * call with one synchronisation -- a new row of the per-wavefunction Gram matrices of the Anderson mixing, or their
 * right-hand sides ("evaluation of overlap matrices").  b_sets_host: HOST array of n_sets DEVICE
 * pointers (n orbitals each); out_host: n_sets * n (re, im) pairs, HOST.  Same kernels and summation order as
 * ptfock_banddot (bit-identical per set).  Synchronises `stream`. */
int ptfock_banddot_many(ptfock_plan *plan, const void *a, const void *const *b_sets_host, int32_t n_sets, int32_t n,
                        double *out_host, void *stream);

/* v_out(r) = v_ext(r) + g rho(r): the local potential of the model Hamiltonian following the density (Alg. 1 line 5,
 * PAPER.md:84 "Update the potential").  v_ext (NULL = 0), rho, v_out: N doubles, DEVICE; v_out may be v_ext or rho.
 * Asynchronous. */
int ptfock_vloc_update(ptfock_plan *plan, const double *v_ext, double g, const double *rho, double *v_out, void *stream);

/* *change_host = (Omega/N) sum_r |rho_a(r) - rho_b(r)|: the density change between two SCF iterations that Alg. 1 line 9
 * monitors.  rho_a, rho_b: N doubles, DEVICE; change_host: HOST.  Deterministic; synchronises `stream`. */
int ptfock_density_change(ptfock_plan *plan, const double *rho_a, const double *rho_b, double *change_host, void *stream);

/* ---- the one entry point that allocates nothing -----------------------------------------------------------------
 * Who needs it: a host code that cannot let this library call cudaMalloc.  Typical cases: an electronic-structure
 * code that has handed all of HBM to its own memory pool at start-up, so that a cudaMalloc from a library simply fails;
 * and a time-step loop whose other streams (copies, NCCL traffic) must keep running, which cudaMalloc / cudaFree
 * would stall because both synchronise the whole device.  Such a caller cannot even build a plan (ptfock_create
 * allocates the tables and the scratch), so this call takes NO plan.
 *
 * What it computes: the per-band inner products of ptfock_banddot, the entries of the per-wavefunction least-squares
 * problems of the Anderson mixing (Sec. 3.4),
 *     out[j] = weight * sum_{r < n_points} conj(a_j(r)) b_j(r),   j < n,
 * by the same two kernels, summed in the same fixed order (bit-identical to ptfock_banddot on a plan with
 * N = n_points and Omega/N = weight).  The kernels need scratch for their per-block partial sums; here it is a
 * fixed array of PTFOCK_STATIC_MAX_BANDS * 64 complex numbers = 4 MiB built into the library image.  Every GPU
 * that loads libptfock.so carries these 4 MiB until the process exits, whether or not this call is ever used.
 *
 *   device   : CUDA ordinal a, b, out live on; left as the caller's current device on return.
 *   n_points : grid points per band (>= 1);  weight: Omega / N for the inner product of this header, or any scale.
 *   a, b     : n bands each, [band][point] complex fp64, DEVICE, 16-byte aligned (inputs, caller-owned).
 *   out      : n complex fp64 (re, im), DEVICE, 16-byte aligned (output, caller-owned).
 *   n        : 1 .. PTFOCK_STATIC_MAX_BANDS; a larger n returns PTFOCK_ERR_TOO_LARGE and launches nothing (split the
 *              bands over several calls on ONE stream instead).
 * Asynchronous on `stream`; nothing is synchronised.  The call itself performs no cudaMalloc / cudaFree /
 * cudaMallocHost and calls no library routine that allocates.
 *
 * First call on each device: the library looks up the device address of its built-in array (one
 * cudaGetSymbolAddress with that device current; this may also make the CUDA runtime load the library's kernels onto
 * the device) and remembers it.  Make that first call during start-up, before any stream capture begins; later calls
 * only launch the two kernels.
 *
 * Sharing: all calls on a device, from every thread and stream, use the SAME array, and it keeps whatever the last
 * call left in it.  Nothing in it has to start at zero: each call overwrites every partial sum before it reads it.
 * Two calls that can overlap on the GPU (different streams without an event between them) race on the array and give
 * wrong results; calls on one stream, or ordered by events, are safe. */
#define PTFOCK_STATIC_MAX_BANDS 4096
int ptfock_banddot_static(int32_t device, int64_t n_points, double weight, const void *a, const void *b, int32_t n,
                          void *out, void *stream);

/* Frees everything the plan owns.  NULL is allowed. */
int ptfock_destroy(ptfock_plan *plan);

/* Static string for an error code. */
const char *ptfock_strerror(int code);

/* The cudaError_t of the most recent PTFOCK_ERR_CUDA on this thread (0 if none). */
int ptfock_last_cuda_error(void);

/* Introspection for the harness (host memory, no device work):
 *   info[0] = block_i, info[1] = block_j in use, info[2] = scratch bytes, info[3] = kernel launches
 *   issued by the most recent apply, info[4] = pair-solves executed by the most recent apply,
 *   info[5] = 1 if the most recent apply used the symmetric schedule, info[6] = total launches since create,
 *   info[7] = kernel family in the low 4 bits: 0 three-stage slab passes + pencil pass, 1 two-stage slab passes +
 *             two-stage pencil pass (64^3, 48^3, 32^3), 2 single-pass on-chip kernel (16^3); bit 4 (value 16) set if the scratch
 *             holds two waves (two waves in flight on the general schedule). */
int ptfock_plan_info(const ptfock_plan *plan, int64_t info[8]);

/* Test hook: W = IFFT[v' * FFT(conj(phi_i) psi_j)] for ONE pair through the same three kernels,
 * v' = -alpha/N * v (so V_X psi_j = sum_i phi_i W_ij).  w_out: one grid, device.  Asynchronous on `stream`
 * (the first call allocates one grid of ones that the plan keeps). */
int ptfock_debug_pair(ptfock_plan *plan, const void *phi_i, const void *psi_j, void *w_out, void *stream);

/* Per-pass device timing for the benchmark harness.  While on, every kernel launch of ptfock_apply is
 * bracketed by cudaEvents on the caller's stream (pass 0 = slab forward "A", 1 = pencil middle "B",
 * 2 = slab inverse + accumulate "C").  ptfock_get_profile waits for the last recorded event, returns the
 * summed milliseconds and launch counts per pass since the last reset, and optionally resets. */
int ptfock_set_profiling(ptfock_plan *plan, int32_t on);
int ptfock_get_profile(ptfock_plan *plan, double ms[3], int64_t launches[3], int32_t reset);

/* Measurement aid (the path sits under two roofs, HBM bandwidth and the plain FP64 pipe, and
 * MEASURED_PEAKS.json records no FP64 number): runs a register-resident DFMA loop on `device` (legacy default
 * stream, synchronous, ~50 ms) and writes the best sustained rate in TFLOP/s (2 flops per DFMA) to HOST memory. */
int ptfock_measure_dfma_peak(int32_t device, double *tflops_host);

/* Same for the FP64 tensor pipe (mma.sync m8n8k4, SASS DMMA.8x8x4): the roof of ptfock_overlap / ptfock_rotate /
 * ptfock_residual / ptfock_orthonormalize, whose contractions run there (csrc/dense_mma.cuh). */
int ptfock_measure_dmma_peak(int32_t device, double *tflops_host);

/* Measurement aid for the scratch-residency question (SURVEY.md 8(d) "a third roof to watch"):
 * copies `bytes` bytes device-to-device `reps` times back to back with a plain 128-bit grid-stride kernel and
 * writes the best read+write rate in GB/s to HOST memory.  A working set (2 * bytes) well under the L2 size
 * measures the L2 copy bandwidth, one well above it the HBM copy bandwidth.  Synchronous, legacy default stream. */
int ptfock_measure_copy_bandwidth(int32_t device, uint64_t bytes, int32_t reps, double *gbs_host);

#ifdef __cplusplus
}
#endif
#endif /* PTFOCK_H */
