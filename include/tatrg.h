/*
 * tatrg.h -- C-ABI of libtatrg: Triad-ATRG coarse-graining of the 4D Ising tensor network
 * on one NVIDIA B200 (sm_100a), FP64.
 *
 * The calls follow the paper's statement of the problem (arXiv:2412.14104,
 * /root/reference/PAPER.md): the model is fixed by the inverse temperature beta
 * (Eqs. 15-17), the method by the bond dimension chi and the oversampling
 * parameter r, the number q of RSVD iterations (Table 1) and the
 * coarse-graining direction ("coarse-graining step along the 1^ direction");
 * the output is the free energy.
 *
 * Conventions
 *   - One process-global context; not thread safe.  The step is enqueued on the stream given
 *     by tatrg_set_stream (default: the legacy default stream); inside coarse_grain the library
 *     forks independent chains of small kernels (squeezers, isometries, factorisations) and the
 *     upload of host-resident inputs onto non-blocking streams of its own and joins them back
 *     with events, so everything a call enqueues is ordered before whatever the caller enqueues
 *     on its stream afterwards.
 *   - The library allocates no device memory: every device buffer lives in the workspace
 *     the caller passes to tatrg_set_workspace (e.g. a torch tensor).  The caller keeps it
 *     alive and unchanged until tatrg_destroy or the next tatrg_set_workspace.  What the library
 *     owns (released by tatrg_destroy): its side streams and events, 64 KB of page-locked host
 *     memory for asynchronous read-backs.
 *   - Status: 0 = OK, negative = error, message via tatrg_last_error().  Errors never abort
 *     the process.  A failed coarse_grain leaves the renormalised tensor (Phi, Psi), the
 *     step count and the ln Z accumulator of the previous step intact.
 *   - "host" / "device" is stated for every pointer.
 */
#ifndef TATRG_H
#define TATRG_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define TATRG_OK 0
#define TATRG_EINVAL (-22)   /* bad argument */
#define TATRG_ENOMEM (-12)   /* workspace too small */
#define TATRG_ESTATE (-1)    /* called before init / before a workspace was set */
#define TATRG_ECUDA (-5)     /* CUDA runtime error (message has the CUDA error string) */
#define TATRG_ENUM (-34)     /* numerical failure (non-finite value, no convergence) */

/* Initial tensor of the 4D Ising model, Eqs. 16-17:
 *   T_{i1..i4 j1..j4} = sum_a e^{beta h s_a} prod_mu W_{a i_mu} prod_mu W_{a j_mu},
 *   W = ((sqrt cosh b, sqrt sinh b), (sqrt cosh b, -sqrt sinh b))  (square roots restored so
 *   that W W^T = e^{beta s s'}; reading G1; field term: reading G2),
 * kept factorised as T = sum_g Phi_{i,g} Psi_{j,g} (bond 2), normalised to |Phi|=|Psi|=1.
 * Resets the step count and the ln Z accumulator.  beta must be finite and > 0, h finite. */
int init_ising_tensor(double beta, double h);

/* One Triad-ATRG coarse-graining step along `direction` (1..4): canonical form
 * A sigma D, RSVD bond swap to Gamma = A X sigma Y D (Eq. 1), oversampled
 * isometries U^A..U^D by RSVD (Eqs. 2-3), triad tensors E..L (Eqs. 4-11), squeezers
 * M^(mu), N^(mu) (Eq. 12), contraction to Phi, Psi (Eqs. 13-14), normalisation.
 *   chi in 1..64 bond dimension, r >= 1 oversampling (internal lines r*chi <= 256: the paper's r = 7 up to
 *   chi = 36), q >= 0 RSVD iterations, seed: master seed of the Gaussian sketches (sub-seeds per
 *   SURVEY.md 8(d)).  Every Gaussian input the caller did not supply with tatrg_set_sketch is generated
 *   on the device by the library's implementation of the shared seeded recipe (tatrg_fill_gauss).
 *   TATRG_EINVAL: bad arguments, or a supplied input whose size is not the one this step needs;
 *   TATRG_ENOMEM: workspace too small; TATRG_ENUM: the tensor or a Gram matrix is numerically zero. */
int coarse_grain(int direction, int chi, int r, int q, uint64_t seed);

/* Same step without the triad decomposition: plain ATRG with bond swapping, O(chi^9)
 * contraction (Table 1); r and q act on the bond-swap RSVD only. */
int coarse_grain_atrg(int direction, int chi, int r, int q, uint64_t seed);

/* ln Z / V = sum_m 2^-m ln c_m + 2^-n ln tTr T^(n)  (Eq. 15 closed periodically
 * after n steps; reading O8).  NaN before init or if the trace is not positive.
 * One device reduction and one scalar device->host copy. */
double log_Z_per_site(void);

/* ---- plumbing (PyTorch owns memory and streams) ------------------------------------- */
int tatrg_set_stream(void *cuda_stream);                     /* cudaStream_t; NULL = default */
int tatrg_set_workspace(void *dev_ptr, size_t bytes);        /* device; 256-byte aligned */
size_t tatrg_workspace_bytes(int chi, int r);                /* upper bound, steady state, coarse_grain */
size_t tatrg_workspace_bytes_atrg(int chi, int r);           /* the same for coarse_grain_atrg (adds the
                                                              * chi^6-sized slices of the O(chi^9) contraction) */

/* Caller-supplied Gaussian inputs for the NEXT coarse_grain call (consumed by it).
 * which: 0 swap sketch [(beta,J), l]; 1..4 isometry sketches A,X,Y,D [(p,q), k];
 *        5 gauge reference for A/D [(i0..i3), a]; 6..8 gauge references of the squeezers.
 * data: n doubles, row-major in the rotated frame;
 * on_device != 0: device pointer, must stay valid until coarse_grain returns;
 * on_device == 0: host pointer (pinned or pageable), copied (H2D) by the library's copy stream inside the next
 * coarse_grain, which does not return before the copy has ended.  n must equal rows * cols of
 * tatrg_sketch_shape for the step that consumes it: a mismatch makes that coarse_grain fail with TATRG_EINVAL
 * (nothing is generated in its place). */
int tatrg_set_sketch(int which, const double *data, size_t n, int on_device);
/* Shape the next coarse_grain(direction, chi, r) will ask for input `which`
 * (rows, cols; 0,0 if unused).  For which = 0,5 the bond after canonicalisation is assumed
 * equal to the current bond (true whenever Phi Psi^T has full numerical rank). */
int tatrg_sketch_shape(int which, int direction, int chi, int r, int64_t *rows, int64_t *cols);

/* Spectra of the LAST step, descending, copied to host_out (host, capacity cap doubles).
 * which: 0 sigma^T (canonical form), 1 sigma (bond swap), 2..5 S^A,S^X,S^Y,S^D (Eq. 3;
 * count 0 when U is the identity), 6..8 squeezer singular values s^(t1..t3), 9: ln c of the
 * step (1 value).  Returns the count (<= cap) or a negative status. */
int tatrg_get_spectrum(int which, double *host_out, int cap);

/* Every stage of coarse_grain has a fast route (used when its conditions hold) and a robust route that
 * follows the oracle's algorithm step by step: mask bit 0 forces the bond swap on the
 * plain chi^4-dimensional operator M instead of its chi^3-dimensional core, bit 1 Householder
 * TSQR instead of Cholesky-QR, bit 2 the squeezers by dense eigendecompositions (PAPER.md:81-86
 * Eq. 12) instead of Cholesky + subspace iteration, bit 3 the four isometries one after the other with
 * synchronous solvers (Eqs. 2-3).  For tests: both routes must give the same step.  Bit 4 feeds the persistent
 * tensor-GEMM tile from TMA (cp.async.bulk.tensor, rank-2 FP64 tensor maps) instead of per-thread cp.async where
 * the operands are plain row-major matrices (an alternative producer, not a fallback).  Bit 5 runs the subspace
 * iteration of the squeezers as separate launches (products, Cholesky-QR passes) instead of the one resident grid
 * of sq_iter.cu.  0 = default; mask in 0..63, else TATRG_EINVAL. */
int tatrg_set_routes(int mask);

/* Phi / Psi split of one step over two GPUs ("two GPUs are used", Fig. 6).
 * The two halves of the contraction, Phi of Eq. 13 and Psi of Eq. 14 (for coarse_grain_atrg the
 * two O(chi^9) products of PAPER.md:92), share no intermediate.  Two processes, one per GPU, run the same steps
 * from the same state with the same seeds (everything up to the squeezers is computed by both: the same kernels
 * on the same inputs give the same bits); sides = 1 makes this process contract Phi only, sides = 2 Psi only,
 * 3 = both (default; an exchange_fn given with 3 is called as an observer of the two finished, not yet normalised
 * tensors, NULL clears it).  After its half the library calls, once per step,
 *     int exchange_fn(void *user, double *phi_dev, double *psi_dev, int64_t n, void *cuda_stream)
 * (exchange_fn is passed as a plain pointer to a function of exactly this type): phi_dev / psi_dev (device) are
 * the new, not yet normalised tensors of n doubles each, this process's half complete in the order of
 * cuda_stream (the library's stream), the other half undefined.  The callback fills the other half (the binding:
 * one NCCL all-gather over NVLink) so that it is complete in the order of cuda_stream when it returns, or after a
 * synchronisation of its own; it returns 0, anything else fails the step with TATRG_ECUDA (state of the previous
 * step intact).  The library then normalises both halves and commits the step as usual, so both processes end on
 * the same state.  The callback must not call into the library.  sides outside 1..3, or one half without an
 * exchange_fn: TATRG_EINVAL.  user is handed back unchanged; both pointers must stay valid until the next
 * tatrg_set_side_split. */
int tatrg_set_side_split(int sides, void *exchange_fn, void *user);

/* Oversampled isometries of the LAST coarse_grain step (Eqs. 2-3; I, J, K, L of Eqs. 8-11),
 * for tests (the projector U U^T is gauge invariant and is what parity compares).  tatrg_keep_isometries(1)
 * makes every following step copy its four isometries to the host (one extra synchronisation per step);
 * tatrg_get_isometry copies U^which (which = 0..3: A, X, Y, D), row-major [(p,q), k] in the rotated
 * frame, rows = d_t1 d_t2, cols = min(r chi, rows) (the identity when cols = rows), to host_out (host,
 * capacity cap doubles; NULL = only rows / cols are returned). */
int tatrg_keep_isometries(int on);
int tatrg_get_isometry(int which, double *host_out, size_t cap, int *rows, int *cols);

/* dims_out[0..3] = leg dimensions d1..d4, dims_out[4] = bond, dims_out[5] = step count. */
int tatrg_get_dims(int dims_out[6]);

/* Copy the current renormalised tensors to the host: phi_out, psi_out each
 * d1*d2*d3*d4*bond doubles, row-major [i1,i2,i3,i4,g] (host).  For tests. */
int tatrg_get_tensors(double *phi_out, double *psi_out, size_t cap_each);

/* Order parameter X^(m) = (Tr A)^2 / Tr(A^2), A_kl = sum T_{i1 i2 i3 k; i1 i2 i3 l}
 * (PAPER.md:177); `leg` = 1..4 is the direction left open (the paper: 4). NaN on error. */
double tatrg_order_parameter(int leg);

/* Per-stage device milliseconds of the last step (CUDA events): out[0..n) for the stages
 * named by tatrg_stage_name(i).  Returns the number of stages. */
int tatrg_get_stage_ms(double *host_out, int cap);
const char *tatrg_stage_name(int i);
/* Host->device upload of the last step's host-resident inputs (tatrg_set_sketch with on_device == 0;
 * the seeded sketches of SURVEY.md 8(d)): *ms_out (host) = device milliseconds between the first and the
 * last copy on the library's copy stream (it runs beside the canonical form and the basis factorisations
 * of the bond swap), *bytes_out (host) = bytes copied.  Either pointer may be NULL. */
int tatrg_get_h2d(double *ms_out, size_t *bytes_out);
/* Per-launch device timing of the tensor-GEMM kernel (CUDA event pairs on the library's stream
 * around the launches inside coarse_grain; a few microseconds of overhead per timed launch).
 * on = 1: only the 128x128-tile launches (the dominant kernel) are timed; on = 2: every tensor-GEMM
 * launch; 0: off.  After a step, tatrg_get_gemm_profile copies, for every stage i and tile class j
 * (0: the 64x64 and 128x64 CTA tiles, 1: 128x128), the triple {milliseconds, FP64 flops, launches}
 * to host_out[(2 i + j) 3 ..]; returns the number of doubles written.  With the environment variable
 * TATRG_TRACE set, every timed launch is also logged on stderr (shape, split, ms, TFLOP/s). */
int tatrg_set_profile(int on);
int tatrg_get_gemm_profile(double *host_out, int cap);
/* Number of kernel launches this library has enqueued since the last call (and reset). */
long long tatrg_launch_count(int reset);
/* FP64 flops of the tensor-GEMM launches since the last reset (2*M*N*K*batch each). */
double tatrg_gemm_flops(int reset);

/* Measured FP64 peak of this GPU: register-resident loop of mode 0: DMMA.8x8x4 (tensor
 * pipe), 1: DFMA (vector pipe), 2: both interleaved.  Runs `iters` outer iterations per
 * warp, returns TFLOP/s (device-timed), <0 on error. */
double tatrg_probe_fp64_peak(int mode, int iters);

/* Stand-alone tensor-GEMM entry (the one contraction kernel the path is built from; PAPER.md:58-67
 * Eqs. 4-7, :90 Eqs. 13-14 are all instances), for tests and roofline measurement:
 *   C[b][cm(m)+cn(n)] (+)= alpha * sum_k A[b][am(m)+ak(k)] * B[b][bk(k)+bn(n)].
 * Every index map is mixed radix over up to four tensor legs:
 *   idx = d0 + n0*(d1 + n1*(d2 + n2*d3))  ->  d0*s0 + d1*s1 + d2*s2 + d3*s3   (element offsets),
 * given as 7 int64 {n0, n1, n2, s0, s1, s2, s3} (radix <= 0 = unused level) in `maps` (host), in
 * the order am, ak, bk, bn, cm, cn, ab, bb, cb (63 values; the last three map the batch index).
 * A, B, C: device.  accumulate: bit 0 set: C += ; bit 1 set: the caller promises B[k][n] = 0 for k > n (a
 * triangular factor applied from the right, as in Q1 = T L^-T of the bond swap's Cholesky-QR; the zeros must be
 * there: the hint only lets the kernel skip whole k tiles of them, the result is the same bit for bit).
 * M, N >= 0, K >= 1, batch in 1..65535. */
int tatrg_tensor_gemm(const double *A, const double *B, double *C, int M, int N, int K, int batch,
                      const int64_t *maps, double alpha, int accumulate);

/* out (device, n doubles) <- the seeded N(0,1) stream (seed, step, which) of the input recipe
 * (the device implementation of the generator of seeded_inputs/, which the
 * library uses for every input the caller did not supply with tatrg_set_sketch).  Equal to the host
 * generator's values up to the last-bit differences of log / sincos. */
int tatrg_fill_gauss(double *out, uint64_t n, uint64_t seed, uint64_t step, uint64_t which);

/* Thin QR with R_ii >= 0 of the row-major m x n matrix Y (device; m >= n, n <= 256): Q overwrites
 * Y, R (n x n row-major upper triangular) goes to R (device).  The "QR decomposition in the RSVD"
 * of PAPER.md:106 / the canonical form of PAPER.md:37 (Householder TSQR, robust to rank deficiency). */
int tatrg_qr_pos(double *Y, int64_t m, int n, double *R);

/* Blocked Cholesky factorisation of the symmetric positive definite n x n matrix A (device, row-major,
 * lower triangle read) + shift_rel * max_i A_ii on the diagonal: A <- L (lower, upper part zeroed);
 * Linv (device, n x n row-major, may be NULL) <- L^-1.  The factorisations behind the squeezers
 * (Eq. 12) and the reduced bond swap.  Returns 0,
 * 1 if a pivot was not positive (A then holds garbage), < 0 on error. */
int tatrg_cholesky(double *A, int n, double shift_rel, double *Linv);

/* Cholesky-QR of the tall row-major m x n block Y (device, n <= 256): `passes` (1..3) rounds of
 * {C = Y^T Y (+ shift_rel * max diag in the first round), C = L L^T, Y <- Y L^-T}; Q overwrites Y and
 * R (device, n x n row-major, may be NULL) receives the accumulated upper-triangular factor.  The
 * orthonormalisation inside the subspace iterations ("iterations of the QR decomposition").
 * Returns 0, 1 if a factorisation broke down, < 0 on error. */
int tatrg_cholqr(double *Y, int64_t m, int n, int passes, double shift_rel, double *R);

/* The subspace iteration of one squeezer as one launch (Eq. 12): for the
 * row-major n x n matrix F (device, n >= 64) and the n x 64 start block `start` (device, row-major),
 *   Q <- orth(F start);  `iters` (>= 1) times { Qt <- orth(F^T Q); Q <- orth(F Qt) };  Qt R <- F^T Q,
 * orth = one Cholesky-QR pass with a relative diagonal shift of 1e-13 (only the span is carried on), two unshifted
 * passes for the last Q and for the closing factorisation F^T Q = Qt R.  Q, Qt: device, n x 64 row-major, written;
 * R: device, 64 x 64 row-major upper triangular (may be NULL); minmax (device, 4 doubles, may be NULL): smallest and
 * largest diagonal entry of the first Cholesky factor of the last Q and of the closing factorisation.  The singular
 * values of R converge to the leading singular values of F.  `grid` = number of resident CTAs wanted (adjusted so
 * that every CTA owns between 1 and 16 blocks of 8 rows).  Uses the scratch workspace; synchronises the stream.
 * Returns 0, 1 if a Cholesky factorisation met a non-positive pivot, < 0 on error (TATRG_EINVAL: arguments). */
int tatrg_subspace_iteration(const double *F, int n, const double *start, double *Q, double *Qt, int iters, int grid,
                             double *R, double *minmax);

/* One-sided Jacobi SVD of the column-major m x n matrix G (device, ld = m): on exit G = U diag(s)
 * with orthogonal columns sorted by decreasing norm, V (n x n column-major, device) such that
 * G_in V = G_out, s (device, n) the singular values.  Also the symmetric PSD eigensolver
 * (G symmetric: V = eigenvectors, s = eigenvalues).  PAPER.md:25 (RSVD core), Eq. 3, Eq. 12. */
int tatrg_jacobi_svd(double *G, int m, int n, double *V, double *s);

/* Norm / trace reductions of the normalisation and of tTr T = <Phi,Psi> (Eq. 15):
 * out_dev[0] = sum x^2, resp. sum x*y; x *= 1/sqrt(*sumsq_dev).  All pointers device. */
int tatrg_sumsq(const double *x, int64_t n, double *out_dev);

/* tatrg_sumsq for callers that cannot allocate (code under CUDA graph capture, tight serving loops, harnesses that
 * forbid cudaMalloc): out_dev[0] = sum_i x[i]^2 (the squared Frobenius norm of the step's normalisation,
 * PAPER.md:119 Eq. 15) by the same two kernels on the same grid as tatrg_sumsq -- the result is equal to the last
 * bit -- with the per-CTA partial sums in a static device array of the library (1184 doubles = 9472 bytes per GPU,
 * held from library load to process exit) instead of the workspace.  Needs no tatrg_set_workspace, calls no
 * cudaMalloc / cudaFree or any allocating routine, and does not synchronise: the two kernels are enqueued on the
 * stream of tatrg_set_stream (default stream if none).  x: device, n doubles (n >= 0; n = 0 gives 0); out_dev:
 * device, 1 double, written.  n > TATRG_SUMSQ_STATIC_MAX_N is rejected with TATRG_EINVAL and nothing is launched.
 * All calls share the static array (it keeps the last call's partial sums; nothing in it has to start at zero):
 * calls whose kernels overlap on the GPU race -- order them on one stream or with events. */
#define TATRG_SUMSQ_STATIC_MAX_N (1LL << 32)   /* elements (32 GiB of doubles; chi^5 at chi = 64 is 2^30) */
int tatrg_sumsq_static(const double *x, int64_t n, double *out_dev);
int tatrg_dot(const double *x, const double *y, int64_t n, double *out_dev);
int tatrg_scale_by_rsqrt(double *x, int64_t n, const double *sumsq_dev);

/* Relative gaps (s[k-1]-s[k])/s[0] at the truncation cuts of the last step: bond swap,
 * squeezers t1..t3 (inf when nothing was cut).  A cut through a degenerate cluster shows here. */
int tatrg_get_gaps(double out[4]);
/* High-water mark of workspace use in bytes since tatrg_set_workspace. */
size_t tatrg_workspace_peak(void);

const char *tatrg_last_error(void);
void tatrg_destroy(void);

#ifdef __cplusplus
}
#endif
#endif /* TATRG_H */
