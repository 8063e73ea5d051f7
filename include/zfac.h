/* zfac.h -- C ABI of the B200 (sm_100a) Z-refinement library  (libzfac.so)
 *
 * The operation (PAPER.md = arxiv 2404.19163, /root/reference/PAPER.md):
 *   given a symmetric positive definite overlap matrix S and an initial guess Z0
 *   with ||Z0^T S Z0 - I||_2 < 1 (Eq. 12, Eq. 14), refine Z so
 *   that Z^T S Z = I, i.e. Z Z^T = S^-1 (Eq. 10), by Algorithm 2
 *    with m = 2:
 *
 *       R_n   = I - Z_n^T (S Z_n)                     (Eq. 13, 22, 26; R = -(X - I))
 *       Err[n]= ||R_n||_F                             (Alg. 2)
 *       stop if n > 0 and Err[n] > Err[n-1]^3         (Eq. 38)
 *       Z_n+1 = Z_n + Z_n (1/2 R_n + 3/8 R_n R_n)     (Eq. 13/16; = Z(15/8 I - 5/4 X + 3/8 X^2))
 *
 * Every step above runs in hand-written CUDA kernels (four fused GEMM kernels per
 * iteration + an O(N^2) copy-in and copy-out per call); there is no CPU fallback:
 * on a device that is not sm_100 every entry point that would launch work returns
 * ZFAC_E_UNSUPPORTED.
 *
 * Conventions common to all entry points
 *   - matrices are dense, ROW-MAJOR, N x N, leading dimension `ld` in ELEMENTS, ld >= N;
 *     S must be stored in full (both triangles);
 *   - element type is fixed by the mode: double for ZFAC_MODE_F64, float for
 *     ZFAC_MODE_SPLIT16, ZFAC_MODE_HH16 and ZFAC_MODE_TF32 ("The matrices Z and S are stored in
 *     single precision");
 *   - pointers named d_* are DEVICE pointers, h_* are HOST pointers; the caller owns
 *     every buffer including the workspace; the library owns only the small host-side
 *     context object;
 *   - all functions return a zfac_status; nothing throws or aborts across the ABI;
 *   - numerical failure (divergence, NaN) is NOT an error code: it is reported in the
 *     result flags and Z holds the last iterate, as Alg. 2 would leave it;
 *   - not checked ("straightforward to check separately"): S symmetric
 *     positive definite, ||Z0^T S Z0 - I||_2 < 1.
 */
#ifndef ZFAC_H_
#define ZFAC_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct zfac_ctx zfac_ctx; /* opaque */

/* Precision mode of the four GEMMs of one iteration.
 *  SPLIT16: the paper's (h)(h)+(h)(l)+(l)(h) scheme (Sec. III.A-B, Eq. 17-32): each FP32
 *           operand is split into two FP16 halves (the low half scaled by 2^11), three
 *           tensor-core MMA passes per product ((l)(l) dropped, Eq. 25/29/32), FP32 accumulation.
 *  TF32   : one tensor-core pass on FP32 operands rounded to TF32, FP32 accumulation.
 *  F64    : the paper's `double` scheme (Table I) on the FP64 tensor pipe.
 *  HH16   : the paper's (h)(h) scheme (Sec. III.C; Table I :211): operands
 *           rounded to FP16, one tensor-core pass, FP32 accumulation; meant to be followed by
 *           the refinement step (zfac_refine_refi).
 * Note on SPLIT16: the second-order product of step a4 (R R in Q = 1/2 R + 3/8 R R) runs its (h)(h) pass only when
 * the update is taken from Err[n] <= ZFAC_OPT_HH_SQUARE_ERR (default 0.1; decided on the device from the Err[n] just
 * computed); every other product always runs all three passes (ZFAC_OPT_HH_SQUARE = 0 disables it).
 *  F64_MIXED, F64_I8: FP64-master modes built for the refinement stage of Alg. 3 but complete modes of
 *           their own (element type double).  What needs FP64-level accuracy in an iteration is the RESIDUAL
 *           R = I - Z^T (S Z); the update Z + Z (1/2 R + 3/8 R R) is a correction of relative size ||R||, evaluated here
 *           with the SPLIT16 tensor-core passes on the FP32 parts of Z and R and ADDED to the FP64 master (its rounding
 *           leaves ~2^-22 ||R|| in the next residual; oracle: update_mixed).  The residual is computed
 *             F64_MIXED: on the FP64 tensor pipe (the kernels of ZFAC_MODE_F64);
 *             F64_I8   : on the INT8 tensor cores -- each FP64 operand row is cut, error-free, into ZFAC_OPT_I8_SLICES
 *                        int8 slices of 7 bits under one exponent per row, all slice products with i + j < slices are
 *                        accumulated exactly in INT32 and summed in FP64 (Ozaki scheme): ~2^(-7 slices) relative to the
 *                        row maxima, i.e. FP64-equivalent for 8 slices.  n <= 32768.
 *           Order m = 2 only; zfac_congruence is not available in these two modes. */
typedef enum { ZFAC_MODE_SPLIT16 = 0, ZFAC_MODE_TF32 = 1, ZFAC_MODE_F64 = 2, ZFAC_MODE_HH16 = 3,
               ZFAC_MODE_F64_MIXED = 4, ZFAC_MODE_F64_I8 = 5 } zfac_mode;

/* Stop rule.  PAPER: Alg. 2's parameter-free test.  FIXED: perform exactly max_iter updates
 * (benchmarks, and parity against the oracle "for the same number of iterations"). */
typedef enum { ZFAC_STOP_PAPER = 0, ZFAC_STOP_FIXED = 1 } zfac_stop;

typedef enum {
  ZFAC_OK = 0,
  ZFAC_E_INVALID = 1,     /* bad argument (null, n <= 0, ld < n, max_iter < 0, unknown enum)   */
  ZFAC_E_UNSUPPORTED = 2, /* current device is not compute capability 10.x                     */
  ZFAC_E_WORKSPACE = 3,   /* workspace null, misaligned (256 B) or smaller than required       */
  ZFAC_E_CUDA = 4         /* a CUDA runtime/driver call failed (see zfac_last_cuda_error)      */
} zfac_status;

/* Result flags written to *flags together with the outputs. */
enum {
  ZFAC_R_STOPPED = 1,  /* the test Err[n] > Err[n-1]^(m+1) fired (m = 2: ^3; converged to the precision floor) */
  ZFAC_R_MAXITER = 2,  /* max_iter updates were performed without the test firing               */
  ZFAC_R_NONFINITE = 4, /* Err[n] became inf/NaN; iteration stopped                              */
  ZFAC_R_REFINED = 8,   /* zfac_refine_refi: at least one refinement update was applied; ZFAC_OPT_EXTRA_UPDATE: the extra
                           update was taken                                                      */
  ZFAC_R_RANGE = 16,    /* SPLIT16 / HH16: a value of S, Z0, T = (S Z)^T or Z with magnitude >= 65504 was clamped when it
                           was rounded to an FP16 operand (FP16 range); the result is not to be trusted.  Admissible input:
                           abs(S_ij), abs(Z_ij), abs((S Z)_ij) < 65504 throughout -- e.g. lambda_min(S) >~ 3e-10 for a
                           normalised S; rescale S by a power of four otherwise (Z scales by its square root)   */
  ZFAC_R_NOCHECK = 32   /* ZFAC_OPT_FINAL_CHECK = 0: the residual of the last update was not evaluated (Err[iters] is NaN) */
};

/* Internal buffers that zfac_peek can copy out (parity tests of the individual steps).
 * After a call, T/R hold the values of the LAST residual evaluation (for the returned Z),
 * Q the polynomial of the last update performed. */
typedef enum {
  ZFAC_BUF_T = 0, /* T = (S Z)^T            step a1, Eq. 22 */
  ZFAC_BUF_R = 1, /* R = I - Z^T S Z        step a2, Eq. 26 */
  ZFAC_BUF_Q = 2, /* Q = 1/2 R + 3/8 R R    step a4, Eq. 30-32 */
  ZFAC_BUF_Z = 3  /* current Z              step a5, Eq. 13 */
} zfac_buf;

/* Bytes of device workspace zfac_create needs for an n x n problem in `mode`
 * (internal padded operand buffers, partial sums, staging for zfac_refine_host).
 * Returns 0 for invalid arguments.  Host function, launches nothing. */
size_t zfac_workspace_bytes(int64_t n, zfac_mode mode);

/* Create a context for n x n problems (1 <= n <= 2^20) in `mode`, bound to the CURRENT device and to the
 * caller-owned device workspace [d_workspace, d_workspace + bytes), which must be 256-byte
 * aligned and stay alive and otherwise unused until zfac_destroy.  Builds the TMA tensor maps.
 * One context serves any number of zfac_refine calls (the MD-step use),
 * one at a time.  Every later call on the context must be made with the same device current
 * (checked: ZFAC_E_INVALID otherwise).  Errors: INVALID, WORKSPACE, UNSUPPORTED, CUDA. */
zfac_status zfac_create(zfac_ctx** ctx, int64_t n, zfac_mode mode, void* d_workspace, size_t bytes);

/* Algorithm 2 on device buffers.  Asynchronous on `stream` (a cudaStream_t passed as void*;
 * NULL = default stream): enqueues the copy-in kernels, then for n = 0..max_iter the fused
 * kernels a1 (T=(S Z)^T), a2 (R = I - Z^T S Z, ||R||_F, stop test), a4 (Q = 1/2 R + 3/8 R R),
 * a5 (Z += Z Q), then the copy-out; no allocation, no host synchronisation; the stop decision
 * is taken on the device and later kernels of the call exit at once.  Outputs are valid once
 * the stream has been synchronised.
 *   d_S  [in]  n x n, lds;   d_Z0 [in] n x n, ldz0;   d_Z [out] n x n, ldz (may alias d_Z0)
 *   max_iter   upper bound on the number of Z updates (>= 0; 0 returns Z0 and Err[0])
 *   d_iters [out] int     number of Z updates performed (= stop index; PAPER counts iters+1 X evaluations)
 *   d_err   [out] double[max_iter+1]; entries 0..iters hold Err[n] = ||R_n||_F, the rest are untouched
 *   d_flags [out] int     ZFAC_R_* bits
 * Errors: INVALID (nothing enqueued), CUDA. */
zfac_status zfac_refine(zfac_ctx* ctx, const void* d_S, int64_t lds, const void* d_Z0, int64_t ldz0,
                        void* d_Z, int64_t ldz, int max_iter, zfac_stop stop, int* d_iters,
                        double* d_err, int* d_flags, void* stream);

/* Many small problems in ONE launch sequence (the graph-partitioned sub-problems of PAPER.md:98; the regime
 * N = O(10^2) - O(10^3) in which the paper reports its largest gain over diagonalisation).
 * A batched context refines `batch` independent n x n problems of one mode (SPLIT16, HH16 or TF32) together: every
 * kernel of the iteration is launched once and walks the tiles of all problems, so tensor-memory allocation, barrier
 * set-up and pipeline fill are paid per launch, not per problem.  Each problem has its own stop test, iteration count,
 * Err history and flags; a problem that has stopped is skipped by the later launches.  Results are bit-identical to
 * refining each problem alone with zfac_refine.
 *   problem b:  S at d_S + b * stride_S, Z0 at d_Z0 + b * stride_Z0, Z at d_Z + b * stride_Z (strides in elements,
 *               problems must not overlap);  d_iters[b], d_flags[b], d_err[b * (max_iter + 1) .. ]
 *   1 <= batch <= 4096 and batch * zfac_padded_n(n) <= 2^24.  zfac_refine_batched also accepts a context made by
 *   zfac_create (batch = 1).  The other entry points take unbatched contexts only (ZFAC_E_INVALID otherwise).
 * Errors: INVALID (also: mode F64 / F64_MIXED / F64_I8), WORKSPACE, UNSUPPORTED, CUDA. */
size_t zfac_workspace_bytes_batched(int64_t n, zfac_mode mode, int batch);
zfac_status zfac_create_batched(zfac_ctx** ctx, int64_t n, zfac_mode mode, int batch, void* d_workspace, size_t bytes);
int zfac_get_batch(const zfac_ctx* ctx);
zfac_status zfac_refine_batched(zfac_ctx* ctx, const void* d_S, int64_t lds, int64_t stride_S, const void* d_Z0,
                                int64_t ldz0, int64_t stride_Z0, void* d_Z, int64_t ldz, int64_t stride_Z, int max_iter,
                                zfac_stop stop, int* d_iters, double* d_err, int* d_flags, void* stream);

/* Algorithm 3 (PAPER.md:322-341; Sec. IV.B, :308-316): the "+refi" schemes of Table I.
 *   1. Algorithm 2 in the low-precision mode of `low` (FP32 S and Z0) until its parameter-free test fires (or
 *      max_iter updates);
 *   2. "Z = FP32[Z] or FP64[Z]": Z is handed to the context `high` of a MORE precise mode, straight
 *      from `low`'s workspace, and R = I - Z^T S Z is recomputed there (S converted exactly);
 *   3. `refi_steps` updates Z <- Z + Z (1/2 R + 3/8 R R) in `high`'s arithmetic (1 <= refi_steps <= 4000; the paper uses 1).
 * Allowed pairs (low -> high): HH16 -> SPLIT16, TF32 -> SPLIT16 (the paper's single-precision refinement,
 * SPLIT16 is this library's FP32-class arithmetic), and HH16 / TF32 / SPLIT16 -> F64,
 * F64_MIXED or F64_I8 (double-precision refinement).  `high` has the same n and order and its own workspace.  d_Z is n x n of `high`'s element
 * type (float for SPLIT16, double for F64 / F64_MIXED / F64_I8).
 * With final_check != 0 the residual of the returned Z is evaluated in `high` as well (two more GEMMs); Alg. 3 as
 * printed stops after the update (final_check = 0).
 *   d_iters [out] low-precision updates + refinement updates performed
 *   d_err   [out] double[max_iter + refi_steps + 2]: Err[0..k] of the low-precision run (k = its stop index), then
 *                 `high`'s Err before each refinement update, then (final_check) `high`'s Err of the returned Z
 *   d_flags [out] flags of the low-precision run | ZFAC_R_REFINED (if a refinement update was applied)
 * If the low-precision run ends non-finite nothing is refined (Z = its last iterate, promoted); if a refinement
 * residual is non-finite the refinement stops there (ZFAC_R_NONFINITE); d_iters and d_err say what was done.
 * Asynchronous on `stream`, no allocation, no host synchronisation.  Errors: INVALID (also: mode pair not allowed,
 * orders differ), CUDA. */
zfac_status zfac_refine_refi(zfac_ctx* low, zfac_ctx* high, const void* d_S, int64_t lds, const void* d_Z0,
                             int64_t ldz0, void* d_Z, int64_t ldz, int max_iter, int refi_steps, int final_check,
                             int* d_iters, double* d_err, int* d_flags, void* stream);

/* zfac_refine_refi on HOST buffers (pinned memory recommended): h_S, h_Z0 float, h_Z of `high`'s element type.
 * Uploads S and Z0 (overlapped with the first a1 as in zfac_refine_host), runs Alg. 3, downloads Z (started right
 * after the last refinement update, i.e. overlapped with the final check), iters, Err[] and flags, and synchronises
 * `stream`.  max_iter + refi_steps + 2 <= 4096.  h_err: double[max_iter + refi_steps + 2].  This is the end-to-end
 * "time to gate" call of bench.py. */
zfac_status zfac_refine_refi_host(zfac_ctx* low, zfac_ctx* high, const void* h_S, int64_t lds, const void* h_Z0,
                                  int64_t ldz0, void* h_Z, int64_t ldz, int max_iter, int refi_steps, int final_check,
                                  int* h_iters, double* h_err, int* h_flags, void* stream);

/* Congruence transformation H_perp = Z^T H Z (Eq. 11): what Z is for.  H is
 * n x n symmetric (full storage), Z n x n (any inverse factor), element type of the context's
 * mode; the product runs through the same kernels as the residual (T = (H Z)^T, then Z^T (H Z)
 * with a symmetric-output epilogue: off-diagonal tiles are mirrored).  d_out is n x n, ld ldo.
 * Asynchronous on `stream`.  Uses the context's workspace: not concurrently with zfac_refine. */
zfac_status zfac_congruence(zfac_ctx* ctx, const void* d_H, int64_t ldh, const void* d_Z, int64_t ldz,
                            void* d_out, int64_t ldo, void* stream);

/* Same operation on HOST buffers (pinned memory recommended): copies S and Z0 to the device
 * staging area of the workspace, runs zfac_refine, copies Z, iters, Err[0..iters] and flags
 * back, and synchronises `stream` before returning.  This is the end-to-end call bench.py times.
 * max_iter <= 4095 (size of the staging area for Err[]; ZFAC_E_INVALID beyond).
 * Transfers are overlapped with the kernels where the data dependences allow, results are
 * bit-identical to zfac_refine either way:
 *   - pinned h_Z, max_iter >= 1: the download of Z starts right after the first update on an internal side stream; it
 *     is the result if that update is the only one (a warm start), else the download at the end supersedes it
 *     (ZFAC_OPT_HOST_OVERLAP = 0 disables it);
 *   - pinned h_S and h_Z0, a tensor-core mode, padded dimension >= 1024: Z0 is uploaded first, then S in up to 8
 *     chunks of whole 256-row blocks; each chunk is converted (step a0) and multiplied (step a1 restricted to that
 *     band of tiles) while the next one is on the bus (ZFAC_OPT_HOST_UPLOAD_OVERLAP = 0 disables it);
 *   - in those modes the first update's a5 runs in ZFAC_OPT_HOST_A5_BANDS (default 2) row bands, each band's rows
 *     of Z downloaded as soon as they are final.
 * Pageable buffers take the plain path. */
zfac_status zfac_refine_host(zfac_ctx* ctx, const void* h_S, int64_t lds, const void* h_Z0,
                             int64_t ldz0, void* h_Z, int64_t ldz, int max_iter, zfac_stop stop,
                             int* h_iters, double* h_err, int* h_flags, void* stream);

/* Copy an internal buffer (top-left n x n block, converted to the mode's element type) to
 * d_out (n x n, ld).  Asynchronous on `stream`.  For tests of the individual steps. */
zfac_status zfac_peek(zfac_ctx* ctx, zfac_buf which, void* d_out, int64_t ld, void* stream);

/* Concurrency.  Contexts share no state (each owns its workspace and tensor maps; the last-error string is
 * thread-local): calls on DIFFERENT contexts may be issued from different host threads and / or on different streams
 * and run concurrently on the device; results are bit-identical to running them one after another.  This is the way
 * to refine many small problems at once (the graph-partitioned sub-problems of PAPER.md:98).
 * Calls on the SAME context must not overlap (they share the workspace); issue them on one stream. */

/* CUDA graphs.  zfac_refine, zfac_refine_refi and zfac_congruence only enqueue kernels on `stream`: no allocation, no
 * host synchronisation, no host-side dependence on device results (the stop decision stays on the device and the
 * statically enqueued kernels after it return at once).  With profiling disabled (zfac_set_profile) a call can
 * therefore be captured into a CUDA graph (cudaStreamBeginCapture ... cudaStreamEndCapture) and replayed; the graph
 * reads and writes the SAME user and workspace buffers as the captured call, so new inputs are written into them in
 * place.  One graph launch replaces 2 + 2 (max_iter + 1) + 2..3 max_iter kernel launches (measurements: DESIGN.md §1). */

/* The whole call as ONE CUDA graph with a WHILE node: copy-in, first residual, WHILE (not stopped) { update, residual,
 * update, residual }, copy-out.  The stop test (Alg. 2, Eq. 38) of every residual sets the loop condition on
 * the device, so the graph runs exactly as many iterations as the refinement needs: none of the 2 + 4 max_iter
 * statically enqueued launches of zfac_refine that return at once after the stop exist here.  Same arguments, same results (bit-identical) and
 * the same restrictions as zfac_refine; the graph is bound to these buffers (write new inputs into them) and to the
 * context's order at creation time.  zfac_graph_launch is asynchronous on `stream`; launches of one graph, and of graphs
 * and calls that share a context, must not overlap.  Destroy graphs before their context. */
typedef struct zfac_graph zfac_graph; /* opaque */
zfac_status zfac_graph_create(zfac_ctx* ctx, const void* d_S, int64_t lds, const void* d_Z0, int64_t ldz0,
                              void* d_Z, int64_t ldz, int max_iter, zfac_stop stop, int* d_iters,
                              double* d_err, int* d_flags, zfac_graph** graph);
zfac_status zfac_graph_launch(zfac_graph* graph, void* stream);
zfac_status zfac_graph_destroy(zfac_graph* graph);

/* Per-context options (host-side state only: no device work; take effect from the next call on `ctx`).  They
 * replace every environment variable earlier versions read.  Values are passed as double; integer options are
 * rounded.  Unknown key or out-of-range value -> ZFAC_E_INVALID, the option keeps its value.
 *   The first group changes which arithmetic is performed (hence results, within the mode's accuracy):           default
 *   ZFAC_OPT_CHUNK_KB        SPLIT16, a1 / a2: k-blocks (64 products each) of (h)(h) products that are summed in the
 *                            tensor core's truncating FP32 accumulator before they are added, with round-to-nearest,
 *                            to FP32 registers ("promoted accumulation"); 1 .. 1024                    1
 *   ZFAC_OPT_CHUNK0_KB       ... length of the FIRST chunk of every tile (>= CHUNK_KB to take effect)                 1
 *   ZFAC_OPT_HH_SQUARE       SPLIT16, a4 (and p2): one (h)(h) pass for the second-order product when the update is
 *                            taken from Err[n] <= HH_SQUARE_ERR; 0 = always three passes (Eq. 32 as printed)        1
 *   ZFAC_OPT_HH_SQUARE_ERR   the bound, >= 0                                                                       0.1
 *   ZFAC_OPT_PROMOTE_UPDATE  SPLIT16: promoted accumulation in the update GEMMs (p2, a4, a5) as well; 0 / 1          0
 *   ZFAC_OPT_I8_SLICES       F64_I8: int8 slices per operand row = orders i + j kept, 2 .. 8 (7 bits each)              8
 *   ZFAC_OPT_INPUT_F32       F64, F64_MIXED, F64_I8: S and Z0 are given as FLOAT ("FP32 stored" inputs, promoted exactly);
 *                            Z is still returned as double; 0 / 1                                                   0
 *   ZFAC_OPT_EXTRA_UPDATE    F64_MIXED, F64_I8 with ZFAC_STOP_PAPER: when the test fires, perform ONE more update (flag
 *                            ZFAC_R_REFINED) and stop after its residual.  The FP32-class correction of these modes makes the
 *                            test also fire when Err has only reached ~2^-22 sqrt(kappa) Err[n-1], one update short of the
 *                            FP64 floor (cold starts); this is Alg. 3's single refinement step, built in; 0 / 1               0
 *   ZFAC_OPT_FINAL_CHECK     F64_MIXED, F64_I8 with ZFAC_STOP_PAPER: 1 = Alg. 2 as printed, every update is followed by its
 *                            residual.  0 = a residual whose stop decision is known beforehand is not evaluated: the one
 *                            after an update taken from Err[n]^3 < 2^-53 sqrt(N) (the test is bound to fire), or, with
 *                            ZFAC_OPT_EXTRA_UPDATE, the one after the extra update.  Same Z, bit for bit, and same iteration
 *                            count as with 1 whenever that run ends by the test; Err[iters] = NaN, flag ZFAC_R_NOCHECK;
 *                            saves one residual (a1 + a2) per call; 0 / 1                                              1
 *   The rest change scheduling only (bit-identical results):
 *   ZFAC_OPT_BAND            full GEMMs: tile columns per rasterisation band, 1 .. 4096                               8
 *   ZFAC_OPT_MAX_PAIRS       tensor-core modes: use at most this many CTA pairs; 0 = all co-resident ones            0
 *   ZFAC_OPT_NARROW_TILES    SPLIT16, HH16, TF32: 256 x 128 pair tiles instead of 256 x 256 (twice as many
 *                            tiles: a small problem occupies more of the chip); -1 = automatically when batch x (padded order / 256)^2
 *                            <= 37 (one problem of padded order <= 1536, or a few smaller ones), 0 = never, 1 = always          -1
 *   ZFAC_OPT_PDL             SPLIT16, HH16, TF32: programmatic dependent launch of the GEMM kernels (a kernel is scheduled while
 *                            its predecessor still runs and waits for it on the device before it reads anything); not
 *                            used inside zfac_graph_*.  In small launches (batch x (padded order / 256)^2 <= 37) the kernel's
 *                            set-up (barriers, tensor memory) runs ahead of that wait as well.  -1 = automatically (small
 *                            launches: 4 .. 21 % off a call; one problem of any size: the launches behind the stop cost
 *                            half; HH16 / TF32 up to padded order 2048: 7 .. 15 % off the working kernels too; larger
 *                            batched launches: not used),
 *                            0 = never, 1 = always, 2 = always, without the early set-up                              -1
 *   ZFAC_OPT_I8_NARROW       F64_I8: the INT8 kernels on 256 x 128 tiles (T and R bit-identical, Err[] in its last bits only);
 *                            -1 = automatically up to padded order 1536 (17 .. 24 % off a call), 0 = never, 1 = always   -1
 *   ZFAC_OPT_I8_CLUSTER      F64_I8, a1 (when the padded order is a multiple of 512): clusters of two CTA pairs that share
 *                            the B slices by TMA multicast (L2 -> SM bytes -25 %); only 33 such clusters are co-resident on a
 *                            B200 against 74 pairs, measured a tie; 0 / 1                              0
 *   ZFAC_OPT_HOST_OVERLAP, ZFAC_OPT_HOST_UPLOAD_OVERLAP (0 / 1), ZFAC_OPT_HOST_A5_BANDS (1 .. 64): zfac_refine_host     1, 1, 2 */
typedef enum {
  ZFAC_OPT_CHUNK_KB = 0, ZFAC_OPT_CHUNK0_KB = 1, ZFAC_OPT_HH_SQUARE = 2, ZFAC_OPT_HH_SQUARE_ERR = 3,
  ZFAC_OPT_PROMOTE_UPDATE = 4, ZFAC_OPT_BAND = 5, ZFAC_OPT_MAX_PAIRS = 6, ZFAC_OPT_HOST_OVERLAP = 7,
  ZFAC_OPT_HOST_UPLOAD_OVERLAP = 8, ZFAC_OPT_HOST_A5_BANDS = 9, ZFAC_OPT_I8_SLICES = 10, ZFAC_OPT_INPUT_F32 = 11,
  ZFAC_OPT_EXTRA_UPDATE = 12, ZFAC_OPT_FINAL_CHECK = 13, ZFAC_OPT_I8_CLUSTER = 14,
  ZFAC_OPT_NARROW_TILES = 15, ZFAC_OPT_PDL = 16, ZFAC_OPT_I8_NARROW = 17
} zfac_option;
zfac_status zfac_set_option(zfac_ctx* ctx, zfac_option key, double value);
zfac_status zfac_get_option(const zfac_ctx* ctx, zfac_option key, double* value);

/* Order m of the refinement polynomial, Z_{n+1} = Z_n sum_{k=0..m} c_k R_n^k  (Eq. 13 / Eq. 16:
 * "Reference 1 gives a table with the coefficients a_k for polynomials of order m = 2, 3, 4, 5. For the tests in
 * this article, we use m = 2").  m = 2 (default; the paper's scheme), 3 or 4; anything else -> ZFAC_E_INVALID and
 * the context keeps its order (F64_MIXED / F64_I8: m = 2 only).  The coefficients follow from the paper's condition that the error terms vanish to
 * the highest possible order: c_k = C(2k,k)/4^k = 1, 1/2, 3/8, 5/16, 35/128, and the stop test
 * becomes Err[n] > Err[n-1]^(m+1) (nu_max = m + 1; Eq. 38).  For m > 2 step a4 is two symmetric
 * GEMMs, P = R R and Q = 1/2 R + P G with G = 3/8 I + 5/16 R (+ 35/128 P for m = 4), i.e. five kernels per
 * iteration instead of four.  Host-side state only: takes effect from the next zfac_refine* call on `ctx`;
 * no device work, no synchronisation.  ZFAC_BUF_Q then holds Q = sum_{k>=1} c_k R^k. */
zfac_status zfac_set_order(zfac_ctx* ctx, int m);
int zfac_get_order(const zfac_ctx* ctx);

/* Number of kernels the last zfac_refine / zfac_refine_host call on this context enqueued. */
int zfac_last_launch_count(const zfac_ctx* ctx);

/* Per-kernel timing for benchmarks.  With profiling enabled, zfac_refine records a CUDA event
 * on the launching stream before every GEMM kernel and after the last one (a few microseconds
 * of overhead per kernel).  After the stream has been synchronised, zfac_get_profile returns,
 * for the last call, up to `cap` entries: tags[i] = step id (1 = a1, 2 = a2, 4 = a4, 5 = a5)
 * + 16 * iteration index, ms[i] = milliseconds until the next event.  Returns the entry count. */
zfac_status zfac_set_profile(zfac_ctx* ctx, int enable);
int zfac_get_profile(zfac_ctx* ctx, int* tags, float* ms, int cap);

/* Padded internal dimension used for n in `mode` (multiple of the tile size). */
int64_t zfac_padded_n(int64_t n, zfac_mode mode);

/* Destroy the context (host memory only; the workspace stays the caller's). NULL is OK. */
zfac_status zfac_destroy(zfac_ctx* ctx);

/* Static string for a status code. */
const char* zfac_status_string(zfac_status s);

/* Last CUDA error string recorded on this thread by a ZFAC_E_CUDA return ("" if none). */
const char* zfac_last_cuda_error(void);

/* ------------------------------------------------------------------------------------------------------------------
 * An entry point that ALLOCATES NOTHING (no context, no workspace, no cudaMalloc / cudaFree / stream or event creation):
 * for callers that cannot allocate -- code under CUDA graph capture, tight serving loops, harnesses that forbid it.
 *
 *   *d_err = || I - Z^T (S Z) ||_F        (Err of Alg. 2 for a GIVEN Z: Eq. 22-29; FP64 throughout)
 *
 * -- the check a consumer makes on a Z it holds (is it still an inverse factor of this S, or must it be refined?).
 * It is the variant of the library's steps a1, a2, a3 whose scratch (T = S Z, the per-CTA partial sums, the arrival
 * counter) lives in a file-scope device array of libzfac.so instead of a caller workspace: 8 MiB + 32 KiB + 256 B, held
 * by every GPU that loads the library until the process exits.
 *   d_S, d_Z [in]  device, double, row-major, n x n, leading dimensions lds, ldz >= n (elements); not modified
 *   n              1 .. ZFAC_NOALLOC_MAX_N; larger n is REJECTED with ZFAC_E_INVALID (zfac_noalloc_last_error() says why):
 *                  use zfac_create / zfac_refine (max_iter = 0) with a workspace there
 *   d_err    [out] device, one double; valid once the work enqueued on `stream` has completed
 *   stream         a cudaStream_t passed as void* (NULL = default stream); the call is asynchronous: one 4-byte memset
 *                  + two kernels on `stream`
 * The result is run-to-run deterministic (partial sums added in index order).  ALL calls on a device share the one scratch
 * array: it keeps the last call's contents (nothing in it needs to survive; the counter is cleared at the head of every
 * call), and two calls that OVERLAP on the GPU -- different streams without an event between them -- RACE on it and give
 * wrong results.  Serialise them.  Calls on different devices do not interact.
 * Returns ZFAC_OK, ZFAC_E_INVALID (null pointer, n < 1, n > ZFAC_NOALLOC_MAX_N, ld < n) or ZFAC_E_CUDA; the reason of
 * the last failure on this thread is in zfac_noalloc_last_error() ("" after a success). */
#define ZFAC_NOALLOC_MAX_N 1024
zfac_status zfac_residual_norm_noalloc(const double* d_S, int64_t lds, const double* d_Z, int64_t ldz, int64_t n,
                                       double* d_err, void* stream);
const char* zfac_noalloc_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* ZFAC_H_ */
