/*
 * cbgmres.h -- C ABI of the B200-native compressed-basis GMRES (CB-GMRES) hot path.
 *
 * Method: arXiv 2009.12101, "Compressed Basis GMRES on High Performance GPUs".  Citations are
 * PAPER.md:<line> (the paper text) and the DESIGN.md reading they rely on.
 *
 * Problem statement: solve A x = b, A in R^{n x n} sparse with nnz nonzeros in
 * CSR (fp64 values + 32-bit indices), by restarted GMRES (Fig. 1)
 * with restart length m, classical Gram-Schmidt with optional re-orthogonalisation threshold eta
 * (PAPER.md:104), stopping when ||b - A x||_2 <= tau ||b||_2.  The Krylov
 * basis is kept in HBM in one of five storage formats while every arithmetic operation is IEEE
 * binary64.
 *
 * Conventions
 *   - Pointers named d_* are DEVICE pointers, h_* are HOST pointers.  All buffers are owned by the
 *     caller (torch tensors in the Python binding); the library only borrows them for the duration
 *     of the call, except the CSR arrays given to cbgmres_set_matrix, which must stay valid until
 *     the next set_matrix / destroy.
 *   - Every call returns a cbgmres_status_t (0 = success).  No exceptions, no errno, no stdout.
 *     On an invalid argument nothing is enqueued.  cbgmres_last_error gives a static string.
 *   - The CUDA stream given to cbgmres_create is borrowed; every call enqueues on it.  Calls that
 *     return results to the host (solve, solve_host) synchronise that stream before returning;
 *     the k_* hooks and set_matrix only enqueue.
 *   - Device memory: cbgmres_create allocates a fixed scratch block (reduction partials and the
 *     solver's control block, a few MB); cbgmres_set_matrix may allocate O(nnz/1024) ints of
 *     row-partition metadata.  cbgmres_solve allocates nothing: the basis and work vectors live in
 *     the caller's workspace.
 *   - One handle per host thread; handles share no mutable state (options, error slots and per-device
 *     kernel attributes are per handle / per device), so several handles -- on one device or on several --
 *     can live in one process.  Basis offsets are 64-bit; CSR indices are 32-bit.
 *   - A basis is stored vector-major: vector c occupies ld entries of the storage type starting
 *     at entry c*ld; ld >= n and ld*bytes(format) must be a multiple of 16, base 16-byte aligned.
 */
#ifndef CBGMRES_H_
#define CBGMRES_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct cbgmres_ctx *cbgmres_handle_t;

/* Storage formats of the basis: <float64>, <float32>, <float16> (IEEE casts,
 * round-to-nearest-even, gradual underflow) and the fixed-point <int32>, <int16> with one scale
 * sigma_j = ||v_j||inf / max_int per vector (readings Q6/Q7). */
typedef enum {
    CBGMRES_FP64 = 0,
    CBGMRES_FP32 = 1,
    CBGMRES_FP16 = 2,
    CBGMRES_INT32 = 3,
    CBGMRES_INT16 = 4
} cbgmres_format_t;

/* Fig. 1 lines 7-11: never, when h_{j+1,j} < eta*omega, or on every step. */
typedef enum { CBGMRES_REORTH_NEVER = 0, CBGMRES_REORTH_COND = 1, CBGMRES_REORTH_ALWAYS = 2 } cbgmres_reorth_t;

typedef enum {
    CBGMRES_OK = 0,
    CBGMRES_E_INVALID = 1,    /* bad argument (null pointer, n <= 0, restart < 1, unknown format ...) */
    CBGMRES_E_NOMATRIX = 2,   /* solve / k_spmv before set_matrix */
    CBGMRES_E_WORKSPACE = 3,  /* workspace too small or misaligned */
    CBGMRES_E_CUDA = 4,       /* a CUDA runtime call failed; see cbgmres_last_error */
    CBGMRES_E_NONFINITE = 5,  /* non-finite residual norm; x holds the last completed cycle */
    CBGMRES_NOT_CONVERGED = 16 /* ran to max_iters; x is valid, result is filled */
} cbgmres_status_t;

/* Right preconditioner M (Fig. 1 l.3 "w := A(M^-1 v_j)", l.17 "x_m := x_0 + M^-1(V_m y_m)").
 * JACOBI: M = diag(A), the setting of every experiment in the paper; a row without a
 * nonzero diagonal entry is left unscaled.  It costs one pass over the matrix per solve and nvals*8 +
 * n*8 more workspace bytes (cbgmres_workspace_bytes accounts for them); the Arnoldi loop is unchanged.
 * BLOCK_JACOBI4: M = the 4 x 4 diagonal blocks of A (rows / columns 4b .. 4b+3; the last block is completed by
 * the identity when 4 does not divide n; a singular block is replaced by the identity), inverted once per solve
 * in fixed (fp64) precision -- the baseline of the paper's section 6.5.  The store kernel
 * hands z = M^-1 v to the next SpMV (l.3) and the cycle end forms x += M^-1 (V_k y) (l.17).  It costs 32 bytes
 * per row and Arnoldi step, and ceil(n/4) * 128 more workspace bytes. */
typedef enum { CBGMRES_PRECOND_NONE = 0, CBGMRES_PRECOND_JACOBI = 1, CBGMRES_PRECOND_BLOCK_JACOBI4 = 2 } cbgmres_precond_t;

#define CBGMRES_MAX_RESTART 512

typedef struct {
    int32_t restart;         /* m, 1..CBGMRES_MAX_RESTART (the paper uses 100, 10..300) */
    int32_t max_iters;       /* bound on Arnoldi steps summed over all restart cycles */
    int32_t format;          /* cbgmres_format_t */
    int32_t reorth;          /* cbgmres_reorth_t */
    double rel_tol;          /* tau */
    double eta;              /* re-orthogonalisation threshold; 0 -> 1/sqrt(2) (reading Q3) */
    double *h_res_history;   /* optional HOST buffer: recurrence residual |g_{j+1}|/||b|| per Arnoldi step */
    int32_t res_history_cap; /* entries available in h_res_history (0 if unused) */
    int32_t precond;         /* cbgmres_precond_t: right preconditioner M of Fig. 1 l.3 / l.17 (0 = none) */
} cbgmres_params;

typedef struct {
    int32_t iters;        /* Arnoldi steps done */
    int32_t restarts;     /* restart cycles started */
    int32_t reorth_count; /* steps on which the second Gram-Schmidt pass ran */
    int32_t breakdown;    /* 1 if the last cycle ended through Fig. 1 line 12 */
    int32_t converged;    /* 1 iff the explicit residual met tau*||b|| */
    int32_t spmv_kernel;  /* which SpMV variant ran (see cbgmres_set_option "spmv_kernel"); 1016 = the whole solve ran as
                           * one kernel of a 16-CTA thread-block cluster (small systems, option "small_path") */
    double rel_res_recurrence; /* |g_{k+1}| / ||b|| at the end of the last cycle */
    double rel_res_true;       /* last explicit ||b - A x|| / ||b|| */
    double b_norm;
    double solve_ms;      /* device time of the whole solve (CUDA events on the stream) */
    double algorithmic_bytes; /* bytes the method must move through HBM for the launches that ran: per Arnoldi step
                               * S1 + S2 + S3 (+ S3' [+ S2'] where l.7 fired) + S4, per cycle S7 + S6 (cbgmres_profile_get
                               * lists the per-kernel figures); divided by solve_ms: the whole solve's achieved GB/s */
} cbgmres_result;

/* ---- the four calls of the problem statement ------------------------------------------------ */

/* Create a handle bound to `device` and to `cuda_stream` (a cudaStream_t, borrowed; NULL = the
 * legacy default stream).  Allocates the handle's fixed scratch block. */
int cbgmres_create(cbgmres_handle_t *out, int device, void *cuda_stream);

/* Register A in CSR: row_ptr int32[n+1], col_idx int32[nnz], vals fp64[nnz], all
 * DEVICE, BORROWED (not copied).  Reads row_ptr once (synchronises the stream) to choose the SpMV
 * variant for the row-length distribution ("automatically selects a CSR kernel"). */
int cbgmres_set_matrix(cbgmres_handle_t h, int64_t n, int64_t nnz, const int32_t *d_row_ptr,
                       const int32_t *d_col_idx, const double *d_vals);

/* Bytes of device workspace cbgmres_solve needs for these params and the registered matrix:
 * (restart+1) basis vectors in the storage format + two fp64 work vectors + small arrays. */
int cbgmres_workspace_bytes(cbgmres_handle_t h, const cbgmres_params *p, size_t *bytes);

/* Restarted CB-GMRES (Fig. 1).  d_b fp64[n]; d_x fp64[n] holds x0 on entry and the solution
 * approximation on exit; d_workspace 256-byte aligned.  Synchronises the stream, fills *out.
 * Returns CBGMRES_OK (converged), CBGMRES_NOT_CONVERGED, or an error. */
int cbgmres_solve(cbgmres_handle_t h, const double *d_b, double *d_x, const cbgmres_params *p, void *d_workspace,
                  size_t workspace_bytes, cbgmres_result *out);

/* Same solve with HOST buffers (the end-to-end path bench.py times): copies the CSR arrays, b and
 * x0 host->device into the workspace, solves, copies x device->host.  Needs
 * cbgmres_workspace_bytes_host bytes.  Host buffers should be pinned for full copy bandwidth.
 * Replaces the handle's registered matrix (it then points into d_workspace). */
int cbgmres_workspace_bytes_host(cbgmres_handle_t h, int64_t n, int64_t nnz, const cbgmres_params *p, size_t *bytes);
int cbgmres_solve_host(cbgmres_handle_t h, int64_t n, int64_t nnz, const int32_t *h_row_ptr, const int32_t *h_col_idx,
                       const double *h_vals, const double *h_b, double *h_x, const cbgmres_params *p,
                       void *d_workspace, size_t workspace_bytes, cbgmres_result *out);

int cbgmres_destroy(cbgmres_handle_t h);

/* Static string describing the last error on this handle (valid until the next call). */
const char *cbgmres_last_error(cbgmres_handle_t h);

/* Tuning / test knobs, by name.  "spmv_kernel": 0 = choose from the row-length statistics,
 * L in {2,4,8,16,32} = L lanes per row, 64 = nnz-balanced streaming kernel, 65 = the same with the matrix stream staged
 * in shared memory by bulk copies, 129/130/132 = row-major kernel with 1/2/4 rows per thread, 146/148/152 = with 2/4/8
 * lanes per row.  "poll": 1 (default)
 * = the host stops launching a cycle's remaining steps once the device reports it left the cycle.
 * "profile": N > 0 = time the kernels of every N-th Arnoldi step of a cycle with CUDA events (see
 * cbgmres_profile_get; 1 = every step), default 0.  "pdl": 1 (default) = launch the step kernels with
 * programmatic stream serialisation (each parks in griddepcontrol.wait until its predecessor is done).
 * "small_path": 1 (default) = a system whose compressed basis, matrix and vectors fit the distributed shared memory of
 * one 16-CTA thread-block cluster (about 3 MB: e.g. n = 4,096, m = 50 in fp64) is solved by ONE kernel launch with
 * cluster barriers in place of kernel boundaries (preconditioner none or scalar Jacobi, restart <= 128); 0 = always the
 * large path.  "orth_fuse": 1 (default) = fuse the first update with the second pass's multi-dot (one read of V).
 * "orth_fused_rows": the fused pass maps warps to rows and adds the update's partial sums with shuffles
 * (orth_fused_kernel) for 2 (default) = the 16-bit formats, 1 = every reduced format, 0 = never (the column-mapped
 * kind of orth_kernel with its shared-memory reduction).
 * "orth_seg_kb": 0 (default, chosen per launch), 1, 2 or 4 = KB per column segment of the
 * Gram-Schmidt passes' row tiles.  "orth_interleave": 0 (default) or 2 = row tiles dealt round-robin to
 * the CTAs, 1 = one contiguous row range per CTA.  Every option belongs to the handle it is set on.
 * Unknown names return CBGMRES_E_INVALID. */
int cbgmres_set_option(cbgmres_handle_t h, const char *name, int64_t value);

/* Number of kernels this handle has launched since creation (bench.py's gpu_launches). */
int64_t cbgmres_launch_count(cbgmres_handle_t h);

/* Per-kernel timing (option "profile" = N): cbgmres_solve brackets the launches (of every N-th step) of the families
 * below with CUDA events on its stream and accumulates, per family, the device time, the
 * ALGORITHMIC bytes of those launches (S1 12 nnz + 4(n+1) + 16 n;
 * S2 j n B + 8 n; S3 j n B + 16 n; S4 (16 + B) n; a fused S3+S2' launch counts j n B + 16 n)
 * and their number.  Launches the device skipped (steps after the cycle's last, second passes that
 * did not fire) are left out.  profile_get reads the totals since the last profile_reset. */
#define CBGMRES_PROF_FAMILIES 7
typedef enum {
    CBGMRES_PROF_SPMV = 0,     /* S1 */
    CBGMRES_PROF_MULTIDOT = 1, /* S2, S2' */
    CBGMRES_PROF_UPDATE = 2,   /* S3, S3' */
    CBGMRES_PROF_STORE = 3,    /* S4 (+ the Givens update riding on it) */
    CBGMRES_PROF_XUPDATE = 4,  /* S6: back substitution + x += V y */
    CBGMRES_PROF_RESIDUAL = 5, /* S7: r = b - A x and the store of v_1 */
    CBGMRES_PROF_UPDATE_DOT = 6 /* S3 + S2' from one read of the basis */
} cbgmres_prof_family_t;
int cbgmres_profile_get(cbgmres_handle_t h, int32_t family, double *ms, double *bytes, int64_t *launches);
int cbgmres_profile_reset(cbgmres_handle_t h);

/* ---- per-kernel hooks (parity is judged per kernel: BASELINE.json north_star) ------------- */

/* enc: d_payload[n] <- storage(d_v[n]); *d_scale <- sigma (1.0 for the
 * floating-point formats).  Bit-exact function of the fp64 input. */
int cbgmres_k_compress(cbgmres_handle_t h, int32_t format, int64_t n, const double *d_v, void *d_payload,
                       double *d_scale);
/* dec: d_v[n] <- fp64(d_payload[n]) * (*d_scale for the integer formats). */
int cbgmres_k_decode(cbgmres_handle_t h, int32_t format, int64_t n, const void *d_payload, const double *d_scale,
                     double *d_v);
/* S2, Fig. 1 line 5: d_h[c] <- sum_i dec(V)[i,c] * d_w[i], c = 0..k-1. */
int cbgmres_k_multidot(cbgmres_handle_t h, int32_t format, int64_t n, int64_t ld, int32_t k, const void *d_V,
                       const double *d_scales, const double *d_w, double *d_h);
/* S3, Fig. 1 lines 5-6: d_w[i] <- d_w[i] - sum_c dec(V)[i,c] * d_h[c];
 * *d_nrm2 <- ||w||_2 and *d_amax <- ||w||_inf of the new w, computed in the same pass. */
int cbgmres_k_update(cbgmres_handle_t h, int32_t format, int64_t n, int64_t ld, int32_t k, const void *d_V,
                     const double *d_scales, const double *d_h, double *d_w, double *d_nrm2, double *d_amax);
/* S3 + S2' fused, Fig. 1 lines 5-8: the update of k_update followed by
 * d_u[c] <- sum_i dec(V)[i,c] * d_w_new[i], from one read of the basis.  k is limited by the
 * shared-memory ring (128 at most; CBGMRES_E_INVALID beyond). */
int cbgmres_k_update_multidot(cbgmres_handle_t h, int32_t format, int64_t n, int64_t ld, int32_t k, const void *d_V,
                              const double *d_scales, const double *d_h, double *d_w, double *d_u, double *d_nrm2,
                              double *d_amax);
/* S4, Fig. 1 lines 13-14: d_v_fp64[i] <- d_w[i] / hnorm;
 * d_payload_col[n] <- enc(v); *d_scale <- sigma.  amax = ||w||_inf (only read by the integer formats). */
int cbgmres_k_store(cbgmres_handle_t h, int32_t format, int64_t n, const double *d_w, double hnorm, double amax,
                    void *d_payload_col, double *d_scale, double *d_v_fp64);
/* Block-Jacobi(4): d_inv[16 b + 4 r + c] <- (A_bb^-1)_{rc} for the 4 x 4 diagonal blocks of the
 * registered matrix, b = 0 .. ceil(n/4)-1 (caller-owned device buffer of ceil(n/4)*16 doubles). */
int cbgmres_k_bj4_setup(cbgmres_handle_t h, double *d_inv);
/* S4 with the block-Jacobi(4) preconditioner: as cbgmres_k_store, but d_z_fp64[i] <- (M^-1 v)_i, the vector the
 * next SpMV multiplies (Fig. 1 l.3), with d_inv from cbgmres_k_bj4_setup.  The payload is enc(v) as before. */
int cbgmres_k_store_bj4(cbgmres_handle_t h, int32_t format, int64_t n, const double *d_w, double hnorm, double amax,
                        const double *d_inv, void *d_payload_col, double *d_scale, double *d_z_fp64);
/* S1, Fig. 1 line 3: d_w <- A d_v with the registered matrix; if d_nrm2 != NULL,
 * *d_nrm2 <- ||w||_2 (omega, line 4) from the same pass. */
int cbgmres_k_spmv(cbgmres_handle_t h, const double *d_v, double *d_w, double *d_nrm2);

/* ---- an entry point that allocates nothing ----------------------------------------------------
 * S2 (Fig. 1 line 5) as cbgmres_k_multidot computes it -- d_h[c] <- sum_i dec(V)[i,c] * d_w[i],
 * the same kernels, the same bits -- for callers that cannot call cudaMalloc (code under CUDA graph capture,
 * serving loops, harnesses that forbid allocation).  It takes no handle (cbgmres_create allocates): the scratch
 * the reduction goes through (CTA partial sums, the last-block-done ticket) is a file-scope device array of
 * CBGMRES_NOALLOC_SCRATCH_BYTES that every GPU loading the library holds until the process exits.
 *   device   CUDA device ordinal the buffers live on (made current); stream: a cudaStream_t of that device
 *            (borrowed; the call only enqueues: a memset of the control block, then one kernel).
 *   format, n, ld, k, d_V, d_scales, d_w, d_h: as cbgmres_k_multidot; all DEVICE pointers, caller-owned.
 *   k > CBGMRES_NOALLOC_MAX_K is rejected with CBGMRES_E_INVALID (nothing enqueued); k == 0 is a no-op.
 * The call makes no cudaMalloc / cudaFree / allocating library call.  All calls on one GPU share the array,
 * which keeps the last call's contents (what must start at zero is cleared on `stream` first): calls that
 * overlap on the GPU -- two streams, two host threads -- race; serialise them.
 * cbgmres_noalloc_setup(device) takes the array's device address (cudaGetSymbolAddress, once per device);
 * the first k_multidot_noalloc call on a device does it itself, so calling it is only needed to keep that
 * one-time step out of a region where it is unwelcome.  Errors: the status code, and a per-thread message
 * from cbgmres_noalloc_last_error(). */
#define CBGMRES_NOALLOC_MAX_K 128
#define CBGMRES_NOALLOC_SCRATCH_BYTES 635392
int cbgmres_noalloc_setup(int32_t device);
int cbgmres_k_multidot_noalloc(int32_t device, void *stream, int32_t format, int64_t n, int64_t ld, int32_t k,
                               const void *d_V, const double *d_scales, const double *d_w, double *d_h);
const char *cbgmres_noalloc_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* CBGMRES_H_ */
