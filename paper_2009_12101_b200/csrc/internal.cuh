// internal.cuh -- shared declarations of the CB-GMRES CUDA library (sm_100a only).
// Nothing in this tree is shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <cuda_fp16.h>
#include <stdint.h>

#include "../../include/cbgmres.h"

namespace cbg {

constexpr int kMaxRestart = CBGMRES_MAX_RESTART;
constexpr int kNumSMs = 148;           // B200: 2 dies x 74 SMs
constexpr int kMaxGrid = kNumSMs * 8;  // upper bound on CTAs of any reduction kernel (partials rows)
constexpr int kLdp = kMaxRestart + 8;  // leading dimension of the multi-dot partials matrix

// Step kinds: the guard every step kernel evaluates from the device-resident control block.
enum Mode : int {
    MODE_HOOK = 0,     // per-kernel test hook: no guard, no solver control
    MODE_ORTH1 = 1,    // first Gram-Schmidt pass of Arnoldi step `step`   (Fig. 1 l.5-6)
    MODE_ORTH2 = 2,    // conditional second pass                           (Fig. 1 l.7-11)
    MODE_XUPDATE = 3,  // x += V_k y at the end of a cycle                  (Fig. 1 l.17)
    MODE_RESIDUAL = 4, // r = b - A x at the start of a cycle               (Fig. 1 l.1)
    MODE_STEP = 5,     // w = A v of Arnoldi step `step`                    (Fig. 1 l.3-4)
    MODE_BNORM = 6,    // ||b|| once per solve
};

// Device-resident control block: every scalar the Arnoldi loop decides on lives here, so the
// host launches a whole restart cycle without reading anything back (one sync per cycle).
struct Ctl {
    // reduction results
    double sumsq_w;   // sum w_i^2 after the SpMV (omega^2) or of the explicit residual
    double amax_w;    // max |w_i| of the explicit residual (feeds the store of V[:,0])
    double omega;     // ||A v||_2 of the current step (Fig. 1 l.4)
    double hn;        // h_{j+1,j} (or beta at cycle start): the divisor of the next store
    double amax;      // ||w||_inf matching hn
    double hook_nrm2; // outputs of the k_update hook
    double hook_amax;
    // solve-wide scalars
    double bnorm, tol_abs, beta, eta, rel_rec, rel_true, rel_tol;
    // control
    int stop_after;   // Arnoldi steps with index > stop_after are skipped in this cycle
    int reorth_flag;  // set by the first pass's finalisation, read by the second pass
    int k;            // Arnoldi steps completed in the current cycle
    int iters, max_iters, reorth_count, breakdown, converged, nonfinite, restarts, done;
    int reorth_mode, m, hist_cap;
    int dir;          // row direction of the next Gram-Schmidt pass (flipped by every pass that runs)
    unsigned tickets[8]; // last-block-done counters, one per kernel family
    unsigned char reorth_log[kMaxRestart + 8]; // reorth_flag of every step of the current cycle
};

// Small dense state of one restart cycle (device memory, < 3 MB at m = 512).
struct CycleState {
    double *h;      // [m+2]  current Hessenberg column (h_{1:j,j}, then rotated in place)
    double *hs;     // [m+2]  sigma_c * h_c: the coefficients the update kernel multiplies payloads with
    double *R;      // [(m+1) * m] rotated Hessenberg, column-major, ld = m+1
    double *cs, *sn; // [m] Givens rotations
    double *g;      // [m+1] rotated right-hand side
    double *y;      // [m]
    double *scales; // [m+1] sigma_c per stored basis vector
    double *hist;   // [hist_cap] recurrence residual per Arnoldi step
};

// Per-handle launch state (host side).  Everything a launcher may change or consult lives here, not in
// process-wide globals: two handles (two devices, two streams, two host threads) do not see each other.
struct LaunchCtx {
    int device = 0;
    int use_pdl = 1;      // "pdl" option: programmatic dependent launch of the step kernels
    int interleave = 0;   // "orth_interleave" option: 0 auto, 1 blocked row ranges, 2 interleaved row tiles
    int fused_rows = 2;   // "orth_fused_rows" option: row-mapped fused update + multi-dot: 0 never, 1 every reduced format, 2 (default) 16-bit formats
    int orth_error = 0;   // CUresult of a failed tensor-map encode (0 = none)
    cudaError_t launch_error = cudaSuccess; // first failed kernel launch since the last take_launch_error
    const char *launch_kernel = "";         // ... and which kernel it was
};

struct Scratch {
    Ctl *ctl;          // device
    double *partials;  // [kMaxGrid * kLdp] multi-dot partial sums, row = CTA
    double *npart;     // [2 * kMaxGrid] sum-of-squares and max partials
    LaunchCtx *lc;     // host: the handle's launch state (never null)
};

// True the first time it is called for (this static mask, device): function attributes
// (cudaFuncSetAttribute, occupancy queries) are per device, not per process.
inline bool first_use_on_device(unsigned long long &mask, int device)
{
    const unsigned long long bit = 1ull << (device & 63);
    if (mask & bit) return false;
    mask |= bit;
    return true;
}

struct BasisView {
    const void *V;     // payload, vector-major
    int64_t ld;        // entries per stored vector
    const double *scales;
    int format;
};

struct CsrView {
    int64_t n, nnz;
    const int32_t *row_ptr, *col_idx;
    const double *vals;
    const int4 *blk_desc;   // [nblk] row blocks of the streaming kernel {row0, row1, nz0, nz1} (may be null)
    int nblk;
    int reduce_lanes;       // lanes sharing a row in the streaming kernel's row reduction (power of two)
    int kernel;             // 2,4,8,16,32 lanes per row, or 64 = streaming
    int slab_nnz;           // nonzeros of the fullest of 16 equal row slabs (small-system path; 0 = not applicable)
};

// ---- launchers (each enqueues on `s` and returns the number of kernels launched) -------------
// Gram-Schmidt passes (orth.cu).  seg_kb: 0 = choose the tile height, else 1, 2 or 4 KB per column segment.
int launch_multidot(cudaStream_t s, const Scratch &sc, const BasisView &b, int64_t n, int k, const double *w,
                    double *h_out, double *hs_out, int mode, int step, int seg_kb);
int launch_update(cudaStream_t s, const Scratch &sc, const BasisView &b, int64_t n, int k, const int *d_k,
                  const double *hs, double *w, int mode, int step, int seg_kb);
// fused update + next multi-dot; returns 0 (nothing launched) if k vectors do not fit the shared-memory ring
int launch_update_multidot(cudaStream_t s, const Scratch &sc, const BasisView &b, int64_t n, int k, const double *hs,
                           double *w, double *h_out, double *hs_out, int mode, int step, int seg_kb);
bool update_multidot_fits(int format, int k, int seg_kb);
int launch_store(cudaStream_t s, const Scratch &sc, int format, int64_t n, const double *w, const double *d_hn,
                 const double *d_amax, double hn_host, double amax_host, void *payload_col, double *scale_out,
                 double *v_out, int mode, int step, const CycleState *cyc, int *h_flag, const double *bj_inv = nullptr);
int launch_decode(cudaStream_t s, int format, int64_t n, const void *payload, const double *d_scale, double *v);
int launch_spmv(cudaStream_t s, const Scratch &sc, const CsrView &A, const double *x, const double *b, double *w,
                int mode, int step, const CycleState *cyc, int *h_flag);
int launch_nrm2(cudaStream_t s, const Scratch &sc, int64_t n, const double *x, int mode);
int launch_backsolve(cudaStream_t s, const Scratch &sc, const CycleState &cyc, int format);
int launch_scale_coeffs(cudaStream_t s, int k, const double *h, const double *scales, double *hs);
int launch_copy_scalars(cudaStream_t s, const double *src0, double *dst0, const double *src1, double *dst1);

int launch_jacobi_setup(cudaStream_t s, const CsrView &A, double *d, double *scaled_vals); // d = diag(A), vals / d[col]
int launch_diag_scale(cudaStream_t s, int64_t n, double *x, const double *d, int inverse);  // x *= d or x /= d

// Block-Jacobi(4) right preconditioner: inv[16 b + 4 r + c] = (A_bb^-1)_{rc} of the 4 x 4 diagonal blocks
int launch_bj4_setup(cudaStream_t s, const CsrView &A, double *inv);
int launch_bj4_axpy(cudaStream_t s, int64_t n, const double *inv, const double *t, double *x); // x += M^-1 t (Fig. 1 l.17)
int launch_fill_zero(cudaStream_t s, int64_t n, double *x);

// Small systems: the whole solve in one kernel of a 16-CTA cluster (cluster.cu)
int small_slab_nnz(cudaStream_t s, int64_t n, const int32_t *d_row_ptr, int *d_scratch);
bool small_fits(int64_t n, int slab_nnz, int m, int format);
int launch_small_solve(cudaStream_t s, const Scratch &sc, const CsrView &A, const double *b, double *x, const CycleState &cyc,
                       int m, int format, int slab_nnz);

int launch_row_stats(cudaStream_t s, int64_t n, const int32_t *d_row_ptr, int *d_out);

// row-partition metadata for the streaming SpMV (set_matrix)
cudaError_t build_row_blocks(cudaStream_t s, int64_t n, int64_t nnz, const int32_t *d_row_ptr, int4 **d_desc_out,
                             int *nblk_out, int kernel);

} // namespace cbg
