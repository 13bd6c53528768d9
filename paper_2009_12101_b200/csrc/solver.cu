// solver.cu -- the C ABI of include/cbgmres.h: handle, matrix registration, the restarted
// CB-GMRES driver loop of Fig. 1 and the per-kernel hooks.
//
// Control flow lives on the device (Ctl in internal.cuh): the host enqueues a whole restart cycle
// -- explicit residual, store of v_1, m x {SpMV, multi-dot, update, [second pass], store+Givens},
// back substitution, x update -- without reading anything back; kernels of steps after the one
// that met the stopping test return at once.  One stream synchronisation per cycle.  A mapped
// host word mirrors the device's "stop after step j" so the host can stop enqueueing early.
#include <climits>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <vector>

#include "internal.cuh"

using namespace cbg;

struct ProfSlot {
    cudaEvent_t a = nullptr, b = nullptr;
    int family = 0, step = 0, pass = 0;
    double bytes = 0.0;
};
struct ProfAcc {
    double ms = 0.0, bytes = 0.0;
    int64_t launches = 0;
};

struct cbgmres_ctx {
    int device = 0;
    cudaStream_t stream = nullptr;
    LaunchCtx lc{};            // per-handle launch options and error slots (no process-wide state)
    Scratch sc{};
    void *scratch_base = nullptr;
    double *hook_hs = nullptr; // [kMaxRestart] coefficients of the k_update hook
    int *d_stats = nullptr;
    Ctl *h_ctl = nullptr;      // pinned host copy for read-back
    int *h_flag = nullptr;     // mapped pinned word
    int *d_flag = nullptr;     // its device alias
    CsrView A{};
    bool has_matrix = false;
    int4 *owned_blk_row = nullptr;
    int opt_spmv_kernel = 0;
    int opt_poll = 1;
    int opt_seg_kb = 0; // column-segment size of the Gram-Schmidt passes (0 = auto)
    int opt_fuse = 1;   // fused update + second-pass multi-dot
    int opt_small = 1;  // small systems: the whole solve in one kernel of a 16-CTA cluster (cluster.cu)
    int64_t launches = 0;
    cudaEvent_t ev0 = nullptr, ev1 = nullptr;
    // optional per-kernel timing ("profile" option): event pairs around the launches of one cycle
    int opt_profile = 0; // 0 = off, N = bracket the launches of every N-th Arnoldi step of a cycle
    bool prof_on = false;
    std::vector<ProfSlot> prof_slots;
    int prof_used = 0;
    int *h_reorth_log = nullptr; // mapped pinned [kMaxRestart + 2]: reorth_flag per step of the cycle
    int *d_reorth_log = nullptr;
    ProfAcc prof[CBGMRES_PROF_FAMILIES]{};
    char err[256] = "no error";
};

namespace {

int fail(cbgmres_ctx *h, int code, const char *msg)
{
    if (h) snprintf(h->err, sizeof(h->err), "%s", msg);
    return code;
}

int fail_cuda(cbgmres_ctx *h, cudaError_t e, const char *where)
{
    if (h) snprintf(h->err, sizeof(h->err), "CUDA error at %s: %s", where, cudaGetErrorString(e));
    return CBGMRES_E_CUDA;
}

#define CK(call)                                                                                                  \
    do {                                                                                                          \
        cudaError_t e_ = (call);                                                                                  \
        if (e_ != cudaSuccess) return fail_cuda(h, e_, #call);                                                    \
    } while (0)

inline int format_bytes(int fmt)
{
    switch (fmt) {
    case CBGMRES_FP64: return 8;
    case CBGMRES_FP32: return 4;
    case CBGMRES_FP16: return 2;
    case CBGMRES_INT32: return 4;
    case CBGMRES_INT16: return 2;
    default: return -1;
    }
}

inline size_t up256(size_t x) { return (x + 255) / 256 * 256; }

struct Layout {
    int64_t ld;
    size_t off_V, off_v, off_w, off_small, total;
    size_t o_h, o_hs, o_R, o_cs, o_sn, o_g, o_y, o_scales, o_hist;
    size_t off_pvals, off_pdiag; // Jacobi: column-scaled values and diag(A) (unused otherwise)
    size_t off_bjinv;            // block-Jacobi(4): the inverted diagonal blocks, 16 doubles per block
};

Layout make_layout(int64_t n, int64_t nnz, const cbgmres_params *p)
{
    Layout L{};
    const int m = p->restart;
    const int B = format_bytes(p->format);
    L.ld = (n + 63) / 64 * 64;
    size_t o = 0;
    L.off_V = o;
    o += up256((size_t)(m + 1) * (size_t)L.ld * (size_t)B);
    L.off_v = o;
    o += up256((size_t)L.ld * 8);
    L.off_w = o;
    o += up256((size_t)L.ld * 8);
    if (p->precond == CBGMRES_PRECOND_JACOBI) {
        L.off_pvals = o;
        o += up256((size_t)nnz * 8);
        L.off_pdiag = o;
        o += up256((size_t)n * 8);
    }
    if (p->precond == CBGMRES_PRECOND_BLOCK_JACOBI4) {
        L.off_bjinv = o;
        o += up256((size_t)((n + 3) / 4) * 16 * 8);
    }
    L.off_small = o;
    size_t s = 0;
    auto take = [&](size_t count) {
        size_t at = s;
        s += up256(count * 8);
        return at;
    };
    L.o_h = take(m + 2);
    L.o_hs = take(m + 2);
    L.o_R = take((size_t)(m + 1) * m);
    L.o_cs = take(m);
    L.o_sn = take(m);
    L.o_g = take(m + 2);
    L.o_y = take(m);
    L.o_scales = take(m + 2);
    L.o_hist = take(p->h_res_history && p->res_history_cap > 0 ? (size_t)p->res_history_cap : 0);
    L.total = o + s;
    return L;
}

int validate_params(cbgmres_ctx *h, const cbgmres_params *p)
{
    if (!p) return fail(h, CBGMRES_E_INVALID, "params is null");
    if (p->restart < 1 || p->restart > CBGMRES_MAX_RESTART) return fail(h, CBGMRES_E_INVALID, "restart out of range");
    if (format_bytes(p->format) < 0) return fail(h, CBGMRES_E_INVALID, "unknown storage format");
    if (p->reorth < 0 || p->reorth > 2) return fail(h, CBGMRES_E_INVALID, "unknown reorth mode");
    if (p->max_iters < 0) return fail(h, CBGMRES_E_INVALID, "max_iters < 0");
    if (!(p->rel_tol >= 0.0)) return fail(h, CBGMRES_E_INVALID, "rel_tol must be >= 0");
    if (!(p->eta >= 0.0) || p->eta > 1.0) return fail(h, CBGMRES_E_INVALID, "eta must be in [0, 1]");
    if (p->res_history_cap < 0) return fail(h, CBGMRES_E_INVALID, "res_history_cap < 0");
    if (p->precond != CBGMRES_PRECOND_NONE && p->precond != CBGMRES_PRECOND_JACOBI &&
        p->precond != CBGMRES_PRECOND_BLOCK_JACOBI4)
        return fail(h, CBGMRES_E_INVALID, "unknown preconditioner");
    return CBGMRES_OK;
}

// ---- optional per-kernel timing ---------------------------------------------------------------
// prof_begin/prof_end bracket one launch with an event pair; prof_collect runs after the cycle's
// stream synchronisation, when the device's control block (k, reorth_log) is back on the host.
void prof_begin(cbgmres_ctx *h, int family, int step, int pass, double bytes)
{
    if (!h->prof_on) return;
    if (h->prof_used == (int)h->prof_slots.size()) {
        ProfSlot sl;
        if (cudaEventCreate(&sl.a) != cudaSuccess || cudaEventCreate(&sl.b) != cudaSuccess) return;
        h->prof_slots.push_back(sl);
    }
    ProfSlot &sl = h->prof_slots[h->prof_used];
    sl.family = family;
    sl.step = step;
    sl.pass = pass;
    sl.bytes = bytes;
    cudaEventRecord(sl.a, h->stream);
}

void prof_end(cbgmres_ctx *h)
{
    if (!h->prof_on || h->prof_used >= (int)h->prof_slots.size()) return;
    cudaEventRecord(h->prof_slots[h->prof_used].b, h->stream);
    h->prof_used += 1;
}

void prof_collect(cbgmres_ctx *h, const Ctl &c, bool cycle_ran)
{
    for (int i = 0; i < h->prof_used; ++i) {
        const ProfSlot &sl = h->prof_slots[i];
        bool ran = true;
        if (sl.step > 0) ran = cycle_ran && sl.step <= c.k && (sl.pass < 2 || c.reorth_log[sl.step]);
        else if (sl.family == CBGMRES_PROF_XUPDATE) ran = cycle_ran && c.k > 0;
        if (!ran) continue;
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, sl.a, sl.b) != cudaSuccess) continue;
        ProfAcc &acc = h->prof[sl.family];
        acc.ms += ms;
        acc.bytes += sl.bytes;
        acc.launches += 1;
    }
    h->prof_used = 0;
}

// A failed kernel launch or tensor-map encode recorded by a launcher since the last call (0 = none).
int take_launch_errors(cbgmres_ctx *h)
{
    LaunchCtx &lc = h->lc;
    int rc = CBGMRES_OK;
    if (lc.launch_error != cudaSuccess) {
        snprintf(h->err, sizeof(h->err), "launch of %s failed: %s", lc.launch_kernel, cudaGetErrorString(lc.launch_error));
        (void)cudaGetLastError(); // clear the sticky-less launch error so that later calls start clean
        rc = CBGMRES_E_CUDA;
    } else if (lc.orth_error) {
        snprintf(h->err, sizeof(h->err), "cuTensorMapEncodeTiled failed for the basis (CUresult %d)", lc.orth_error);
        rc = CBGMRES_E_CUDA;
    }
    lc.launch_error = cudaSuccess;
    lc.launch_kernel = "";
    lc.orth_error = 0;
    return rc;
}

int choose_spmv_kernel(cbgmres_ctx *h, int64_t n, int64_t nnz, int max_len)
{
    if (h->opt_spmv_kernel) return h->opt_spmv_kernel;
    const double mean = n > 0 ? (double)nnz / (double)n : 0.0;
    // irregular row lengths (power-law): stream nonzeros in storage order, reduce rows from shared memory
    if (max_len > 64 && (double)max_len > 8.0 * mean) return 64;
    // regular: row-major from shared memory; blocks of 256 RPT / LPR rows must hold <= 3584 nonzeros
    const int len = (int)std::fmin((double)max_len, std::ceil(2.0 * mean));
    // (halving the row blocks when a CTA gets fewer than twelve -- C2, n = 1e6: 6.6 blocks per CTA -- measured no gain:
    // 31.4 against 29.7 us, L2 flushed)
    if (len <= 3) return 132;  // 4 rows per thread
    if (len <= 7) return 130;  // 2 rows per thread
    if (len <= 14) return 129; // 1 row per thread
    if (len <= 28) return 146; // 2 lanes per row
    if (len <= 56) return 148; // 4 lanes per row
    if (len <= 112) return 152; // 8 lanes per row
    return 32;                 // a warp per row
}

int register_matrix(cbgmres_ctx *h, int64_t n, int64_t nnz, const int32_t *rp, const int32_t *ci, const double *va)
{
    if (n <= 0 || nnz < 0 || n >= INT32_MAX || nnz >= INT32_MAX) return fail(h, CBGMRES_E_INVALID, "bad n / nnz");
    if (!rp || !ci || !va) return fail(h, CBGMRES_E_INVALID, "null CSR pointer");
    if (h->owned_blk_row) {
        cudaFree(h->owned_blk_row);
        h->owned_blk_row = nullptr;
    }
    h->has_matrix = false;
    h->A = CsrView{};
    h->A.n = n;
    h->A.nnz = nnz;
    h->A.row_ptr = rp;
    h->A.col_idx = ci;
    h->A.vals = va;
    h->launches += launch_row_stats(h->stream, n, rp, h->d_stats);
    int max_len = 0;
    CK(cudaMemcpyAsync(&max_len, h->d_stats, sizeof(int), cudaMemcpyDeviceToHost, h->stream));
    CK(cudaStreamSynchronize(h->stream));
    h->A.kernel = choose_spmv_kernel(h, n, nnz, max_len);
    if (h->A.kernel == 64 || h->A.kernel == 65) {
        int nblk = 0;
        CK(build_row_blocks(h->stream, n, nnz, rp, &h->owned_blk_row, &nblk, h->A.kernel));
        h->launches += 1;
        h->A.blk_desc = h->owned_blk_row;
        h->A.nblk = nblk;
        const double mean = (double)nnz / (double)n; // about 4 products per lane
        h->A.reduce_lanes = mean <= 6.0 ? 1 : mean <= 12.0 ? 2 : mean <= 24.0 ? 4 : mean <= 48.0 ? 8 : mean <= 96.0 ? 16 : 32;
    }
    // small systems: how many nonzeros the fullest of 16 equal row slabs holds (decides whether the cluster path fits)
    h->A.slab_nnz = small_slab_nnz(h->stream, n, rp, h->d_stats + 16);
    if (h->A.slab_nnz) h->launches += 1;
    h->has_matrix = true;
    return CBGMRES_OK;
}

} // namespace

extern "C" {

int cbgmres_create(cbgmres_handle_t *out, int device, void *cuda_stream)
{
    if (!out) return CBGMRES_E_INVALID;
    *out = nullptr;
    cbgmres_ctx *h = new (std::nothrow) cbgmres_ctx();
    if (!h) return CBGMRES_E_INVALID;
    h->device = device;
    h->lc.device = device;
    h->sc.lc = &h->lc;
    h->stream = reinterpret_cast<cudaStream_t>(cuda_stream);
    cudaError_t e = cudaSetDevice(device);
    if (e != cudaSuccess) {
        delete h;
        return CBGMRES_E_CUDA;
    }
    const size_t b_ctl = up256(sizeof(Ctl));
    const size_t b_part = up256((size_t)kMaxGrid * kLdp * 8);
    const size_t b_np = up256((size_t)2 * kMaxGrid * 8);
    const size_t b_hs = up256((size_t)(kMaxRestart + 8) * 8);
    const size_t b_stats = 256;
    e = cudaMalloc(&h->scratch_base, b_ctl + b_part + b_np + b_hs + b_stats);
    if (e != cudaSuccess) {
        delete h;
        return CBGMRES_E_CUDA;
    }
    char *base = static_cast<char *>(h->scratch_base);
    h->sc.ctl = reinterpret_cast<Ctl *>(base);
    h->sc.partials = reinterpret_cast<double *>(base + b_ctl);
    h->sc.npart = reinterpret_cast<double *>(base + b_ctl + b_part);
    h->hook_hs = reinterpret_cast<double *>(base + b_ctl + b_part + b_np);
    h->d_stats = reinterpret_cast<int *>(base + b_ctl + b_part + b_np + b_hs);
    cudaMemsetAsync(h->scratch_base, 0, b_ctl + b_part + b_np + b_hs + b_stats, h->stream);
    if (cudaHostAlloc(&h->h_ctl, sizeof(Ctl), cudaHostAllocDefault) != cudaSuccess ||
        cudaHostAlloc(&h->h_flag, 64, cudaHostAllocMapped) != cudaSuccess ||
        cudaHostGetDevicePointer(reinterpret_cast<void **>(&h->d_flag), h->h_flag, 0) != cudaSuccess ||
        cudaEventCreate(&h->ev0) != cudaSuccess || cudaEventCreate(&h->ev1) != cudaSuccess) {
        cbgmres_destroy(h);
        return CBGMRES_E_CUDA;
    }
    *h->h_flag = INT_MAX;
    *out = h;
    return CBGMRES_OK;
}

int cbgmres_destroy(cbgmres_handle_t h)
{
    if (!h) return CBGMRES_E_INVALID;
    cudaSetDevice(h->device);
    if (h->stream) cudaStreamSynchronize(h->stream);
    else cudaDeviceSynchronize();
    if (h->owned_blk_row) cudaFree(h->owned_blk_row);
    if (h->scratch_base) cudaFree(h->scratch_base);
    if (h->h_ctl) cudaFreeHost(h->h_ctl);
    if (h->h_flag) cudaFreeHost(h->h_flag);
    if (h->ev0) cudaEventDestroy(h->ev0);
    if (h->ev1) cudaEventDestroy(h->ev1);
    for (ProfSlot &sl : h->prof_slots) {
        if (sl.a) cudaEventDestroy(sl.a);
        if (sl.b) cudaEventDestroy(sl.b);
    }
    delete h;
    return CBGMRES_OK;
}

const char *cbgmres_last_error(cbgmres_handle_t h) { return h ? h->err : "null handle"; }

int64_t cbgmres_launch_count(cbgmres_handle_t h) { return h ? h->launches : -1; }

int cbgmres_set_option(cbgmres_handle_t h, const char *name, int64_t value)
{
    if (!h || !name) return CBGMRES_E_INVALID;
    if (!strcmp(name, "spmv_kernel")) {
        if (value != 0 && value != 2 && value != 4 && value != 8 && value != 16 && value != 32 && value != 64 && value != 65 &&
            value != 129 && value != 130 && value != 132 && value != 146 && value != 148 && value != 152)
            return fail(h, CBGMRES_E_INVALID, "spmv_kernel must be 0, 2, 4, 8, 16, 32, 64, 65, 129, 130, 132, 146, 148 or 152");
        h->opt_spmv_kernel = (int)value;
        return CBGMRES_OK;
    }
    if (!strcmp(name, "poll")) {
        h->opt_poll = value != 0;
        return CBGMRES_OK;
    }
    if (!strcmp(name, "orth_seg_kb")) {
        if (value != 0 && value != 1 && value != 2 && value != 4)
            return fail(h, CBGMRES_E_INVALID, "orth_seg_kb must be 0, 1, 2 or 4");
        h->opt_seg_kb = (int)value;
        return CBGMRES_OK;
    }
    if (!strcmp(name, "orth_interleave")) {
        if (value < 0 || value > 2) return fail(h, CBGMRES_E_INVALID, "orth_interleave must be 0, 1 or 2");
        h->lc.interleave = (int)value;
        return CBGMRES_OK;
    }
    if (!strcmp(name, "orth_fuse")) {
        h->opt_fuse = value != 0;
        return CBGMRES_OK;
    }
    if (!strcmp(name, "small_path")) {
        h->opt_small = value != 0;
        return CBGMRES_OK;
    }
    if (!strcmp(name, "orth_fused_rows")) {
        if (value < 0 || value > 2) return fail(h, CBGMRES_E_INVALID, "orth_fused_rows must be 0, 1 or 2");
        h->lc.fused_rows = (int)value;
        return CBGMRES_OK;
    }
    if (!strcmp(name, "pdl")) {
        h->lc.use_pdl = value != 0;
        return CBGMRES_OK;
    }
    if (!strcmp(name, "profile")) {
        if (value < 0 || value > 1024) return fail(h, CBGMRES_E_INVALID, "profile must be 0..1024");
        h->opt_profile = (int)value;
        return CBGMRES_OK;
    }
    return fail(h, CBGMRES_E_INVALID, "unknown option");
}

int cbgmres_set_matrix(cbgmres_handle_t h, int64_t n, int64_t nnz, const int32_t *d_row_ptr, const int32_t *d_col_idx,
                       const double *d_vals)
{
    if (!h) return CBGMRES_E_INVALID;
    CK(cudaSetDevice(h->device));
    return register_matrix(h, n, nnz, d_row_ptr, d_col_idx, d_vals);
}

int cbgmres_workspace_bytes(cbgmres_handle_t h, const cbgmres_params *p, size_t *bytes)
{
    if (!h || !bytes) return CBGMRES_E_INVALID;
    if (!h->has_matrix) return fail(h, CBGMRES_E_NOMATRIX, "set_matrix has not been called");
    const int rc = validate_params(h, p);
    if (rc) return rc;
    *bytes = make_layout(h->A.n, h->A.nnz, p).total;
    return CBGMRES_OK;
}

// The restarted CB-GMRES driver (Fig. 1).  Everything numerical happens in kernels; this loop only
// orders launches.
int cbgmres_solve(cbgmres_handle_t h, const double *d_b, double *d_x, const cbgmres_params *p, void *d_workspace,
                  size_t workspace_bytes, cbgmres_result *out)
{
    if (!h) return CBGMRES_E_INVALID;
    if (!h->has_matrix) return fail(h, CBGMRES_E_NOMATRIX, "set_matrix has not been called");
    int rc = validate_params(h, p);
    if (rc) return rc;
    if (!d_b || !d_x || !d_workspace || !out) return fail(h, CBGMRES_E_INVALID, "null pointer argument");
    if (reinterpret_cast<uintptr_t>(d_workspace) % 256 != 0) return fail(h, CBGMRES_E_WORKSPACE, "workspace not 256-byte aligned");
    if (reinterpret_cast<uintptr_t>(d_b) % 16 != 0 || reinterpret_cast<uintptr_t>(d_x) % 16 != 0)
        return fail(h, CBGMRES_E_INVALID, "b and x must be 16-byte aligned");
    const int64_t n = h->A.n;
    const Layout L = make_layout(n, h->A.nnz, p);
    if (workspace_bytes < L.total) return fail(h, CBGMRES_E_WORKSPACE, "workspace too small");
    CK(cudaSetDevice(h->device));
    cudaStream_t s = h->stream;
    const int m = p->restart, fmt = p->format, B = format_bytes(fmt);
    char *ws = static_cast<char *>(d_workspace);
    char *Vp = ws + L.off_V;
    double *v = reinterpret_cast<double *>(ws + L.off_v);
    double *w = reinterpret_cast<double *>(ws + L.off_w);
    char *sm = ws + L.off_small;
    CycleState cy{};
    cy.h = reinterpret_cast<double *>(sm + L.o_h);
    cy.hs = reinterpret_cast<double *>(sm + L.o_hs);
    cy.R = reinterpret_cast<double *>(sm + L.o_R);
    cy.cs = reinterpret_cast<double *>(sm + L.o_cs);
    cy.sn = reinterpret_cast<double *>(sm + L.o_sn);
    cy.g = reinterpret_cast<double *>(sm + L.o_g);
    cy.y = reinterpret_cast<double *>(sm + L.o_y);
    cy.scales = reinterpret_cast<double *>(sm + L.o_scales);
    const int hist_cap = (p->h_res_history && p->res_history_cap > 0) ? p->res_history_cap : 0;
    cy.hist = hist_cap ? reinterpret_cast<double *>(sm + L.o_hist) : nullptr;
    BasisView bv{Vp, L.ld, cy.scales, fmt};
    Ctl *dctl = h->sc.ctl;

    memset(out, 0, sizeof(*out));
    out->spmv_kernel = h->A.kernel;
    const int64_t launches0 = h->launches;
    CK(cudaEventRecord(h->ev0, s));

    // control block for this solve
    Ctl c0{};
    c0.eta = (p->eta > 0.0) ? p->eta : 0.70710678118654752440;
    c0.rel_tol = p->rel_tol;
    c0.max_iters = p->max_iters;
    c0.reorth_mode = p->reorth;
    c0.m = m;
    c0.hist_cap = hist_cap;
    c0.stop_after = 0;
    *h->h_ctl = c0;
    CK(cudaMemcpyAsync(dctl, h->h_ctl, sizeof(Ctl), cudaMemcpyHostToDevice, s));
    // ||b||_2 and the absolute threshold tau * ||b||_2
    h->launches += launch_nrm2(s, h->sc, n, d_b, MODE_BNORM);
    CK(cudaMemcpyAsync(h->h_ctl, dctl, sizeof(Ctl), cudaMemcpyDeviceToHost, s));
    CK(cudaStreamSynchronize(s));
    const double bnorm = h->h_ctl->bnorm;
    out->b_norm = bnorm;
    if (bnorm == 0.0) { // reading Q9: b = 0 => x = 0
        CK(cudaMemsetAsync(d_x, 0, (size_t)n * 8, s));
        CK(cudaEventRecord(h->ev1, s));
        CK(cudaStreamSynchronize(s));
        out->converged = 1;
        float ms = 0.f;
        cudaEventElapsedTime(&ms, h->ev0, h->ev1);
        out->solve_ms = ms;
        return CBGMRES_OK;
    }
    if (!std::isfinite(bnorm)) return fail(h, CBGMRES_E_NONFINITE, "||b|| is not finite");

    // Scalar Jacobi: GMRES on A D^-1 in u = D x (small.cu); d_x holds u until the end.
    // Block-Jacobi(4): the store kernel hands z = M^-1 v to the SpMV (l.3) and the cycle end
    // forms x += M^-1 (V_k y) (l.17); x stays in the original variable.
    const bool jacobi = p->precond == CBGMRES_PRECOND_JACOBI;
    const bool bj4 = p->precond == CBGMRES_PRECOND_BLOCK_JACOBI4;
    CsrView A = h->A;
    double *pdiag = nullptr, *bjinv = nullptr;
    if (jacobi) {
        double *pvals = reinterpret_cast<double *>(ws + L.off_pvals);
        pdiag = reinterpret_cast<double *>(ws + L.off_pdiag);
        h->launches += launch_jacobi_setup(s, h->A, pdiag, pvals);
        h->launches += launch_diag_scale(s, n, d_x, pdiag, 0);
        A.vals = pvals;
    }
    if (bj4) {
        bjinv = reinterpret_cast<double *>(ws + L.off_bjinv);
        h->launches += launch_bj4_setup(s, h->A, bjinv);
    }
    volatile int *flag = h->h_flag;
    const double dn = (double)n, dB = (double)B;
    const double bytes_spmv = 12.0 * (double)h->A.nnz + 4.0 * (dn + 1.0) + 16.0 * dn;
    const double bytes_store = (16.0 + dB) * dn + (bj4 ? 32.0 * dn : 0.0);
    const int sk = h->opt_seg_kb;
    double alg_bytes = 0.0;
    // The restart cycles.  Any failure leaves through `return`; the caller below undoes the Jacobi change of
    // variable on EVERY exit, so d_x never stays in the variable u = D x.
    auto cycles = [&]() -> int {
    for (;;) {
        *flag = INT_MAX;
        h->prof_used = 0;
        const int restarts_before = h->h_ctl->restarts;
        h->prof_on = h->opt_profile != 0;
        // l.1: r0 = b - A x, beta, the stopping test on the explicit residual; v1 = r0 / beta
        prof_begin(h, CBGMRES_PROF_RESIDUAL, 0, 0, bytes_spmv + 8.0 * dn + bytes_store);
        h->launches += launch_spmv(s, h->sc, A, d_x, d_b, w, MODE_RESIDUAL, 0, &cy, h->d_flag);
        h->launches += launch_store(s, h->sc, fmt, n, w, &dctl->hn, &dctl->amax, 0.0, 0.0, Vp, cy.scales, v,
                                    MODE_RESIDUAL, 1, nullptr, nullptr, bjinv);
        prof_end(h);
        for (int j = 1; j <= m; ++j) {
            if (h->opt_poll && *flag < j) break; // the device already left this cycle
            h->prof_on = h->opt_profile && (j % h->opt_profile == 0);
            const double bytes_dot = (double)j * dn * dB + 8.0 * dn, bytes_upd = (double)j * dn * dB + 16.0 * dn;
            // l.3-4: w = A v, omega = ||w||
            prof_begin(h, CBGMRES_PROF_SPMV, j, 0, bytes_spmv);
            h->launches += launch_spmv(s, h->sc, A, v, nullptr, w, MODE_STEP, j, nullptr, nullptr);
            prof_end(h);
            // l.5: h = V^T w
            prof_begin(h, CBGMRES_PROF_MULTIDOT, j, 1, bytes_dot);
            h->launches += launch_multidot(s, h->sc, bv, n, j, w, cy.h, cy.hs, MODE_ORTH1, j, sk);
            prof_end(h);
            if (p->reorth == CBGMRES_REORTH_NEVER) {
                // l.5-6: w -= V h ; h_{j+1,j} = ||w||
                prof_begin(h, CBGMRES_PROF_UPDATE, j, 1, bytes_upd);
                h->launches += launch_update(s, h->sc, bv, n, j, nullptr, cy.hs, w, MODE_ORTH1, j, sk);
                prof_end(h);
            } else if (h->opt_fuse && update_multidot_fits(fmt, j, sk)) {
                // l.5-8 from one read of V: w -= V h, ||w||, and u = V^T w for the second pass;
                // l.7 is decided on the device, u is dropped if the second pass does not fire
                prof_begin(h, CBGMRES_PROF_UPDATE_DOT, j, 1, bytes_upd);
                h->launches += launch_update_multidot(s, h->sc, bv, n, j, cy.hs, w, cy.h, cy.hs, MODE_ORTH1, j, sk);
                prof_end(h);
                // l.8-10: w -= V u ; h_{j+1,j} = ||w||   (skipped on the device unless flagged)
                prof_begin(h, CBGMRES_PROF_UPDATE, j, 2, bytes_upd);
                h->launches += launch_update(s, h->sc, bv, n, j, nullptr, cy.hs, w, MODE_ORTH2, j, sk);
                prof_end(h);
            } else {
                prof_begin(h, CBGMRES_PROF_UPDATE, j, 1, bytes_upd);
                h->launches += launch_update(s, h->sc, bv, n, j, nullptr, cy.hs, w, MODE_ORTH1, j, sk);
                prof_end(h);
                prof_begin(h, CBGMRES_PROF_MULTIDOT, j, 2, bytes_dot);
                h->launches += launch_multidot(s, h->sc, bv, n, j, w, cy.h, cy.hs, MODE_ORTH2, j, sk);
                prof_end(h);
                prof_begin(h, CBGMRES_PROF_UPDATE, j, 2, bytes_upd);
                h->launches += launch_update(s, h->sc, bv, n, j, nullptr, cy.hs, w, MODE_ORTH2, j, sk);
                prof_end(h);
            }
            // l.13-14: v = w / h_{j+1,j}; V[:, j] = enc(v); + Givens update and stopping test
            prof_begin(h, CBGMRES_PROF_STORE, j, 0, bytes_store);
            h->launches += launch_store(s, h->sc, fmt, n, w, &dctl->hn, &dctl->amax, 0.0, 0.0,
                                        Vp + (size_t)j * (size_t)L.ld * (size_t)B, cy.scales + j, v, MODE_ORTH1, j, &cy,
                                        h->d_flag, bjinv);
            prof_end(h);
            if (h->lc.launch_error != cudaSuccess || h->lc.orth_error) break; // a launch of this step failed: stop enqueueing
        }
        // l.16-17: R y = g ; x += M^-1 (V_k y)  (k read on the device)
        h->prof_on = h->opt_profile != 0;
        prof_begin(h, CBGMRES_PROF_XUPDATE, 0, 0, 0.0);
        h->launches += launch_backsolve(s, h->sc, cy, fmt);
        if (bj4) { // t = V_k y in the (now free) work vector, then x += M^-1 t
            h->launches += launch_fill_zero(s, n, w);
            h->launches += launch_update(s, h->sc, bv, n, m, &dctl->k, cy.hs, w, MODE_XUPDATE, 0, sk);
            h->launches += launch_bj4_axpy(s, n, bjinv, w, d_x);
        } else {
            h->launches += launch_update(s, h->sc, bv, n, m, &dctl->k, cy.hs, d_x, MODE_XUPDATE, 0, sk);
        }
        prof_end(h);
        CK(cudaMemcpyAsync(h->h_ctl, dctl, sizeof(Ctl), cudaMemcpyDeviceToHost, s));
        CK(cudaStreamSynchronize(s));
        {
            const int lrc = take_launch_errors(h);
            if (lrc) return lrc;
        }
        CK(cudaGetLastError());
        if (h->h_ctl->restarts > restarts_before) { // algorithmic bytes of the launches that ran
            const Ctl &c = *h->h_ctl;
            double by = bytes_spmv + 8.0 * dn + bytes_store; // l.1: residual + store of v_1
            for (int j = 1; j <= c.k; ++j) {
                const double dot = (double)j * dn * dB + 8.0 * dn, upd = (double)j * dn * dB + 16.0 * dn;
                const bool fused = p->reorth != CBGMRES_REORTH_NEVER && h->opt_fuse && update_multidot_fits(fmt, j, sk);
                by += bytes_spmv + dot + upd + bytes_store;          // S1, S2, S3 (fused: S3 + S2' from one read), S4
                if (c.reorth_log[j]) by += fused ? upd : dot + upd;  // S3' (and a separate S2' where the fusion does not fit)
            }
            if (c.k > 0) by += (double)c.k * dn * dB + 16.0 * dn;    // S6: x += V_k y
            alg_bytes += by;
        }
        if (h->opt_profile) {
            const bool cycle_ran = h->h_ctl->restarts > restarts_before;
            // the x update's bytes depend on k, known only now
            for (int i = 0; i < h->prof_used; ++i)
                if (h->prof_slots[i].family == CBGMRES_PROF_XUPDATE)
                    h->prof_slots[i].bytes = (double)h->h_ctl->k * dn * dB + 16.0 * dn;
            prof_collect(h, *h->h_ctl, cycle_ran);
        }
        if (h->h_ctl->done) break;
    }
    return CBGMRES_OK;
    };
    // Small systems (basis + matrix + vectors within the distributed shared memory of one 16-CTA cluster): the whole
    // solve is ONE kernel (cluster.cu).  -1 = not applicable / launch refused: the large path runs.
    auto small = [&]() -> int {
        if (!h->opt_small || bj4 || !small_fits(n, h->A.slab_nnz, m, fmt)) return -1;
        const int nl = launch_small_solve(s, h->sc, A, d_b, d_x, cy, m, fmt, h->A.slab_nnz);
        if (!nl) { // e.g. no room for a 16-CTA cluster on this device right now: not an error, use the large path
            h->lc.launch_error = cudaSuccess;
            h->lc.launch_kernel = "";
            (void)cudaGetLastError();
            return -1;
        }
        h->launches += nl;
        CK(cudaMemcpyAsync(h->h_ctl, dctl, sizeof(Ctl), cudaMemcpyDeviceToHost, s));
        CK(cudaStreamSynchronize(s));
        CK(cudaGetLastError());
        out->spmv_kernel = 1016;
        return CBGMRES_OK;
    };
    rc = small();
    if (rc == -1) rc = cycles();
    if (jacobi) { // l.17: x = M^-1 u -- on every exit, also the failed ones (x then holds the last iterate reached)
        h->launches += launch_diag_scale(s, n, d_x, pdiag, 1);
        if (rc != CBGMRES_OK) cudaStreamSynchronize(s);
    }
    if (rc != CBGMRES_OK) return rc;
    if (hist_cap) {
        const int cnt = h->h_ctl->iters < hist_cap ? h->h_ctl->iters : hist_cap;
        if (cnt > 0) CK(cudaMemcpyAsync(p->h_res_history, cy.hist, (size_t)cnt * 8, cudaMemcpyDeviceToHost, s));
    }
    CK(cudaEventRecord(h->ev1, s));
    CK(cudaStreamSynchronize(s));
    float ms = 0.f;
    cudaEventElapsedTime(&ms, h->ev0, h->ev1);
    const Ctl &c = *h->h_ctl;
    out->iters = c.iters;
    out->restarts = c.restarts;
    out->reorth_count = c.reorth_count;
    out->breakdown = c.breakdown;
    out->converged = c.converged;
    out->rel_res_recurrence = c.rel_rec;
    out->rel_res_true = c.rel_true;
    out->solve_ms = ms;
    out->algorithmic_bytes = alg_bytes;
    (void)launches0;
    if (c.nonfinite) return fail(h, CBGMRES_E_NONFINITE, "non-finite residual norm");
    return c.converged ? CBGMRES_OK : CBGMRES_NOT_CONVERGED;
}

int cbgmres_workspace_bytes_host(cbgmres_handle_t h, int64_t n, int64_t nnz, const cbgmres_params *p, size_t *bytes)
{
    if (!h || !bytes) return CBGMRES_E_INVALID;
    const int rc = validate_params(h, p);
    if (rc) return rc;
    if (n <= 0 || nnz < 0) return fail(h, CBGMRES_E_INVALID, "bad n / nnz");
    *bytes = up256((size_t)(n + 1) * 4) + up256((size_t)nnz * 4) + up256((size_t)nnz * 8) + 2 * up256((size_t)n * 8) +
             make_layout(n, nnz, p).total;
    return CBGMRES_OK;
}

int cbgmres_solve_host(cbgmres_handle_t h, int64_t n, int64_t nnz, const int32_t *h_row_ptr, const int32_t *h_col_idx,
                       const double *h_vals, const double *h_b, double *h_x, const cbgmres_params *p,
                       void *d_workspace, size_t workspace_bytes, cbgmres_result *out)
{
    if (!h) return CBGMRES_E_INVALID;
    if (!h_row_ptr || !h_col_idx || !h_vals || !h_b || !h_x || !d_workspace || !out)
        return fail(h, CBGMRES_E_INVALID, "null pointer argument");
    size_t need = 0;
    int rc = cbgmres_workspace_bytes_host(h, n, nnz, p, &need);
    if (rc) return rc;
    if (workspace_bytes < need) return fail(h, CBGMRES_E_WORKSPACE, "workspace too small");
    if (reinterpret_cast<uintptr_t>(d_workspace) % 256 != 0) return fail(h, CBGMRES_E_WORKSPACE, "workspace not 256-byte aligned");
    CK(cudaSetDevice(h->device));
    cudaStream_t s = h->stream;
    char *ws = static_cast<char *>(d_workspace);
    size_t o = 0;
    int32_t *d_rp = reinterpret_cast<int32_t *>(ws + o);
    o += up256((size_t)(n + 1) * 4);
    int32_t *d_ci = reinterpret_cast<int32_t *>(ws + o);
    o += up256((size_t)nnz * 4);
    double *d_va = reinterpret_cast<double *>(ws + o);
    o += up256((size_t)nnz * 8);
    double *d_b = reinterpret_cast<double *>(ws + o);
    o += up256((size_t)n * 8);
    double *d_x = reinterpret_cast<double *>(ws + o);
    o += up256((size_t)n * 8);
    CK(cudaMemcpyAsync(d_rp, h_row_ptr, (size_t)(n + 1) * 4, cudaMemcpyHostToDevice, s));
    CK(cudaMemcpyAsync(d_ci, h_col_idx, (size_t)nnz * 4, cudaMemcpyHostToDevice, s));
    CK(cudaMemcpyAsync(d_va, h_vals, (size_t)nnz * 8, cudaMemcpyHostToDevice, s));
    CK(cudaMemcpyAsync(d_b, h_b, (size_t)n * 8, cudaMemcpyHostToDevice, s));
    CK(cudaMemcpyAsync(d_x, h_x, (size_t)n * 8, cudaMemcpyHostToDevice, s));
    rc = register_matrix(h, n, nnz, d_rp, d_ci, d_va);
    if (rc) return rc;
    rc = cbgmres_solve(h, d_b, d_x, p, ws + o, workspace_bytes - o, out);
    if (rc != CBGMRES_OK && rc != CBGMRES_NOT_CONVERGED && rc != CBGMRES_E_NONFINITE) return rc;
    CK(cudaMemcpyAsync(h_x, d_x, (size_t)n * 8, cudaMemcpyDeviceToHost, s));
    CK(cudaStreamSynchronize(s));
    return rc;
}

int cbgmres_profile_get(cbgmres_handle_t h, int32_t family, double *ms, double *bytes, int64_t *launches)
{
    if (!h) return CBGMRES_E_INVALID;
    if (family < 0 || family >= CBGMRES_PROF_FAMILIES) return fail(h, CBGMRES_E_INVALID, "unknown kernel family");
    if (ms) *ms = h->prof[family].ms;
    if (bytes) *bytes = h->prof[family].bytes;
    if (launches) *launches = h->prof[family].launches;
    return CBGMRES_OK;
}

int cbgmres_profile_reset(cbgmres_handle_t h)
{
    if (!h) return CBGMRES_E_INVALID;
    for (ProfAcc &a : h->prof) a = ProfAcc{};
    return CBGMRES_OK;
}

// ---- per-kernel hooks -------------------------------------------------------------------------------
// Every hook ends here: a launch that failed (recorded by launch_chain with the kernel's name), a failed
// tensor-map encode, or any other pending CUDA error becomes this call's status.
static int finish_hook(cbgmres_ctx *h)
{
    const int lrc = take_launch_errors(h);
    if (lrc) return lrc;
    CK(cudaGetLastError());
    return CBGMRES_OK;
}

static int check_basis_args(cbgmres_ctx *h, int32_t format, int64_t n, int64_t ld, int32_t k, const void *V)
{
    const int B = format_bytes(format);
    if (B < 0) return fail(h, CBGMRES_E_INVALID, "unknown storage format");
    if (n <= 0 || ld < n || k < 0 || k > CBGMRES_MAX_RESTART) return fail(h, CBGMRES_E_INVALID, "bad n / ld / k");
    if (((size_t)ld * (size_t)B) % 16 != 0 || reinterpret_cast<uintptr_t>(V) % 16 != 0)
        return fail(h, CBGMRES_E_INVALID, "basis vectors must be 16-byte aligned (ld*bytes % 16 == 0)");
    return CBGMRES_OK;
}

int cbgmres_k_compress(cbgmres_handle_t h, int32_t format, int64_t n, const double *d_v, void *d_payload,
                       double *d_scale)
{
    if (!h) return CBGMRES_E_INVALID;
    if (format_bytes(format) < 0 || n <= 0 || !d_v || !d_payload || !d_scale)
        return fail(h, CBGMRES_E_INVALID, "bad argument");
    if (reinterpret_cast<uintptr_t>(d_v) % 16 != 0 || reinterpret_cast<uintptr_t>(d_payload) % 16 != 0)
        return fail(h, CBGMRES_E_INVALID, "buffers must be 16-byte aligned");
    CK(cudaSetDevice(h->device));
    // ||v||_inf first (exact under any reduction order), then v / 1.0 == v through the store kernel
    h->launches += launch_nrm2(h->stream, h->sc, n, d_v, MODE_HOOK);
    h->launches += launch_store(h->stream, h->sc, format, n, d_v, nullptr, &h->sc.ctl->hook_amax, 1.0, 0.0, d_payload,
                                d_scale, nullptr, MODE_HOOK, 0, nullptr, nullptr);
    return finish_hook(h);
}

int cbgmres_k_decode(cbgmres_handle_t h, int32_t format, int64_t n, const void *d_payload, const double *d_scale,
                     double *d_v)
{
    if (!h) return CBGMRES_E_INVALID;
    if (format_bytes(format) < 0 || n <= 0 || !d_v || !d_payload) return fail(h, CBGMRES_E_INVALID, "bad argument");
    if ((format == CBGMRES_INT32 || format == CBGMRES_INT16) && !d_scale)
        return fail(h, CBGMRES_E_INVALID, "fixed-point formats need d_scale");
    CK(cudaSetDevice(h->device));
    h->launches += launch_decode(h->stream, format, n, d_payload, d_scale, d_v);
    return finish_hook(h);
}

int cbgmres_k_multidot(cbgmres_handle_t h, int32_t format, int64_t n, int64_t ld, int32_t k, const void *d_V,
                       const double *d_scales, const double *d_w, double *d_h)
{
    if (!h) return CBGMRES_E_INVALID;
    const int rc = check_basis_args(h, format, n, ld, k, d_V);
    if (rc) return rc;
    if (!d_V || !d_w || !d_h) return fail(h, CBGMRES_E_INVALID, "null pointer argument");
    if ((format == CBGMRES_INT32 || format == CBGMRES_INT16) && !d_scales)
        return fail(h, CBGMRES_E_INVALID, "fixed-point formats need d_scales");
    if (k == 0) return CBGMRES_OK;
    CK(cudaSetDevice(h->device));
    BasisView bv{d_V, ld, d_scales, format};
    h->launches += launch_multidot(h->stream, h->sc, bv, n, k, d_w, d_h, nullptr, MODE_HOOK, 0, h->opt_seg_kb);
    return finish_hook(h);
}

int cbgmres_k_update(cbgmres_handle_t h, int32_t format, int64_t n, int64_t ld, int32_t k, const void *d_V,
                     const double *d_scales, const double *d_h, double *d_w, double *d_nrm2, double *d_amax)
{
    if (!h) return CBGMRES_E_INVALID;
    const int rc = check_basis_args(h, format, n, ld, k, d_V);
    if (rc) return rc;
    if (!d_V || !d_w || !d_h) return fail(h, CBGMRES_E_INVALID, "null pointer argument");
    if (reinterpret_cast<uintptr_t>(d_w) % 16 != 0) return fail(h, CBGMRES_E_INVALID, "w must be 16-byte aligned");
    const bool scaled = (format == CBGMRES_INT32 || format == CBGMRES_INT16);
    if (scaled && !d_scales) return fail(h, CBGMRES_E_INVALID, "fixed-point formats need d_scales");
    if (k == 0) return fail(h, CBGMRES_E_INVALID, "k must be >= 1");
    CK(cudaSetDevice(h->device));
    BasisView bv{d_V, ld, d_scales, format};
    h->launches += launch_scale_coeffs(h->stream, k, d_h, scaled ? d_scales : nullptr, h->hook_hs);
    h->launches += launch_update(h->stream, h->sc, bv, n, k, nullptr, h->hook_hs, d_w, MODE_HOOK, 0, h->opt_seg_kb);
    if (d_nrm2 || d_amax)
        h->launches += launch_copy_scalars(h->stream, &h->sc.ctl->hook_nrm2, d_nrm2, &h->sc.ctl->hook_amax, d_amax);
    return finish_hook(h);
}

int cbgmres_k_update_multidot(cbgmres_handle_t h, int32_t format, int64_t n, int64_t ld, int32_t k, const void *d_V,
                              const double *d_scales, const double *d_h, double *d_w, double *d_u, double *d_nrm2,
                              double *d_amax)
{
    if (!h) return CBGMRES_E_INVALID;
    const int rc = check_basis_args(h, format, n, ld, k, d_V);
    if (rc) return rc;
    if (!d_V || !d_w || !d_h || !d_u) return fail(h, CBGMRES_E_INVALID, "null pointer argument");
    if (reinterpret_cast<uintptr_t>(d_w) % 16 != 0) return fail(h, CBGMRES_E_INVALID, "w must be 16-byte aligned");
    const bool scaled = (format == CBGMRES_INT32 || format == CBGMRES_INT16);
    if (scaled && !d_scales) return fail(h, CBGMRES_E_INVALID, "fixed-point formats need d_scales");
    if (k == 0) return fail(h, CBGMRES_E_INVALID, "k must be >= 1");
    if (!update_multidot_fits(format, k, h->opt_seg_kb))
        return fail(h, CBGMRES_E_INVALID, "k vectors do not fit the fused pass (use k_update + k_multidot)");
    CK(cudaSetDevice(h->device));
    BasisView bv{d_V, ld, d_scales, format};
    h->launches += launch_scale_coeffs(h->stream, k, d_h, scaled ? d_scales : nullptr, h->hook_hs);
    h->launches += launch_update_multidot(h->stream, h->sc, bv, n, k, h->hook_hs, d_w, d_u, nullptr, MODE_HOOK, 0,
                                          h->opt_seg_kb);
    if (d_nrm2 || d_amax)
        h->launches += launch_copy_scalars(h->stream, &h->sc.ctl->hook_nrm2, d_nrm2, &h->sc.ctl->hook_amax, d_amax);
    return finish_hook(h);
}

int cbgmres_k_store(cbgmres_handle_t h, int32_t format, int64_t n, const double *d_w, double hnorm, double amax,
                    void *d_payload_col, double *d_scale, double *d_v_fp64)
{
    if (!h) return CBGMRES_E_INVALID;
    if (format_bytes(format) < 0 || n <= 0 || !d_w || !d_payload_col || !d_scale)
        return fail(h, CBGMRES_E_INVALID, "bad argument");
    if (reinterpret_cast<uintptr_t>(d_w) % 16 != 0 || reinterpret_cast<uintptr_t>(d_payload_col) % 16 != 0 ||
        reinterpret_cast<uintptr_t>(d_v_fp64) % 16 != 0)
        return fail(h, CBGMRES_E_INVALID, "buffers must be 16-byte aligned");
    CK(cudaSetDevice(h->device));
    h->launches += launch_store(h->stream, h->sc, format, n, d_w, nullptr, nullptr, hnorm, amax, d_payload_col, d_scale,
                                d_v_fp64, MODE_HOOK, 0, nullptr, nullptr);
    return finish_hook(h);
}

int cbgmres_k_bj4_setup(cbgmres_handle_t h, double *d_inv)
{
    if (!h) return CBGMRES_E_INVALID;
    if (!h->has_matrix) return fail(h, CBGMRES_E_NOMATRIX, "set_matrix has not been called");
    if (!d_inv || reinterpret_cast<uintptr_t>(d_inv) % 16 != 0) return fail(h, CBGMRES_E_INVALID, "d_inv must be a 16-byte aligned device buffer");
    CK(cudaSetDevice(h->device));
    h->launches += launch_bj4_setup(h->stream, h->A, d_inv);
    return finish_hook(h);
}

int cbgmres_k_store_bj4(cbgmres_handle_t h, int32_t format, int64_t n, const double *d_w, double hnorm, double amax,
                        const double *d_inv, void *d_payload_col, double *d_scale, double *d_z_fp64)
{
    if (!h) return CBGMRES_E_INVALID;
    if (format_bytes(format) < 0 || n <= 0 || !d_w || !d_payload_col || !d_scale || !d_inv || !d_z_fp64)
        return fail(h, CBGMRES_E_INVALID, "bad argument");
    if (reinterpret_cast<uintptr_t>(d_w) % 16 != 0 || reinterpret_cast<uintptr_t>(d_payload_col) % 16 != 0 ||
        reinterpret_cast<uintptr_t>(d_z_fp64) % 16 != 0 || reinterpret_cast<uintptr_t>(d_inv) % 16 != 0)
        return fail(h, CBGMRES_E_INVALID, "buffers must be 16-byte aligned");
    CK(cudaSetDevice(h->device));
    h->launches += launch_store(h->stream, h->sc, format, n, d_w, nullptr, nullptr, hnorm, amax, d_payload_col, d_scale,
                                d_z_fp64, MODE_HOOK, 0, nullptr, nullptr, d_inv);
    return finish_hook(h);
}

int cbgmres_k_spmv(cbgmres_handle_t h, const double *d_v, double *d_w, double *d_nrm2)
{
    if (!h) return CBGMRES_E_INVALID;
    if (!h->has_matrix) return fail(h, CBGMRES_E_NOMATRIX, "set_matrix has not been called");
    if (!d_v || !d_w) return fail(h, CBGMRES_E_INVALID, "null pointer argument");
    CK(cudaSetDevice(h->device));
    h->launches += launch_spmv(h->stream, h->sc, h->A, d_v, nullptr, d_w, MODE_HOOK, 0, nullptr, nullptr);
    if (d_nrm2) h->launches += launch_copy_scalars(h->stream, &h->sc.ctl->hook_nrm2, d_nrm2, nullptr, nullptr);
    return finish_hook(h);
}

} // extern "C"
