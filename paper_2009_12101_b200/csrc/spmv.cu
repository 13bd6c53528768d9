// spmv.cu -- S1: w = A v (Fig. 1 line 3) with omega^2 = sum w_i^2 from the same pass
// (line 4), and S7: r = b - A x with ||r||_2, ||r||_inf (Fig. 1 line 1), on CSR
// with fp64 values and int32 indices.
//
// Bound: HBM.  Algorithmic bytes per launch: 12 nnz + 4(n+1) + 8n (v, once) + 8n (w).
//
// Two variants, chosen in set_matrix from the row-length distribution:
//   * L lanes per row (L in 2..32): regular matrices (stencils).  Consecutive rows sit in
//     consecutive lane groups, so a warp's loads of col_idx / vals cover one contiguous range.
//   * nnz-balanced streaming: the matrix is cut at multiples of T nonzeros (whole rows per CTA);
//     a CTA streams its nonzeros with fully dense coalesced loads, leaves the products in shared
//     memory and then reduces rows from there (thread per short row, warp per long row).
//     Irregular matrices (power-law row lengths) keep every lane busy this way.
#include "device_utils.cuh"

namespace cbg {

struct SpmvArgs {
    CsrView A;
    const double *x, *b;
    double *w;
    Ctl *ctl;
    double *npart;
    CycleState cyc;
    int has_cyc;
    int mode, step;
    int *h_flag;
};

// Norm finalisation shared by all SpMV variants and the plain norm kernel: called by every thread
// of the CTA that arrived last, with this CTA's (sum of squares, max) partial already in npart.
__device__ __forceinline__ void finalize_norms(const SpmvArgs &a)
{
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (warp != 0) return;
    double t = 0.0, m = 0.0;
    for (int b = lane; b < (int)gridDim.x; b += 32) {
        t += __ldcg(&a.npart[b]);
        m = fmax(m, __ldcg(&a.npart[kMaxGrid + b]));
    }
    t = warp_sum(t);
    m = warp_max(m);
    if (lane != 0) return;
    Ctl *ctl = a.ctl;
    const double nrm = sqrt(t);
    switch (a.mode) {
    case MODE_HOOK:
        ctl->hook_nrm2 = nrm;
        ctl->hook_amax = m;
        break;
    case MODE_STEP: // Fig. 1 l.4: omega := ||w||_2
        ctl->sumsq_w = t;
        ctl->omega = nrm;
        break;
    case MODE_BNORM:
        ctl->bnorm = nrm;
        ctl->tol_abs = ctl->rel_tol * nrm;
        break;
    case MODE_RESIDUAL: { // Fig. 1 l.1 and the stopping test on the explicit residual
        const double beta = nrm;
        ctl->beta = beta;
        ctl->rel_true = beta / ctl->bnorm;
        ctl->k = 0;
        int stop_after = 0;
        if (!isfinite(beta)) {
            ctl->nonfinite = 1;
            ctl->done = 1;
        } else if (beta <= ctl->tol_abs) {
            ctl->converged = 1;
            ctl->done = 1;
        } else if (ctl->iters >= ctl->max_iters) {
            ctl->done = 1;
        } else {
            ctl->restarts += 1;
            ctl->breakdown = 0; // reported for the last cycle that ran (Fig. 1 l.12)
            stop_after = ctl->m;
            ctl->hn = beta; // v_1 := r_0 / beta through the same store kernel
            ctl->amax = m;
            a.cyc.g[0] = beta;
        }
        ctl->stop_after = stop_after;
        if (a.h_flag) {
            *reinterpret_cast<volatile int *>(a.h_flag) = stop_after;
            __threadfence_system();
        }
        break;
    }
    default: break;
    }
}

__device__ __forceinline__ void block_norm_partials(const SpmvArgs &a, double ss, double am, unsigned *ticket)
{
    __shared__ double s_ss[32], s_am[32];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nw = blockDim.x >> 5;
    ss = warp_sum(ss);
    am = warp_max(am);
    if (lane == 0) {
        s_ss[warp] = ss;
        s_am[warp] = am;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0, m = 0.0;
        for (int i = 0; i < nw; ++i) {
            t += s_ss[i];
            m = fmax(m, s_am[i]);
        }
        a.npart[blockIdx.x] = t;
        a.npart[kMaxGrid + blockIdx.x] = m;
    }
    if (last_block_done(ticket)) finalize_norms(a);
}

// ---- variant 1: LANES lanes per row ---------------------------------------------------------------
template <int LANES> __global__ void __launch_bounds__(256) spmv_vec_kernel(const SpmvArgs a)
{
    if (a.mode == MODE_STEP && a.step > a.ctl->stop_after) return;
    constexpr int RPB = 256 / LANES;
    const int sub = threadIdx.x / LANES, sl = threadIdx.x % LANES;
    const int32_t *__restrict__ rp = a.A.row_ptr;
    const int32_t *__restrict__ ci = a.A.col_idx;
    const double *__restrict__ va = a.A.vals;
    const double *__restrict__ x = a.x;
    double ss = 0.0, am = 0.0;
    const int64_t nrows_pad = (a.A.n + RPB - 1) / RPB * RPB; // keep whole warps in the shuffles
    for (int64_t row = (int64_t)blockIdx.x * RPB + sub; row < nrows_pad; row += (int64_t)gridDim.x * RPB) {
        double s = 0.0;
        if (row < a.A.n) {
            const int p1 = rp[row + 1];
            for (int p = rp[row] + sl; p < p1; p += LANES) s = fma(va[p], x[ci[p]], s);
        }
#pragma unroll
        for (int o = LANES / 2; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
        if (sl == 0 && row < a.A.n) {
            const double val = (a.mode == MODE_RESIDUAL) ? a.b[row] - s : s;
            a.w[row] = val;
            ss = fma(val, val, ss);
            am = fmax(am, fabs(val));
        }
    }
    block_norm_partials(a, ss, am, &a.ctl->tickets[2]);
}

// ---- variant 2: nnz-balanced streaming ---------------------------------------------------------------
constexpr int kStreamT = 4096;      // target nonzeros per CTA (blocks are cut at multiples of T, whole rows)
constexpr int kStreamBuf = 6000;    // product buffer: T + the overhang of the block's last row (static smem <= 48 KB)
constexpr int kStreamThreads = 256;
constexpr int kLongRow = 64;        // rows longer than this are reduced by a whole warp

__global__ void __launch_bounds__(kStreamThreads) spmv_stream_kernel(const SpmvArgs a)
{
    if (a.mode == MODE_STEP && a.step > a.ctl->stop_after) return;
    __shared__ double prod[kStreamBuf];
    const int32_t *__restrict__ rp = a.A.row_ptr;
    const int32_t *__restrict__ ci = a.A.col_idx;
    const double *__restrict__ va = a.A.vals;
    const double *__restrict__ x = a.x;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    double ss = 0.0, am = 0.0;
    for (int blk = blockIdx.x; blk < a.A.nblk; blk += gridDim.x) {
        const int r0 = a.A.blk_row[blk], r1 = a.A.blk_row[blk + 1];
        if (r0 >= r1) continue;
        const int p0 = rp[r0], p1 = rp[r1];
        if (p1 - p0 <= kStreamBuf) {
            __syncthreads();
            for (int p = p0 + threadIdx.x; p < p1; p += kStreamThreads) prod[p - p0] = va[p] * x[ci[p]];
            __syncthreads();
            // short rows: one thread each, sequential over the row's products; a long row is reduced
            // by the whole warp that found it (ballot), so the order of every sum is fixed
            for (int rb = r0; rb < r1; rb += kStreamThreads) {
                const int r = rb + threadIdx.x;
                const bool valid = r < r1;
                const int q0 = valid ? rp[r] - p0 : 0, q1 = valid ? rp[r + 1] - p0 : 0;
                const bool is_long = (q1 - q0) > kLongRow;
                if (valid && !is_long) {
                    double s = 0.0;
                    for (int q = q0; q < q1; ++q) s += prod[q];
                    const double val = (a.mode == MODE_RESIDUAL) ? a.b[r] - s : s;
                    a.w[r] = val;
                    ss = fma(val, val, ss);
                    am = fmax(am, fabs(val));
                }
                unsigned mask = __ballot_sync(0xffffffffu, is_long);
                while (mask) {
                    const int src = __ffs(mask) - 1;
                    mask &= mask - 1;
                    const int rr = rb + warp * 32 + src;
                    const int qq0 = __shfl_sync(0xffffffffu, q0, src), qq1 = __shfl_sync(0xffffffffu, q1, src);
                    double s = 0.0;
                    for (int q = qq0 + lane; q < qq1; q += 32) s += prod[q];
                    s = warp_sum(s);
                    if (lane == 0) {
                        const double val = (a.mode == MODE_RESIDUAL) ? a.b[rr] - s : s;
                        a.w[rr] = val;
                        ss = fma(val, val, ss);
                        am = fmax(am, fabs(val));
                    }
                }
            }
        } else {
            // a block whose rows do not fit the product buffer (a single very long row, or a long row
            // next to short ones): one warp per row straight from global memory
            for (int r = r0 + warp; r < r1; r += kStreamThreads / 32) {
                double s = 0.0;
                for (int p = rp[r] + lane; p < rp[r + 1]; p += 32) s = fma(va[p], x[ci[p]], s);
                s = warp_sum(s);
                if (lane == 0) {
                    const double val = (a.mode == MODE_RESIDUAL) ? a.b[r] - s : s;
                    a.w[r] = val;
                    ss = fma(val, val, ss);
                    am = fmax(am, fabs(val));
                }
            }
        }
    }
    block_norm_partials(a, ss, am, &a.ctl->tickets[2]);
}

// Row partition of the streaming kernel: blk_row[b] = first row r with row_ptr[r] >= b*T, so block b
// holds whole rows and about T nonzeros.
__global__ void row_blocks_kernel(int64_t n, const int32_t *__restrict__ rp, int T, int nblk, int32_t *blk_row)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b > nblk) return;
    if (b == nblk) {
        blk_row[b] = (int32_t)n;
        return;
    }
    const int64_t target = (int64_t)b * T;
    int64_t lo = 0, hi = n; // first r in [0, n] with rp[r] >= target
    while (lo < hi) {
        const int64_t mid = (lo + hi) >> 1;
        if (rp[mid] >= target) hi = mid;
        else lo = mid + 1;
    }
    blk_row[b] = (int32_t)lo;
}

cudaError_t build_row_blocks(cudaStream_t s, int64_t n, int64_t nnz, const int32_t *d_row_ptr, int nnz_per_block,
                             int32_t **d_blk_row_out, int *nblk_out)
{
    (void)nnz_per_block;
    const int nblk = (int)((nnz + kStreamT - 1) / kStreamT) + 1;
    int32_t *blk = nullptr;
    cudaError_t e = cudaMalloc(&blk, (size_t)(nblk + 1) * sizeof(int32_t));
    if (e != cudaSuccess) return e;
    row_blocks_kernel<<<(nblk + 1 + 255) / 256, 256, 0, s>>>(n, d_row_ptr, kStreamT, nblk, blk);
    *d_blk_row_out = blk;
    *nblk_out = nblk;
    return cudaGetLastError();
}

// Row-length statistics for the kernel choice in set_matrix: out[0] = max row length.
__global__ void row_stats_kernel(int64_t n, const int32_t *__restrict__ rp, int *out)
{
    int mx = 0;
    for (int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; r < n; r += (int64_t)gridDim.x * blockDim.x)
        mx = max(mx, rp[r + 1] - rp[r]);
    for (int o = 16; o > 0; o >>= 1) mx = max(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    if ((threadIdx.x & 31) == 0) atomicMax(out, mx);
}

int launch_row_stats(cudaStream_t s, int64_t n, const int32_t *d_row_ptr, int *d_out)
{
    cudaMemsetAsync(d_out, 0, sizeof(int), s);
    int64_t grid = (n + 255) / 256;
    if (grid > kNumSMs * 8) grid = kNumSMs * 8;
    if (grid < 1) grid = 1;
    row_stats_kernel<<<(int)grid, 256, 0, s>>>(n, d_row_ptr, d_out);
    return 1;
}

// ---- plain norm kernel (||b||, and the amax of the k_compress hook) ------------------------------------
__global__ void __launch_bounds__(256) nrm2_kernel(const SpmvArgs a, int64_t n)
{
    double ss = 0.0, am = 0.0;
    for (int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x; i < n; i += (int64_t)gridDim.x * 256) {
        const double v = a.x[i];
        ss = fma(v, v, ss);
        am = fmax(am, fabs(v));
    }
    block_norm_partials(a, ss, am, &a.ctl->tickets[3]);
}

int launch_nrm2(cudaStream_t s, const Scratch &sc, int64_t n, const double *x, int mode)
{
    SpmvArgs a{};
    a.x = x;
    a.ctl = sc.ctl;
    a.npart = sc.npart;
    a.mode = mode;
    int64_t grid = (n + 1023) / 1024;
    if (grid > kNumSMs * 4) grid = kNumSMs * 4;
    if (grid < 1) grid = 1;
    nrm2_kernel<<<(int)grid, 256, 0, s>>>(a, n);
    return 1;
}

template <int LANES> static void launch_vec(cudaStream_t s, const SpmvArgs &a)
{
    constexpr int RPB = 256 / LANES;
    int64_t grid = (a.A.n + RPB - 1) / RPB;
    const int64_t cap = (int64_t)kNumSMs * 8;
    if (grid > cap) grid = cap;
    spmv_vec_kernel<LANES><<<(int)grid, 256, 0, s>>>(a);
}

int launch_spmv(cudaStream_t s, const Scratch &sc, const CsrView &A, const double *x, const double *b, double *w,
                int mode, int step, const CycleState *cyc, int *h_flag)
{
    SpmvArgs a{};
    a.A = A;
    a.x = x;
    a.b = b;
    a.w = w;
    a.ctl = sc.ctl;
    a.npart = sc.npart;
    a.has_cyc = cyc != nullptr;
    if (cyc) a.cyc = *cyc;
    a.mode = mode;
    a.step = step;
    a.h_flag = h_flag;
    switch (A.kernel) {
    case 2: launch_vec<2>(s, a); break;
    case 4: launch_vec<4>(s, a); break;
    case 8: launch_vec<8>(s, a); break;
    case 16: launch_vec<16>(s, a); break;
    case 32: launch_vec<32>(s, a); break;
    case 64: {
        int grid = A.nblk < kNumSMs * 6 ? A.nblk : kNumSMs * 6;
        if (grid < 1) grid = 1;
        spmv_stream_kernel<<<grid, kStreamThreads, 0, s>>>(a);
        break;
    }
    default: return 0;
    }
    return 1;
}

} // namespace cbg
