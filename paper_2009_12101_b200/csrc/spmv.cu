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

// Gather of one entry of x.  x is the fp64 v that the preceding store kernel wrote; under programmatic
// dependent launch this grid can be resident while that kernel is still running, so x is NOT read-only
// for this kernel's lifetime and must not go through ld.global.nc (which `const __restrict__` or __ldg
// would select).  A plain L1-cached load issued after griddepcontrol.wait sees the predecessor's writes;
// L1 matters for the stencils, where the diagonals of consecutive rows share lines.  Only the matrix
// arrays, which no kernel ever writes, use the non-coherent path.
__device__ __forceinline__ double ld_x(const double *p)
{
    double r;
    asm volatile("ld.global.ca.f64 %0, [%1];" : "=d"(r) : "l"(p));
    return r;
}

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
// U rows per lane group are in flight at once: all row pointers first, then all (col, val) pairs,
// then all gathers of x -- three rounds of independent loads instead of 3 U dependent ones.
template <int LANES, int U> __global__ void __launch_bounds__(256) spmv_vec_kernel(const SpmvArgs a)
{
    pdl_wait();
    pdl_launch_dependents();
    if (a.mode == MODE_STEP && a.step > a.ctl->stop_after) return;
    constexpr int RPB = 256 / LANES;
    const int sub = threadIdx.x / LANES, sl = threadIdx.x % LANES;
    const int32_t *__restrict__ rp = a.A.row_ptr;
    const int32_t *__restrict__ ci = a.A.col_idx;
    const double *__restrict__ va = a.A.vals;
    const double *__restrict__ x = a.x;
    double ss = 0.0, am = 0.0;
    const int64_t n = a.A.n;
    const int64_t nrows_pad = (n + RPB - 1) / RPB * RPB; // keep whole warps in the shuffles
    const int64_t stride = (int64_t)gridDim.x * RPB;
    for (int64_t row0 = (int64_t)blockIdx.x * RPB + sub; row0 < nrows_pad; row0 += stride * U) {
        int p[U], p1[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int64_t row = row0 + u * stride;
            p[u] = 0;
            p1[u] = 0;
            if (row < n) {
                p[u] = rp[row] + sl;
                p1[u] = rp[row + 1];
            }
        }
        double s[U];
        bool more = false;
        int c[U];
        double v[U];
#pragma unroll
        for (int u = 0; u < U; ++u) { // first LANES entries of every row: the whole row for short rows
            s[u] = 0.0;
            c[u] = 0;
            v[u] = 0.0;
            if (p[u] < p1[u]) {
                c[u] = ci[p[u]];
                v[u] = va[p[u]];
            }
            more |= p[u] + LANES < p1[u];
        }
#pragma unroll
        for (int u = 0; u < U; ++u) s[u] = v[u] * ld_x(x + c[u]);
        if (__any_sync(0xffffffffu, more)) {
#pragma unroll
            for (int u = 0; u < U; ++u)
                for (int q = p[u] + LANES; q < p1[u]; q += LANES) s[u] = fma(va[q], ld_x(x + ci[q]), s[u]);
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
#pragma unroll
            for (int o = LANES / 2; o > 0; o >>= 1) s[u] += __shfl_xor_sync(0xffffffffu, s[u], o);
            const int64_t row = row0 + u * stride;
            if (sl == 0 && row < n) {
                const double val = (a.mode == MODE_RESIDUAL) ? a.b[row] - s[u] : s[u];
                a.w[row] = val;
                ss = fma(val, val, ss);
                am = fmax(am, fabs(val));
            }
        }
    }
    block_norm_partials(a, ss, am, &a.ctl->tickets[2]);
}

// ---- variant 2: nnz-balanced streaming (irregular row lengths) ------------------------------------------
// A block is a run of whole rows holding about T nonzeros (descriptors made once in set_matrix).
// Phase 1 streams the block's col_idx / vals with dense coalesced loads -- every thread first issues
// ALL of its loads (T/256 index + value pairs, then as many gathers of x), so a CTA has ~T
// independent requests in flight -- and leaves the products in shared memory.  Phase 2 reduces rows
// from there (g lanes per row, a warp per very long row), in a fixed order.  The matrix is read once
// per Arnoldi step and the basis passes stream hundreds of MB in between, so its lines are marked
// evict-first in L2: the 126 MB L2 is kept for the basis and the vectors.
// What bounds it on a power-law matrix is how many scattered 8-byte gathers of x an SM has in flight and for how much
// of the time (ncu on C4, n = 2e6, nnz = 4.2e7, before round 2: issue slots 15 % busy, 0.25 eligible warps per scheduler,
// no unit above 30 % of its peak; 587 us against 217 us for a bare torch.index_select of the same entries).  Round 2:
//  (1) the gathers are volatile asm like the index / value loads.  Written as plain loads the compiler interleaved
//      gather -> multiply -> store per item to save registers (40 registers, two or three gathers in flight per thread:
//      the "all loads first" of the source was not what ran): 587 -> 385 us;
//  (2) the values go global -> shared memory with cp.async, so no register holds them while the gathers are in flight
//      (64 registers: four CTAs per SM with twelve gathers per thread), and the row pointers of a pass of phase 2 are
//      fetched under the previous pass (volatile loads again): 385 -> 333 us (372 us with L2 flushed; 359 us inside
//      a Jacobi-preconditioned C4 solve, 630 us before).
// Tried on top and dropped: the next block's descriptor and column indices prefetched into shared memory with cp.async
// while this block's gathers are in flight (18 KB more shared memory and a spill at four CTAs per SM: 478 us; 351 us at
// three CTAs per SM); eight items at five or six CTAs per SM (335 - 369 us).
constexpr int kStreamThreads = 256;
#ifndef CBG_STREAM_ITEMS
#define CBG_STREAM_ITEMS 12
#endif
#ifndef CBG_STREAM_MINCTAS
#define CBG_STREAM_MINCTAS 4
#endif
constexpr int kStreamItems = CBG_STREAM_ITEMS;            // nonzeros per thread and batch
constexpr int kStreamT = kStreamThreads * kStreamItems;   // 3072 nonzeros per block
constexpr int kStreamBuf = kStreamT + kStreamT / 2;       // + the overhang of the block's last row (36 KB)
constexpr int kLongRow = 64;                              // rows longer than 64 g are reduced by a whole warp

__device__ __forceinline__ uint64_t policy_evict_first()
{
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
__device__ __forceinline__ int ldg_stream_i32(const int32_t *p, uint64_t pol)
{
    int r;
    asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.b32 %0, [%1], %2;" : "=r"(r) : "l"(p), "l"(pol));
    return r;
}

// 8-byte asynchronous copy global -> shared (LDGSTS): no register holds the value while it is in flight
__device__ __forceinline__ void cp_async8_hint(void *dst_smem, const void *src, uint64_t pol)
{
    asm volatile("cp.async.ca.shared.global.L2::cache_hint [%0], [%1], 8, %2;" ::"r"(smem_u32(dst_smem)), "l"(src), "l"(pol) : "memory");
}
// row pointers: volatile, so that the loads are issued where they are written (ahead of the phase that needs them)
__device__ __forceinline__ int ldg_rowptr(const int32_t *p)
{
    int r;
    asm volatile("ld.global.nc.b32 %0, [%1];" : "=r"(r) : "l"(p));
    return r;
}

// Gather of one entry of x by the streaming kernel.  Random columns find nothing in L1 (x is 16 MB), so
// the gathers go to L2 directly (ld.global.cg): C4, n = 2e6: 387 -> 369 us against ld.global.nc through
// L1; the .L1::no_allocate form of the nc load was far slower (545 us).  -DCBG_GATHER=0 / 2 select those.
#ifndef CBG_GATHER
#define CBG_GATHER 1
#endif
#ifndef CBG_GATHER_VOLATILE
#define CBG_GATHER_VOLATILE 1
#endif
__device__ __forceinline__ double gather_x(const double *p)
{
#if CBG_GATHER == 1
#if CBG_GATHER_VOLATILE
    // volatile: keeps the program order "all index / value loads, then all gathers, then the products" -- the
    // compiler otherwise interleaves gather -> multiply -> store per item to save registers
    double r;
    asm volatile("ld.global.cg.f64 %0, [%1];" : "=d"(r) : "l"(p));
    return r;
#else
    return __ldcg(p);
#endif
#elif CBG_GATHER == 2
    double r;
    asm volatile("ld.global.nc.L1::no_allocate.f64 %0, [%1];" : "=d"(r) : "l"(p));
    return r;
#else
    return ld_x(p);
#endif
}

__global__ void __launch_bounds__(kStreamThreads, CBG_STREAM_MINCTAS) spmv_stream_kernel(const SpmvArgs a)
{
    pdl_wait();
    pdl_launch_dependents();
    if (a.mode == MODE_STEP && a.step > a.ctl->stop_after) return;
    __shared__ double prod[kStreamBuf];
    const int32_t *__restrict__ rp = a.A.row_ptr;
    const int32_t *__restrict__ ci = a.A.col_idx;
    const double *__restrict__ va = a.A.vals;
    const double *__restrict__ x = a.x;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const uint64_t pol = policy_evict_first();
    // g consecutive lanes share a row in phase 2 (a power of two <= 32 chosen from the mean row length):
    // lane l of the group adds products l, l+g, ... and a butterfly adds the g partial sums.
    const int g = a.A.reduce_lanes, gl = tid & (g - 1), rows_per_pass = kStreamThreads / g;
    double ss = 0.0, am = 0.0;
    for (int blk = blockIdx.x; blk < a.A.nblk; blk += gridDim.x) {
        const int4 d = a.A.blk_desc[blk]; // {first row, end row, first nonzero, end nonzero}
        const int r0 = d.x, r1 = d.y, p0 = d.z, cnt = d.w - d.z;
        if (r0 >= r1) continue;
        if (cnt <= kStreamBuf) {
            // row pointers of this thread's first row of phase 2: on their way while phase 1 runs
            int rr = r0 + tid / g;
            int pa0 = p0, pa1 = p0;
            if (rr < r1) {
                pa0 = ldg_rowptr(rp + rr);
                pa1 = ldg_rowptr(rp + rr + 1);
            }
            __syncthreads(); // the previous block's phase 2 has finished with prod[]
            for (int off = 0; off < cnt; off += kStreamT) {
                // values: global -> shared memory without passing through registers (the registers go to the gathers)
#pragma unroll
                for (int i = 0; i < kStreamItems; ++i) {
                    const int q = off + i * kStreamThreads + tid;
                    if (q < cnt) cp_async8_hint(&prod[q], va + p0 + q, pol);
                }
                asm volatile("cp.async.commit_group;" ::: "memory");
                int c[kStreamItems];
#pragma unroll
                for (int i = 0; i < kStreamItems; ++i) {
                    const int q = off + i * kStreamThreads + tid;
                    c[i] = 0;
                    if (q < cnt) c[i] = ldg_stream_i32(ci + p0 + q, pol);
                }
                double xv[kStreamItems];
#pragma unroll
                for (int i = 0; i < kStreamItems; ++i) xv[i] = gather_x(x + c[i]);
                asm volatile("cp.async.wait_group 0;" ::: "memory");
#pragma unroll
                for (int i = 0; i < kStreamItems; ++i) {
                    const int q = off + i * kStreamThreads + tid;
                    if (q < cnt) prod[q] *= xv[i]; // the thread that copied value q multiplies it: no barrier in between
                }
            }
            __syncthreads();
            for (int rb = r0; rb < r1; rb += rows_per_pass) {
                const int r = rb + tid / g;
                const bool valid = r < r1;
                const int a0 = pa0 - p0, a1 = pa1 - p0;
                // the next pass's row pointers (an L2 round trip each) are fetched under this pass's reduction
                rr = r + rows_per_pass;
                pa0 = pa1 = p0;
                if (rr < r1) {
                    pa0 = ldg_rowptr(rp + rr);
                    pa1 = ldg_rowptr(rp + rr + 1);
                }
                const double bv = (valid && a.mode == MODE_RESIDUAL) ? a.b[r] : 0.0;
                const bool is_long = valid && (a1 - a0) > kLongRow * g;
                double s = 0.0;
                if (valid && !is_long) { // two independent chains: LDS -> DADD latency is the cost of a long-ish row
                    double s1 = 0.0;
                    int q = a0 + gl;
                    for (; q + g < a1; q += 2 * g) {
                        s += prod[q];
                        s1 += prod[q + g];
                    }
                    if (q < a1) s += prod[q];
                    s += s1;
                }
                for (int o = g >> 1; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
                if (valid && !is_long && gl == 0) {
                    const double val = (a.mode == MODE_RESIDUAL) ? bv - s : s;
                    a.w[r] = val;
                    ss = fma(val, val, ss);
                    am = fmax(am, fabs(val));
                }
                unsigned mask = __ballot_sync(0xffffffffu, is_long && gl == 0);
                while (mask) { // a very long row is reduced by the whole warp that found it: fixed order
                    const int src = __ffs(mask) - 1;
                    mask &= mask - 1;
                    const int rr = __shfl_sync(0xffffffffu, r, src);
                    const int qq0 = __shfl_sync(0xffffffffu, a0, src), qq1 = __shfl_sync(0xffffffffu, a1, src);
                    const double bb = __shfl_sync(0xffffffffu, bv, src);
                    double t = 0.0;
                    for (int q = qq0 + lane; q < qq1; q += 32) t += prod[q];
                    t = warp_sum(t);
                    if (lane == 0) {
                        const double val = (a.mode == MODE_RESIDUAL) ? bb - t : t;
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
                for (int p = rp[r] + lane; p < rp[r + 1]; p += 32) s = fma(va[p], ld_x(x + ci[p]), s);
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

// ---- variant 2b: nnz-balanced streaming with the matrix stream on the TMA engine -------------------------------
// The bound of variant 2 on C4 is not a bandwidth: ncu shows L1 34 %, L2 29 %, DRAM 14 % of peak.  What limits it is
// how many scattered 8-byte loads an SM keeps in flight: 4.2e7 gathers of x from L2 / 148 SMs / 369 us = 770 sectors per
// us and SM, and in variant 2 the same LSU / L1 miss path also carries the 12 bytes per nonzero of the matrix stream.
// Here a producer warp moves each block's col_idx / vals / row pointers into a two-stage shared-memory ring with bulk
// copies (cp.async.bulk: no LSU, no L1 miss slots, fetched one block ahead), so the load/store path of the SM carries
// the gathers and nothing else -- the situation of a bare gather kernel (torch.index_select of the same entries:
// 214 us).  Consumers: phase 1 reads the indices from shared memory, issues all gathers of a batch together and leaves
// the products IN PLACE of the staged values; phase 2 reduces the rows from there with the staged row pointers
// (no global loads at all in phase 2); one named barrier between the phases, stage handed back after phase 2.
// Blocks (built once in set_matrix) hold whole rows and about kTmaT nonzeros; a block that does not fit a stage
// (a very long row) is done warp-per-row from global memory as in variant 2.
// Measured on C4 (n = 2e6, nnz = 4.2e7; this round's box, where variant 2 takes 587 us stand-alone and 630 us inside a
// solve -- 369 us on round 1's box; torch.index_select of the same gathers 222 us on both): 509 us stand-alone with x in
// L2, 637 us with L2 flushed, 630 us inside a solve: no gain where it counts, so variant 2 stays the default for
// irregular matrices and this one is option 65.  Neither the load path of the gathers (.cg / .ca / .nc no-allocate:
// 587 / 621 / 795 us) nor smaller blocks at four CTAs per SM (634 us) moves the bound.
constexpr int kTmaThreads = 256;                 // consumers
constexpr int kTmaCta = kTmaThreads + 32;        // + the producer warp
#ifndef CBG_TMA_ITEMS
#define CBG_TMA_ITEMS 8
#endif
constexpr int kTmaItems = CBG_TMA_ITEMS;         // gathers in flight per thread and batch
constexpr int kTmaT = kTmaThreads * kTmaItems;   // 2048 nonzeros per block
constexpr int kTmaBuf = kTmaT + kTmaT / 2;       // + the overhang of the block's last row
constexpr int kTmaMaxRows = kTmaBuf;             // rows of a staged block (rows may be as short as one entry)
constexpr int kTmaStages = 2;

struct TmaStage {
    int32_t ci[kTmaBuf + 4];
    int32_t rp[kTmaMaxRows + 8];
    double va[kTmaBuf + 2];
};
struct TmaSmem {
    uint64_t full[kTmaStages], empty[kTmaStages];
    TmaStage st[kTmaStages];
};

__global__ void __launch_bounds__(kTmaCta, 2) spmv_stream_tma_kernel(const SpmvArgs a)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    TmaSmem &sm = *reinterpret_cast<TmaSmem *>(smem_raw);
    const int32_t *__restrict__ rp = a.A.row_ptr;
    const int32_t *__restrict__ ci = a.A.col_idx;
    const double *__restrict__ va = a.A.vals;
    const double *x = a.x;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const bool is_producer = warp == kTmaThreads / 32;
    const int safe_ci = (int)(a.A.nnz & ~(int64_t)3), safe_va = (int)(a.A.nnz & ~(int64_t)1);
    const int safe_rp = (int)((a.A.n + 1) & ~(int64_t)3);
    if (tid == 0) {
        for (int s = 0; s < kTmaStages; ++s) {
            mbar_init(&sm.full[s], 1);
            mbar_init(&sm.empty[s], kTmaThreads / 32);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    double ss = 0.0, am = 0.0;
    const int nblk = a.A.nblk, stride = gridDim.x;
    auto staged = [&](const int4 &d) { return d.w - d.z <= kTmaBuf && d.y - d.x <= kTmaMaxRows; };

    if (is_producer) {
        // the matrix is never written by a predecessor kernel: the first blocks are fetched BEFORE the grid dependency resolves
        Ring ring;
        const uint64_t pol = policy_evict_first();
        int issued = 0;
        bool waited = false;
        auto dependency = [&]() {
            pdl_wait();
            pdl_launch_dependents();
            waited = true;
            if (a.mode == MODE_STEP && a.step > a.ctl->stop_after) {
                if (lane == 0)
                    for (int s2 = 0; s2 < issued && s2 < kTmaStages; ++s2) mbar_wait(&sm.full[s2], 0u);
                return false;
            }
            return true;
        };
        for (int blk = blockIdx.x; blk < nblk; blk += stride) {
            if (!waited && issued == kTmaStages && !dependency()) return;
            const int4 d = a.A.blk_desc[blk];
            if (lane == 0) {
                mbar_wait(&sm.empty[ring.s], ring.ph ^ 1u);
                TmaStage &st = sm.st[ring.s];
                uint32_t bytes_ci = 0, bytes_va = 0, bytes_rp = 0;
                if (d.x < d.y && staged(d)) {
                    const int pc = d.z & ~3, pv = d.z & ~1, ra = d.x & ~3;
                    bytes_ci = (uint32_t)max(0, min((d.w + 3) & ~3, safe_ci) - pc) * 4u;
                    bytes_va = (uint32_t)max(0, min((d.w + 1) & ~1, safe_va) - pv) * 8u;
                    bytes_rp = (uint32_t)max(0, min((d.y + 1 + 3) & ~3, safe_rp) - ra) * 4u;
                    mbar_expect_tx(&sm.full[ring.s], bytes_ci + bytes_va + bytes_rp);
                    if (bytes_ci) bulk_g2s_hint(st.ci, ci + pc, bytes_ci, &sm.full[ring.s], pol);
                    if (bytes_va) bulk_g2s_hint(st.va, va + pv, bytes_va, &sm.full[ring.s], pol);
                    if (bytes_rp) bulk_g2s(st.rp, rp + ra, bytes_rp, &sm.full[ring.s]);
                }
                if (bytes_ci + bytes_va + bytes_rp == 0) mbar_arrive(&sm.full[ring.s]); // nothing to stage: the phase still completes
            }
            __syncwarp();
            ring.advance(kTmaStages);
            ++issued;
        }
        if (!waited && !dependency()) return;
    } else {
        pdl_wait();
        pdl_launch_dependents();
        if (a.mode == MODE_STEP && a.step > a.ctl->stop_after) return;
        const int g = a.A.reduce_lanes, gl = tid & (g - 1), rows_per_pass = kTmaThreads / g;
        Ring ring;
        for (int blk = blockIdx.x; blk < nblk; blk += stride) {
            const int4 d = a.A.blk_desc[blk];
            const int r0 = d.x, r1 = d.y, p0 = d.z, cnt = d.w - d.z;
            mbar_wait(&sm.full[ring.s], ring.ph);
            TmaStage &st = sm.st[ring.s];
            if (r0 < r1 && staged(d)) {
                const int pc = p0 & ~3, pv = p0 & ~1, ra = r0 & ~3;
                const int32_t *sci = st.ci + (p0 - pc);
                double *sva = st.va + (p0 - pv);
                // ---- phase 1: products in place of the staged values --------------------------------------------
                for (int off = 0; off < cnt; off += kTmaT) {
                    int c[kTmaItems];
                    double xv[kTmaItems];
#pragma unroll
                    for (int i = 0; i < kTmaItems; ++i) {
                        const int q = off + i * kTmaThreads + tid;
                        c[i] = 0;
                        if (q < cnt) c[i] = (p0 + q < safe_ci) ? sci[q] : ci[p0 + q]; // (the matrix's last few entries are not staged)
                    }
#pragma unroll
                    for (int i = 0; i < kTmaItems; ++i) xv[i] = gather_x(x + c[i]);
#pragma unroll
                    for (int i = 0; i < kTmaItems; ++i) {
                        const int q = off + i * kTmaThreads + tid;
                        if (q < cnt) sva[q] = ((p0 + q < safe_va) ? sva[q] : va[p0 + q]) * xv[i];
                    }
                }
                asm volatile("bar.sync 1, %0;" ::"n"(kTmaThreads) : "memory");
                // ---- phase 2: rows from shared memory, g lanes per row, fixed order -------------------------------
                auto rowptr = [&](int r) { return r < safe_rp ? st.rp[r - ra] : rp[r]; };
                for (int rb = r0; rb < r1; rb += rows_per_pass) {
                    const int r = rb + tid / g;
                    const bool valid = r < r1;
                    const int a0 = valid ? rowptr(r) - p0 : 0, a1 = valid ? rowptr(r + 1) - p0 : 0;
                    const double bv = (valid && a.mode == MODE_RESIDUAL) ? a.b[r] : 0.0;
                    const bool is_long = valid && (a1 - a0) > kLongRow * g;
                    double s = 0.0;
                    if (valid && !is_long) {
                        double s1 = 0.0;
                        int q = a0 + gl;
                        for (; q + g < a1; q += 2 * g) {
                            s += sva[q];
                            s1 += sva[q + g];
                        }
                        if (q < a1) s += sva[q];
                        s += s1;
                    }
                    for (int o = g >> 1; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
                    if (valid && !is_long && gl == 0) {
                        const double val = (a.mode == MODE_RESIDUAL) ? bv - s : s;
                        a.w[r] = val;
                        ss = fma(val, val, ss);
                        am = fmax(am, fabs(val));
                    }
                    unsigned mask = __ballot_sync(0xffffffffu, is_long && gl == 0);
                    while (mask) {
                        const int src = __ffs(mask) - 1;
                        mask &= mask - 1;
                        const int rr = __shfl_sync(0xffffffffu, r, src);
                        const int qq0 = __shfl_sync(0xffffffffu, a0, src), qq1 = __shfl_sync(0xffffffffu, a1, src);
                        const double bb = __shfl_sync(0xffffffffu, bv, src);
                        double t = 0.0;
                        for (int q = qq0 + lane; q < qq1; q += 32) t += sva[q];
                        t = warp_sum(t);
                        if (lane == 0) {
                            const double val = (a.mode == MODE_RESIDUAL) ? bb - t : t;
                            a.w[rr] = val;
                            ss = fma(val, val, ss);
                            am = fmax(am, fabs(val));
                        }
                    }
                }
                // the stage goes back once this warp is through phase 2 (the products live in the stage; they were written
                // through the generic proxy and the refill is an async-proxy write: fence between the two)
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                __syncwarp();
                if (lane == 0) mbar_arrive(&sm.empty[ring.s]);
            } else {
                __syncwarp();
                if (lane == 0) mbar_arrive(&sm.empty[ring.s]);
                for (int r = r0 + warp; r < r1; r += kTmaThreads / 32) { // oversized block: warp per row from global memory
                    double t = 0.0;
                    for (int p = rp[r] + lane; p < rp[r + 1]; p += 32) t = fma(va[p], ld_x(x + ci[p]), t);
                    t = warp_sum(t);
                    if (lane == 0) {
                        const double val = (a.mode == MODE_RESIDUAL) ? a.b[r] - t : t;
                        a.w[r] = val;
                        ss = fma(val, val, ss);
                        am = fmax(am, fabs(val));
                    }
                }
            }
            ring.advance(kTmaStages);
        }
    }
    block_norm_partials(a, ss, am, &a.ctl->tickets[2]);
}

// ---- variant 3: row-major from shared memory (regular matrices: stencils, banded, FEM) --------------
// Blocks of RB = 256 RPT / LPR consecutive rows, sized so that a block's nonzeros fit a stage:
// RPT rows per thread (short rows) or LPR lanes per row (long rows), at most ~14 nonzeros per thread.
// Two persistent CTAs per SM; a producer warp streams each block's col_idx / vals / row pointers
// into a two-stage shared-memory ring with bulk TMA copies (up to 43 KB per stage).  The consumer
// threads walk their rows in CSR order straight from shared memory, so the 32 lanes of a warp read
// THE SAME DIAGONALS of consecutive rows and the gathers of x coalesce into a few 128-byte lines --
// instead of the 8-16 lines a warp touches when it walks the nonzeros in storage order.  All of a
// thread's gathers (16) are issued before the first is used: one exposed latency per block.
// No CTA barrier: warps only meet at the mbarriers.
constexpr int kRowsThreads = 256;
constexpr int kRowsCta = kRowsThreads + 32;
constexpr int kRowsBuf = 3584;  // nonzeros per stage (256 threads x 14)
constexpr int kRowsMaxRows = 1024;
constexpr int kRowsStages = 2;
constexpr int kRowsGathers = 16; // gathers in flight per thread and round

struct RowsStage {
    int32_t ci[kRowsBuf + 4];
    int32_t rp[kRowsMaxRows + 8];
    double va[kRowsBuf + 2];
};
struct RowsSmem {
    uint64_t full[kRowsStages], empty[kRowsStages];
    RowsStage st[kRowsStages];
};

template <int RPT, int LPR> __global__ void __launch_bounds__(kRowsCta, 2) spmv_rows_kernel(const SpmvArgs a)
{
    // The matrix is never written by a predecessor kernel: the producer warp fetches its first
    // blocks BEFORE the grid dependency resolves (while the predecessor's tail is still running);
    // everything else -- x, the control block -- is read after the wait.
    const bool is_producer = (threadIdx.x >> 5) == kRowsThreads / 32;
    constexpr int RB = kRowsThreads * RPT / LPR, KU = kRowsGathers / RPT, RSTRIDE = kRowsThreads / LPR;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    RowsSmem &sm = *reinterpret_cast<RowsSmem *>(smem_raw);
    const int32_t *__restrict__ rp = a.A.row_ptr;
    const int32_t *__restrict__ ci = a.A.col_idx;
    const double *__restrict__ va = a.A.vals;
    const double *__restrict__ x = a.x;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int n = (int)a.A.n;
    const int safe_ci = (int)(a.A.nnz & ~(int64_t)3), safe_va = (int)(a.A.nnz & ~(int64_t)1);
    const int safe_rp = (int)((a.A.n + 1) & ~(int64_t)3);
    if (tid == 0) {
        for (int s = 0; s < kRowsStages; ++s) {
            mbar_init(&sm.full[s], 1);
            mbar_init(&sm.empty[s], kRowsThreads / 32);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (!is_producer) {
        pdl_wait();
        pdl_launch_dependents();
        if (a.mode == MODE_STEP && a.step > a.ctl->stop_after) return;
    }
    double ss = 0.0, am = 0.0;
    const int nblk = (n + RB - 1) / RB, stride = gridDim.x;

    if (warp == kRowsThreads / 32) {
        // ---- producer ----------------------------------------------------------------------------------
        Ring ring;
        const uint64_t pol = policy_evict_first(); // the matrix is read once per step: keep the L2 for basis and vectors
        int np0 = 0, np1 = 0;
        if ((int)blockIdx.x < nblk) {
            np0 = rp[blockIdx.x * RB];
            np1 = rp[min(n, (int)(blockIdx.x + 1) * RB)];
        }
        int issued = 0;
        bool waited = false;
        auto dependency = [&]() { // returns false if this step is skipped: drain the copies in flight and leave
            pdl_wait();
            pdl_launch_dependents();
            waited = true;
            if (a.mode == MODE_STEP && a.step > a.ctl->stop_after) {
                if (lane == 0)
                    for (int s2 = 0; s2 < issued; ++s2) mbar_wait(&sm.full[s2], 0u);
                return false;
            }
            return true;
        };
        for (int blk = blockIdx.x; blk < nblk; blk += stride) {
            if (!waited && issued == kRowsStages && !dependency()) return;
            const int r0 = blk * RB, r1 = min(n, r0 + RB), p0 = np0, p1 = np1;
            if (blk + stride < nblk) { // row pointers of the next block, one iteration ahead
                np0 = rp[(blk + stride) * RB];
                np1 = rp[min(n, (blk + stride + 1) * RB)];
            }
            if (lane == 0) {
                mbar_wait(&sm.empty[ring.s], ring.ph ^ 1u);
                RowsStage &st = sm.st[ring.s];
                uint32_t bytes_ci = 0, bytes_va = 0, bytes_rp = 0;
                const int pc = p0 & ~3, pv = p0 & ~1, ra = r0 & ~3;
                bytes_rp = (uint32_t)max(0, min((r1 + 1 + 3) & ~3, safe_rp) - ra) * 4u;
                if (p1 - p0 <= kRowsBuf) { // else: the consumers take this block straight from global memory
                    bytes_ci = (uint32_t)max(0, min((p1 + 3) & ~3, safe_ci) - pc) * 4u;
                    bytes_va = (uint32_t)max(0, min((p1 + 1) & ~1, safe_va) - pv) * 8u;
                }
                mbar_expect_tx(&sm.full[ring.s], bytes_ci + bytes_va + bytes_rp);
                if (bytes_ci) bulk_g2s_hint(st.ci, ci + pc, bytes_ci, &sm.full[ring.s], pol);
                if (bytes_va) bulk_g2s_hint(st.va, va + pv, bytes_va, &sm.full[ring.s], pol);
                if (bytes_rp) bulk_g2s(st.rp, rp + ra, bytes_rp, &sm.full[ring.s]);
            }
            __syncwarp();
            ring.advance(kRowsStages);
            ++issued;
        }
        if (!waited && !dependency()) return;
    } else {
        // ---- consumers: lane group tid / LPR owns rows r0 + tid / LPR + u * RSTRIDE of the block ----------
        const int gl = tid % LPR;
        Ring ring;
        for (int blk = blockIdx.x; blk < nblk; blk += stride) {
            const int r0 = blk * RB, r1 = min(n, r0 + RB), ra = r0 & ~3;
            mbar_wait(&sm.full[ring.s], ring.ph);
            const RowsStage &st = sm.st[ring.s];
            auto rowptr = [&](int r) { return r < safe_rp ? st.rp[r - ra] : rp[r]; };
            const int p0 = rowptr(r0), p1 = rowptr(r1);
            if (p1 - p0 <= kRowsBuf) {
                const int oc = -(p0 & ~3), ov = -(p0 & ~1); // stage index = offset + global index
                int q[RPT], e[RPT];
                double s[RPT];
#pragma unroll
                for (int u = 0; u < RPT; ++u) {
                    const int row = r0 + u * RSTRIDE + tid / LPR;
                    q[u] = e[u] = 0;
                    s[u] = 0.0;
                    if (row < r1) {
                        q[u] = rowptr(row) + gl;
                        e[u] = rowptr(row + 1);
                    }
                }
                // The index and value arrays of a block lie wholly inside the staged (16-byte aligned) part of
                // the matrix except in the last block(s) of the matrix: a block-uniform flag picks the loop
                // whose guards are predicates on shared-memory loads (no divergence, ~10 instructions per
                // nonzero) and keeps the per-element shared/global select for that tail only.
                const bool tail_blk = p1 > safe_ci || p1 > safe_va;
                bool more = true;
                if (!tail_blk) {
                    const int32_t *sci = st.ci + oc;
                    const double *sva = st.va + ov;
                    while (more) {
                        int c[RPT][KU];
#pragma unroll
                        for (int u = 0; u < RPT; ++u)
#pragma unroll
                            for (int k = 0; k < KU; ++k) {
                                const int g = q[u] + k * LPR;
                                c[u][k] = (g < e[u]) ? sci[g] : 0;
                            }
                        double xv[RPT][KU];
#pragma unroll
                        for (int u = 0; u < RPT; ++u)
#pragma unroll
                            for (int k = 0; k < KU; ++k) xv[u][k] = ld_x(x + c[u][k]);
                        more = false;
#pragma unroll
                        for (int u = 0; u < RPT; ++u) {
#pragma unroll
                            for (int k = 0; k < KU; ++k) {
                                const int g = q[u] + k * LPR;
                                const double av = (g < e[u]) ? sva[g] : 0.0;
                                s[u] = fma(av, xv[u][k], s[u]);
                            }
                            q[u] += KU * LPR;
                            more |= q[u] < e[u];
                        }
                        more = __any_sync(0xffffffffu, more);
                    }
                }
                while (more) {
                    int c[RPT][KU];
#pragma unroll
                    for (int u = 0; u < RPT; ++u)
#pragma unroll
                        for (int k = 0; k < KU; ++k) {
                            const int g = q[u] + k * LPR;
                            c[u][k] = 0;
                            if (g < e[u]) c[u][k] = g < safe_ci ? st.ci[oc + g] : ci[g];
                        }
                    double xv[RPT][KU];
#pragma unroll
                    for (int u = 0; u < RPT; ++u)
#pragma unroll
                        for (int k = 0; k < KU; ++k) xv[u][k] = ld_x(x + c[u][k]);
                    more = false;
#pragma unroll
                    for (int u = 0; u < RPT; ++u) {
#pragma unroll
                        for (int k = 0; k < KU; ++k) {
                            const int g = q[u] + k * LPR;
                            if (g < e[u]) s[u] = fma(g < safe_va ? st.va[ov + g] : va[g], xv[u][k], s[u]);
                        }
                        q[u] += KU * LPR;
                        more |= q[u] < e[u];
                    }
                    more = __any_sync(0xffffffffu, more);
                }
                { // hand the stage back once its loads have been USED (device_utils.cuh): the sums depend on all of them
                    unsigned dep = 0;
#pragma unroll
                    for (int u = 0; u < RPT; ++u) dep ^= dep_bits(s[u]);
                    mbar_arrive_after_use(&sm.empty[ring.s], lane, dep);
                }
#pragma unroll
                for (int u = 0; u < RPT; ++u) {
#pragma unroll
                    for (int o = LPR / 2; o > 0; o >>= 1) s[u] += __shfl_xor_sync(0xffffffffu, s[u], o);
                    const int row = r0 + u * RSTRIDE + tid / LPR;
                    if (row < r1 && gl == 0) {
                        const double val = (a.mode == MODE_RESIDUAL) ? a.b[row] - s[u] : s[u];
                        a.w[row] = val;
                        ss = fma(val, val, ss);
                        am = fmax(am, fabs(val));
                    }
                }
            } else {
                __syncwarp();
                if (lane == 0) mbar_arrive(&sm.empty[ring.s]);
                for (int r = r0 + warp; r < r1; r += kRowsThreads / 32) { // oversized block: warp per row from global
                    double t = 0.0;
                    for (int p = rp[r] + lane; p < rp[r + 1]; p += 32) t = fma(va[p], ld_x(x + ci[p]), t);
                    t = warp_sum(t);
                    if (lane == 0) {
                        const double val = (a.mode == MODE_RESIDUAL) ? a.b[r] - t : t;
                        a.w[r] = val;
                        ss = fma(val, val, ss);
                        am = fmax(am, fabs(val));
                    }
                }
            }
            ring.advance(kRowsStages);
        }
    }
    block_norm_partials(a, ss, am, &a.ctl->tickets[2]);
}

template <int RPT, int LPR> static void launch_rows(cudaStream_t s, const Scratch &sc, const SpmvArgs &a)
{
    static unsigned long long attr_set = 0; // per device
    if (first_use_on_device(attr_set, sc.lc->device))
        cudaFuncSetAttribute(spmv_rows_kernel<RPT, LPR>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(RowsSmem));
    constexpr int RB = kRowsThreads * RPT / LPR;
    const int64_t nblk = (a.A.n + RB - 1) / RB;
    const int grid = (int)(nblk < 2 * kNumSMs ? nblk : 2 * kNumSMs); // persistent: two CTAs per SM
    launch_chain(sc, "spmv_rows_kernel", spmv_rows_kernel<RPT, LPR>, dim3(grid), dim3(kRowsCta), sizeof(RowsSmem), s, a);
}

// Row partition of the streaming kernel: block b = rows [R(b), R(b+1)) with R(b) the first row r with
// row_ptr[r] >= b*T, so a block holds whole rows and about T nonzeros.  One descriptor per block:
// {first row, end row, first nonzero, end nonzero}.
__global__ void row_blocks_kernel(int64_t n, const int32_t *__restrict__ rp, int T, int nblk, int4 *desc)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= nblk) return;
    auto first_row = [&](int64_t target) { // first r in [0, n] with rp[r] >= target
        int64_t lo = 0, hi = n;
        while (lo < hi) {
            const int64_t mid = (lo + hi) >> 1;
            if (rp[mid] >= target) hi = mid;
            else lo = mid + 1;
        }
        return (int)lo;
    };
    const int r0 = first_row((int64_t)b * T);
    const int r1 = (b == nblk - 1) ? (int)n : first_row((int64_t)(b + 1) * T);
    desc[b] = make_int4(r0, r1, rp[r0], rp[r1]);
}

cudaError_t build_row_blocks(cudaStream_t s, int64_t n, int64_t nnz, const int32_t *d_row_ptr, int4 **d_desc_out,
                             int *nblk_out, int kernel)
{
    const int T = (kernel == 65) ? kTmaT : kStreamT; // nonzeros per block of the variant that will read the descriptors
    const int nblk = (int)((nnz + T - 1) / T) + 1;
    int4 *desc = nullptr;
    cudaError_t e = cudaMalloc(&desc, (size_t)nblk * sizeof(int4));
    if (e != cudaSuccess) return e;
    row_blocks_kernel<<<(nblk + 255) / 256, 256, 0, s>>>(n, d_row_ptr, T, nblk, desc);
    *d_desc_out = desc;
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

template <int LANES> static void launch_vec(cudaStream_t s, const Scratch &sc, const SpmvArgs &a)
{
    constexpr int RPB = 256 / LANES, U = 4;
    int64_t grid = (a.A.n + RPB * U - 1) / (RPB * U);
    const int64_t cap = (int64_t)kNumSMs * 8;
    if (grid > cap) grid = cap;
    if (grid < 1) grid = 1;
    launch_chain(sc, "spmv_vec_kernel", spmv_vec_kernel<LANES, U>, dim3((unsigned)grid), dim3(256), 0, s, a);
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
    case 2: launch_vec<2>(s, sc, a); break;
    case 4: launch_vec<4>(s, sc, a); break;
    case 8: launch_vec<8>(s, sc, a); break;
    case 16: launch_vec<16>(s, sc, a); break;
    case 32: launch_vec<32>(s, sc, a); break;
    case 64: {
        static int per_sm = 0; // persistent grid: exactly the CTAs that are resident at once (one more per SM
                               // and the stragglers run as a second wave: +25 % on C4); the same on every B200
        if (!per_sm) {
            if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, spmv_stream_kernel, kStreamThreads, 0) != cudaSuccess || per_sm < 1)
                per_sm = 1;
        }
        int grid = A.nblk < kNumSMs * per_sm ? A.nblk : kNumSMs * per_sm;
        if (grid < 1) grid = 1;
        launch_chain(sc, "spmv_stream_kernel", spmv_stream_kernel, dim3(grid), dim3(kStreamThreads), 0, s, a);
        break;
    }
    case 65: {
        static unsigned long long attr_set = 0; // per device
        if (first_use_on_device(attr_set, sc.lc->device))
            cudaFuncSetAttribute(spmv_stream_tma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(TmaSmem));
        int grid = A.nblk < 2 * kNumSMs ? A.nblk : 2 * kNumSMs; // persistent: two CTAs per SM (four CTAs of half-size blocks: 634 against 509 us)
        if (grid < 1) grid = 1;
        launch_chain(sc, "spmv_stream_tma_kernel", spmv_stream_tma_kernel, dim3(grid), dim3(kTmaCta), sizeof(TmaSmem), s, a);
        break;
    }
    // row-major kernel: 128 + rows per thread, or 144 + lanes per row
    case 129: launch_rows<1, 1>(s, sc, a); break;
    case 130: launch_rows<2, 1>(s, sc, a); break;
    case 132: launch_rows<4, 1>(s, sc, a); break;
    case 146: launch_rows<1, 2>(s, sc, a); break;
    case 148: launch_rows<1, 4>(s, sc, a); break;
    case 152: launch_rows<1, 8>(s, sc, a); break;
    default: return 0;
    }
    return 1;
}

} // namespace cbg
