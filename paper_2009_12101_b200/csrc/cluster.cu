// cluster.cu -- the whole restarted CB-GMRES solve (Fig. 1) of a SMALL system in ONE kernel launch:
// a thread-block cluster of 16 CTAs keeps the compressed Krylov basis, the matrix and every vector in its
// distributed shared memory (16 x ~200 KB = 3.2 MB) and replaces every kernel boundary of the Arnoldi step by a
// hardware cluster barrier.
//
// Why: BASELINE.json's C1 (5-point Laplacian 64^2, n = 4,096, m = 50) moves ~2 MB per Arnoldi step -- nothing a
// bandwidth roofline says applies; with one launch per kernel the step costs five dependent-launch latencies
// (~31 us per step measured, SURVEY.md section 7 step 6 "launch-latency work").  Here a step is 3 (5 when l.7 fires)
// all-to-all exchanges of a few hundred bytes through distributed shared memory plus the arithmetic on 256 rows per
// CTA out of shared memory.
//
// Mapping.  CTA c of the cluster owns rows [c nr, (c+1) nr) of A, b, x, w and of every basis vector (nr = ceil(n / 16)).
// Its slab of the basis is stored in shared memory IN THE STORAGE FORMAT (enc on store, decode on every read, as in
// the large path: PAPER.md:133, 169-181), vector-major.  The fp64 v that the SpMV multiplies (reading Q1) is
// replicated: after the store every CTA writes its nr entries into all 16 copies (st.shared::cluster).  Reductions
// (h = V^T w, norms) are all-to-all: every CTA writes its partial sums into slot [its rank] of every CTA's buffer,
// one cluster barrier, and every CTA adds the 16 partials in rank order -- the same bits everywhere, so every CTA takes
// the decisions of l.7 / l.12 / the stopping tests on its own and no broadcast of control flow is needed.  The small
// Hessenberg recurrences (Givens) run redundantly in one thread per CTA; rank 0 alone keeps R in global
// memory, solves R y = g at the end of a cycle and sends y to the others.
//
// Used by cbgmres_solve when the problem fits (small_fits below) and the preconditioner is none or scalar Jacobi (the
// column-scaled copy of the values is what is loaded); otherwise the large path runs.  Option "small_path" = 0 turns it off.
#include <cooperative_groups.h>

#include "device_utils.cuh"

namespace cg = cooperative_groups;

namespace cbg {

constexpr int kClusterCtas = 16;   // non-portable cluster size (opt-in), all of one GPC's worth of SMs
constexpr int kSmallThreads = 256; // 8 warps x up to 255 registers: the many shared-memory pointers of the kernel stay in registers
constexpr int kSmallMaxRestart = 128;
constexpr int kSmallSmemBytes = 200 * 1024;

struct SmallArgs {
    CsrView A;
    const double *b;
    double *x;       // in: x0, out: x
    Ctl *ctl;        // bnorm, tol_abs, eta, max_iters, reorth_mode, m, hist_cap set by the host; results written back
    CycleState cyc;  // R (rank 0 only), hist
    int64_t n;
    int nr;          // rows per CTA
    int m;
    int slab_nnz;    // capacity of the matrix slab (max over the CTAs)
    int format;
};

// shared-memory carve-up of one CTA (bytes, every region 16-byte aligned)
struct SmallLayout {
    int o_basis, o_sigma, o_rp, o_ci, o_va, o_vfull, o_w, o_x, o_b, o_part, o_h, o_hs, o_cs, o_sn, o_g, o_y, o_misc, total;
};
__host__ __device__ inline int up16(int x) { return (x + 15) & ~15; }
__host__ __device__ inline SmallLayout small_layout(int64_t n, int nr, int m, int slab_nnz, int B)
{
    SmallLayout L;
    int o = 0;
    L.o_basis = o;  o += up16((m + 1) * nr * B);
    L.o_sigma = o;  o += up16((m + 2) * 8);
    L.o_rp = o;     o += up16((nr + 1) * 4);
    L.o_ci = o;     o += up16(slab_nnz * 4);
    L.o_va = o;     o += up16(slab_nnz * 8);
    L.o_vfull = o;  o += up16((int)(kClusterCtas * nr) * 8);
    L.o_w = o;      o += up16(nr * 8);
    L.o_x = o;      o += up16(nr * 8);
    L.o_b = o;      o += up16(nr * 8);
    L.o_part = o;   o += up16(2 * kClusterCtas * (m + 4) * 8); // two buffers of [16 ranks][m + 4] partial sums
    L.o_h = o;      o += up16((m + 4) * 8);
    L.o_hs = o;     o += up16((m + 4) * 8);
    L.o_cs = o;     o += up16((m + 2) * 8);
    L.o_sn = o;     o += up16((m + 2) * 8);
    L.o_g = o;      o += up16((m + 2) * 8);
    L.o_y = o;      o += up16((m + 2) * 8);
    L.o_misc = o;   o += 512;
    L.total = o;
    (void)n;
    return L;
}

template <int FMT> __device__ __forceinline__ void small_store_entry(unsigned char *col, int r, double v, double s)
{
    if constexpr (FMT == CBGMRES_FP64) reinterpret_cast<double *>(col)[r] = v;
    else if constexpr (Fmt<FMT>::BYTES == 4) reinterpret_cast<unsigned *>(col)[r] = enc_bits<FMT>(v, s);
    else reinterpret_cast<unsigned short *>(col)[r] = (unsigned short)enc_bits<FMT>(v, s);
}

template <int FMT> __global__ void __launch_bounds__(kSmallThreads, 1) small_solve_kernel(const SmallArgs a)
{
    using Fm = Fmt<FMT>;
    constexpr int B = Fm::BYTES, T = kSmallThreads, NW = T / 32, C = kClusterCtas;
    cg::cluster_group cluster = cg::this_cluster();
    const int rank = (int)cluster.block_rank();
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    extern __shared__ __align__(16) unsigned char sm[];
    const int nr = a.nr, m = a.m, pstride = m + 4;
    const int64_t n = a.n;
    const SmallLayout L = small_layout(n, nr, m, a.slab_nnz, B);
    unsigned char *basis = sm + L.o_basis;
    double *sigma = reinterpret_cast<double *>(sm + L.o_sigma);
    int *rp_s = reinterpret_cast<int *>(sm + L.o_rp);
    int *ci_s = reinterpret_cast<int *>(sm + L.o_ci);
    double *va_s = reinterpret_cast<double *>(sm + L.o_va);
    double *vfull = reinterpret_cast<double *>(sm + L.o_vfull);
    double *w = reinterpret_cast<double *>(sm + L.o_w);
    double *xs = reinterpret_cast<double *>(sm + L.o_x);
    double *bs = reinterpret_cast<double *>(sm + L.o_b);
    double *part = reinterpret_cast<double *>(sm + L.o_part);
    double *h = reinterpret_cast<double *>(sm + L.o_h);   // Hessenberg column (then rotated in place)
    double *hs = reinterpret_cast<double *>(sm + L.o_hs); // sigma_c * coefficient: what multiplies the raw payload
    double *cs = reinterpret_cast<double *>(sm + L.o_cs);
    double *sn = reinterpret_cast<double *>(sm + L.o_sn);
    double *g = reinterpret_cast<double *>(sm + L.o_g);
    double *y = reinterpret_cast<double *>(sm + L.o_y);
    double *misc = reinterpret_cast<double *>(sm + L.o_misc); // [0..15] warp sums, [16..31] warp maxima, [32] the recurrence residual
    __shared__ double loc[kSmallMaxRestart + 4]; // this CTA's partial sums of the exchange in flight
    __shared__ double tot[kSmallMaxRestart + 4]; // ... and the totals over the cluster
    __shared__ int s_stop;

    const int64_t row0 = (int64_t)rank * nr;
    const int rows = (int)max((int64_t)0, min((int64_t)nr, n - row0));
    Ctl *ctl = a.ctl;
    const double bnorm = ctl->bnorm, tol_abs = ctl->tol_abs, eta = ctl->eta;
    const int max_iters = ctl->max_iters, reorth_mode = ctl->reorth_mode, hist_cap = ctl->hist_cap;

    // ---- this CTA's slab of the problem into shared memory ----------------------------------------------------
    const int p0 = rows > 0 ? a.A.row_ptr[row0] : 0;
    if (rows > 0) {
        for (int r = tid; r <= rows; r += T) rp_s[r] = a.A.row_ptr[row0 + r] - p0;
    } else if (tid == 0) rp_s[0] = 0;
    const int slab = rows > 0 ? a.A.row_ptr[row0 + rows] - p0 : 0;
    for (int q = tid; q < slab; q += T) {
        ci_s[q] = a.A.col_idx[p0 + q];
        va_s[q] = a.A.vals[p0 + q];
    }
    for (int r = tid; r < nr; r += T) {
        bs[r] = r < rows ? a.b[row0 + r] : 0.0;
        xs[r] = r < rows ? a.x[row0 + r] : 0.0;
    }
    for (int c = tid; c < m + 2; c += T) sigma[c] = 1.0;
    cluster.sync(); // every CTA of the cluster is resident: its shared memory may be written from now on

    int pbuf = 0; // which of the two exchange buffers the next exchange writes
    // All-to-all reduction of loc[0 .. count): every CTA ends with tot[i] = sum (or max for i == max_slot) over the
    // ranks, added in rank order -- the same bits in every CTA.  One cluster barrier.
    auto exchange = [&](int count, int max_slot) {
        __syncthreads(); // loc[] complete
        double *mine = part + ((size_t)pbuf * C + rank) * pstride;
        for (int dst = warp; dst < C; dst += NW) { // warp q sends this CTA's partial sums to CTAs q, q + 8: all in flight together
            double *remote = cluster.map_shared_rank(mine, dst);
            for (int i = lane; i < count; i += 32) remote[i] = loc[i];
        }
        cluster.sync();
        const double *buf = part + (size_t)pbuf * C * pstride;
        for (int i = tid; i < count; i += T) {
            double t = buf[i];
            if (i == max_slot) {
                for (int q = 1; q < C; ++q) t = fmax(t, buf[q * pstride + i]);
            } else {
                for (int q = 1; q < C; ++q) t += buf[q * pstride + i];
            }
            tot[i] = t;
        }
        pbuf ^= 1;
        __syncthreads();
    };
    // this CTA's sum / max of a per-thread pair -> loc[slot_s], loc[slot_m]
    auto block_pair = [&](double s, double mx, int slot_s, int slot_m) {
        s = warp_sum(s);
        mx = warp_max(mx);
        if (lane == 0) {
            misc[warp] = s;
            misc[16 + warp] = mx;
        }
        __syncthreads();
        if (tid == 0) {
            double ts = 0.0, tm = 0.0;
            for (int q = 0; q < NW; ++q) {
                ts += misc[q];
                tm = fmax(tm, misc[16 + q]);
            }
            loc[slot_s] = ts;
            if (slot_m >= 0) loc[slot_m] = tm;
        }
    };
    // own rows of a vector into every CTA's copy of the full vector (the caller separates it from readers by a barrier)
    auto allgather = [&](const double *own) {
        for (int dst = warp; dst < C; dst += NW) { // warp q -> CTAs q, q + 8
            double *remote = cluster.map_shared_rank(vfull, dst) + (size_t)rank * nr;
            if ((nr & 1) == 0) {
                for (int r = 2 * lane; r < nr; r += 64) *reinterpret_cast<double2 *>(remote + r) = *reinterpret_cast<const double2 *>(own + r);
            } else {
                for (int r = lane; r < nr; r += 32) remote[r] = own[r];
            }
        }
    };
    auto spmv_rows = [&](bool residual, double &ss, double &am) { // w = A vfull (or b - A vfull) on the own rows
        ss = 0.0;
        am = 0.0;
        for (int r = tid; r < rows; r += T) {
            double s = 0.0;
            for (int q = rp_s[r]; q < rp_s[r + 1]; ++q) s = fma(va_s[q], vfull[ci_s[q]], s);
            const double val = residual ? bs[r] - s : s;
            w[r] = val;
            ss = fma(val, val, ss);
            am = fmax(am, fabs(val));
        }
    };
    // partial inner products of the stored vectors 0 .. j-1 with w over the own rows -> loc[0 .. j)
    auto dots = [&](int j) {
        // a warp takes four columns at a time: four independent chains per lane and four shuffle reductions in flight
        for (int c0 = 4 * warp; c0 < j; c0 += 4 * NW) {
            double s4[4] = {0.0, 0.0, 0.0, 0.0};
            const unsigned char *col[4];
#pragma unroll
            for (int q = 0; q < 4; ++q) col[q] = basis + (size_t)min(c0 + q, j - 1) * nr * B;
            for (int r = lane; r < rows; r += 32) {
                const double wr = w[r];
#pragma unroll
                for (int q = 0; q < 4; ++q) s4[q] = fma(Fm::decode_one(col[q], r), wr, s4[q]);
            }
#pragma unroll
            for (int q = 0; q < 4; ++q) s4[q] = warp_sum(s4[q]);
            if (lane == 0) {
#pragma unroll
                for (int q = 0; q < 4; ++q)
                    if (c0 + q < j) loc[c0 + q] = s4[q];
            }
        }
    };
    // w_r -= sum_c payload[r, c] * hs_c on the own rows; partial norms of the new w
    auto update = [&](int j, double *vec, double &ss, double &am) {
        ss = 0.0;
        am = 0.0;
        for (int r = tid; r < rows; r += T) {
            double p0a = 0.0, p1a = 0.0;
            int c = 0;
            for (; c + 1 < j; c += 2) {
                p0a = fma(Fm::decode_one(basis + (size_t)c * nr * B, r), hs[c], p0a);
                p1a = fma(Fm::decode_one(basis + (size_t)(c + 1) * nr * B, r), hs[c + 1], p1a);
            }
            if (c < j) p0a = fma(Fm::decode_one(basis + (size_t)c * nr * B, r), hs[c], p0a);
            const double val = vec[r] - (p0a + p1a);
            vec[r] = val;
            ss = fma(val, val, ss);
            am = fmax(am, fabs(val));
        }
    };
    // v = w / hn -> stored column `col` (enc) and every CTA's copy of the full fp64 v (reading Q1)
    auto store = [&](int col, double hn, double amax_w) {
        double s = 0.0, sg = 1.0;
        if (Fm::SCALED) {
            const double av = amax_w / hn;
            if (av > 0.0 && isfinite(av)) {
                s = fmt_maxint<FMT>() / av;
                sg = av / fmt_maxint<FMT>();
            } else {
                s = 0.0;
                sg = 0.0;
            }
        }
        if (tid == 0) sigma[col] = sg;
        unsigned char *cptr = basis + (size_t)col * nr * B;
        for (int r = tid; r < nr; r += T) {
            const double v = r < rows ? w[r] / hn : 0.0; // IEEE division per element (reading Q8)
            w[r] = v;
            small_store_entry<FMT>(cptr, r, v, s);
        }
        __syncthreads();
        allgather(w);
    };

    // ---- the solve: restart cycles until the explicit residual decides -----------------------
    int iters = 0, restarts = 0, reorth_count = 0, breakdown = 0, converged = 0, nonfinite = 0, k = 0;
    double rel_true = 0.0, rel_rec = 0.0;
    for (;;) {
        // l.1: r0 = b - A x; beta = ||r0||_2
        allgather(xs);
        cluster.sync();
        double ss, am;
        spmv_rows(true, ss, am);
        block_pair(ss, am, 0, 1);
        exchange(2, 1);
        const double beta = sqrt(tot[0]), amax0 = tot[1];
        rel_true = beta / bnorm;
        k = 0;
        if (!isfinite(beta)) {
            nonfinite = 1;
            break;
        }
        if (beta <= tol_abs) {
            converged = 1;
            break;
        }
        if (iters >= max_iters) break;
        restarts += 1;
        breakdown = 0;
        if (tid == 0) {
            for (int c = 1; c <= m; ++c) g[c] = 0.0;
            g[0] = beta;
        }
        store(0, beta, amax0); // v_1 = r0 / beta
        cluster.sync();
        for (int j = 1; j <= m; ++j) {
            // l.3-4: w = A v; omega = ||w||_2 -- l.5: h = V^T w, both from one exchange
            spmv_rows(false, ss, am);
            block_pair(ss, 0.0, j, -1); // (ends with every w[r] written: block_pair synchronises the CTA)
            __syncthreads();
            dots(j);
            exchange(j + 1, -1);
            const double omega = sqrt(tot[j]);
            for (int c = tid; c < j; c += T) {
                const double hc = tot[c] * sigma[c]; // h_c = sigma_c * sum q w (the scale leaves the inner loop)
                h[c] = hc;
                hs[c] = hc * sigma[c];
            }
            __syncthreads();
            // l.5-6: w -= V h; h_{j+1,j} = ||w||_2, ||w||_inf
            // ... and, in the same exchange, u = V^T w of the second pass (l.8), dropped if l.7 does not fire: one cluster
            // barrier less per re-orthogonalised step (the large path's fused update + multi-dot, in small)
            update(j, w, ss, am);
            block_pair(ss, am, j, j + 1);
            const bool may_reorth = reorth_mode != CBGMRES_REORTH_NEVER;
            if (may_reorth) dots(j); // (block_pair has synchronised the CTA: every w[r] is the new one)
            exchange(j + 2, j + 1);
            double hn = sqrt(tot[j]), amax = tot[j + 1];
            // l.7: re-orthogonalise iff h_{j+1,j} < eta * omega
            const bool flag = reorth_mode == CBGMRES_REORTH_ALWAYS || (reorth_mode == CBGMRES_REORTH_COND && hn < eta * omega);
            breakdown = (hn == 0.0);
            if (!isfinite(hn)) nonfinite = 1;
            if (flag) {
                // l.8-10: u = V^T w (already here); w -= V u; h += u; new norm
                for (int c = tid; c < j; c += T) {
                    const double uc = tot[c] * sigma[c];
                    h[c] += uc; // l.9
                    hs[c] = uc * sigma[c];
                }
                __syncthreads();
                update(j, w, ss, am);
                block_pair(ss, am, 0, 1);
                exchange(2, 1);
                const double omega1 = hn;
                hn = sqrt(tot[0]);
                amax = tot[1];
                reorth_count += 1;
                breakdown = (hn == 0.0) || (hn < eta * omega1); // l.12 (reading Q4)
                if (!isfinite(hn)) nonfinite = 1;
            }
            // "updating technique": rotations 1..j-1 on the new column, rotation j, g; the stopping tests.
            // Every CTA runs the same recurrence on the same bits; rank 0 keeps R and the history in global memory.
            if (tid == 0) {
                double hc = h[0];
                for (int c = 0; c < j - 1; ++c) {
                    const double hnext = h[c + 1];
                    const double a1 = sn[c] * hnext, a2 = cs[c] * hnext;
                    const double t = fma(cs[c], hc, a1);
                    hc = fma(-sn[c], hc, a2);
                    h[c] = t;
                }
                const double rho = hypot(hc, hn);
                double cj = 1.0, sj = 0.0;
                if (rho != 0.0) {
                    cj = hc / rho;
                    sj = hn / rho;
                }
                cs[j - 1] = cj;
                sn[j - 1] = sj;
                h[j - 1] = rho;
                const double gj = g[j - 1];
                g[j] = -sj * gj;
                g[j - 1] = cj * gj;
                const double rec = fabs(sj * gj);
                if (rank == 0) {
                    double *Rcol = a.cyc.R + (size_t)(j - 1) * (m + 1);
                    for (int c = 0; c < j; ++c) Rcol[c] = h[c];
                    if (a.cyc.hist && iters < hist_cap) a.cyc.hist[iters] = rec / bnorm;
                }
                misc[32] = rec;
                s_stop = (rec <= tol_abs) || breakdown || (iters + 1 >= max_iters) || nonfinite || !isfinite(rec);
            }
            __syncthreads();
            const double rec = misc[32];
            iters += 1;
            k = j;
            rel_rec = rec / bnorm;
            if (!isfinite(rec)) nonfinite = 1;
            const int stop = s_stop;
            // l.13-14: v = w / h_{j+1,j}; V[:, j] = enc(v)
            if (hn > 0.0) store(j, hn, amax);
            cluster.sync(); // the new v is in every CTA's copy before the next SpMV; also separates this step's reads of vfull
            if (stop) break;
        }
        // l.16-17: R y = g (rank 0), y to everyone, x += V_k y
        if (k > 0 && !nonfinite) {
            if (rank == 0) {
                if (warp == 0) {
                    for (int i = lane; i < k; i += 32) y[i] = g[i];
                    __syncwarp();
                    for (int i = k - 1; i >= 0; --i) {
                        const double *Rc = a.cyc.R + (size_t)i * (m + 1);
                        const double yi = y[i] / Rc[i];
                        __syncwarp();
                        if (lane == 0) y[i] = yi;
                        for (int l = lane; l < i; l += 32) y[l] = fma(-Rc[l], yi, y[l]);
                        __syncwarp();
                    }
                }
                __syncthreads();
                for (int dst = 1; dst < C; ++dst) {
                    double *remote = cluster.map_shared_rank(y, dst);
                    for (int i = tid; i < k; i += T) remote[i] = y[i];
                }
            }
            cluster.sync();
            for (int c = tid; c < k; c += T) hs[c] = -sigma[c] * y[c];
            __syncthreads();
            update(k, xs, ss, am); // x -= V (-sigma y)
            __syncthreads();
        } else {
            cluster.sync(); // keep the barrier count of the cluster in step
        }
    }
    // ---- results ------------------------------------------------------------------------------------------------
    for (int r = tid; r < rows; r += T) a.x[row0 + r] = xs[r];
    if (rank == 0 && tid == 0) {
        ctl->iters = iters;
        ctl->restarts = restarts;
        ctl->reorth_count = reorth_count;
        ctl->breakdown = breakdown;
        ctl->converged = converged;
        ctl->nonfinite = nonfinite;
        ctl->rel_true = rel_true;
        ctl->rel_rec = rel_rec;
        ctl->k = k;
        ctl->done = 1;
    }
    cluster.sync(); // no CTA leaves while another may still write into its shared memory
}

// ---- host side ---------------------------------------------------------------------------------------------------
__global__ void slab_bounds_kernel(int64_t n, const int32_t *__restrict__ rp, int nr, int *out)
{
    const int c = threadIdx.x;
    if (c <= kClusterCtas) {
        const int64_t r = min(n, (int64_t)c * nr);
        out[c] = rp[r];
    }
}

// nonzeros of the fullest of the 16 row slabs (0 if the rows cannot be cut this way); enqueues on s and synchronises it
int small_slab_nnz(cudaStream_t s, int64_t n, const int32_t *d_row_ptr, int *d_scratch /* >= 17 ints */)
{
    if (n <= 0 || n > (int64_t)kClusterCtas * 65536) return 0;
    const int nr = (int)((n + kClusterCtas - 1) / kClusterCtas);
    slab_bounds_kernel<<<1, 32, 0, s>>>(n, d_row_ptr, nr, d_scratch);
    int hb[kClusterCtas + 1];
    if (cudaMemcpyAsync(hb, d_scratch, sizeof(hb), cudaMemcpyDeviceToHost, s) != cudaSuccess) return 0;
    if (cudaStreamSynchronize(s) != cudaSuccess) return 0;
    int mx = 0;
    for (int c = 0; c < kClusterCtas; ++c) mx = hb[c + 1] - hb[c] > mx ? hb[c + 1] - hb[c] : mx;
    return mx > 0 ? mx : 1;
}

static inline int small_fmt_bytes(int format) { return format == CBGMRES_FP64 ? 8 : (format == CBGMRES_FP32 || format == CBGMRES_INT32) ? 4 : 2; }

// Does the whole solve fit the distributed shared memory of one cluster?
bool small_fits(int64_t n, int slab_nnz, int m, int format)
{
    if (slab_nnz <= 0 || m < 1 || m > kSmallMaxRestart || n <= 0 || n > (int64_t)kClusterCtas * 65536) return false;
    const int nr = (int)((n + kClusterCtas - 1) / kClusterCtas);
    const long long basis = (long long)(m + 1) * nr * small_fmt_bytes(format);
    if (basis > kSmallSmemBytes) return false;
    return small_layout(n, nr, m, slab_nnz, small_fmt_bytes(format)).total + 4096 <= kSmallSmemBytes;
}

template <int FMT> static cudaError_t launch_small_t(cudaStream_t s, const Scratch &sc, const SmallArgs &a, int smem)
{
    static unsigned long long attr_set = 0; // per device
    if (first_use_on_device(attr_set, sc.lc->device)) {
        cudaError_t e = cudaFuncSetAttribute(small_solve_kernel<FMT>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(small_solve_kernel<FMT>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmallSmemBytes);
        if (e != cudaSuccess) return e;
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(kClusterCtas);
    cfg.blockDim = dim3(kSmallThreads);
    cfg.dynamicSmemBytes = (size_t)smem;
    cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = kClusterCtas;
    at[0].val.clusterDim.y = 1;
    at[0].val.clusterDim.z = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, small_solve_kernel<FMT>, a);
}

// One launch = the whole solve.  Returns the number of kernels launched (0 and a recorded launch error on failure).
int launch_small_solve(cudaStream_t s, const Scratch &sc, const CsrView &A, const double *b, double *x, const CycleState &cyc,
                       int m, int format, int slab_nnz)
{
    SmallArgs a{};
    a.A = A;
    a.b = b;
    a.x = x;
    a.ctl = sc.ctl;
    a.cyc = cyc;
    a.n = A.n;
    a.nr = (int)((A.n + kClusterCtas - 1) / kClusterCtas);
    a.m = m;
    a.slab_nnz = slab_nnz;
    a.format = format;
    const int smem = small_layout(A.n, a.nr, m, slab_nnz, small_fmt_bytes(format)).total;
    cudaError_t e;
    switch (format) {
    case CBGMRES_FP64: e = launch_small_t<CBGMRES_FP64>(s, sc, a, smem); break;
    case CBGMRES_FP32: e = launch_small_t<CBGMRES_FP32>(s, sc, a, smem); break;
    case CBGMRES_FP16: e = launch_small_t<CBGMRES_FP16>(s, sc, a, smem); break;
    case CBGMRES_INT32: e = launch_small_t<CBGMRES_INT32>(s, sc, a, smem); break;
    case CBGMRES_INT16: e = launch_small_t<CBGMRES_INT16>(s, sc, a, smem); break;
    default: e = cudaErrorInvalidValue;
    }
    if (e != cudaSuccess) {
        if (sc.lc->launch_error == cudaSuccess) {
            sc.lc->launch_error = e;
            sc.lc->launch_kernel = "small_solve_kernel";
        }
        return 0;
    }
    return 1;
}

} // namespace cbg
