// store.cu -- S4: v := w / h_{j+1,j}; V_{j+1} := [V_j, enc(v)]  (Fig. 1 lines 13-14, PAPER.md:87,
// 169-181), keeping the fp64 v for the next SpMV (reading Q1); plus the incremental
// Givens QR of the Hessenberg matrix ("updating technique") run by one extra CTA of
// the same launch, and the decode kernel of the per-kernel hooks.
//
// Bound: HBM.  Algorithmic bytes per launch: 8n (w) + B*n (payload) + 8n (v).
#include "device_utils.cuh"

namespace cbg {

struct StoreArgs {
    const double *w;
    const double *d_hn, *d_amax; // device scalars (solver) or null -> host values below (hooks)
    double hn_host, amax_host;
    void *payload;
    double *scale_out;
    double *v_out;               // may be null (k_compress hook)
    int64_t n;
    Ctl *ctl;
    CycleState cyc;
    int has_cyc;
    int mode, step;
    int *h_flag;                 // mapped host word: mirrors ctl->stop_after (may be null)
    const double *bj_inv;        // block-Jacobi(4): inverted diagonal blocks [ceil(n/4)][16]; v_out then receives M^-1 v
};

// The control CTA: apply rotations 1..j-1 to the new column, form rotation j, rotate g, decide
// whether the cycle goes on (recurrence residual; breakdown, Fig. 1 l.12; iteration
// bound).  The column and the rotations are staged in shared memory by all threads (one round trip
// to global memory); the recurrence itself is inherently sequential and runs in one thread.
__device__ void givens_step(const StoreArgs &a)
{
    __shared__ double s_h[kMaxRestart + 2], s_cs[kMaxRestart], s_sn[kMaxRestart];
    Ctl *ctl = a.ctl;
    const CycleState &cy = a.cyc;
    const int j = a.step, m = ctl->m, tid = threadIdx.x, nt = blockDim.x;
    for (int c = tid; c < j; c += nt) s_h[c] = cy.h[c];
    for (int c = tid; c < j - 1; c += nt) {
        s_cs[c] = cy.cs[c];
        s_sn[c] = cy.sn[c];
    }
    __syncthreads();
    if (tid == 0) {
        // scalars of the control block, fetched together (L2 round trips) before the recurrence
        const double hn = __ldcg(&ctl->hn), bnorm = __ldcg(&ctl->bnorm), tol_abs = __ldcg(&ctl->tol_abs);
        const double gj = __ldcg(&cy.g[j - 1]);
        const int iters0 = __ldcg(&ctl->iters), max_iters = __ldcg(&ctl->max_iters), hist_cap = __ldcg(&ctl->hist_cap);
        const int bd = __ldcg(&ctl->breakdown), nonfin = __ldcg(&ctl->nonfinite);
        double hc = s_h[0]; // h_c after the rotations applied so far
        for (int c = 0; c < j - 1; ++c) {
            // one FMA per rotation on the critical path: the products with h_{c+1} do not depend on hc
            const double hnext = s_h[c + 1];
            const double a1 = s_sn[c] * hnext, a2 = s_cs[c] * hnext;
            const double t = fma(s_cs[c], hc, a1);
            hc = fma(-s_sn[c], hc, a2);
            s_h[c] = t;
        }
        const double rho = hypot(hc, hn);
        double cj = 1.0, sj = 0.0;
        if (rho != 0.0) {
            cj = hc / rho;
            sj = hn / rho;
        }
        cy.cs[j - 1] = cj;
        cy.sn[j - 1] = sj;
        s_h[j - 1] = rho;
        cy.g[j] = -sj * gj;
        cy.g[j - 1] = cj * gj;
        const double rec = fabs(sj * gj);
        const int iters = iters0 + 1;
        ctl->iters = iters;
        ctl->k = j;
        ctl->rel_rec = rec / bnorm;
        if (cy.hist && iters - 1 < hist_cap) cy.hist[iters - 1] = rec / bnorm;
        if (!isfinite(rec)) ctl->nonfinite = 1;
        const bool stop = (rec <= tol_abs) || bd || (iters >= max_iters) || nonfin || !isfinite(rec);
        if (stop) {
            ctl->stop_after = j; // later steps of this cycle see step > stop_after and return at once
            if (a.h_flag) {
                *reinterpret_cast<volatile int *>(a.h_flag) = j;
                __threadfence_system();
            }
        }
    }
    __syncthreads();
    double *Rcol = cy.R + (size_t)(j - 1) * (m + 1);
    for (int c = tid; c < j; c += nt) Rcol[c] = s_h[c];
}

// BJ: with the block-Jacobi(4) right preconditioner the vector the next SpMV multiplies is
// z = M^-1 v (Fig. 1 l.3), so the store writes z instead of v: the thread that holds the four entries of
// a block multiplies them by the block's inverse (a.bj_inv, 16 doubles per block, row-major) -- 32 bytes
// more per row and no extra launch.  A thread then owns RT = max(VEC, 4) consecutive rows.
template <int FMT, int THREADS, bool BJ> __global__ void __launch_bounds__(THREADS) store_kernel(const StoreArgs a)
{
    using F = Fmt<FMT>;
    constexpr int VEC = F::VEC;
    constexpr int GROUPS = (BJ && VEC < 4) ? 4 / VEC : 1; // 16-byte payload words per thread and iteration
    constexpr int RT = VEC * GROUPS;                       // rows per thread and iteration
    pdl_wait();
    // A successor may fetch basis columns before ITS grid dependency resolves (orth.cu); inside a solve
    // the successor of a store is never a Gram-Schmidt pass, but after the k_compress / k_store hooks it
    // can be: there the successor is only released when this kernel has completed.
    if (a.mode != MODE_HOOK) pdl_launch_dependents();
    // this thread's first rows of w and the control words, fetched together (each is an L2 round trip)
    const bool has_ctl_cta = a.has_cyc && a.mode == MODE_ORTH1;
    const int bid = has_ctl_cta ? (int)blockIdx.x - 1 : (int)blockIdx.x;
    const int nblk = has_ctl_cta ? gridDim.x - 1 : gridDim.x;
    const int64_t nunits = (a.n + RT - 1) / RT;
    const int64_t g0 = (int64_t)bid * THREADS + threadIdx.x;
    double2 w0[RT / 2];
    if (bid >= 0 && g0 < nunits && g0 * RT + RT <= a.n) {
#pragma unroll
        for (int r = 0; r < RT; r += 2) w0[r / 2] = *reinterpret_cast<const double2 *>(a.w + g0 * RT + r);
    }
    const int stop_after = (a.mode != MODE_HOOK) ? __ldcg(&a.ctl->stop_after) : 0;
    const double hn_dev = a.d_hn ? __ldcg(a.d_hn) : 0.0, amax_dev = a.d_amax ? __ldcg(a.d_amax) : 0.0;
    if (a.mode != MODE_HOOK && a.step > stop_after) return;
    if (has_ctl_cta && blockIdx.x == 0) { // the control CTA: first to be scheduled, its serial chain overlaps the streaming
        givens_step(a);
        return;
    }
    const double hn = a.d_hn ? hn_dev : a.hn_host;
    const double amax_w = a.d_amax ? amax_dev : a.amax_host;
    if (!(hn > 0.0)) return; // Fig. 1 l.12: h_{j+1,j} = 0 -> no new vector
    double s = 0.0, sigma = 1.0;
    if (F::SCALED) {
        // sigma = ||v||inf / max_int with ||v||inf = fl(||w||inf / hn): division by a positive
        // constant is monotone, so this equals max_i fl(|w_i| / hn) exactly.
        const double av = amax_w / hn;
        if (av > 0.0 && isfinite(av)) {
            s = fmt_maxint<FMT>() / av;
            sigma = av / fmt_maxint<FMT>();
        } else {
            s = 0.0;
            sigma = 0.0;
        }
    }
    if (bid == 0 && threadIdx.x == 0) *a.scale_out = sigma;

    for (int64_t g = g0; g < nunits; g += (int64_t)nblk * THREADS) {
        const int64_t row = g * RT;
        if (row + RT <= a.n) {
            double v[RT];
#pragma unroll
            for (int r = 0; r < RT; r += 2) {
                const double2 t = (g == g0) ? w0[r / 2] : *reinterpret_cast<const double2 *>(a.w + row + r);
                v[r] = t.x / hn; // IEEE division per element (reading Q8)
                v[r + 1] = t.y / hn;
            }
            if (a.v_out) {
                if constexpr (BJ) {
#pragma unroll
                    for (int q = 0; q < RT / 4; ++q) { // z = A_bb^-1 v_b for the blocks this thread holds
                        const double2 *iv = reinterpret_cast<const double2 *>(a.bj_inv + (row / 4 + q) * 16);
                        double2 m[8];
#pragma unroll
                        for (int i = 0; i < 8; ++i) m[i] = __ldg(iv + i); // written once per solve, before the cycle loop
                        double z[4];
#pragma unroll
                        for (int r = 0; r < 4; ++r)
                            z[r] = fma(m[2 * r + 1].y, v[4 * q + 3], fma(m[2 * r + 1].x, v[4 * q + 2], fma(m[2 * r].y, v[4 * q + 1], m[2 * r].x * v[4 * q])));
                        *reinterpret_cast<double2 *>(a.v_out + row + 4 * q) = make_double2(z[0], z[1]);
                        *reinterpret_cast<double2 *>(a.v_out + row + 4 * q + 2) = make_double2(z[2], z[3]);
                    }
                } else {
#pragma unroll
                    for (int r = 0; r < RT; r += 2)
                        *reinterpret_cast<double2 *>(a.v_out + row + r) = make_double2(v[r], v[r + 1]);
                }
            }
#pragma unroll
            for (int q = 0; q < GROUPS; ++q) {
                const double *vq = v + q * VEC;
                uint4 out;
                if constexpr (FMT == CBGMRES_FP64) {
                    out.x = (unsigned)__double2loint(vq[0]);
                    out.y = (unsigned)__double2hiint(vq[0]);
                    out.z = (unsigned)__double2loint(vq[1]);
                    out.w = (unsigned)__double2hiint(vq[1]);
                } else if constexpr (VEC == 4) {
                    out.x = enc_bits<FMT>(vq[0], s);
                    out.y = enc_bits<FMT>(vq[1], s);
                    out.z = enc_bits<FMT>(vq[2], s);
                    out.w = enc_bits<FMT>(vq[3], s);
                } else {
                    out.x = enc_bits<FMT>(vq[0], s) | (enc_bits<FMT>(vq[1], s) << 16);
                    out.y = enc_bits<FMT>(vq[2], s) | (enc_bits<FMT>(vq[3], s) << 16);
                    out.z = enc_bits<FMT>(vq[4], s) | (enc_bits<FMT>(vq[5], s) << 16);
                    out.w = enc_bits<FMT>(vq[6], s) | (enc_bits<FMT>(vq[7], s) << 16);
                }
                *reinterpret_cast<uint4 *>(reinterpret_cast<char *>(a.payload) + (g * GROUPS + q) * 16) = out;
            }
        } else { // the last, incomplete unit: row by row
            double v[RT];
            for (int r = 0; r < RT && row + r < a.n; ++r) {
                v[r] = a.w[row + r] / hn;
                if (a.v_out && !BJ) a.v_out[row + r] = v[r];
                if constexpr (FMT == CBGMRES_FP64) reinterpret_cast<double *>(a.payload)[row + r] = v[r];
                else if constexpr (F::BYTES == 4) reinterpret_cast<unsigned *>(a.payload)[row + r] = enc_bits<FMT>(v[r], s);
                else reinterpret_cast<unsigned short *>(a.payload)[row + r] = (unsigned short)enc_bits<FMT>(v[r], s);
            }
            if (BJ && a.v_out) { // the last block is completed by the identity: only its real rows and columns count
                for (int r = 0; r < RT && row + r < a.n; ++r) {
                    const int q = r / 4;
                    const double *iv = a.bj_inv + (row / 4 + q) * 16 + (r & 3) * 4;
                    double z = 0.0;
                    for (int c = 0; c < 4 && row + 4 * q + c < a.n; ++c) z = fma(iv[c], v[4 * q + c], z);
                    a.v_out[row + r] = z;
                }
            }
        }
    }
}

template <int FMT> static int launch_store_t(cudaStream_t s, const Scratch &sc, const StoreArgs &a)
{
    constexpr int THREADS = 256;
    using F = Fmt<FMT>;
    const int RT = (a.bj_inv && F::VEC < 4) ? 4 : F::VEC;
    const int64_t nunits = (a.n + RT - 1) / RT;
    int64_t grid = (nunits + THREADS - 1) / THREADS;
    const int64_t cap = (int64_t)kNumSMs * 8;
    if (grid > cap) grid = cap;
    if (grid < 1) grid = 1;
    if (a.has_cyc && a.mode == MODE_ORTH1) grid += 1; // + the control CTA (Givens update)
    if (a.bj_inv) launch_chain(sc, "store_kernel", store_kernel<FMT, THREADS, true>, dim3((unsigned)grid), dim3(THREADS), 0, s, a);
    else launch_chain(sc, "store_kernel", store_kernel<FMT, THREADS, false>, dim3((unsigned)grid), dim3(THREADS), 0, s, a);
    return 1;
}

int launch_store(cudaStream_t s, const Scratch &sc, int format, int64_t n, const double *w, const double *d_hn,
                 const double *d_amax, double hn_host, double amax_host, void *payload_col, double *scale_out,
                 double *v_out, int mode, int step, const CycleState *cyc, int *h_flag, const double *bj_inv)
{
    StoreArgs a{};
    a.w = w;
    a.d_hn = d_hn;
    a.d_amax = d_amax;
    a.hn_host = hn_host;
    a.amax_host = amax_host;
    a.payload = payload_col;
    a.scale_out = scale_out;
    a.v_out = v_out;
    a.n = n;
    a.ctl = sc.ctl;
    a.has_cyc = cyc != nullptr;
    if (cyc) a.cyc = *cyc;
    a.mode = mode;
    a.step = step;
    a.h_flag = h_flag;
    a.bj_inv = bj_inv;
    switch (format) {
    case CBGMRES_FP64: return launch_store_t<CBGMRES_FP64>(s, sc, a);
    case CBGMRES_FP32: return launch_store_t<CBGMRES_FP32>(s, sc, a);
    case CBGMRES_FP16: return launch_store_t<CBGMRES_FP16>(s, sc, a);
    case CBGMRES_INT32: return launch_store_t<CBGMRES_INT32>(s, sc, a);
    case CBGMRES_INT16: return launch_store_t<CBGMRES_INT16>(s, sc, a);
    default: return 0;
    }
}

// ---- decode hook: v_i = fp64(payload_i) * sigma ----------------------------------------------------
template <int FMT> __global__ void decode_kernel(const void *payload, const double *d_scale, double *v, int64_t n)
{
    using F = Fmt<FMT>;
    const double sigma = F::SCALED ? *d_scale : 1.0;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const double d = F::decode_one(payload, i);
        v[i] = F::SCALED ? d * sigma : d;
    }
}

int launch_decode(cudaStream_t s, int format, int64_t n, const void *payload, const double *d_scale, double *v)
{
    int64_t grid = (n + 255) / 256;
    if (grid > kNumSMs * 16) grid = kNumSMs * 16;
    if (grid < 1) grid = 1;
    switch (format) {
    case CBGMRES_FP64: decode_kernel<CBGMRES_FP64><<<(int)grid, 256, 0, s>>>(payload, d_scale, v, n); break;
    case CBGMRES_FP32: decode_kernel<CBGMRES_FP32><<<(int)grid, 256, 0, s>>>(payload, d_scale, v, n); break;
    case CBGMRES_FP16: decode_kernel<CBGMRES_FP16><<<(int)grid, 256, 0, s>>>(payload, d_scale, v, n); break;
    case CBGMRES_INT32: decode_kernel<CBGMRES_INT32><<<(int)grid, 256, 0, s>>>(payload, d_scale, v, n); break;
    case CBGMRES_INT16: decode_kernel<CBGMRES_INT16><<<(int)grid, 256, 0, s>>>(payload, d_scale, v, n); break;
    default: return 0;
    }
    return 1;
}

} // namespace cbg
