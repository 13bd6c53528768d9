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

template <int FMT, int THREADS> __global__ void __launch_bounds__(THREADS) store_kernel(const StoreArgs a)
{
    using F = Fmt<FMT>;
    constexpr int VEC = F::VEC;
    pdl_wait();
    // A successor may fetch basis columns before ITS grid dependency resolves (orth.cu); inside a solve
    // the successor of a store is never a Gram-Schmidt pass, but after the k_compress / k_store hooks it
    // can be: there the successor is only released when this kernel has completed.
    if (a.mode != MODE_HOOK) pdl_launch_dependents();
    // this thread's first rows of w and the control words, fetched together (each is an L2 round trip)
    const bool has_ctl_cta0 = a.has_cyc && a.mode == MODE_ORTH1;
    const int bid0 = has_ctl_cta0 ? (int)blockIdx.x - 1 : (int)blockIdx.x;
    const int nblk = has_ctl_cta0 ? gridDim.x - 1 : gridDim.x;
    const int64_t ngroups = (a.n + VEC - 1) / VEC;
    const int64_t g0 = (int64_t)bid0 * THREADS + threadIdx.x;
    double2 w0[VEC / 2];
    if (bid0 >= 0 && g0 < ngroups && g0 * VEC + VEC <= a.n) {
#pragma unroll
        for (int r = 0; r < VEC; r += 2) w0[r / 2] = *reinterpret_cast<const double2 *>(a.w + g0 * VEC + r);
    }
    const int stop_after = (a.mode != MODE_HOOK) ? __ldcg(&a.ctl->stop_after) : 0;
    const double hn_dev = a.d_hn ? __ldcg(a.d_hn) : 0.0, amax_dev = a.d_amax ? __ldcg(a.d_amax) : 0.0;
    if (a.mode != MODE_HOOK && a.step > stop_after) return;
    const bool has_ctl_cta = a.has_cyc && a.mode == MODE_ORTH1;
    if (has_ctl_cta && blockIdx.x == 0) { // the control CTA: first to be scheduled, its serial chain overlaps the streaming
        givens_step(a);
        return;
    }
    const int bid = has_ctl_cta ? blockIdx.x - 1 : blockIdx.x;
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

    for (int64_t g = g0; g < ngroups; g += (int64_t)nblk * THREADS) {
        const int64_t row = g * VEC;
        if (row + VEC <= a.n) {
            double v[VEC];
#pragma unroll
            for (int r = 0; r < VEC; r += 2) {
                const double2 t = (g == g0) ? w0[r / 2] : *reinterpret_cast<const double2 *>(a.w + row + r);
                v[r] = t.x / hn; // IEEE division per element (reading Q8)
                v[r + 1] = t.y / hn;
            }
            if (a.v_out) {
#pragma unroll
                for (int r = 0; r < VEC; r += 2)
                    *reinterpret_cast<double2 *>(a.v_out + row + r) = make_double2(v[r], v[r + 1]);
            }
            uint4 out;
            if constexpr (FMT == CBGMRES_FP64) {
                out.x = (unsigned)__double2loint(v[0]);
                out.y = (unsigned)__double2hiint(v[0]);
                out.z = (unsigned)__double2loint(v[1]);
                out.w = (unsigned)__double2hiint(v[1]);
            } else if constexpr (VEC == 4) {
                out.x = enc_bits<FMT>(v[0], s);
                out.y = enc_bits<FMT>(v[1], s);
                out.z = enc_bits<FMT>(v[2], s);
                out.w = enc_bits<FMT>(v[3], s);
            } else {
                out.x = enc_bits<FMT>(v[0], s) | (enc_bits<FMT>(v[1], s) << 16);
                out.y = enc_bits<FMT>(v[2], s) | (enc_bits<FMT>(v[3], s) << 16);
                out.z = enc_bits<FMT>(v[4], s) | (enc_bits<FMT>(v[5], s) << 16);
                out.w = enc_bits<FMT>(v[6], s) | (enc_bits<FMT>(v[7], s) << 16);
            }
            *reinterpret_cast<uint4 *>(reinterpret_cast<char *>(a.payload) + g * 16) = out;
        } else {
            for (int r = 0; r < VEC && row + r < a.n; ++r) {
                const double v = a.w[row + r] / hn;
                if (a.v_out) a.v_out[row + r] = v;
                if constexpr (FMT == CBGMRES_FP64) reinterpret_cast<double *>(a.payload)[row + r] = v;
                else if constexpr (F::BYTES == 4) reinterpret_cast<unsigned *>(a.payload)[row + r] = enc_bits<FMT>(v, s);
                else reinterpret_cast<unsigned short *>(a.payload)[row + r] = (unsigned short)enc_bits<FMT>(v, s);
            }
        }
    }
}

template <int FMT> static int launch_store_t(cudaStream_t s, const StoreArgs &a)
{
    constexpr int THREADS = 256;
    using F = Fmt<FMT>;
    const int64_t ngroups = (a.n + F::VEC - 1) / F::VEC;
    int64_t grid = (ngroups + THREADS - 1) / THREADS;
    const int64_t cap = (int64_t)kNumSMs * 8;
    if (grid > cap) grid = cap;
    if (grid < 1) grid = 1;
    if (a.has_cyc && a.mode == MODE_ORTH1) grid += 1; // + the control CTA (Givens update)
    launch_chain(store_kernel<FMT, THREADS>, dim3((unsigned)grid), dim3(THREADS), 0, s, a);
    return 1;
}

int launch_store(cudaStream_t s, const Scratch &sc, int format, int64_t n, const double *w, const double *d_hn,
                 const double *d_amax, double hn_host, double amax_host, void *payload_col, double *scale_out,
                 double *v_out, int mode, int step, const CycleState *cyc, int *h_flag)
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
    switch (format) {
    case CBGMRES_FP64: return launch_store_t<CBGMRES_FP64>(s, a);
    case CBGMRES_FP32: return launch_store_t<CBGMRES_FP32>(s, a);
    case CBGMRES_FP16: return launch_store_t<CBGMRES_FP16>(s, a);
    case CBGMRES_INT32: return launch_store_t<CBGMRES_INT32>(s, a);
    case CBGMRES_INT16: return launch_store_t<CBGMRES_INT16>(s, a);
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
