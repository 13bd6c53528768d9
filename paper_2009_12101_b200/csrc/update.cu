// update.cu -- S3: w_i <- w_i - sum_c dec(V)[i,c] * h_c, returning ||w||_2 and ||w||_inf of the new
// w from the same pass (Fig. 1 lines 5-6 and 8-10; "both norms can be computed
// simultaneously").  The same kernel applies the solution update x += V_k y of
// Fig. 1 line 17 with coefficients -sigma_c y_c.
//
// Bound: HBM.  Algorithmic bytes per launch: k*n*B + 16n.
//
// Mapping.  One thread owns VEC = 16/B consecutive rows (one 128-bit payload word per vector),
// keeps their VEC fp64 accumulators in registers, and walks the k vectors U at a time so that U
// independent 128-bit loads are in flight per thread.  The coefficients (already multiplied by
// the fixed-point scale sigma_c, negated) sit in shared memory and are broadcast.  Norm partials
// go through warp shuffles, one shared-memory stage and a last-block-done final stage.
#include "device_utils.cuh"

namespace cbg {

struct UpdateArgs {
    const void *V;
    int64_t ld;
    const double *hs; // [k] sigma_c * h_c
    const int *d_k;   // if non-null, the vector count is read from the device (cycle end)
    double *w;
    int64_t n;
    int k;
    Ctl *ctl;
    double *npart;
    int mode, step;
};

template <int FMT, int U, int THREADS>
__global__ void __launch_bounds__(THREADS) update_kernel(const UpdateArgs a)
{
    using F = Fmt<FMT>;
    constexpr int VEC = F::VEC;
    Ctl *ctl = a.ctl;
    if (a.mode == MODE_ORTH1 || a.mode == MODE_ORTH2) {
        if (a.step > ctl->stop_after) return;
        if (a.mode == MODE_ORTH2 && !ctl->reorth_flag) return;
    }
    const int k = a.d_k ? *a.d_k : a.k;
    if (a.mode == MODE_XUPDATE && k <= 0) return;

    extern __shared__ __align__(16) unsigned char smem_raw[];
    double *nhs = reinterpret_cast<double *>(smem_raw); // -hs[c], zero padded to a multiple of U
    const int kpad = (k + U - 1) / U * U;
    for (int c = threadIdx.x; c < kpad; c += THREADS) nhs[c] = (c < k) ? -a.hs[c] : 0.0;
    __syncthreads();

    const int64_t col_stride = a.ld * F::BYTES;
    const int64_t ngroups = (a.n + VEC - 1) / VEC;
    const int kfull = k / U * U;
    double ss = 0.0, am = 0.0;

    for (int64_t g = (int64_t)blockIdx.x * THREADS + threadIdx.x; g < ngroups; g += (int64_t)gridDim.x * THREADS) {
        const int64_t row = g * VEC;
        double acc[VEC];
        if (row + VEC <= a.n) {
#pragma unroll
            for (int r = 0; r < VEC; r += 2) {
                const double2 t = *reinterpret_cast<const double2 *>(a.w + row + r);
                acc[r] = t.x;
                acc[r + 1] = t.y;
            }
            const char *p = reinterpret_cast<const char *>(a.V) + g * 16;
            int c = 0;
            for (; c < kfull; c += U) {
                uint4 raw[U];
#pragma unroll
                for (int u = 0; u < U; ++u) raw[u] = ldg_stream128(p + (int64_t)(c + u) * col_stride);
#pragma unroll
                for (int u = 0; u < U; ++u) {
                    double d[VEC];
                    F::decode(raw[u], d);
                    const double coef = nhs[c + u];
#pragma unroll
                    for (int r = 0; r < VEC; ++r) acc[r] = fma(d[r], coef, acc[r]);
                }
            }
            if (c < k) {
                uint4 raw[U];
#pragma unroll
                for (int u = 0; u < U; ++u)
                    if (c + u < k) raw[u] = ldg_stream128(p + (int64_t)(c + u) * col_stride);
#pragma unroll
                for (int u = 0; u < U; ++u) {
                    if (c + u < k) {
                        double d[VEC];
                        F::decode(raw[u], d);
                        const double coef = nhs[c + u];
#pragma unroll
                        for (int r = 0; r < VEC; ++r) acc[r] = fma(d[r], coef, acc[r]);
                    }
                }
            }
#pragma unroll
            for (int r = 0; r < VEC; r += 2)
                *reinterpret_cast<double2 *>(a.w + row + r) = make_double2(acc[r], acc[r + 1]);
#pragma unroll
            for (int r = 0; r < VEC; ++r) {
                ss = fma(acc[r], acc[r], ss);
                am = fmax(am, fabs(acc[r]));
            }
        } else { // the one ragged group at the end of the vector: element-wise, never reads beyond n
            for (int r = 0; r < VEC && row + r < a.n; ++r) {
                double s = a.w[row + r];
                for (int c = 0; c < k; ++c) {
                    const char *col = reinterpret_cast<const char *>(a.V) + (int64_t)c * col_stride;
                    s = fma(F::decode_one(col, row + r), nhs[c], s);
                }
                a.w[row + r] = s;
                ss = fma(s, s, ss);
                am = fmax(am, fabs(s));
            }
        }
    }
    if (a.mode == MODE_XUPDATE) return; // no norms needed for x

    // ---- norms: warp -> CTA -> last CTA, fixed order ----------------------------------------------
    __shared__ double s_ss[THREADS / 32], s_am[THREADS / 32];
    ss = warp_sum(ss);
    am = warp_max(am);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (lane == 0) {
        s_ss[warp] = ss;
        s_am[warp] = am;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0, m = 0.0;
        for (int i = 0; i < THREADS / 32; ++i) {
            t += s_ss[i];
            m = fmax(m, s_am[i]);
        }
        a.npart[blockIdx.x] = t;
        a.npart[kMaxGrid + blockIdx.x] = m;
    }
    if (!last_block_done(&ctl->tickets[1])) return;
    if (warp == 0) {
        double t = 0.0, m = 0.0;
        for (int b = lane; b < (int)gridDim.x; b += 32) {
            t += __ldcg(&a.npart[b]);
            m = fmax(m, __ldcg(&a.npart[kMaxGrid + b]));
        }
        t = warp_sum(t);
        m = warp_max(m);
        if (lane == 0) {
            const double hn = sqrt(t);
            if (a.mode == MODE_HOOK) {
                ctl->hook_nrm2 = hn;
                ctl->hook_amax = m;
            } else if (a.mode == MODE_ORTH1) {
                // Fig. 1 l.6-7: h_{j+1,j} := ||w||_2 ; re-orthogonalise iff h_{j+1,j} < eta * omega
                ctl->hn = hn;
                ctl->amax = m;
                ctl->breakdown = (hn == 0.0);
                ctl->reorth_flag = (ctl->reorth_mode == CBGMRES_REORTH_ALWAYS) ||
                                   (ctl->reorth_mode == CBGMRES_REORTH_COND && hn < ctl->eta * ctl->omega);
                ctl->reorth_log[a.step] = (unsigned char)ctl->reorth_flag;
                if (!isfinite(hn)) ctl->nonfinite = 1;
            } else { // MODE_ORTH2, Fig. 1 l.10-12: new norm; breakdown if it again fell below eta * (norm before)
                const double omega1 = ctl->hn;
                ctl->hn = hn;
                ctl->amax = m;
                ctl->reorth_count += 1;
                ctl->breakdown = (hn == 0.0) || (hn < ctl->eta * omega1);
                if (!isfinite(hn)) ctl->nonfinite = 1;
            }
        }
    }
}

template <int FMT, int U> static int launch_t(cudaStream_t s, const UpdateArgs &a, int kmax)
{
    constexpr int THREADS = 256;
    using F = Fmt<FMT>;
    const int64_t ngroups = (a.n + F::VEC - 1) / F::VEC;
    int64_t grid = (ngroups + THREADS - 1) / THREADS;
    const int64_t cap = (int64_t)kNumSMs * 8;
    if (grid > cap) grid = cap;
    if (grid < 1) grid = 1;
    const size_t smem = (size_t)((kmax + U - 1) / U * U) * 8;
    update_kernel<FMT, U, THREADS><<<(int)grid, THREADS, smem, s>>>(a);
    return 1;
}

int launch_update(cudaStream_t s, const Scratch &sc, const BasisView &b, int64_t n, int k, const int *d_k,
                  const double *hs, double *w, int mode, int step)
{
    if (k <= 0 && !d_k) return 0;
    UpdateArgs a{};
    a.V = b.V;
    a.ld = b.ld;
    a.hs = hs;
    a.d_k = d_k;
    a.w = w;
    a.n = n;
    a.k = k;
    a.ctl = sc.ctl;
    a.npart = sc.npart;
    a.mode = mode;
    a.step = step;
    const int kmax = d_k ? kMaxRestart : k;
    switch (b.format) {
    case CBGMRES_FP64: return launch_t<CBGMRES_FP64, 8>(s, a, kmax);
    case CBGMRES_FP32: return launch_t<CBGMRES_FP32, 8>(s, a, kmax);
    case CBGMRES_FP16: return launch_t<CBGMRES_FP16, 8>(s, a, kmax);
    case CBGMRES_INT32: return launch_t<CBGMRES_INT32, 8>(s, a, kmax);
    case CBGMRES_INT16: return launch_t<CBGMRES_INT16, 8>(s, a, kmax);
    default: return 0;
    }
}

} // namespace cbg
