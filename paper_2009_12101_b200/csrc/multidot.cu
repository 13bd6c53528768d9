// multidot.cu -- S2: h_c = sum_i dec(V)[i,c] * w_i for c = 0..k-1  (Fig. 1 line 5 / line 8,
// PAPER.md:70, 76; the basis is read in its storage format and widened in registers).
//
// Shape: tall-skinny, n up to ~4e6 rows, k <= 512 vectors, each vector contiguous in HBM.
// Bound: HBM.  Algorithmic bytes per launch: k*n*B + 8n  (B = bytes per stored entry).
//
// Mapping.  Every WARP owns a contiguous segment of rows (n split evenly over all warps of a
// one-wave grid), stages its slice of w once in shared memory, and then streams the same rows of
// every vector, CT vectors at a time: per lane and iteration CT independent 128-bit loads are in
// flight, the w values are reused from registers across the CT vectors, and CT fp64 accumulators
// live in registers.  There is no CTA-wide barrier inside the streaming loop.  After each
// (segment, CT-vector tile) a transposing butterfly leaves one warp total per vector; totals are
// accumulated in the warp's private row of a shared-memory table, reduced across the CTA's warps
// once at the end, written as one row of `partials`, and the last CTA to finish adds the rows in
// a fixed order (deterministic, no fp64 atomics) and applies the per-vector scale.
#include "device_utils.cuh"

namespace cbg {

struct MultidotArgs {
    const void *V;
    int64_t ld;
    const double *scales;
    const double *w;
    int64_t n;
    int k;
    Ctl *ctl;
    double *partials;
    double *h_out;
    double *hs_out;
    int mode, step;
    int64_t seg_rows; // rows per warp segment (multiple of 64)
    int chunk_rows;   // rows of w staged per pass (multiple of 64)
    int kpad;         // k rounded up to CT
};

template <int FMT, int CT, bool FULL>
__device__ __forceinline__ void tile_pass(const char *__restrict__ tile_base, int64_t col_stride, int ncols,
                                          const double *__restrict__ wbuf, int ngroups_full, int lane,
                                          double (&acc)[CT])
{
    using F = Fmt<FMT>;
    for (int g = lane; g < ngroups_full; g += 32) {
        uint4 raw[CT];
#pragma unroll
        for (int c = 0; c < CT; ++c)
            if (FULL || c < ncols) raw[c] = ldg_stream128(tile_base + (int64_t)c * col_stride + (int64_t)g * 16);
        double wv[F::VEC];
#pragma unroll
        for (int r = 0; r < F::VEC; r += 2) {
            const double2 t = *reinterpret_cast<const double2 *>(wbuf + g * F::VEC + r);
            wv[r] = t.x;
            wv[r + 1] = t.y;
        }
#pragma unroll
        for (int c = 0; c < CT; ++c) {
            if (FULL || c < ncols) {
                double d[F::VEC];
                F::decode(raw[c], d);
#pragma unroll
                for (int r = 0; r < F::VEC; ++r) acc[c] = fma(d[r], wv[r], acc[c]);
            }
        }
    }
}

template <int FMT, int CT, int WARPS>
__global__ void __launch_bounds__(WARPS * 32) multidot_kernel(const MultidotArgs a)
{
    using F = Fmt<FMT>;
    if (a.mode != MODE_HOOK) {
        if (a.step > a.ctl->stop_after) return;
        if (a.mode == MODE_ORTH2 && !a.ctl->reorth_flag) return;
    }
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double *smem = reinterpret_cast<double *>(smem_raw);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    double *wbuf = smem + (size_t)warp * a.chunk_rows;
    double *hacc = smem + (size_t)WARPS * a.chunk_rows + (size_t)warp * a.kpad;
    for (int c = lane; c < a.kpad; c += 32) hacc[c] = 0.0;

    const int64_t gw = (int64_t)blockIdx.x * WARPS + warp;
    const int64_t r0 = gw * a.seg_rows;
    const int64_t r1 = min(a.n, r0 + a.seg_rows);
    const int64_t col_stride = a.ld * F::BYTES;
    const int ntiles = a.kpad / CT;

    for (int64_t c0 = r0; c0 < r1; c0 += a.chunk_rows) {
        const int cr = (int)min((int64_t)a.chunk_rows, r1 - c0);
        const int crp = (cr + F::VEC - 1) / F::VEC * F::VEC;
        __syncwarp();
        for (int i = lane; i < crp; i += 32) wbuf[i] = (i < cr) ? a.w[c0 + i] : 0.0;
        __syncwarp();
        const int ngroups = crp / F::VEC;
        // only the last group of the whole vector can straddle n (c0 and chunk_rows are multiples of 64)
        const bool ragged = (c0 + (int64_t)ngroups * F::VEC > a.n);
        const int ngroups_full = ragged ? ngroups - 1 : ngroups;
        const char *base = reinterpret_cast<const char *>(a.V) + c0 * F::BYTES;
        for (int t = 0; t < ntiles; ++t) {
            double acc[CT];
#pragma unroll
            for (int c = 0; c < CT; ++c) acc[c] = 0.0;
            const int ncols = min(CT, a.k - t * CT);
            const char *tile_base = base + (int64_t)t * CT * col_stride;
            if (ncols == CT) tile_pass<FMT, CT, true>(tile_base, col_stride, ncols, wbuf, ngroups_full, lane, acc);
            else tile_pass<FMT, CT, false>(tile_base, col_stride, ncols, wbuf, ngroups_full, lane, acc);
            if (ragged && lane == 0) { // element-wise tail: never reads a payload entry at or beyond n
                const int g = ngroups - 1;
                for (int c = 0; c < ncols; ++c) {
                    const char *col = reinterpret_cast<const char *>(a.V) + (int64_t)(t * CT + c) * col_stride;
                    for (int r = 0; r < F::VEC; ++r) {
                        const int64_t row = c0 + (int64_t)g * F::VEC + r;
                        if (row < a.n) acc[c] = fma(F::decode_one(col, row), wbuf[g * F::VEC + r], acc[c]);
                    }
                }
            }
            const double tot = butterfly_rec<CT, 16>(acc, lane);
            const int col = butterfly_col<CT>(lane);
            if (butterfly_owner<CT>(lane)) hacc[t * CT + col] += tot;
        }
    }
    __syncthreads();
    // CTA row of partials: fixed warp order
    const double *hall = smem + (size_t)WARPS * a.chunk_rows;
    for (int c = threadIdx.x; c < a.k; c += WARPS * 32) {
        double s = 0.0;
#pragma unroll
        for (int wq = 0; wq < WARPS; ++wq) s += hall[(size_t)wq * a.kpad + c];
        a.partials[(size_t)blockIdx.x * kLdp + c] = s;
    }
    if (!last_block_done(&a.ctl->tickets[0])) return;

    // ---- final stage (one CTA): rows of `partials` added in a fixed order -----------------------
    __shared__ double red[WARPS][33];
    const int nb = gridDim.x;
    for (int cg = 0; cg < a.k; cg += 32) {
        const int col = cg + lane;
        double s = 0.0;
        if (col < a.k)
            for (int b = warp; b < nb; b += WARPS) s += __ldcg(&a.partials[(size_t)b * kLdp + col]);
        red[warp][lane] = s;
        __syncthreads();
        if (warp == 0 && col < a.k) {
            double tot = 0.0;
#pragma unroll
            for (int wq = 0; wq < WARPS; ++wq) tot += red[wq][lane];
            const double sigma = F::SCALED ? a.scales[col] : 1.0;
            const double h = tot * sigma; // h_c = sigma_c * sum_i q_ic w_i
            if (a.mode == MODE_ORTH2) a.h_out[col] += h; // Fig. 1 l.9: h_{1:j,j} += u
            else a.h_out[col] = h;
            if (a.hs_out) a.hs_out[col] = h * sigma;     // coefficient of the raw payload in the update
        }
        __syncthreads();
    }
}

template <int FMT, int CT, int WARPS> static int launch_t(cudaStream_t s, const MultidotArgs &a0, int ctas_per_sm)
{
    using F = Fmt<FMT>;
    MultidotArgs a = a0;
    a.kpad = (a.k + CT - 1) / CT * CT;
    // one wave: ctas_per_sm CTAs on each of the 148 SMs, rows split evenly over all warps
    const int64_t min_seg = 512; // do not spread tiny vectors over the whole chip
    int grid = kNumSMs * ctas_per_sm;
    int64_t seg = (a.n + (int64_t)grid * WARPS - 1) / ((int64_t)grid * WARPS);
    seg = (seg + 63) / 64 * 64;
    if (seg < min_seg) seg = min_seg;
    grid = (int)((a.n + seg * WARPS - 1) / (seg * WARPS));
    if (grid < 1) grid = 1;
    a.seg_rows = seg;
    // shared memory: WARPS * (chunk_rows + kpad) doubles, at most ~220 KB / ctas_per_sm
    const size_t budget = (size_t)(220 * 1024) / ctas_per_sm;
    const size_t hacc_bytes = (size_t)WARPS * a.kpad * 8;
    int64_t chunk = ((int64_t)(budget - hacc_bytes) / (WARPS * 8)) / 64 * 64;
    if (chunk > seg) chunk = seg;
    if (chunk < 64) chunk = 64;
    a.chunk_rows = (int)chunk;
    const size_t smem = (size_t)WARPS * ((size_t)a.chunk_rows + a.kpad) * 8;
    static bool attr_set = false;
    if (!attr_set) {
        cudaFuncSetAttribute(multidot_kernel<FMT, CT, WARPS>, cudaFuncAttributeMaxDynamicSharedMemorySize, 222 * 1024); // + ~2 KB static <= 227 KB
        attr_set = true;
    }
    (void)sizeof(F);
    multidot_kernel<FMT, CT, WARPS><<<grid, WARPS * 32, smem, s>>>(a);
    return 1;
}

int launch_multidot(cudaStream_t s, const Scratch &sc, const BasisView &b, int64_t n, int k, const double *w,
                    double *h_out, double *hs_out, int mode, int step)
{
    if (k <= 0) return 0;
    MultidotArgs a{};
    a.V = b.V;
    a.ld = b.ld;
    a.scales = b.scales;
    a.w = w;
    a.n = n;
    a.k = k;
    a.ctl = sc.ctl;
    a.partials = sc.partials;
    a.h_out = h_out;
    a.hs_out = hs_out;
    a.mode = mode;
    a.step = step;
    constexpr int W = 8;
    switch (b.format) {
    case CBGMRES_FP64: return launch_t<CBGMRES_FP64, 8, W>(s, a, 2);
    case CBGMRES_FP32: return launch_t<CBGMRES_FP32, 8, W>(s, a, 2);
    case CBGMRES_FP16: return launch_t<CBGMRES_FP16, 8, W>(s, a, 2);
    case CBGMRES_INT32: return launch_t<CBGMRES_INT32, 8, W>(s, a, 2);
    case CBGMRES_INT16: return launch_t<CBGMRES_INT16, 8, W>(s, a, 2);
    default: return 0;
    }
}

} // namespace cbg
