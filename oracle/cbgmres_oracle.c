/*
 * cbgmres_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, obviously-correct CPU restatement of compressed-basis GMRES (CB-GMRES),
 * written from /root/reference/PAPER.md (arXiv 2009.12101) only.  All arithmetic is IEEE
 * binary64; the Krylov basis is really encoded to the storage format
 * on store and decoded on every read.  Nothing here is shared with,
 * imported by, or derived from the CUDA path under paper_2009_12101_b200/.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may call it.
 *
 * Build: gcc -O2 -fopenmp -ffp-contract=off -fno-fast-math -shared -fPIC (see oracle/build.py).
 * -ffp-contract=off: no FMA contraction, so every line below rounds exactly as written.
 *
 * Pins (tests/test_oracle_*.py, all `-m "not gpu"`): see the table in DESIGN.md §"Oracle pins".
 *   - codecs: numpy astype (library), exhaustive fp16 round trip + midpoint ties, closed forms and
 *     exact rational brute force for the fixed-point formats;
 *   - SpMV: scipy.sparse, row sums;
 *   - GMRES (fp64 storage): numpy.linalg.solve on tiny systems, <= n-step convergence, Arnoldi
 *     relation, basis orthogonality, recurrence == explicit residual, scipy.sparse.linalg.gmres;
 *   - GMRES (compressed storage): mixed Arnoldi relation, |V^| <= 1, explicit residual <= tol.
 *   - right preconditioner M = diag(A) (orc_gmres_m): numpy.linalg.solve on badly scaled systems,
 *     residual history equal to plain GMRES on the explicitly formed A D^-1, constant-diagonal no-op.
 *   - right preconditioner M = blockdiag_4(A) (orc_block_jacobi4, orc_gmres_p): every inverted
 *     block against numpy.linalg.inv, numpy.linalg.solve on dense systems, residual history equal to plain
 *     GMRES on the explicitly formed A M^-1, reduction to scalar Jacobi for block-diagonal-free matrices.
 *   - Fig. 1 l.12 (second-pass breakdown, reading Q4): a matrix with an exact invariant subspace and a
 *     quantised basis, where the clause hn < eta * omega1 -- and not hn == 0 -- ends the cycle.
 *   - PARITY UNPINNED: exact iteration counts of the compressed formats on the synthetic configs
 *     (the paper prints no value for any of them; only Table 2's qualitative ratios apply).
 *
 * Storage format codes: 0 <float64>, 1 <float32>, 2 <float16>,
 * 3 <int32> fixed point, 4 <int16> fixed point.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

enum { ORC_F64 = 0, ORC_F32 = 1, ORC_F16 = 2, ORC_I32 = 3, ORC_I16 = 4 };
enum { ORC_REORTH_NEVER = 0, ORC_REORTH_COND = 1, ORC_REORTH_ALWAYS = 2 };

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* Thread count of the following calls (t <= 0: leave as is).  It only changes the order in which
 * dot() adds its per-thread block sums, i.e. the last bits of each inner product: tests use it to
 * measure how far the oracle's OWN iteration counts move under rounding-level perturbations
 * (reading Q11). */
void orc_set_num_threads(int t)
{
#ifdef _OPENMP
    if (t > 0) omp_set_num_threads(t);
#else
    (void)t;
#endif
}

int64_t orc_format_bytes(int fmt)
{
    switch (fmt) {
    case ORC_F64: return 8;
    case ORC_F32: return 4;
    case ORC_F16: return 2;
    case ORC_I32: return 4;
    case ORC_I16: return 2;
    default: return -1;
    }
}

/* ------------------------------------------------------------------------------------------
 * Codecs (readings Q6, Q7 in DESIGN.md).
 * ---------------------------------------------------------------------------------------- */

/* IEEE binary64 -> binary16 in ONE rounding, round-to-nearest-even, gradual underflow
 * (reading Q7).  Written out on the bit patterns so that no intermediate binary32 exists. */
static uint16_t f64_to_f16_bits(double x)
{
    uint64_t u;
    memcpy(&u, &x, 8);
    uint16_t sign = (uint16_t)((u >> 48) & 0x8000u);
    int e = (int)((u >> 52) & 0x7FF);
    uint64_t m = u & 0xFFFFFFFFFFFFFull;
    if (e == 0x7FF) return (uint16_t)(sign | 0x7C00u | (m ? 0x200u : 0u)); /* inf / nan */
    if (e == 0) return sign;              /* |x| < 2^-1022: far below half's 2^-25 tie point */
    int E = e - 1023;                     /* x = S * 2^(E-52), S = 2^52 + m                  */
    if (E > 15) return (uint16_t)(sign | 0x7C00u);
    /* normal half (E >= -14) keeps 10 fraction bits -> drop 42; subnormal half has the fixed
     * unit 2^-24 -> drop 42 + (-14 - E). */
    int shift = (E >= -14) ? 42 : 42 + (-14 - E);
    if (shift > 63) return sign;          /* S < 2^53 <= half a unit */
    uint64_t S = (1ull << 52) | m;
    uint64_t q = S >> shift;
    uint64_t rem = S & ((1ull << shift) - 1);
    uint64_t half = 1ull << (shift - 1);
    if (rem > half || (rem == half && (q & 1))) q++;
    /* normal: q in [2^10, 2^11]; adding it to the (E+14) exponent field carries correctly,
     * including the carry into infinity at E = 15.  subnormal: q in [0, 2^10]. */
    uint16_t bits = (E >= -14) ? (uint16_t)(((unsigned)(E + 14) << 10) + q) : (uint16_t)q;
    return (uint16_t)(sign | bits);
}

/* binary16 -> binary64 is exact.  Normal halves: same sign, exponent re-biased (e - 15 + 1023), the
 * 10 fraction bits become the top 10 of the 52.  Subnormal halves: m * 2^-24. */
static double f16_bits_to_f64(uint16_t h)
{
    const uint64_t s = (uint64_t)(h >> 15) & 1u;
    const int e = (h >> 10) & 0x1F;
    const uint64_t m = h & 0x3FFu;
    double v;
    if (e == 0) {
        v = (double)m * 0x1p-24;
        return s ? -v : v;
    }
    if (e == 31) return m ? NAN : (s ? -INFINITY : INFINITY);
    const uint64_t bits = (s << 63) | ((uint64_t)(e - 15 + 1023) << 52) | (m << 42);
    memcpy(&v, &bits, 8);
    return v;
}

/* enc: fp64[n] -> (payload, sigma).  sigma is 1 for the floating-point formats.
 * Fixed point: sigma_j = (||w||inf/||w||2)/max_int for the un-normalised w,
 * i.e. sigma = ||v||inf / max_int for the unit vector v = w/||w||2 that is passed in here; the
 * stored integer is v_i / sigma rounded to nearest-even and clamped to +-max_int (reading Q6). */
int orc_enc(int fmt, int64_t n, const double *v, void *payload, double *sigma)
{
    int64_t i;
    switch (fmt) {
    case ORC_F64:
        memcpy(payload, v, (size_t)n * 8);
        *sigma = 1.0;
        return 0;
    case ORC_F32: {
        float *p = (float *)payload;
#pragma omp parallel for schedule(static)
        for (i = 0; i < n; i++) p[i] = (float)v[i]; /* cvtsd2ss: RNE, gradual underflow */
        *sigma = 1.0;
        return 0;
    }
    case ORC_F16: {
        uint16_t *p = (uint16_t *)payload;
#pragma omp parallel for schedule(static)
        for (i = 0; i < n; i++) p[i] = f64_to_f16_bits(v[i]);
        *sigma = 1.0;
        return 0;
    }
    case ORC_I32:
    case ORC_I16: {
        const double maxint = (fmt == ORC_I32) ? 2147483647.0 : 32767.0;
        double a = 0.0;
        for (i = 0; i < n; i++) {
            double t = fabs(v[i]);
            if (t > a) a = t;
        }
        if (!(a > 0.0) || !isfinite(a)) { /* zero (or non-finite) vector: nothing to scale */
            memset(payload, 0, (size_t)n * (size_t)orc_format_bytes(fmt));
            *sigma = 0.0;
            return 0;
        }
        double s = maxint / a;
#pragma omp parallel for schedule(static)
        for (i = 0; i < n; i++) {
            double q = nearbyint(v[i] * s); /* default rounding mode: to nearest, ties to even */
            if (q > maxint) q = maxint;
            if (q < -maxint) q = -maxint;
            if (fmt == ORC_I32) ((int32_t *)payload)[i] = (int32_t)q;
            else ((int16_t *)payload)[i] = (int16_t)q;
        }
        *sigma = a / maxint;
        return 0;
    }
    default:
        return -1;
    }
}

/* dec: (payload, sigma) -> fp64[n]; "any subsequent access ... implies an intrinsic
 * post-multiplication by a diagonal matrix" of the scaling factors. */
int orc_dec(int fmt, int64_t n, const void *payload, double sigma, double *out)
{
    int64_t i;
    switch (fmt) {
    case ORC_F64: memcpy(out, payload, (size_t)n * 8); return 0;
    case ORC_F32:
#pragma omp parallel for schedule(static)
        for (i = 0; i < n; i++) out[i] = (double)((const float *)payload)[i];
        return 0;
    case ORC_F16:
#pragma omp parallel for schedule(static)
        for (i = 0; i < n; i++) out[i] = f16_bits_to_f64(((const uint16_t *)payload)[i]);
        return 0;
    case ORC_I32:
#pragma omp parallel for schedule(static)
        for (i = 0; i < n; i++) out[i] = (double)((const int32_t *)payload)[i] * sigma;
        return 0;
    case ORC_I16:
#pragma omp parallel for schedule(static)
        for (i = 0; i < n; i++) out[i] = (double)((const int16_t *)payload)[i] * sigma;
        return 0;
    default: return -1;
    }
}

/* ------------------------------------------------------------------------------------------
 * Plain fp64 building blocks.
 * ---------------------------------------------------------------------------------------- */

/* y = A x, CSR, fp64 values + int32 indices. */
void orc_spmv(int64_t n, const int32_t *rp, const int32_t *ci, const double *va, const double *x, double *y)
{
    int64_t i;
#pragma omp parallel for schedule(static)
    for (i = 0; i < n; i++) {
        double s = 0.0;
        for (int32_t p = rp[i]; p < rp[i + 1]; p++) s += va[p] * x[ci[p]];
        y[i] = s;
    }
}

/* Dot product.  Each thread sums one contiguous block of the index range (static schedule) and
 * the per-thread sums are added in thread order, so the result is reproducible run to run for a
 * fixed thread count (an OpenMP reduction clause leaves the combination order unspecified). */
#define ORC_MAX_THREADS 1024
static double dot(int64_t n, const double *a, const double *b)
{
    double part[ORC_MAX_THREADS];
    int nt = 1;
#pragma omp parallel
    {
#ifdef _OPENMP
        const int t = omp_get_thread_num(), T = omp_get_num_threads();
#else
        const int t = 0, T = 1;
#endif
        const int64_t lo = n * t / T, hi = n * (t + 1) / T;
        double s = 0.0;
        for (int64_t i = lo; i < hi; i++) s += a[i] * b[i];
        part[t] = s;
        if (t == 0) nt = T;
    }
    double s = 0.0;
    for (int t = 0; t < nt; t++) s += part[t];
    return s;
}

static double nrm2(int64_t n, const double *a) { return sqrt(dot(n, a, a)); }

static double amax(int64_t n, const double *a)
{
    double m = 0.0;
    int64_t i;
#pragma omp parallel for schedule(static) reduction(max : m)
    for (i = 0; i < n; i++) {
        double t = fabs(a[i]);
        if (t > m) m = t;
    }
    return m;
}

/* y += alpha * x */
static void axpy(int64_t n, double alpha, const double *x, double *y)
{
    int64_t i;
#pragma omp parallel for schedule(static)
    for (i = 0; i < n; i++) y[i] += alpha * x[i];
}

double orc_nrm2(int64_t n, const double *a) { return nrm2(n, a); }
double orc_amax(int64_t n, const double *a) { return amax(n, a); }

/* ------------------------------------------------------------------------------------------
 * Per-kernel references with extended accumulation (x87 long double, 64-bit significand), so
 * that the 1e-12 parity budget belongs to the GPU kernels.
 * V is k stored vectors, vector c at payload + c*ld*bytes(fmt); sigma[c] per vector.
 * ---------------------------------------------------------------------------------------- */
static double dec_one(int fmt, const void *payload, int64_t i, double sigma)
{
    switch (fmt) {
    case ORC_F64: return ((const double *)payload)[i];
    case ORC_F32: return (double)((const float *)payload)[i];
    case ORC_F16: return f16_bits_to_f64(((const uint16_t *)payload)[i]);
    case ORC_I32: return (double)((const int32_t *)payload)[i] * sigma;
    default: return (double)((const int16_t *)payload)[i] * sigma;
    }
}

/* h_c = sum_i dec(V)[i,c] * w_i   (Fig. 1 line 5) */
void orc_ref_multidot(int fmt, int64_t n, int64_t ld, int k, const void *V, const double *sigma, const double *w,
                      double *h)
{
    int c;
    int64_t B = orc_format_bytes(fmt);
#pragma omp parallel for schedule(dynamic, 1)
    for (c = 0; c < k; c++) {
        const char *col = (const char *)V + (size_t)c * (size_t)ld * (size_t)B;
        long double s = 0.0L;
        for (int64_t i = 0; i < n; i++) s += (long double)dec_one(fmt, col, i, sigma[c]) * (long double)w[i];
        h[c] = (double)s;
    }
}

/* w_i <- w_i - sum_c dec(V)[i,c] * h_c ; returns sum w_i^2 and max |w_i| of the new w
 * (Fig. 1 lines 5-6; both norms together). */
void orc_ref_update(int fmt, int64_t n, int64_t ld, int k, const void *V, const double *sigma, const double *h,
                    double *w, double *nrm2sq, double *amax_out)
{
    int64_t B = orc_format_bytes(fmt);
    long double ss = 0.0L;
    double mx = 0.0;
    int64_t i;
#pragma omp parallel for schedule(static) reduction(+ : ss) reduction(max : mx)
    for (i = 0; i < n; i++) {
        long double s = (long double)w[i];
        for (int c = 0; c < k; c++) {
            const char *col = (const char *)V + (size_t)c * (size_t)ld * (size_t)B;
            s -= (long double)dec_one(fmt, col, i, sigma[c]) * (long double)h[c];
        }
        w[i] = (double)s;
        ss += (long double)w[i] * (long double)w[i];
        if (fabs(w[i]) > mx) mx = fabs(w[i]);
    }
    *nrm2sq = (double)ss;
    *amax_out = mx;
}

/* y = A x with long double row sums; also rowabs_i = sum_k |a_ik x_k| (the error scale). */
void orc_ref_spmv(int64_t n, const int32_t *rp, const int32_t *ci, const double *va, const double *x, double *y,
                  double *rowabs)
{
    int64_t i;
#pragma omp parallel for schedule(static)
    for (i = 0; i < n; i++) {
        long double s = 0.0L, a = 0.0L;
        for (int32_t p = rp[i]; p < rp[i + 1]; p++) {
            long double t = (long double)va[p] * (long double)x[ci[p]];
            s += t;
            a += fabsl(t);
        }
        y[i] = (double)s;
        if (rowabs) rowabs[i] = (double)a;
    }
}

/* ------------------------------------------------------------------------------------------
 * Restarted CB-GMRES, step by step in the order and notation of Fig. 1, with
 * M = I (reading Q12), the explicit residual at every restart and the
 * confirmation of convergence by the explicit residual.  Line numbers "l.N" are
 * those the paper's prose uses (reconstruction Q2 in DESIGN.md).
 * ---------------------------------------------------------------------------------------- */
typedef struct {
    int32_t restart;   /* m */
    int32_t max_iters; /* bound on the total number of Arnoldi steps */
    int32_t format;    /* storage format of the basis */
    int32_t reorth;    /* ORC_REORTH_* */
    double rel_tol;    /* tau: stop when ||b - A x||_2 <= tau * ||b||_2 */
    double eta;        /* re-orthogonalisation threshold (reading Q3: 1/sqrt 2) */
} orc_params;

typedef struct {
    int32_t iters;        /* Arnoldi steps, summed over cycles */
    int32_t restarts;     /* restart cycles started */
    int32_t reorth_count; /* steps on which l.7-11 ran */
    int32_t breakdown;    /* 1 if the last cycle left through l.12 */
    int32_t converged;    /* 1 iff the explicit residual met the threshold */
    int32_t pad_;
    double rel_res_recurrence; /* |g_{k+1}| / ||b|| at the end of the last cycle */
    double rel_res_true;       /* last explicit ||b - A x|| / ||b|| */
    double b_norm;
} orc_result;

typedef struct {      /* optional capture of one restart cycle, for the pins */
    int32_t cycle;    /* in : 0-based index of the cycle to capture */
    int32_t k;        /* out: Arnoldi steps done in that cycle */
    double beta;      /* out: ||r_0|| of that cycle */
    double *Vhat;     /* out: (m+1) x n, row c = dec(stored vector c) */
    double *Vfp64;    /* out: (m+1) x n, row c = the fp64 vector before compression */
    double *Hbar;     /* out: (m+1) x m, column-major, the UNROTATED Hessenberg matrix (l.16) */
    double *y;        /* out: m, the minimiser of l.17 */
    double *g;        /* out: m+1, rotated right-hand side at the end of the cycle */
    int32_t *reorth_log; /* out: m, 1 where l.7 fired at that step of the cycle (may be NULL) */
    double *omega;    /* out: m, omega = ||A M^-1 v_j||_2 of l.4 at that step (may be NULL) */
} orc_capture;

/* Scalar Jacobi preconditioner M = diag(A) ("a scalar Jacobi preconditioner" in every
 * experiment): d_i = a_ii; a missing or zero diagonal entry leaves that row unscaled (d_i = 1). */
void orc_jacobi_diag(int64_t n, const int32_t *rp, const int32_t *ci, const double *va, double *d)
{
    for (int64_t i = 0; i < n; i++) {
        d[i] = 1.0;
        for (int32_t p = rp[i]; p < rp[i + 1]; p++)
            if (ci[p] == i && va[p] != 0.0) d[i] = va[p];
    }
}

/* Block-Jacobi preconditioner with blocks of size 4 (section 6.5: "a block-Jacobi
 * preconditioning scheme with block-size 4"), fixed (fp64) precision: M = blockdiag(A_00, A_11, ...),
 * A_bb = rows and columns 4b .. 4b+3 of A (entries absent from the pattern are 0; the last block has
 * n mod 4 rows when 4 does not divide n and is completed by the identity).  Each block is inverted
 * by plain Gaussian elimination with partial pivoting on [A_bb | I] (Gauss-Jordan); a block that turns
 * out singular (a zero pivot column) is replaced by the identity, as the scalar variant leaves a row
 * with a zero diagonal unscaled.  inv[16 b + 4 r + c] = (A_bb^-1)_{rc}. */
void orc_block_jacobi4(int64_t n, const int32_t *rp, const int32_t *ci, const double *va, double *inv)
{
    const int64_t nb = (n + 3) / 4;
    for (int64_t b = 0; b < nb; b++) {
        double a[4][8];
        for (int r = 0; r < 4; r++)
            for (int c = 0; c < 8; c++) a[r][c] = (c == r + 4) ? 1.0 : 0.0;
        for (int r = 0; r < 4; r++) {
            const int64_t i = 4 * b + r;
            if (i >= n) { a[r][r] = 1.0; continue; } /* ragged last block: identity */
            for (int32_t p = rp[i]; p < rp[i + 1]; p++) {
                const int64_t c = (int64_t)ci[p] - 4 * b;
                if (c >= 0 && c < 4) a[r][c] += va[p];
            }
        }
        int singular = 0;
        for (int k = 0; k < 4 && !singular; k++) {
            int piv = k;
            for (int r = k + 1; r < 4; r++)
                if (fabs(a[r][k]) > fabs(a[piv][k])) piv = r;
            if (a[piv][k] == 0.0 || !isfinite(a[piv][k])) { singular = 1; break; }
            if (piv != k)
                for (int c = 0; c < 8; c++) { double t = a[k][c]; a[k][c] = a[piv][c]; a[piv][c] = t; }
            const double d = a[k][k];
            for (int c = 0; c < 8; c++) a[k][c] = a[k][c] / d;
            for (int r = 0; r < 4; r++) {
                if (r == k) continue;
                const double f = a[r][k];
                if (f == 0.0) continue;
                for (int c = 0; c < 8; c++) a[r][c] = a[r][c] - f * a[k][c];
            }
        }
        for (int r = 0; r < 4; r++)
            for (int c = 0; c < 4; c++) inv[16 * b + 4 * r + c] = singular ? (r == c ? 1.0 : 0.0) : a[r][c + 4];
    }
}

/* z := M^-1 v for the preconditioner kinds below (l.3 and l.17 of Fig. 1). */
enum { ORC_PRECOND_NONE = 0, ORC_PRECOND_JACOBI = 1, ORC_PRECOND_BLOCK_JACOBI4 = 2 };
static void apply_minv(int kind, const double *pdata, int64_t n, const double *v, double *z)
{
    int64_t i;
    if (kind == ORC_PRECOND_JACOBI) { /* pdata = d, d_i = a_ii */
#pragma omp parallel for schedule(static)
        for (i = 0; i < n; i++) z[i] = v[i] / pdata[i];
    } else if (kind == ORC_PRECOND_BLOCK_JACOBI4) { /* pdata = the inverted blocks of orc_block_jacobi4 */
        const int64_t nb = (n + 3) / 4;
#pragma omp parallel for schedule(static)
        for (i = 0; i < nb; i++) {
            for (int r = 0; r < 4; r++) {
                if (4 * i + r >= n) break;
                double s = 0.0;
                for (int c = 0; c < 4; c++)
                    if (4 * i + c < n) s += pdata[16 * i + 4 * r + c] * v[4 * i + c];
                z[4 * i + r] = s;
            }
        }
    } else {
        memcpy(z, v, (size_t)n * 8);
    }
}
void orc_apply_minv(int kind, const double *pdata, int64_t n, const double *v, double *z) { apply_minv(kind, pdata, n, v, z); }

/* Fig. 1 with a right preconditioner M (kind = ORC_PRECOND_*, pdata as apply_minv reads it; kind 0: M = I):
 * l.3 "w := A (M^-1 v_j)" and l.17 "x_m := x_0 + M^-1 (V_m y_m)"; the residual
 * of l.1 and the stopping test are those of the ORIGINAL system A x = b (right preconditioning
 * leaves the residual unchanged). */
int orc_gmres_p(int64_t n, const int32_t *rp, const int32_t *ci, const double *va, int kind, const double *pdata,
                const double *b, double *x, const orc_params *prm, orc_result *res, double *rec_hist,
                int32_t rec_hist_cap, double *expl_hist, int32_t expl_hist_cap, orc_capture *cap);

/* M = diag(mdiag) (mdiag == NULL: M = I). */
int orc_gmres_m(int64_t n, const int32_t *rp, const int32_t *ci, const double *va, const double *mdiag,
                const double *b, double *x, const orc_params *prm, orc_result *res, double *rec_hist,
                int32_t rec_hist_cap, double *expl_hist, int32_t expl_hist_cap, orc_capture *cap)
{
    return orc_gmres_p(n, rp, ci, va, mdiag ? ORC_PRECOND_JACOBI : ORC_PRECOND_NONE, mdiag, b, x, prm, res, rec_hist,
                       rec_hist_cap, expl_hist, expl_hist_cap, cap);
}

int orc_gmres(int64_t n, const int32_t *rp, const int32_t *ci, const double *va, const double *b, double *x,
              const orc_params *prm, orc_result *res, double *rec_hist, int32_t rec_hist_cap, double *expl_hist,
              int32_t expl_hist_cap, orc_capture *cap)
{
    return orc_gmres_p(n, rp, ci, va, ORC_PRECOND_NONE, NULL, b, x, prm, res, rec_hist, rec_hist_cap, expl_hist,
                       expl_hist_cap, cap);
}

int orc_gmres_p(int64_t n, const int32_t *rp, const int32_t *ci, const double *va, int kind, const double *pdata,
                const double *b, double *x, const orc_params *prm, orc_result *res, double *rec_hist,
                int32_t rec_hist_cap, double *expl_hist, int32_t expl_hist_cap, orc_capture *cap)
{
    const int m = prm->restart, fmt = prm->format;
    const int64_t B = orc_format_bytes(fmt);
    if (n <= 0 || m < 1 || B < 0 || prm->max_iters < 0) return 1;
    const double tau = prm->rel_tol, eta = prm->eta;

    char *V = (char *)malloc((size_t)(m + 1) * (size_t)n * (size_t)B); /* stored basis, vector-major */
    double *sigma = (double *)calloc((size_t)m + 1, 8);
    double *v = (double *)malloc((size_t)n * 8);   /* fp64 copy of the newest basis vector (reading Q1) */
    double *w = (double *)malloc((size_t)n * 8);
    double *tmp = (double *)malloc((size_t)n * 8); /* one decoded basis vector */
    double *z = (double *)malloc((size_t)n * 8);   /* M^-1 v (l.3) / V_k y (l.17) when preconditioned */
    double *h = (double *)calloc((size_t)m + 2, 8), *u = (double *)calloc((size_t)m + 2, 8);
    double *R = (double *)calloc((size_t)(m + 1) * (size_t)m, 8); /* rotated H, column-major ld m+1 */
    double *cs = (double *)calloc((size_t)m, 8), *sn = (double *)calloc((size_t)m, 8);
    double *g = (double *)calloc((size_t)m + 1, 8), *y = (double *)calloc((size_t)m, 8);
    if (!V || !sigma || !v || !w || !tmp || !z || !h || !u || !R || !cs || !sn || !g || !y) return 2;
#define VCOL(c) (V + (size_t)(c) * (size_t)n * (size_t)B)

    memset(res, 0, sizeof(*res));
    const double bnorm = nrm2(n, b);
    res->b_norm = bnorm;
    int iters = 0, cycles = 0, nexpl = 0;
    int64_t i;
    if (bnorm == 0.0) { /* reading Q9: b = 0 => x = 0 */
        memset(x, 0, (size_t)n * 8);
        res->converged = 1;
        goto done;
    }
    for (;;) {
        /* l.1: r_0 := b - A x_0, beta := ||r_0||_2 */
        orc_spmv(n, rp, ci, va, x, w);
#pragma omp parallel for schedule(static)
        for (i = 0; i < n; i++) w[i] = b[i] - w[i];
        const double beta = nrm2(n, w);
        res->rel_res_true = beta / bnorm;
        if (expl_hist && nexpl < expl_hist_cap) expl_hist[nexpl] = beta / bnorm;
        nexpl++;
        if (!isfinite(beta)) { res->converged = 0; break; }
        if (beta <= tau * bnorm) { res->converged = 1; break; }
        if (iters >= prm->max_iters) { res->converged = 0; break; }
        const int capture = cap && cap->cycle == cycles;
        cycles++;
        /* l.1: v := r_0 / beta, V_1 = [v]  (store through the codec) */
#pragma omp parallel for schedule(static)
        for (i = 0; i < n; i++) v[i] = w[i] / beta;
        orc_enc(fmt, n, v, VCOL(0), &sigma[0]);
        memset(g, 0, ((size_t)m + 1) * 8);
        g[0] = beta;
        if (capture) {
            cap->beta = beta;
            memcpy(cap->Vfp64, v, (size_t)n * 8);
            orc_dec(fmt, n, VCOL(0), sigma[0], cap->Vhat);
            memset(cap->Hbar, 0, (size_t)(m + 1) * (size_t)m * 8);
        }
        int k = 0, breakdown = 0;
        for (int j = 1; j <= m; j++) {
            /* l.3: w := A (M^-1 v)   (the fp64 v, reading Q1) */
            if (kind != ORC_PRECOND_NONE) {
                apply_minv(kind, pdata, n, v, z);
                orc_spmv(n, rp, ci, va, z, w);
            } else {
                orc_spmv(n, rp, ci, va, v, w);
            }
            /* l.4: omega := ||w||_2 */
            const double omega = nrm2(n, w);
            /* l.5: h_{1:j,j} := V_j^T w  (classical Gram-Schmidt: all j dots from the same w) */
            for (int c = 0; c < j; c++) {
                orc_dec(fmt, n, VCOL(c), sigma[c], tmp);
                h[c] = dot(n, tmp, w);
            }
            /*      w := w - V_j h_{1:j,j} */
            for (int c = 0; c < j; c++) {
                orc_dec(fmt, n, VCOL(c), sigma[c], tmp);
                axpy(n, -h[c], tmp, w);
            }
            /* l.6: h_{j+1,j} := ||w||_2 */
            double hn = nrm2(n, w);
            breakdown = (hn == 0.0);
            if (capture && cap->omega) cap->omega[j - 1] = omega;
            if (capture && cap->reorth_log) cap->reorth_log[j - 1] = 0;
            /* l.7: if h_{j+1,j} < eta * omega then re-orthogonalise (one extra pass, reading Q3) */
            if (prm->reorth == ORC_REORTH_ALWAYS || (prm->reorth == ORC_REORTH_COND && hn < eta * omega)) {
                const double omega1 = hn; /* norm before the second pass (reading Q4) */
                if (capture && cap->reorth_log) cap->reorth_log[j - 1] = 1;
                /* l.8: u := V_j^T w, w := w - V_j u */
                for (int c = 0; c < j; c++) {
                    orc_dec(fmt, n, VCOL(c), sigma[c], tmp);
                    u[c] = dot(n, tmp, w);
                }
                for (int c = 0; c < j; c++) {
                    orc_dec(fmt, n, VCOL(c), sigma[c], tmp);
                    axpy(n, -u[c], tmp, w);
                }
                /* l.9: h_{1:j,j} += u ; l.10: h_{j+1,j} := ||w||_2 */
                for (int c = 0; c < j; c++) h[c] += u[c];
                hn = nrm2(n, w);
                res->reorth_count++;
                /* l.12: breakdown if the second pass again lost more than the factor eta */
                breakdown = (hn == 0.0) || (hn < eta * omega1);
            }
            iters++;
            if (capture) {
                for (int c = 0; c < j; c++) cap->Hbar[(size_t)(j - 1) * (m + 1) + c] = h[c];
                cap->Hbar[(size_t)(j - 1) * (m + 1) + j] = hn;
            }
            /* l.16-17 "updating technique": apply the previous rotations to the
             * new column, form rotation j, rotate the right-hand side. */
            h[j] = hn;
            for (int c = 0; c < j - 1; c++) {
                const double t = cs[c] * h[c] + sn[c] * h[c + 1];
                h[c + 1] = -sn[c] * h[c] + cs[c] * h[c + 1];
                h[c] = t;
            }
            const double rho = hypot(h[j - 1], h[j]);
            if (rho == 0.0) { cs[j - 1] = 1.0; sn[j - 1] = 0.0; }
            else { cs[j - 1] = h[j - 1] / rho; sn[j - 1] = h[j] / rho; }
            h[j - 1] = rho;
            h[j] = 0.0;
            for (int c = 0; c < j; c++) R[(size_t)(j - 1) * (m + 1) + c] = h[c];
            g[j] = -sn[j - 1] * g[j - 1];
            g[j - 1] = cs[j - 1] * g[j - 1];
            /* l.13-14: v := w / h_{j+1,j}; V_{j+1} := [V_j, v] */
            if (hn > 0.0) {
#pragma omp parallel for schedule(static)
                for (i = 0; i < n; i++) v[i] = w[i] / hn;
                orc_enc(fmt, n, v, VCOL(j), &sigma[j]);
                if (capture) {
                    memcpy(cap->Vfp64 + (size_t)j * n, v, (size_t)n * 8);
                    orc_dec(fmt, n, VCOL(j), sigma[j], cap->Vhat + (size_t)j * n);
                }
            }
            k = j;
            if (rec_hist && iters - 1 < rec_hist_cap) rec_hist[iters - 1] = fabs(g[j]) / bnorm;
            /* recurrence residual |g_{j+1}| tracks ||b - A x_j|| */
            if (fabs(g[j]) <= tau * bnorm || breakdown || iters >= prm->max_iters) break;
        }
        res->breakdown = breakdown;
        res->rel_res_recurrence = fabs(g[k]) / bnorm;
        /* l.17: y := argmin ||beta e_1 - Hbar y||  <=>  R_{1:k,1:k} y = g_{1:k} */
        for (int r = k - 1; r >= 0; r--) {
            double s = g[r];
            for (int c = r + 1; c < k; c++) s -= R[(size_t)c * (m + 1) + r] * y[c];
            y[r] = s / R[(size_t)r * (m + 1) + r];
        }
        /*       x := x_0 + M^-1 (V_k y)   (decoded basis) */
        if (kind == ORC_PRECOND_JACOBI) {
            memset(z, 0, (size_t)n * 8);
            for (int c = 0; c < k; c++) {
                orc_dec(fmt, n, VCOL(c), sigma[c], tmp);
                axpy(n, y[c], tmp, z);
            }
#pragma omp parallel for schedule(static)
            for (i = 0; i < n; i++) x[i] += z[i] / pdata[i];
        } else if (kind != ORC_PRECOND_NONE) {
            memset(z, 0, (size_t)n * 8);
            for (int c = 0; c < k; c++) {
                orc_dec(fmt, n, VCOL(c), sigma[c], tmp);
                axpy(n, y[c], tmp, z);
            }
            apply_minv(kind, pdata, n, z, tmp);
#pragma omp parallel for schedule(static)
            for (i = 0; i < n; i++) x[i] += tmp[i];
        } else {
            for (int c = 0; c < k; c++) {
                orc_dec(fmt, n, VCOL(c), sigma[c], tmp);
                axpy(n, y[c], tmp, x);
            }
        }
        if (capture) {
            cap->k = k;
            memcpy(cap->y, y, (size_t)k * 8);
            memcpy(cap->g, g, ((size_t)m + 1) * 8);
        }
        /* l.18: go to step 1 (the explicit residual decides) */
    }
done:
    res->iters = iters;
    res->restarts = cycles;
#undef VCOL
    free(V); free(sigma); free(v); free(w); free(tmp); free(z); free(h); free(u); free(R); free(cs); free(sn); free(g); free(y);
    return 0;
}
