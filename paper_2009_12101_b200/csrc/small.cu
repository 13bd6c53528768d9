// small.cu -- the tiny dense pieces that stay on the device (north_star: "small Hessenberg Givens
// rotations and the triangular solve, kept on the device"): the back substitution R y = g of
// Fig. 1 line 17 and two marshalling kernels used by the per-kernel hooks.
#include "device_utils.cuh"

namespace cbg {

// Column-oriented back substitution on the k x k upper-triangular R (column-major, ld = m+1):
// y_i = g_i / R_ii, then g_{0..i-1} -= R_{0..i-1,i} y_i with the lanes of warp 0 striding the rows.
// For k <= kBackStage the upper triangle is first staged in shared memory (packed by columns) by all
// threads -- one round of global loads instead of two dependent L2 round trips per column
// (80 -> ~10 us at k = 100); larger k reads R column by column from global memory.
// Leaves hs_c = -sigma_c * y_c, the coefficients with which the update kernel forms x += V_k y.
constexpr int kBackStage = 100;
constexpr int kBackThreads = 256;
template <bool SCALED> __global__ void __launch_bounds__(kBackThreads) backsolve_kernel(Ctl *ctl, CycleState cy)
{
    pdl_wait();
    pdl_launch_dependents();
    const int k = ctl->k;
    if (k <= 0 || ctl->nonfinite) return; // a non-finite norm: x stays at the last completed cycle (cbgmres.h)
    __shared__ double t[kMaxRestart + 1];
    __shared__ double Rs[kBackStage * (kBackStage + 1) / 2]; // column i at offset i (i + 1) / 2, rows 0..i
    const int tid = threadIdx.x, lane = tid & 31, m = ctl->m;
    const bool staged = k <= kBackStage;
    for (int i = tid; i < k; i += kBackThreads) t[i] = cy.g[i];
    if (staged) {
        for (int c = 0; c < k; ++c) {
            const double *Rc = cy.R + (size_t)c * (m + 1);
            for (int l = tid; l <= c; l += kBackThreads) Rs[c * (c + 1) / 2 + l] = Rc[l];
        }
    }
    __syncthreads();
    if (tid < 32) {
        for (int i = k - 1; i >= 0; --i) {
            const double *Rc = staged ? Rs + i * (i + 1) / 2 : cy.R + (size_t)i * (m + 1);
            const double yi = t[i] / Rc[i];
            __syncwarp();
            if (lane == 0) t[i] = yi;
            for (int l = lane; l < i; l += 32) t[l] = fma(-Rc[l], yi, t[l]);
            __syncwarp();
        }
    }
    __syncthreads();
    for (int i = tid; i < k; i += kBackThreads) {
        cy.y[i] = t[i];
        cy.hs[i] = -(SCALED ? cy.scales[i] : 1.0) * t[i];
    }
}

int launch_backsolve(cudaStream_t s, const Scratch &sc, const CycleState &cyc, int format)
{
    if (format == CBGMRES_INT32 || format == CBGMRES_INT16) launch_chain(sc, "backsolve_kernel", backsolve_kernel<true>, dim3(1), dim3(kBackThreads), 0, s, sc.ctl, cyc);
    else launch_chain(sc, "backsolve_kernel", backsolve_kernel<false>, dim3(1), dim3(kBackThreads), 0, s, sc.ctl, cyc);
    return 1;
}

__global__ void scale_coeffs_kernel(int k, const double *h, const double *scales, double *hs)
{
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c < k) hs[c] = scales ? h[c] * scales[c] : h[c];
}

int launch_scale_coeffs(cudaStream_t s, int k, const double *h, const double *scales, double *hs)
{
    scale_coeffs_kernel<<<(k + 127) / 128, 128, 0, s>>>(k, h, scales, hs);
    return 1;
}

__global__ void copy_scalars_kernel(const double *s0, double *d0, const double *s1, double *d1)
{
    if (d0 && s0) *d0 = *s0;
    if (d1 && s1) *d1 = *s1;
}

int launch_copy_scalars(cudaStream_t s, const double *src0, double *dst0, const double *src1, double *dst1)
{
    copy_scalars_kernel<<<1, 1, 0, s>>>(src0, dst0, src1, dst1);
    return 1;
}

// ---- scalar Jacobi right preconditioner M = diag(A) (Fig. 1 l.3 and l.17) ---------------
// Applied by a change of variable, at no cost inside the Arnoldi loop: GMRES runs on A D^-1 (a
// column-scaled copy of the values, made once per solve in the caller's workspace) in the variable
// u = D x; the residual b - (A D^-1) u = b - A x is that of the original system, so every stopping
// test is unchanged, and x = D^-1 u is formed once at the end.
__global__ void jacobi_diag_kernel(int64_t n, const int32_t *__restrict__ rp, const int32_t *__restrict__ ci,
                                   const double *__restrict__ va, double *__restrict__ d)
{
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        double di = 1.0; // a row without a (nonzero) diagonal entry stays unscaled
        for (int32_t p = rp[i]; p < rp[i + 1]; ++p)
            if (ci[p] == i && va[p] != 0.0) di = va[p];
        d[i] = di;
    }
}

__global__ void jacobi_scale_vals_kernel(int64_t n, const int32_t *__restrict__ rp, const int32_t *__restrict__ ci,
                                         const double *__restrict__ va, const double *__restrict__ d, double *__restrict__ out)
{
    const int64_t nnz = rp[n];
    for (int64_t p = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; p < nnz; p += (int64_t)gridDim.x * blockDim.x)
        out[p] = va[p] / d[ci[p]];
}

// x_i *= d_i (inverse = 0) or x_i /= d_i (inverse = 1)
__global__ void diag_scale_kernel(int64_t n, double *__restrict__ x, const double *__restrict__ d, int inverse)
{
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
        x[i] = inverse ? x[i] / d[i] : x[i] * d[i];
}

int launch_jacobi_setup(cudaStream_t s, const CsrView &A, double *d, double *scaled_vals)
{
    jacobi_diag_kernel<<<kNumSMs * 8, 256, 0, s>>>(A.n, A.row_ptr, A.col_idx, A.vals, d);
    jacobi_scale_vals_kernel<<<kNumSMs * 8, 256, 0, s>>>(A.n, A.row_ptr, A.col_idx, A.vals, d, scaled_vals);
    return 2;
}

int launch_diag_scale(cudaStream_t s, int64_t n, double *x, const double *d, int inverse)
{
    diag_scale_kernel<<<kNumSMs * 8, 256, 0, s>>>(n, x, d, inverse);
    return 1;
}

// ---- block-Jacobi right preconditioner, block size 4 (section 6.5) -------------------------
// M = blockdiag(A_bb), A_bb = rows and columns 4b .. 4b+3 of A (absent entries are zero; the last block is
// completed by the identity when 4 does not divide n).  One thread gathers one block from its four CSR
// rows and inverts it by Gauss-Jordan elimination with partial pivoting; a singular block is replaced by
// the identity (as the scalar variant leaves a row with a zero diagonal unscaled).  Once per solve.
// In the loop, M^-1 is applied by the store kernel (store.cu: the next SpMV multiplies z = M^-1 v, Fig. 1
// l.3); at the end of a cycle x += M^-1 (V_k y) (l.17) by bj4_axpy_kernel below.
__global__ void __launch_bounds__(128) bj4_setup_kernel(int64_t n, const int32_t *__restrict__ rp, const int32_t *__restrict__ ci,
                                                        const double *__restrict__ va, double *__restrict__ inv)
{
    const int64_t nb = (n + 3) / 4;
    for (int64_t b = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; b < nb; b += (int64_t)gridDim.x * blockDim.x) {
        double a[4][8];
#pragma unroll
        for (int r = 0; r < 4; ++r)
#pragma unroll
            for (int c = 0; c < 8; ++c) a[r][c] = (c == r + 4) ? 1.0 : 0.0;
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            const int64_t i = 4 * b + r;
            if (i >= n) {
                a[r][r] = 1.0;
                continue;
            }
            for (int32_t p = rp[i]; p < rp[i + 1]; ++p) {
                const int64_t c = (int64_t)ci[p] - 4 * b;
                if (c >= 0 && c < 4) {
#pragma unroll
                    for (int cc = 0; cc < 4; ++cc) // static register indexing
                        if (cc == c) a[r][cc] += va[p];
                }
            }
        }
        bool singular = false;
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            if (singular) continue;
            int piv = k;
            double best = fabs(a[k][k]);
#pragma unroll
            for (int r = k + 1; r < 4; ++r)
                if (fabs(a[r][k]) > best) {
                    best = fabs(a[r][k]);
                    piv = r;
                }
            if (best == 0.0 || !isfinite(best)) {
                singular = true;
                continue;
            }
#pragma unroll
            for (int r = k + 1; r < 4; ++r)
                if (r == piv) {
#pragma unroll
                    for (int c = 0; c < 8; ++c) {
                        const double t = a[k][c];
                        a[k][c] = a[r][c];
                        a[r][c] = t;
                    }
                }
            const double d = a[k][k];
#pragma unroll
            for (int c = 0; c < 8; ++c) a[k][c] = a[k][c] / d;
#pragma unroll
            for (int r = 0; r < 4; ++r) {
                if (r == k) continue;
                const double f = a[r][k];
#pragma unroll
                for (int c = 0; c < 8; ++c) a[r][c] = fma(-f, a[k][c], a[r][c]);
            }
        }
#pragma unroll
        for (int r = 0; r < 4; ++r)
#pragma unroll
            for (int c = 0; c < 4; ++c) inv[16 * b + 4 * r + c] = singular ? (r == c ? 1.0 : 0.0) : a[r][c + 4];
    }
}

// x_b += A_bb^-1 t_b, one block per thread (Fig. 1 l.17 with M = blockdiag: x := x + M^-1 (V_k y), t = V_k y)
__global__ void __launch_bounds__(256) bj4_axpy_kernel(int64_t n, const double *__restrict__ inv, const double *__restrict__ t, double *__restrict__ x)
{
    const int64_t nb = (n + 3) / 4;
    for (int64_t b = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; b < nb; b += (int64_t)gridDim.x * blockDim.x) {
        double tv[4];
#pragma unroll
        for (int c = 0; c < 4; ++c) tv[c] = (4 * b + c < n) ? t[4 * b + c] : 0.0;
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            if (4 * b + r >= n) break;
            const double *iv = inv + 16 * b + 4 * r;
            const double z = fma(iv[3], tv[3], fma(iv[2], tv[2], fma(iv[1], tv[1], iv[0] * tv[0])));
            x[4 * b + r] += z;
        }
    }
}

__global__ void fill_zero_kernel(int64_t n, double *__restrict__ x)
{
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) x[i] = 0.0;
}

int launch_bj4_setup(cudaStream_t s, const CsrView &A, double *inv)
{
    const int64_t nb = (A.n + 3) / 4;
    int64_t grid = (nb + 127) / 128;
    if (grid > kNumSMs * 16) grid = kNumSMs * 16;
    bj4_setup_kernel<<<(int)grid, 128, 0, s>>>(A.n, A.row_ptr, A.col_idx, A.vals, inv);
    return 1;
}

int launch_bj4_axpy(cudaStream_t s, int64_t n, const double *inv, const double *t, double *x)
{
    const int64_t nb = (n + 3) / 4;
    int64_t grid = (nb + 255) / 256;
    if (grid > kNumSMs * 8) grid = kNumSMs * 8;
    bj4_axpy_kernel<<<(int)grid, 256, 0, s>>>(n, inv, t, x);
    return 1;
}

int launch_fill_zero(cudaStream_t s, int64_t n, double *x)
{
    fill_zero_kernel<<<kNumSMs * 8, 256, 0, s>>>(n, x);
    return 1;
}

} // namespace cbg
