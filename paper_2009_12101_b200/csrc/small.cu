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
    if (k <= 0) return;
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
    if (format == CBGMRES_INT32 || format == CBGMRES_INT16) launch_chain(backsolve_kernel<true>, dim3(1), dim3(kBackThreads), 0, s, sc.ctl, cyc);
    else launch_chain(backsolve_kernel<false>, dim3(1), dim3(kBackThreads), 0, s, sc.ctl, cyc);
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

} // namespace cbg
