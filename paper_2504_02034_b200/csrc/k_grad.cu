// k_grad.cu -- lambda-gradients of log L (SURVEY 8(f) NEXT-4; PAPER.md:132 "automatic differentiation", :175 Hamiltonian MCMC)
// by central differences with one Richardson step, evaluated THROUGH the batched hot path: the path is batched over lambda, so
// the 60 displaced points of a gradient are 60 more rows of the batch.
//   row 0            lambda
//   rows 1 + 4k + s  lambda + d_s h_k e_k,  d = (+1, -1, +1/2, -1/2),  h_k = rel_step |lambda_k| (rel_step if lambda_k = 0)
//   D(h) = [f(+h) - f(-h)] / 2h;   dlogL/dlambda_k = [4 D(h/2) - D(h)] / 3 + O(h^4)
// k_grad_expand writes the rows, chim_loglike_batch evaluates them, k_grad_combine forms the derivatives (fp64).
#include "chim_internal.cuh"

namespace chim {

constexpr int kGradRows = 1 + 4 * CHIM_N_LAMBDA_PARAMS;

__device__ __forceinline__ double grad_step(double v, double rel) { return (v != 0.0) ? rel * fabs(v) : rel; }

__global__ void k_grad_expand(const double* __restrict__ lam, int n_lambda, double rel, double* __restrict__ ext) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;       // one thread per (lambda, row)
    if (i >= n_lambda * kGradRows) return;
    const int l = i / kGradRows, r = i - l * kGradRows;
    const double* src = lam + (size_t)l * CHIM_N_LAMBDA_PARAMS;
    double* dst = ext + (size_t)i * CHIM_N_LAMBDA_PARAMS;
#pragma unroll
    for (int k = 0; k < CHIM_N_LAMBDA_PARAMS; ++k) dst[k] = src[k];
    if (r > 0) {
        const int k = (r - 1) >> 2, s = (r - 1) & 3;
        const double h = grad_step(src[k], rel);
        dst[k] = src[k] + ((s & 1) ? -1.0 : 1.0) * ((s & 2) ? 0.5 : 1.0) * h;
    }
}

__global__ void k_grad_combine(const double* __restrict__ lam, int n_lambda, double rel, const double* __restrict__ ll,
                               const uint32_t* __restrict__ fl, double* __restrict__ out_ll, double* __restrict__ out_grad,
                               uint32_t* __restrict__ out_fl) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;       // one thread per (lambda, parameter)
    if (i >= n_lambda * CHIM_N_LAMBDA_PARAMS) return;
    const int l = i / CHIM_N_LAMBDA_PARAMS, k = i - l * CHIM_N_LAMBDA_PARAMS;
    const double* f = ll + (size_t)l * kGradRows;
    const double h = grad_step(lam[(size_t)l * CHIM_N_LAMBDA_PARAMS + k], rel);
    const double d1 = (f[1 + 4 * k] - f[2 + 4 * k]) / (2.0 * h), d2 = (f[3 + 4 * k] - f[4 + 4 * k]) / h;
    out_grad[i] = (4.0 * d2 - d1) / 3.0;                        // NaN / inf rows propagate: the derivative is undefined there
    if (k == 0) {
        out_ll[l] = f[0];
        if (out_fl) {
            uint32_t a = 0;
            for (int r = 0; r < kGradRows; ++r) a |= fl[(size_t)l * kGradRows + r];
            out_fl[l] = a;
        }
    }
}

cudaError_t launch_grad_expand(const double* lam, int n_lambda, double rel, double* ext, cudaStream_t st) {
    const int n = n_lambda * kGradRows;
    if (n <= 0) return cudaSuccess;
    k_grad_expand<<<(n + 255) / 256, 256, 0, st>>>(lam, n_lambda, rel, ext);
    return cudaGetLastError();
}
cudaError_t launch_grad_combine(const double* lam, int n_lambda, double rel, const double* ll, const uint32_t* fl, double* out_ll,
                                double* out_grad, uint32_t* out_fl, cudaStream_t st) {
    const int n = n_lambda * CHIM_N_LAMBDA_PARAMS;
    if (n <= 0) return cudaSuccess;
    k_grad_combine<<<(n + 255) / 256, 256, 0, st>>>(lam, n_lambda, rel, ll, fl, out_ll, out_grad, out_fl);
    return cudaGetLastError();
}
int grad_rows() { return kGradRows; }

}  // namespace chim
