// pointwise.cuh -- the stand-alone one-pass optic operators (no transform):
//   quadratic phase factor  u[b][j][k] *= Q_b[j] * Q_b[k]            (Eq. 2; separable table)
//   optic phasor            u[b][j][k] *= A[j][k] * exp(2 pi i OPD[j][k] / lambda_b)   (Eq. 3)
// In a propagation these ride on the load of the row pass (pass_kernel.cuh); this kernel serves
// fresnel_apply_qpf / fresnel_apply_mask and the z == 0 case of fresnel_surface_as.
// Streaming, 16 bytes per thread per access, grid-stride over rows.
#pragma once
#include "pass_kernel.cuh"

namespace fresnel {

template <typename T>
__global__ void __launch_bounds__(256) pointwise_kernel(typename cplx_of<T>::type *wf, const typename cplx_of<T>::type *__restrict__ tab,
                                                        const T *__restrict__ amp, const T *__restrict__ opd,
                                                        const double *__restrict__ inv_lambda, int N)
{
    using C = typename cplx_of<T>::type;
    const int b = blockIdx.z;
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= N) return;
    const C *q = tab ? tab + (size_t)b * N : nullptr;
    C qk;
    if (q) qk = ldg_c(q + k);
    const T il = opd ? (T)inv_lambda[b] : (T)0;
    for (int j = blockIdx.y; j < N; j += gridDim.y) {
        const size_t o = (size_t)j * N + k;
        C *e = wf + (size_t)b * N * N + o;
        C u = *e;
        if (q) u = cmul(u, cmul(ldg_c(q + j), qk));
        if (opd) u = cmul(u, phasor_turns(opd[o] * il));
        if (amp) { T s = amp[o]; u.x *= s; u.y *= s; }
        *e = u;
    }
}

template <typename T>
cudaError_t launch_pointwise(typename cplx_of<T>::type *wf, const typename cplx_of<T>::type *tab, const T *amp, const T *opd,
                             const double *inv_lambda, int N, int batch, cudaStream_t stream)
{
    const int threads = N < 256 ? N : 256;
    int rows = N < 1024 ? N : 1024;          // row-blocks in flight; each walks N/rows rows
    dim3 grid((N + threads - 1) / threads, rows, batch);
    pointwise_kernel<T><<<grid, threads, 0, stream>>>(wf, tab, amp, opd, inv_lambda, N);
    return cudaGetLastError();
}

// ---- broadband image -----------------------------------------
//   image[j][k] += sum_b weight[b] * |wf[b][j][k]|^2
// One streaming pass: every thread owns two adjacent pixels (16 or 32 bytes of wavefront per access), walks the
// batch with the running sum in double, and touches the image once.  Weights ride in the kernel parameters.
constexpr int kIntensityMaxBatch = 64;
struct IntensityWeights { double w[kIntensityMaxBatch]; };

template <typename T>
__global__ void __launch_bounds__(256) intensity_kernel(const typename cplx_of<T>::type *__restrict__ wf, T *__restrict__ image,
                                                        IntensityWeights wt, int nb, size_t plane /* N*N */)
{
    using C = typename cplx_of<T>::type;
    const size_t stride = (size_t)gridDim.x * blockDim.x * 2;
    for (size_t i = ((size_t)blockIdx.x * blockDim.x + threadIdx.x) * 2; i < plane; i += stride) {
        const bool two = i + 1 < plane;                 // an odd grid has an odd number of pixels
        double a0 = (double)image[i], a1 = two ? (double)image[i + 1] : 0.0;
        for (int b = 0; b < nb; ++b) {
            const C u0 = wf[(size_t)b * plane + i];
            a0 = fma(wt.w[b], (double)u0.x * (double)u0.x + (double)u0.y * (double)u0.y, a0);
            if (two) {
                const C u1 = wf[(size_t)b * plane + i + 1];
                a1 = fma(wt.w[b], (double)u1.x * (double)u1.x + (double)u1.y * (double)u1.y, a1);
            }
        }
        image[i] = (T)a0;
        if (two) image[i + 1] = (T)a1;
    }
}

template <typename T>
cudaError_t launch_intensity(const typename cplx_of<T>::type *wf, T *image, const double *weight, int N, int batch, int sms,
                             cudaStream_t stream, unsigned long long *launches)
{
    const size_t plane = (size_t)N * N;
    for (int b0 = 0; b0 < batch; b0 += kIntensityMaxBatch) {
        IntensityWeights wt;
        const int nb = batch - b0 < kIntensityMaxBatch ? batch - b0 : kIntensityMaxBatch;
        for (int b = 0; b < nb; ++b) wt.w[b] = weight[b0 + b];
        const size_t want = ((plane + 1) / 2 + 255) / 256;
        const int grid = (int)(want < (size_t)sms * 8 ? want : (size_t)sms * 8);
        intensity_kernel<T><<<grid, 256, 0, stream>>>(wf + (size_t)b0 * plane, image, wt, nb, plane);
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return e;
        ++*launches;
    }
    return cudaSuccess;
}

} // namespace fresnel
