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

} // namespace fresnel
