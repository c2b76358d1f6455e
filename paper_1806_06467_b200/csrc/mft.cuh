// mft.cuh -- Fraunhofer propagation by a matrix Fourier transform (PAPER.md:27
// "discrete matrix Fourier transforms of modest sized arrays", :119): the one dense contraction of the path.
//
//     V[p,q] = s * sum_j sum_k E[p,j] U[j,k] E[q,k],     E[q,k] = exp(-+ 2 pi i x_k x'_q / (lambda f)),  s = dx^2/(+- i lambda f)
//
// for an na x na input of pitch dx and ANY nb x nb output grid of pitch dx' (both centred on pixel n/2).  Two complex
// GEMMs on the FP64 TENSOR CORES (mma.sync m8n8k4 f64: DMMA -- tcgen05 has no FP64 kind, and the north-star tolerance
// of 1e-11 rules out the narrower tensor formats; complex64 plans convert on load and round on store, so they are
// computed in FP64 too):
//     T^t[q,j] = sum_k U[j,k] E[q,k]          (M = na, N = nb, K = na; stored transposed)
//     V[p,q]   = s sum_j E[p,j] T^t[q,j]      (M = nb, N = nb, K = na)
// both of the form C[m,n] = alpha sum_k A[m,k] B[n,k] with K contiguous in A and B.  The kernel matrix E is built once
// per call by mft_matrix_kernel: the phase m n c with the integer product m n exact and c = dx dx'/(lambda f) (turns)
// a double-double from the host, reduced to +-1/2 turn before sincospi -- the same device as the chirp tables.
#pragma once
#include <cuda_runtime.h>
#include <cstdint>
#include "fft_core.cuh"

namespace fresnel {

// E[b][q][k], q < nb, k < na (double2, row-major)
struct MftMatrixArgs {
    double2 *out;
    int na, nb, batch;
    int sign;                    // -1: forward kernel exp(-...), +1: inverse kernel
    const double *c_hi, *c_lo;   // [batch] device: dx dx'/(lambda f) in turns, double-double
};

__global__ void __launch_bounds__(256) mft_matrix_kernel(MftMatrixArgs a)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    const int q = blockIdx.y, b = blockIdx.z;
    if (k >= a.na) return;
    const double m = (double)(k - a.na / 2) * (double)(q - a.nb / 2);      // exact: |m| < 2^24
    const double ch = a.c_hi[b], cl = a.c_lo[b];
    const double hi = m * ch;
    const double err = fma(m, ch, -hi);
    const double lo = fma(m, cl, err);
    const double r = (hi - rint(hi)) + lo;
    double s, c;
    sincospi(2.0 * r, &s, &c);
    a.out[((size_t)b * a.nb + q) * a.na + k] = make_double2(c, a.sign < 0 ? -s : s);
}

FR_DEV void dmma8x8x4(double &d0, double &d1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};" : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

template <typename CIN> FR_DEV double2 mft_load(const CIN *p) { return make_double2((double)p->x, (double)p->y); }
FR_DEV void mft_store(double2 *p, double2 v) { *p = v; }
FR_DEV void mft_store(float2 *p, double2 v) { *p = make_float2((float)v.x, (float)v.y); }

// C[m,n] = alpha_b * sum_k A[m,k] B[n,k]   (complex; A: [M][K], B: [N][K], K contiguous; TRANS: C stored as [N][M])
struct MftGemmArgs {
    const void *A;
    const double2 *B;
    void *C;
    int M, N, K;
    size_t strideA, strideB, strideC;     // batch strides in elements
    const double2 *alpha;                 // [batch] device, or nullptr for 1
};

constexpr int kMftBM = 32, kMftBN = 32, kMftBK = 16, kMftLD = kMftBK + 4;   // row stride 20 double2: conflict-free fragment loads

template <typename CIN, typename COUT, bool TRANS>
__global__ void __launch_bounds__(128) mft_gemm_kernel(MftGemmArgs g)
{
    __shared__ double2 As[kMftBM][kMftLD];
    __shared__ double2 Bs[kMftBN][kMftLD];
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int b = blockIdx.z;
    const int m0 = blockIdx.y * kMftBM, n0 = blockIdx.x * kMftBN;
    const CIN *A = reinterpret_cast<const CIN *>(g.A) + (size_t)b * g.strideA;
    const double2 *B = g.B + (size_t)b * g.strideB;
    COUT *C = reinterpret_cast<COUT *>(g.C) + (size_t)b * g.strideC;
    const int wm = (warp >> 1) * 16, wn = (warp & 1) * 16;       // this warp's 16 x 16 corner of the CTA tile
    const int fr = lane >> 2, fk = lane & 3;                     // fragment row (m or n) and k of this lane
    double cr[2][2][2], ci[2][2][2];                             // [m-tile][n-tile][2 columns of the C fragment]
#pragma unroll
    for (int i = 0; i < 2; ++i)
#pragma unroll
        for (int j = 0; j < 2; ++j) { cr[i][j][0] = cr[i][j][1] = 0.0; ci[i][j][0] = ci[i][j][1] = 0.0; }

    for (int k0 = 0; k0 < g.K; k0 += kMftBK) {
        // ---- stage the two tiles (zero beyond the matrix edges) ----
#pragma unroll
        for (int i = 0; i < (kMftBM * kMftBK) / 128; ++i) {
            const int e = tid + i * 128, r = e / kMftBK, c = e % kMftBK;
            const bool ok = (k0 + c) < g.K;
            As[r][c] = (ok && m0 + r < g.M) ? mft_load(A + (size_t)(m0 + r) * g.K + k0 + c) : make_double2(0.0, 0.0);
            Bs[r][c] = (ok && n0 + r < g.N) ? B[(size_t)(n0 + r) * g.K + k0 + c] : make_double2(0.0, 0.0);
        }
        __syncthreads();
#pragma unroll
        for (int kk = 0; kk < kMftBK; kk += 4) {
            double2 af[2], bf[2];
#pragma unroll
            for (int i = 0; i < 2; ++i) {
                af[i] = As[wm + 8 * i + fr][kk + fk];
                bf[i] = Bs[wn + 8 * i + fr][kk + fk];
            }
#pragma unroll
            for (int i = 0; i < 2; ++i)
#pragma unroll
                for (int j = 0; j < 2; ++j) {
                    dmma8x8x4(cr[i][j][0], cr[i][j][1], af[i].x, bf[j].x);        // + Ar Br
                    dmma8x8x4(cr[i][j][0], cr[i][j][1], -af[i].y, bf[j].y);       // - Ai Bi
                    dmma8x8x4(ci[i][j][0], ci[i][j][1], af[i].x, bf[j].y);        // + Ar Bi
                    dmma8x8x4(ci[i][j][0], ci[i][j][1], af[i].y, bf[j].x);        // + Ai Br
                }
        }
        __syncthreads();
    }
    // ---- epilogue: C fragment element (row = lane/4, col = 2*(lane%4) + e) ----
    double2 al = make_double2(1.0, 0.0);
    if (g.alpha != nullptr) al = g.alpha[b];
#pragma unroll
    for (int i = 0; i < 2; ++i)
#pragma unroll
        for (int j = 0; j < 2; ++j)
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int m = m0 + wm + 8 * i + fr, n = n0 + wn + 8 * j + 2 * fk + e;
                if (m < g.M && n < g.N) {
                    const double xr = cr[i][j][e], xi = ci[i][j][e];
                    const double2 v = make_double2(xr * al.x - xi * al.y, xr * al.y + xi * al.x);
                    if (TRANS) mft_store(C + (size_t)n * g.M + m, v);
                    else       mft_store(C + (size_t)m * g.N + n, v);
                }
            }
}

template <typename CIN, typename COUT, bool TRANS>
cudaError_t launch_mft_gemm(const MftGemmArgs &g, int batch, cudaStream_t stream)
{
    dim3 grid((g.N + kMftBN - 1) / kMftBN, (g.M + kMftBM - 1) / kMftBM, batch);
    mft_gemm_kernel<CIN, COUT, TRANS><<<grid, 128, 0, stream>>>(g);
    return cudaGetLastError();
}

} // namespace fresnel
