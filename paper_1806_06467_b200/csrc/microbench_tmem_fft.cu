// microbench_tmem_fft.cu -- stand-alone prototype (not part of libfresnel.so): a 2048-point complex128 transform whose
// FIRST exchange goes through tensor memory (X1 = tcgen05.st.32x32b + tcgen05.ld.16x128b) and whose
// second goes through shared memory; checked bit for bit against fft_line and timed in-SM beside it, together with
// the two kinds of exchange alone.   Build + run: python -m paper_1806_06467_b200.build --microbench && ./paper_1806_06467_b200/microbench_tmem_fft
#include <cstdio>
#include <cstdint>
#include <cmath>
#include <vector>
#include "fft_core.cuh"
using namespace fresnel;
typedef double2 C;
constexpr int N = 2048, TL = 128, P2 = 130;     // P2: row pitch of the second (shared-memory) exchange

#define TST4(addr, a, b, c, d) asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(a), "r"(b), "r"(c), "r"(d) : "memory")
__device__ __forceinline__ void tld8(uint32_t addr, uint32_t (&r)[8])
{
    asm volatile("tcgen05.ld.sync.aligned.16x128b.x4.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]) : "r"(addr) : "memory");
}
__device__ __forceinline__ uint32_t word_of(const C &z, int p)
{
    const double d = (p < 2) ? z.x : z.y;
    return (p & 1) ? (uint32_t)__double2hiint(d) : (uint32_t)__double2loint(d);
}

// powers w^1..w^15 applied to v[1..15] (forward: multiply by w^q; DIR>0: by conj)
template <int DIR> __device__ __forceinline__ void mul_powers(C (&v)[16], C p1)
{
    v[1] = twmul<DIR>(v[1], p1);
    const C p2 = csq(p1), p3 = cmul(p2, p1), p4 = csq(p2);
    v[2] = twmul<DIR>(v[2], p2); v[3] = twmul<DIR>(v[3], p3);
    C g4 = p4;
#pragma unroll
    for (int mm = 1; mm < 4; ++mm) {
        v[4 * mm] = twmul<DIR>(v[4 * mm], g4);
        v[4 * mm + 1] = twmul<DIR>(v[4 * mm + 1], cmul(g4, p1));
        v[4 * mm + 2] = twmul<DIR>(v[4 * mm + 2], cmul(g4, p2));
        v[4 * mm + 3] = twmul<DIR>(v[4 * mm + 3], cmul(g4, p3));
        if (mm < 3) g4 = (mm == 1) ? csq(g4) : cmul(g4, p4);
    }
}

// v: thread j = 32 m + l, register r <-> element j + 128 r, in and out (natural order both sides)
template <int DIR>
__device__ __forceinline__ void fft2048_tmem(C (&v)[16], int m, int l, C *sbuf, uint32_t tm, const C *__restrict__ tw, const C *__restrict__ tw_old, int bar)
{
    // ---- stage 0: radix 16 over n1 (registers); thread = (n2, n3): n2 = (m, l4 l3), n3 = l2 l1 l0 ----
    dft16<DIR>(v);                                   // v[k1]
    // ---- exchange 1 through tensor memory: registers <- n2, thread <- (n3; k1) ----
#pragma unroll
    for (int p = 0; p < 4; ++p)
#pragma unroll
        for (int q = 0; q < 4; ++q)
            TST4(tm + p * 64 + 16 * q + 4 * m, word_of(v[4 * q], p), word_of(v[4 * q + 1], p), word_of(v[4 * q + 2], p), word_of(v[4 * q + 3], p));
    asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    asm volatile("bar.sync %0, 128;" ::"r"(bar) : "memory");
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    uint32_t wds[4][2][8];
#pragma unroll
    for (int p = 0; p < 4; ++p)
#pragma unroll
        for (int h = 0; h < 2; ++h) tld8(tm + ((uint32_t)(16 * h) << 16) + p * 64 + 16 * m, wds[p][h]);
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
    for (int k = 0; k < 4; ++k)
#pragma unroll
        for (int h = 0; h < 2; ++h)
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int n2 = 4 * k + 2 * h + e;
                v[n2].x = __hiloint2double((int)wds[1][h][2 * k + e], (int)wds[0][h][2 * k + e]);
                v[n2].y = __hiloint2double((int)wds[3][h][2 * k + e], (int)wds[2][h][2 * k + e]);
            }
    const int k1 = 4 * m + (l & 3), n3 = l >> 2;
    // ---- twiddle W_256^(n2 k1), stage 1: radix 16 over n2 ----
    mul_powers<DIR>(v, ldg_c(tw + 8 * k1));
    dft16<DIR>(v);                                   // v[k2]
    // ---- exchange 2 through shared memory: registers <- (n3, k2[3]); thread j' = (k2[2:0], k1) ----
#pragma unroll
    for (int r = 0; r < 16; ++r) sbuf[((r >> 3) + 2 * n3) * P2 + (r & 7) * 16 + k1] = v[r];
    asm volatile("bar.sync %0, 128;" ::"r"(bar) : "memory");
    const int j = 32 * m + l;
#pragma unroll
    for (int r = 0; r < 16; ++r) v[r] = sbuf[r * P2 + j];
    // ---- stage 2: twiddle W_2048^(n3 (k1 + 16 k2)) = (W_2048^(j + 128 b))^n3 and two radix-8 butterflies: the last
    // stage of the plain factorisation, unchanged ----
    fft_stage_compute<double, N, 2, DIR>(v, j, tw_old);
}

template <int VAR>   // 0: fft_line pair (shared memory only), 1: tmem-hybrid pair
__global__ void __launch_bounds__(512, 1) k(int iters, const C *tw_old, const C *tw, const C *in, C *out)
{
    extern __shared__ __align__(16) unsigned char smraw[];
    __shared__ uint32_t tbase;
    const int tid = threadIdx.x, warp = tid >> 5, l = tid & 31;
    const int g = warp & 3, m = warp >> 2, j = 32 * m + l;
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"((uint32_t)__cvta_generic_to_shared(&tbase)), "r"(256u) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tm = tbase + (((uint32_t)(32 * g)) << 16);
    C *sb = reinterpret_cast<C *>(smraw) + (size_t)g * ((VAR == 1 || VAR == 2) ? 16 * P2 : fr_padded_len(N));
    const C *src = in + (size_t)(blockIdx.x * 4 + g) * N;
    C v[16];
#pragma unroll
    for (int r = 0; r < 16; ++r) v[r] = src[j + r * TL];
    for (int it = 0; it < iters; ++it) {
        int mm = m, ll = l; asm volatile("" : "+r"(mm), "+r"(ll));
        const C *t = VAR ? tw : tw_old; asm volatile("" : "+l"(t));
        if (VAR == 0) {
            fft_line<double, N, -1, false, 1, TL>(v, sb, 0, 32 * mm + ll, t, 1 + g);
            if (iters > 1) { asm volatile("" : "+l"(t)); fft_line<double, N, +1, false, 1, TL>(v, sb, 0, 32 * mm + ll, t, 1 + g); }
        } else if (VAR == 2) {
#pragma unroll 1
            for (int rep = 0; rep < 4; ++rep) {
#pragma unroll
                for (int p = 0; p < 4; ++p)
#pragma unroll
                    for (int q = 0; q < 4; ++q)
                        TST4(tm + p * 64 + 16 * q + 4 * mm, word_of(v[4 * q], p), word_of(v[4 * q + 1], p), word_of(v[4 * q + 2], p), word_of(v[4 * q + 3], p));
                asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
                asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
                asm volatile("bar.sync %0, 128;" ::"r"(1 + g) : "memory");
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                uint32_t wds[4][2][8];
#pragma unroll
                for (int p = 0; p < 4; ++p)
#pragma unroll
                    for (int h = 0; h < 2; ++h) tld8(tm + ((uint32_t)(16 * h) << 16) + p * 64 + 16 * mm, wds[p][h]);
                asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
                for (int kk = 0; kk < 4; ++kk)
#pragma unroll
                    for (int h = 0; h < 2; ++h)
#pragma unroll
                        for (int e = 0; e < 2; ++e) {
                            const int n2 = 4 * kk + 2 * h + e;
                            v[n2].x = __hiloint2double((int)wds[1][h][2 * kk + e], (int)wds[0][h][2 * kk + e]);
                            v[n2].y = __hiloint2double((int)wds[3][h][2 * kk + e], (int)wds[2][h][2 * kk + e]);
                        }
                asm volatile("bar.sync %0, 128;" ::"r"(1 + g) : "memory");
            }
        } else if (VAR == 3) {
#pragma unroll 1
            for (int rep = 0; rep < 4; ++rep) {
                fft_stage_scatter<double, N, 0, false, 1>(v, sb, 0, 32 * mm + ll); fr_sync<TL>(1 + g);
                fft_stage_gather<double, N, false, 1>(v, sb, 0, 32 * mm + ll); fr_sync<TL>(1 + g);
            }
        } else {
            fft2048_tmem<-1>(v, mm, ll, sb, tm, t, tw_old, 1 + g);
            if (iters > 1) { asm volatile("" : "+l"(t)); fft2048_tmem<+1>(v, mm, ll, sb, tm, t, tw_old, 1 + g); }
        }
        if (iters > 1) {
#pragma unroll
            for (int r = 0; r < 16; ++r) { v[r].x *= 1.0 / N; v[r].y *= 1.0 / N; }
        }
    }
    C *dst = out + (size_t)(blockIdx.x * 4 + g) * N;
#pragma unroll
    for (int r = 0; r < 16; ++r) dst[j + r * TL] = v[r];
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tbase), "r"(256u) : "memory");
}

int main()
{
    const int lines = 148 * 4;
    std::vector<C> hin((size_t)lines * N), tw(N), two(4096, C{0, 0});
    for (size_t i = 0; i < hin.size(); ++i) { hin[i].x = sin(0.37 * i) + 0.1 * (i % 7); hin[i].y = cos(0.11 * i) - 0.05 * (i % 5); }
    const long double PI = 3.14159265358979323846264338327950288L;
    for (int kk = 0; kk < N; ++kk) { tw[kk].x = (double)cosl(-2 * PI * kk / N); tw[kk].y = (double)sinl(-2 * PI * kk / N); }
    // stage tables of the existing code for N = 2048: stage 1 (NS=16): W_256^k, k<16 at offset 0; stage 2 (NS=256, R=8): W_2048^k, k<256 at offset 16
    for (int kk = 0; kk < 16; ++kk) { two[kk].x = (double)cosl(-2 * PI * kk / 256); two[kk].y = (double)sinl(-2 * PI * kk / 256); }
    for (int kk = 0; kk < 256; ++kk) { two[16 + kk].x = (double)cosl(-2 * PI * kk / 2048); two[16 + kk].y = (double)sinl(-2 * PI * kk / 2048); }
    C *din, *dtw, *dtwo, *o0, *o1;
    cudaMalloc(&din, hin.size() * sizeof(C)); cudaMalloc(&o0, hin.size() * sizeof(C)); cudaMalloc(&o1, hin.size() * sizeof(C));
    cudaMalloc(&dtw, N * sizeof(C)); cudaMalloc(&dtwo, 4096 * sizeof(C));
    cudaMemcpy(din, hin.data(), hin.size() * sizeof(C), cudaMemcpyHostToDevice);
    cudaMemcpy(dtw, tw.data(), N * sizeof(C), cudaMemcpyHostToDevice);
    cudaMemcpy(dtwo, two.data(), 4096 * sizeof(C), cudaMemcpyHostToDevice);
    const int smem0 = 4 * fr_padded_len(N) * sizeof(C), smem1 = 4 * 16 * P2 * sizeof(C);
    cudaFuncSetAttribute(k<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem0);
    cudaFuncSetAttribute(k<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem1);
    // correctness: one forward transform each
    k<0><<<148, 512, smem0>>>(1, dtwo, dtw, din, o0);
    k<1><<<148, 512, smem1>>>(1, dtwo, dtw, din, o1);
    cudaError_t e = cudaDeviceSynchronize();
    std::vector<C> h0(hin.size()), h1(hin.size());
    cudaMemcpy(h0.data(), o0, h0.size() * sizeof(C), cudaMemcpyDeviceToHost);
    cudaMemcpy(h1.data(), o1, h1.size() * sizeof(C), cudaMemcpyDeviceToHost);
    double num = 0, den = 0;
    for (size_t i = 0; i < h0.size(); ++i) { num += (h0[i].x - h1[i].x) * (h0[i].x - h1[i].x) + (h0[i].y - h1[i].y) * (h0[i].y - h1[i].y); den += h0[i].x * h0[i].x + h0[i].y * h0[i].y; }
    printf("forward transform, tmem-hybrid vs fft_line: relative L2 difference %.3e  (%s)\n", sqrt(num / den), cudaGetErrorString(e));
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    const int iters = 400;
    for (int var = 0; var < 2; ++var) {
        float best = 1e30f;
        for (int rep = 0; rep < 3; ++rep) {
            cudaEventRecord(e0);
            if (var == 0) k<0><<<148, 512, smem0>>>(iters, dtwo, dtw, din, o0); else k<1><<<148, 512, smem1>>>(iters, dtwo, dtw, din, o1);
            cudaEventRecord(e1); e = cudaEventSynchronize(e1);
            float ms; cudaEventElapsedTime(&ms, e0, e1); if (ms < best) best = ms;
        }
        printf("%s transform pair, 4 lines per SM: %.3f clk/element/SM  (%s)\n", var ? "tmem-hybrid" : "fft_line   ", best * 1e-3 * 1.965e9 / iters / (4.0 * N), cudaGetErrorString(e));
    }
    cudaFuncSetAttribute(k<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem1);
    cudaFuncSetAttribute(k<3>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem0);
    for (int var = 2; var < 4; ++var) {
        float best = 1e30f;
        for (int rep = 0; rep < 3; ++rep) {
            cudaEventRecord(e0);
            if (var == 2) k<2><<<148, 512, smem1>>>(iters, dtwo, dtw, din, o0); else k<3><<<148, 512, smem0>>>(iters, dtwo, dtw, din, o0);
            cudaEventRecord(e1); e = cudaEventSynchronize(e1);
            float ms; cudaEventElapsedTime(&ms, e0, e1); if (ms < best) best = ms;
        }
        printf("%s exchange alone (x4 per iteration), 4 lines per SM: %.3f clk/element/SM per exchange (%s)\n", var == 2 ? "tensor-memory" : "shared-memory", best * 1e-3 * 1.965e9 / iters / (4.0 * N) / 4, cudaGetErrorString(e));
    }
    // round trip check of the hybrid (fwd + inv + 1/N repeated keeps the input)
    cudaMemcpy(h1.data(), o1, h1.size() * sizeof(C), cudaMemcpyDeviceToHost);
    num = den = 0;
    for (size_t i = 0; i < h1.size(); ++i) { num += (hin[i].x - h1[i].x) * (hin[i].x - h1[i].x) + (hin[i].y - h1[i].y) * (hin[i].y - h1[i].y); den += hin[i].x * hin[i].x + hin[i].y * hin[i].y; }
    printf("tmem-hybrid: %d round trips reproduce the input to %.3e\n", iters, sqrt(num / den));
    return 0;
}
