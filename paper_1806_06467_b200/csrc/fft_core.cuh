// fft_core.cuh -- register-resident Stockham FFT building blocks for sm_100a.
//
// One FFT "line" of N points (N = 64 .. 8192, power of two) is held by N/16 threads, 16 complex
// elements per thread.  Invariant before and after a whole transform:
//        thread j (0 <= j < N/16), register r (0 <= r < 16)  <->  element index  j + r * N/16
// which is exactly the coalesced global-memory access pattern, so a transform can be followed by a
// pointwise multiply and another transform without any reshuffle (the fused angular-spectrum pass).
//
// The transform is the decimation-in-time Stockham autosort factorisation N = R_1 * R_2 * ... with
// R = 16 for every stage but the last (the remainder 2/4/8/16).  Stage s (Ns = R_1*...*R_{s-1}):
//        for butterfly jb:  k = jb mod Ns;  v_t = y[jb + t*N/R] * W_{Ns*R}^{t*k};  z = DFT_R(v);
//                           y'[(jb-k)*R + k + q*Ns] = z_q
// Between stages the line lives in shared memory (one exchange = one store + one load per
// element); butterflies, twiddles and pointwise multiplies all happen in registers.
// Twiddles W_{Ns*R}^{t*k} are precomputed on the host in long double (tables.cu) -- never by
// recurrence -- and read through the read-only path.
#pragma once
#include <cuda_runtime.h>

namespace fresnel {

template <typename T> struct cplx_of;
template <> struct cplx_of<float>  { using type = float2; };
template <> struct cplx_of<double> { using type = double2; };

#define FR_DEV __device__ __forceinline__

template <typename C> FR_DEV C cadd(C a, C b) { C r; r.x = a.x + b.x; r.y = a.y + b.y; return r; }
template <typename C> FR_DEV C csub(C a, C b) { C r; r.x = a.x - b.x; r.y = a.y - b.y; return r; }
template <typename C> FR_DEV C cmul(C a, C b) { C r; r.x = a.x * b.x - a.y * b.y; r.y = a.x * b.y + a.y * b.x; return r; }
// a * conj(b)
template <typename C> FR_DEV C cmulc(C a, C b) { C r; r.x = a.x * b.x + a.y * b.y; r.y = a.y * b.x - a.x * b.y; return r; }

// DIR = -1: forward kernel exp(-2 pi i ...); DIR = +1: inverse kernel.  Tables hold FORWARD twiddles.
template <int DIR, typename C> FR_DEV C twmul(C a, C w) { return DIR < 0 ? cmul(a, w) : cmulc(a, w); }
// w * w
template <typename C> FR_DEV C csq(C w) { C r; r.x = w.x * w.x - w.y * w.y; r.y = (w.x + w.x) * w.y; return r; }

// multiply by -i (DIR<0) or +i (DIR>0):  the radix-4 quarter turn
template <int DIR, typename C> FR_DEV C rot90(C a)
{
    C r;
    if (DIR < 0) { r.x = a.y; r.y = -a.x; } else { r.x = -a.y; r.y = a.x; }
    return r;
}

// cos(2 pi m / 16), sin(2 pi m / 16), m = 0..15, to 25 digits
template <typename T> struct W16 {
    __host__ __device__ static constexpr T c(int m)
    {
        constexpr double t[16] = {1.0, 0.9238795325112867561281832, 0.7071067811865475244008444, 0.3826834323650897717284600,
                                  0.0, -0.3826834323650897717284600, -0.7071067811865475244008444, -0.9238795325112867561281832,
                                  -1.0, -0.9238795325112867561281832, -0.7071067811865475244008444, -0.3826834323650897717284600,
                                  0.0, 0.3826834323650897717284600, 0.7071067811865475244008444, 0.9238795325112867561281832};
        return (T)t[m & 15];
    }
    __host__ __device__ static constexpr T s(int m) { return c((m + 12) & 15); }   // sin(x) = cos(x - pi/2)
};

// a * W16^M  (forward: exp(-2 pi i M/16); inverse: conjugate), M a compile-time constant
template <int M, int DIR, typename C> FR_DEV C mulw16(C a)
{
    using T = decltype(a.x);
    constexpr int m = M & 15;
    if constexpr (m == 0) return a;
    else if constexpr (m == 4) return rot90<DIR>(a);
    else if constexpr (m == 8) { C r; r.x = -a.x; r.y = -a.y; return r; }
    else if constexpr (m == 12) return rot90<-DIR>(a);
    else {
        constexpr T c = W16<T>::c(m);
        constexpr T s = (DIR < 0 ? -1 : 1) * W16<T>::s(m);
        C r;
        r.x = a.x * c - a.y * s;
        r.y = a.x * s + a.y * c;
        return r;
    }
}

template <int DIR, typename C> FR_DEV void dft2(C &a, C &b)
{
    C t = a;
    a = cadd(t, b);
    b = csub(t, b);
}

// natural order in, natural order out
template <int DIR, typename C> FR_DEV void dft4(C &a0, C &a1, C &a2, C &a3)
{
    C s0 = cadd(a0, a2), d0 = csub(a0, a2);
    C s1 = cadd(a1, a3), d1 = rot90<DIR>(csub(a1, a3));
    a0 = cadd(s0, s1);
    a2 = csub(s0, s1);
    a1 = cadd(d0, d1);
    a3 = csub(d0, d1);
}

template <int DIR, typename C> FR_DEV void dft8(C &a0, C &a1, C &a2, C &a3, C &a4, C &a5, C &a6, C &a7)
{
    // t = 2*t1 + t0: radix-4 over the evens and over the odds, twiddle W8^q on the odds, radix-2
    dft4<DIR>(a0, a2, a4, a6);
    dft4<DIR>(a1, a3, a5, a7);
    C o1 = mulw16<2, DIR>(a3), o2 = mulw16<4, DIR>(a5), o3 = mulw16<6, DIR>(a7);
    C e0 = a0, e1 = a2, e2 = a4, e3 = a6, o0 = a1;
    a0 = cadd(e0, o0); a4 = csub(e0, o0);
    a1 = cadd(e1, o1); a5 = csub(e1, o1);
    a2 = cadd(e2, o2); a6 = csub(e2, o2);
    a3 = cadd(e3, o3); a7 = csub(e3, o3);
}

// 16-point DFT on v[0..15], natural order in and out (4 x 4 with the W16 twiddles in between)
template <int DIR, typename C> FR_DEV void dft16(C (&v)[16])
{
    // step 1: for each t0, radix-4 over t1 (elements t0, t0+4, t0+8, t0+12) -> y[t0][q1] in v[t0 + 4*q1]
#pragma unroll
    for (int t0 = 0; t0 < 4; ++t0) dft4<DIR>(v[t0], v[t0 + 4], v[t0 + 8], v[t0 + 12]);
    // step 2: y[t0][q1] *= W16^(t0*q1)
    v[5] = mulw16<1, DIR>(v[5]);   v[9] = mulw16<2, DIR>(v[9]);   v[13] = mulw16<3, DIR>(v[13]);
    v[6] = mulw16<2, DIR>(v[6]);   v[10] = mulw16<4, DIR>(v[10]); v[14] = mulw16<6, DIR>(v[14]);
    v[7] = mulw16<3, DIR>(v[7]);   v[11] = mulw16<6, DIR>(v[11]); v[15] = mulw16<9, DIR>(v[15]);
    // step 3: for each q1, radix-4 over t0 (elements 4*q1 + t0) -> X[q1 + 4*q0] in v[4*q1 + q0]
#pragma unroll
    for (int q1 = 0; q1 < 4; ++q1) dft4<DIR>(v[4 * q1], v[4 * q1 + 1], v[4 * q1 + 2], v[4 * q1 + 3]);
    // step 4: un-transpose (compile-time register renaming): v[4*q1 + q0] holds X[q1 + 4*q0]
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int b = a + 1; b < 4; ++b) {
            C t = v[4 * a + b];
            v[4 * a + b] = v[4 * b + a];
            v[4 * b + a] = t;
        }
}

// ---- compile-time factorisation -----------------------------------------------------------------
// N = 16 * 16 * ... * last, last in {2, 4, 8, 16}
__host__ __device__ constexpr int fr_num_stages(int N)
{
    int s = 0;
    while (N > 1) { N /= (N >= 16 ? 16 : N); ++s; }
    return s;
}
__host__ __device__ constexpr int fr_radix(int N, int stage)   // stage = 0-based
{
    int r = 1;
    for (int s = 0; s <= stage; ++s) { r = (N >= 16 ? 16 : N); N /= r; }
    return r;
}
__host__ __device__ constexpr int fr_ns(int N, int stage)      // product of the radices before `stage`
{
    int ns = 1;
    for (int s = 0; s < stage; ++s) { int r = (N >= 16 ? 16 : N); N /= r; ns *= r; }
    return ns;
}
// offset (in complex elements) of stage `stage`'s twiddle table inside the per-N table; stage >= 1.
// A stage table holds only the BASE twiddles w_k = W_{Ns*R}^k, k = 0..Ns-1 (exactly rounded, built
// in long double on the host).  The powers w_k^t, t = 2..R-1, are generated in registers by at most
// five chained multiplications: one 16-byte load costs the load/store pipe as much as eight FP64
// instructions cost the FP64 pipe, a complex multiply is four.
__host__ __device__ constexpr int fr_tw_offset(int N, int stage)
{
    int off = 0;
    for (int s = 1; s < stage; ++s) off += fr_ns(N, s);
    return off;
}
__host__ __device__ constexpr int fr_tw_total(int N) { return fr_tw_offset(N, fr_num_stages(N)); }

// padded shared-memory position: one spare element every 16 keeps both the strided scatter of a
// stage and the contiguous gather of the next free of bank conflicts
__host__ __device__ constexpr int fr_pad(int a) { return a + (a >> 4); }
__host__ __device__ constexpr int fr_padded_len(int N) { return N + N / 16; }

// Shared-memory slot of padded position `p` of line `line`:
//   column pass (COL): lines interleaved (a warp holds W adjacent columns of the same rows),
//   row pass:          lines back to back (a warp stays inside one line).
template <int N, bool COL, int W> FR_DEV int fr_slot(int p, int line)
{
    return COL ? p * W + line : line * fr_padded_len(N) + p;
}

template <typename C> FR_DEV C ldg_c(const C *p) { return __ldg(p); }

// Barrier among the threads that share one exchange buffer.  GT = 0: the whole CTA;
// GT = 32: one warp; otherwise a named barrier over GT threads (id 1..15) so that the line
// groups of a CTA run independently of one another.
template <int GT> FR_DEV void fr_sync(int bar_id)
{
    if constexpr (GT == 0) __syncthreads();
    else if constexpr (GT == 32) __syncwarp();
    else asm volatile("bar.sync %0, %1;" ::"r"(bar_id), "n"(GT) : "memory");
}

// One Stockham stage = compute (twiddles + butterflies, registers only) -> scatter -> barrier ->
// gather -> barrier.  STAGE is 0-based.
// v[b + q*B] *= w^q, w = W_{Ns*R}^k, k = (j + b*N/16) mod Ns  (none in stage 0: Ns = 1)
template <typename T, int N, int STAGE, int DIR>
FR_DEV void fft_stage_twiddle(typename cplx_of<T>::type (&v)[16], int j, const typename cplx_of<T>::type *__restrict__ tw)
{
    using C = typename cplx_of<T>::type;
    constexpr int TL = N / 16;
    constexpr int R = fr_radix(N, STAGE);
    constexpr int NS = fr_ns(N, STAGE);
    constexpr int B = 16 / R;
    if constexpr (STAGE > 0) {
        const C *t = tw + fr_tw_offset(N, STAGE);
#pragma unroll
        for (int b = 0; b < B; ++b) {
            const int k = (j + b * TL) & (NS - 1);
            const C p1 = ldg_c(t + k);
            v[b + B] = twmul<DIR>(v[b + B], p1);
            if constexpr (R >= 4) {
                const C p2 = csq(p1), p3 = cmul(p2, p1);
                v[b + 2 * B] = twmul<DIR>(v[b + 2 * B], p2);
                v[b + 3 * B] = twmul<DIR>(v[b + 3 * B], p3);
                if constexpr (R >= 8) {
                    const C p4 = csq(p2);
                    C g = p4;                                        // w^(4m)
#pragma unroll
                    for (int m = 1; m < R / 4; ++m) {                // block m: w^(4m) .. w^(4m+3)
                        v[b + (4 * m) * B] = twmul<DIR>(v[b + (4 * m) * B], g);
                        v[b + (4 * m + 1) * B] = twmul<DIR>(v[b + (4 * m + 1) * B], cmul(g, p1));
                        v[b + (4 * m + 2) * B] = twmul<DIR>(v[b + (4 * m + 2) * B], cmul(g, p2));
                        v[b + (4 * m + 3) * B] = twmul<DIR>(v[b + (4 * m + 3) * B], cmul(g, p3));
                        if (m + 1 < R / 4) g = (m == 1) ? csq(g) : cmul(g, p4);   // w^8 = (w^4)^2, w^12 = w^8 * w^4
                    }
                }
            }
        }
    }
}

// B = 16/R butterflies of radix R over v[b + q*B], q = 0..R-1
template <typename T, int N, int STAGE, int DIR>
FR_DEV void fft_stage_butterfly(typename cplx_of<T>::type (&v)[16])
{
    constexpr int R = fr_radix(N, STAGE);
    constexpr int B = 16 / R;
    constexpr bool LAST = (STAGE == fr_num_stages(N) - 1);
    static_assert(LAST || R == 16, "only the last stage may have a radix below 16");
    if constexpr (R == 16) {
        dft16<DIR>(v);
    } else if constexpr (R == 8) {
#pragma unroll
        for (int b = 0; b < B; ++b)
            dft8<DIR>(v[b], v[b + B], v[b + 2 * B], v[b + 3 * B], v[b + 4 * B], v[b + 5 * B], v[b + 6 * B], v[b + 7 * B]);
    } else if constexpr (R == 4) {
#pragma unroll
        for (int b = 0; b < B; ++b) dft4<DIR>(v[b], v[b + B], v[b + 2 * B], v[b + 3 * B]);
    } else {
#pragma unroll
        for (int b = 0; b < B; ++b) dft2<DIR>(v[b], v[b + B]);
    }
}

// decimation in time: twiddles on the inputs, then the butterflies
template <typename T, int N, int STAGE, int DIR>
FR_DEV void fft_stage_compute(typename cplx_of<T>::type (&v)[16], int j, const typename cplx_of<T>::type *__restrict__ tw)
{
    fft_stage_twiddle<T, N, STAGE, DIR>(v, j, tw);
    fft_stage_butterfly<T, N, STAGE, DIR>(v);
}

// scatter the outputs of stage STAGE (not the last) into the exchange buffer
template <typename T, int N, int STAGE, bool COL, int W>
FR_DEV void fft_stage_scatter(const typename cplx_of<T>::type (&v)[16], typename cplx_of<T>::type *buf, int line, int j)
{
    constexpr int NS = fr_ns(N, STAGE);
    const int k = j & (NS - 1);
    const int base = (j - k) * 16 + k;          // + q*NS ; NS is 1 or a multiple of 16
    if constexpr (NS == 1) {
        const int p0 = j * 17;                  // fr_pad(16*j + q) = 17*j + q
#pragma unroll
        for (int q = 0; q < 16; ++q) buf[fr_slot<N, COL, W>(p0 + q, line)] = v[q];
    } else {
        const int p0 = fr_pad(base);
#pragma unroll
        for (int q = 0; q < 16; ++q) buf[fr_slot<N, COL, W>(p0 + q * (NS + NS / 16), line)] = v[q];
    }
}

// gather the inputs of the next stage: element j + r*N/16 into register r
template <typename T, int N, bool COL, int W>
FR_DEV void fft_stage_gather(typename cplx_of<T>::type (&v)[16], const typename cplx_of<T>::type *buf, int line, int j)
{
    constexpr int TL = N / 16;
    if constexpr (TL % 16 == 0) {
        const int p0 = fr_pad(j);
#pragma unroll
        for (int r = 0; r < 16; ++r) v[r] = buf[fr_slot<N, COL, W>(p0 + r * (TL + TL / 16), line)];
    } else {
#pragma unroll
        for (int r = 0; r < 16; ++r) v[r] = buf[fr_slot<N, COL, W>(fr_pad(j + r * TL), line)];
    }
}

template <typename T, int N, int STAGE, int DIR, bool COL, int W, int GT = 0>
FR_DEV void fft_stage(typename cplx_of<T>::type (&v)[16], typename cplx_of<T>::type *buf, int line, int j,
                      const typename cplx_of<T>::type *__restrict__ tw, int bar_id = 0)
{
    constexpr bool LAST = (STAGE == fr_num_stages(N) - 1);
    fft_stage_compute<T, N, STAGE, DIR>(v, j, tw);
    // ---- exchange through shared memory (the last stage's output is already in place) ----
    if constexpr (!LAST) {
        fft_stage_scatter<T, N, STAGE, COL, W>(v, buf, line, j);
        fr_sync<GT>(bar_id);
        fft_stage_gather<T, N, COL, W>(v, buf, line, j);
        fr_sync<GT>(bar_id);
    }
}

// Whole transform of one line: v in, v out, both in the (thread j, register r) <-> j + r*N/16 layout.
template <typename T, int N, int DIR, bool COL, int W, int GT = 0>
FR_DEV void fft_line(typename cplx_of<T>::type (&v)[16], typename cplx_of<T>::type *buf, int line, int j,
                     const typename cplx_of<T>::type *__restrict__ tw, int bar_id = 0)
{
    constexpr int S = fr_num_stages(N);
    fft_stage<T, N, 0, DIR, COL, W, GT>(v, buf, line, j, tw, bar_id);
    if constexpr (S > 1) fft_stage<T, N, 1, DIR, COL, W, GT>(v, buf, line, j, tw, bar_id);
    if constexpr (S > 2) fft_stage<T, N, 2, DIR, COL, W, GT>(v, buf, line, j, tw, bar_id);
    if constexpr (S > 3) fft_stage<T, N, 3, DIR, COL, W, GT>(v, buf, line, j, tw, bar_id);
}

} // namespace fresnel
