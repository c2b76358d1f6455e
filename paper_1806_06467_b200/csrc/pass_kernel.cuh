// pass_kernel.cuh -- ONE HBM round trip of the Fresnel hot path.
//
// A pass reads every line (row or column) of a [batch][N][N] wavefront once, and on chip does
//     [optic phasor A*exp(2 pi i OPD/lambda)]  (row pass only; Eq. 3)
//  -> [x pre[n]]                                (1-D chirp table: lens / Fresnel QPF, Eq. 2)
//  -> FFT (MODE_FWD, MODE_CONV) or inverse FFT (MODE_INV)
//  -> [x mid[k]]                                (transfer function H1 / output chirp / 1/N / signs)
//  -> inverse FFT                               (MODE_CONV only)
//  -> [x scale] [x rowfac[row]]               (row pass: the y-part of the input chirp, constant along a row)
//  -> MODE_CONV2 only: the optic of the NEXT surface -- [optic phasor] [x lens2[n] x lens2[line]] -- and a second
//     convolution FFT -> x mid2[k] -> inverse FFT (fused trains, see fresnel_system_run)
// and writes the line back in place.  Angular-spectrum propagation is MODE_CONV over rows then
// over columns (H is separable); fft2d and direct Fresnel are MODE_FWD/MODE_INV over rows then
// columns.  Shifts are folded into the tables ((-1)^n signs) and never touch memory.
//
// MODE_CONV2 (train-level fusion).  The row and the column convolution of a surface commute, so a train
// of angular-spectrum surfaces can be ordered  rows_0 | cols_0, optic_1, cols_1 | rows_1, optic_2, rows_2 | ...:
// the last convolution of surface s-1 and the first of surface s run along the same direction and, with the
// optic of surface s between them, on ONE resident line -- n+1 passes over the wavefront instead of 2n.
#pragma once
#include <atomic>
#include <cstdint>
#include "fft_core.cuh"

namespace fresnel {

enum PassMode { MODE_FWD = 0, MODE_INV = 1, MODE_CONV = 2, MODE_CONV2 = 3 };

template <typename T> struct PassArgs {
    using C = typename cplx_of<T>::type;
    C *wf;                    // [batch][N][N]
    const C *pre;             // [batch][N] or nullptr
    const C *mid;             // [batch][N] or nullptr
    const C *rowfac;          // [batch][N] or nullptr (row pass only): row i of the result is multiplied by rowfac[i]
    const C *tw;              // FFT twiddle tables of this N
    const T *amp;             // [N][N] or nullptr (row pass only)
    const T *opd;             // [N][N] or nullptr (row pass only)
    const double *inv_lambda; // [batch] 1/lambda (only read when opd != nullptr)
    T scale;                  // applied last when != 1
    int prefetch_distance;    // tiles ahead to prefetch into L2 (0: off); ~ number of resident CTAs
    int pdl;                  // launched with programmatic stream serialization
    // MODE_CONV2: the optic between the two convolutions and the second transfer function
    const C *lens2;           // [batch][N] lens chirp of the in-between optic (applied as lens2[n] * lens2[line]) or nullptr
    const C *mid2;            // [batch][N] transfer function (with 1/N) of the second convolution
    const T *amp2;            // [N][N] or nullptr.  TMA column pass: only null / non-null matters (the tile comes
    const T *opd2;            //                     through the tensor maps given to the launcher)
};

// Programmatic dependent launch: every pass kernel depends on ALL of the previous pass (a 2-D transform is
// two global transposes), so kernels cannot overlap their work -- but the next kernel's launch latency and
// prologue can hide under the previous kernel's last wave.  A pass kernel lets its dependents launch at once
// and waits for its own predecessor right before its first global access.
FR_DEV void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
FR_DEV void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

template <typename... KArgs, typename... Args>
cudaError_t launch_pdl(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t stream, bool pdl, Args... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kern, args...);
}

// cudaFuncSetAttribute(MaxDynamicSharedMemorySize) is a per-device setting: every launcher keeps one bit per
// device ordinal (setting the attribute twice is harmless, so two threads racing here are too)
inline bool fr_needs_configuring(const std::atomic<unsigned long long> &mask)
{
    int dev = 0;
    cudaGetDevice(&dev);
    return !((mask.load(std::memory_order_acquire) >> (dev & 63)) & 1ull);
}
inline void fr_mark_configured(std::atomic<unsigned long long> &mask)
{
    int dev = 0;
    cudaGetDevice(&dev);
    mask.fetch_or(1ull << (dev & 63), std::memory_order_release);
}

// bulk L2 prefetch of a contiguous range (bytes: multiple of 16)
FR_DEV void l2_prefetch_bulk(const void *p, uint32_t bytes)
{
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p), "r"(bytes) : "memory");
}

// exp(2 pi i u) for a phase u given in turns (optic phasor, Eq. 3).  Surface maps are a small fraction of a
// wave, so the common case |u| <= 1/8 is a pair of Taylor polynomials in u^2 with coefficients (2 pi)^n / n!
// (truncation < 1e-19 double, < 3e-9 float): no range reduction, no quadrant logic, no branch.  Larger phases
// go through phasor_turns_any (out of line, so that the common path stays small).
FR_DEV double2 phasor_turns_small(double u)
{
    const double t = u * u;
    double s = 0.1042291622081398411727104, c = 0.2820059684557912150702702;
    s = fma(s, t, -0.7181223017785005122317403);  c = fma(c, t, -1.714390711088672065421586);
    s = fma(s, t, 3.819952584848282127733792);    c = fma(c, t, 7.903536371318468804212103);
    s = fma(s, t, -15.09464257682299039182662);   c = fma(c, t, -26.42625678337439745290065);
    s = fma(s, t, 42.05869394489765314498681);    c = fma(c, t, 60.24464137187666036272111);
    s = fma(s, t, -76.70585975306138584163064);   c = fma(c, t, -85.45681720669372773601951);
    s = fma(s, t, 81.60524927607505420339768);    c = fma(c, t, 64.93939402266829149096022);
    s = fma(s, t, -41.34170224039976023396842);   c = fma(c, t, -19.73920880217871723766898);
    s = fma(s, t, 6.283185307179586476925287);    c = fma(c, t, 1.0);
    return make_double2(c, s * u);
}
FR_DEV float2 phasor_turns_small(float u)
{
    const float t = u * u;
    float s = -15.09464257682299039182662f, c = -26.42625678337439745290065f;
    s = fmaf(s, t, 42.05869394489765314498681f);   c = fmaf(c, t, 60.24464137187666036272111f);
    s = fmaf(s, t, -76.70585975306138584163064f);  c = fmaf(c, t, -85.45681720669372773601951f);
    s = fmaf(s, t, 81.60524927607505420339768f);   c = fmaf(c, t, 64.93939402266829149096022f);
    s = fmaf(s, t, -41.34170224039976023396842f);  c = fmaf(c, t, -19.73920880217871723766898f);
    s = fmaf(s, t, 6.283185307179586476925287f);   c = fmaf(c, t, 1.0f);
    return make_float2(c, s * u);
}
static __device__ __noinline__ double2 phasor_turns_any(double u)
{
    double s, c;
    sincospi(2.0 * u, &s, &c);
    return make_double2(c, s);
}
static __device__ __noinline__ float2 phasor_turns_any(float u)
{
    float s, c;
    sincospif(2.0f * u, &s, &c);
    return make_float2(c, s);
}
FR_DEV bool phasor_is_small(double u) { return fabs(u) <= 0.125; }
FR_DEV bool phasor_is_small(float u) { return fabsf(u) <= 0.125f; }
template <typename T> FR_DEV typename cplx_of<T>::type phasor_turns(T u)
{
    return phasor_is_small(u) ? phasor_turns_small(u) : phasor_turns_any(u);
}

// v[r] *= exp(2 pi i * opd[r*stride] * inv_lambda), r = 0..15: polynomial for all sixteen, then the rare
// large phases one by one
template <typename T>
FR_DEV void apply_opd16(typename cplx_of<T>::type (&v)[16], const T *__restrict__ o, size_t stride, T inv_lambda)
{
    T u[16];
    bool all_small = true;
#pragma unroll
    for (int r = 0; r < 16; ++r) {
        u[r] = o[r * stride] * inv_lambda;
        all_small = all_small && phasor_is_small(u[r]);
    }
    if (all_small) {
#pragma unroll
        for (int r = 0; r < 16; ++r) v[r] = cmul(v[r], phasor_turns_small(u[r]));
    } else {
#pragma unroll
        for (int r = 0; r < 16; ++r) v[r] = cmul(v[r], phasor_turns_any(u[r]));
    }
}

// The transforms of one resident line, for every mode, as a ROLLED loop over ONE copy of the forward transform:
// an inverse transform is conj o forward o conj, and the conjugations fold into the neighbouring multiplies
// (bit-identical to a transform with conjugated twiddles: negation is exact).  One copy keeps the instruction
// footprint at a quarter of the unrolled fused kernel, and -- what matters -- keeps ptxas from spilling: four
// inlined transforms cost 150-350 bytes of spill traffic per thread on the load/store pipe the exchanges need.
//   MODE_FWD   F, [x mid]                         MODE_INV   conj, F, conj, [x mid]
//   MODE_CONV  F, x mid, conj, F, conj            MODE_CONV2 the same twice, optic2(v) in between, then mid2
template <typename T, int N, int MODE, bool COL, int W, int GT, typename Optic2>
FR_DEV void line_transforms(typename cplx_of<T>::type (&v)[16], typename cplx_of<T>::type *buf, int line, int j, int b,
                            const PassArgs<T> &a, int bar_id, Optic2 &&optic2)
{
    using C = typename cplx_of<T>::type;
    constexpr int TL = N / 16;
    constexpr int NIT = MODE == MODE_CONV2 ? 4 : (MODE == MODE_CONV ? 2 : 1);
    const C *m = a.mid != nullptr ? a.mid + (size_t)b * N : nullptr;
    if constexpr (MODE == MODE_INV) {
#pragma unroll
        for (int r = 0; r < 16; ++r) v[r].y = -v[r].y;
    }
#pragma unroll 1
    for (int it = 0; it < NIT; ++it) {
        fft_line<T, N, -1, COL, W, GT>(v, buf, line, j, a.tw, bar_id);
        if constexpr (MODE == MODE_FWD) {
            if (m != nullptr) {
#pragma unroll
                for (int r = 0; r < 16; ++r) v[r] = cmul(v[r], ldg_c(m + j + r * TL));
            }
        } else if constexpr (MODE == MODE_INV) {
            if (m != nullptr) {
#pragma unroll
                for (int r = 0; r < 16; ++r) v[r] = cmulc(ldg_c(m + j + r * TL), v[r]);      // mid * conj(v)
            } else {
#pragma unroll
                for (int r = 0; r < 16; ++r) v[r].y = -v[r].y;
            }
        } else if ((it & 1) == 0) {
            // x transfer function, conjugated for the inverse transform that follows.  (m is never null here; the
            // branch keeps the 16 table loads from being hoisted into the transform, where they would cost registers)
            if (m != nullptr) {
#pragma unroll
                for (int r = 0; r < 16; ++r) {
                    const C t = cmul(v[r], ldg_c(m + j + r * TL));
                    v[r].x = t.x; v[r].y = -t.y;
                }
            }
        } else {
#pragma unroll
            for (int r = 0; r < 16; ++r) v[r].y = -v[r].y;
            if constexpr (MODE == MODE_CONV2) {
                if (it == 1) {
                    optic2(v);
                    m = a.mid2 + (size_t)b * N;
                }
            }
        }
    }
}

template <typename T, int N, bool COL, int W, int MODE, int MINB>
__global__ void __launch_bounds__(W *(N / 16), MINB) pass_kernel(PassArgs<T> a)
{
    using C = typename cplx_of<T>::type;
    constexpr int TL = N / 16;
    extern __shared__ __align__(16) unsigned char fr_smem[];
    C *buf = reinterpret_cast<C *>(fr_smem);

    const int tid = threadIdx.x;
    const int line = COL ? tid % W : tid / TL;
    const int j = COL ? tid / W : tid % TL;
    const int b = blockIdx.y;
    const int idx = blockIdx.x * W + line;                    // row (row pass) or column (column pass)
    const size_t gstride = COL ? (size_t)N : (size_t)1;
    C *g = a.wf + (size_t)b * N * N + (COL ? (size_t)idx : (size_t)idx * N);

    pdl_launch_dependents();
    pdl_wait();
    C v[16];
#pragma unroll
    for (int r = 0; r < 16; ++r) v[r] = g[(size_t)(j + r * TL) * gstride];

    if constexpr (!COL) {
        // L2 prefetch of the rows (and map rows) a later CTA will load: one bulk request per row
        if (j == 0 && a.prefetch_distance > 0) {
            const int nx = (int)gridDim.x;
            int t = (int)blockIdx.x + a.prefetch_distance, bb = b;
            while (t >= nx) { t -= nx; ++bb; }
            if (bb < (int)gridDim.y) {
                const size_t row = (size_t)t * W + line;
                l2_prefetch_bulk(a.wf + (size_t)bb * N * N + row * N, (uint32_t)(N * sizeof(C)));
                if (a.opd != nullptr) l2_prefetch_bulk(a.opd + row * N, (uint32_t)(N * sizeof(T)));
                if (a.amp != nullptr) l2_prefetch_bulk(a.amp + row * N, (uint32_t)(N * sizeof(T)));
            }
        }
    }
    if constexpr (!COL && MODE == MODE_CONV2) {
        // the map rows of the in-between optic are needed one convolution from now: ask L2 for them
        if (j == 0) {
            if (a.opd2 != nullptr) l2_prefetch_bulk(a.opd2 + (size_t)idx * N, (uint32_t)(N * sizeof(T)));
            if (a.amp2 != nullptr) l2_prefetch_bulk(a.amp2 + (size_t)idx * N, (uint32_t)(N * sizeof(T)));
        }
    }
    if constexpr (!COL) {
        if (a.opd != nullptr) {
            apply_opd16<T>(v, a.opd + (size_t)idx * N + j, TL, (T)a.inv_lambda[b]);
        }
        if (a.amp != nullptr) {
            const T *m = a.amp + (size_t)idx * N;
#pragma unroll
            for (int r = 0; r < 16; ++r) {
                T s = m[j + r * TL];
                v[r].x *= s; v[r].y *= s;
            }
        }
    }
    if (a.pre != nullptr) {
        const C *p = a.pre + (size_t)b * N;
#pragma unroll
        for (int r = 0; r < 16; ++r) v[r] = cmul(v[r], ldg_c(p + j + r * TL));
    }

    line_transforms<T, N, MODE, COL, W, 0>(v, buf, line, j, b, a, 0, [&](C (&u)[16]) {
        // MODE_CONV2: the optic of the next surface on the resident line
        const size_t mstride = COL ? (size_t)TL * N : (size_t)TL;
        const size_t m0 = COL ? (size_t)j * N + idx : (size_t)idx * N + j;
        if (a.opd2 != nullptr) apply_opd16<T>(u, a.opd2 + m0, mstride, (T)a.inv_lambda[b]);
        if (a.amp2 != nullptr) {
#pragma unroll
            for (int r = 0; r < 16; ++r) {
                T s = a.amp2[m0 + r * mstride];
                u[r].x *= s; u[r].y *= s;
            }
        }
        if (a.lens2 != nullptr) {
            const C *l = a.lens2 + (size_t)b * N;
            const C c = ldg_c(l + idx);
#pragma unroll
            for (int r = 0; r < 16; ++r) u[r] = cmul(u[r], cmul(ldg_c(l + j + r * TL), c));
        }
    });

    if (a.scale != (T)1) {
#pragma unroll
        for (int r = 0; r < 16; ++r) { v[r].x *= a.scale; v[r].y *= a.scale; }
    }
    if constexpr (!COL) {
        // the y-part of a separable input chirp is one factor per row: applied here, after the (linear) row
        // transform, it saves the column pass a table load and a multiply on its critical path
        if (a.rowfac != nullptr) {
            const C c = ldg_c(a.rowfac + (size_t)b * N + idx);
#pragma unroll
            for (int r = 0; r < 16; ++r) v[r] = cmul(v[r], c);
        }
    }
#pragma unroll
    for (int r = 0; r < 16; ++r) g[(size_t)(j + r * TL) * gstride] = v[r];
}

// ---- launch geometry -------------------------------------------------------------------------------
// Lines per CTA.  Row pass: enough rows to make a CTA of >= 128 threads.  Column pass: W adjacent
// columns, so that a row of the tile is W*sizeof(complex) contiguous bytes (>= one 32 B sector),
// chosen so that at least two CTAs fit an SM wherever the register file allows (the tile lives in
// registers, 16 elements per thread; co-resident CTAs are what overlaps one tile's loads with
// another tile's butterflies).  Override per build with -DFR_COLW_F64=<W> / -DFR_COLW_F32=<W>.
__host__ __device__ constexpr int fr_col_lines(int N, int elem_bytes)
{
    const int TL = N / 16;
    if (elem_bytes == 16) {
#ifdef FR_COLW_F64
        if (FR_COLW_F64 * TL <= 512) return FR_COLW_F64;
#endif
        return N <= 1024 ? 4 : (N <= 4096 ? 2 : 1);
    }
#ifdef FR_COLW_F32
    if (FR_COLW_F32 * TL <= 1024) return FR_COLW_F32;
#endif
    return N <= 1024 ? 8 : (N <= 4096 ? 4 : 2);
}
__host__ __device__ constexpr int fr_row_lines(int N, int elem_bytes)
{
    const int TL = N / 16;
#ifdef FR_ROWL_F64
    if (elem_bytes == 16 && FR_ROWL_F64 * TL <= 512 && FR_ROWL_F64 * TL >= 128) return FR_ROWL_F64;
#endif
#ifdef FR_ROWL_F32
    if (elem_bytes == 8 && FR_ROWL_F32 * TL <= 1024 && FR_ROWL_F32 * TL >= 128) return FR_ROWL_F32;
#endif
    return TL >= 128 ? 1 : 128 / TL;
}

template <typename T, int N, bool COL> struct PassGeom {
    static constexpr int TL = N / 16;
    static constexpr int ES = (int)sizeof(typename cplx_of<T>::type);
    static constexpr int row_lines = fr_row_lines(N, ES);
    static constexpr int W = COL ? fr_col_lines(N, ES) : row_lines;
    static constexpr int threads = W * TL;
    static_assert(threads <= 1024, "CTA too large");
    static constexpr size_t smem = (size_t)W * fr_padded_len(N) * ES;
    // resident CTAs per SM the register budget is tuned for
#ifndef FR_REGS_F64
#define FR_REGS_F64 128
#endif
#ifndef FR_REGS_F32
#define FR_REGS_F32 64
#endif
    // complex64 at N <= 512: a pass is a single wave of one CTA per SM, i.e. pure latency, and the handful of spills that
    // a 64-register cap costs the convolution kernel sit on that critical path as first-touch local-memory accesses
    // (N = 512 row pass 14.4 -> 10.0 us with 72 registers)
    static constexpr int regs_per_thread_goal = sizeof(T) == 8 ? FR_REGS_F64 : (N <= 512 && FR_REGS_F32 < 72 ? 72 : FR_REGS_F32);
    static constexpr int minb_regs = 65536 / (threads * regs_per_thread_goal);
    static constexpr int minb_smem = (int)((227 * 1024) / smem);
    static constexpr int minb0 = minb_regs < minb_smem ? minb_regs : minb_smem;
    static constexpr int MINB = minb0 < 1 ? 1 : (minb0 > 8 ? 8 : minb0);
};

template <typename T, int N, bool COL, int MODE>
cudaError_t launch_pass(const PassArgs<T> &a, int batch, cudaStream_t stream)
{
    using G = PassGeom<T, N, COL>;
    auto kern = pass_kernel<T, N, COL, G::W, MODE, G::MINB>;
    static std::atomic<unsigned long long> configured{0};      // one bit per device: the attribute is per device
    if (fr_needs_configuring(configured)) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)G::smem);
        if (e != cudaSuccess) return e;
        fr_mark_configured(configured);
    }
    dim3 grid(N / G::W, batch, 1);
    PassArgs<T> b = a;
    if (b.prefetch_distance < 0) b.prefetch_distance = -b.prefetch_distance * G::MINB;
    return launch_pdl(kern, grid, dim3(G::threads), G::smem, stream, b.pdl != 0, b);
}

} // namespace fresnel
