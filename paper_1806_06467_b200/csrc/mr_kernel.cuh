// mr_kernel.cuh -- REGISTER-RESIDENT mixed-radix pass for selected grids that are not a power of two.
//
// The paper ran N = 2800 and found it faster than 4096 (Fig. 2 row 2800 at :172).  gen_kernel.cuh takes any
// N but pays a shared-memory round trip for every stage AND every pointwise step; here a line of N = R_0 R_1 ... R_{L-1}
// points (2800 = 5 * 5 * 7 * 16) is held in registers by TPL threads exactly as in fft_core.cuh, and only the exchanges
// between stages go through shared memory:
//   * stage s has N/R_s butterflies of radix R_s; thread j takes butterflies b = j, j + TPL, ... (ceil(N/R_s / TPL) rounds),
//     so a thread holds rounds * R_s <= 16 elements in every stage (2800, TPL = 200: 3 x 5, 3 x 5, 2 x 7, 1 x 16);
//   * Stockham autosort: butterfly b of a stage reads elements b + t N/R_s -- for fixed t adjacent threads take adjacent
//     elements, which is the coalesced global access pattern -- and the LAST stage writes q-th output to b + q N/R_s:
//     the read pattern of a FIRST stage of the same radix.  So the forward transform runs its stages in the order
//     (R_0 .. R_{L-1}) and the inverse transform of a convolution in the REVERSED order (R_{L-1} .. R_0): the spectrum
//     stays in registers between them (x transfer function, no exchange), and the result comes out in the pattern the line
//     was loaded in.  Any stage order computes the same DFT (twiddles W_{Ns R}^{t k} follow the order).
//   * an inverse transform is conj o forward o conj, the conjugations folded into the neighbouring multiplies;
//   * odd radices in their symmetric form (dft_odd, gen_kernel.cuh); twiddles: one load of W_N^m from the plan's root table
//     per butterfly, the powers generated in registers.
// Row pass: loads and stores straight from / to registers (optic phasor, chirp table, per-row factor as in pass_kernel.cuh).
// Column pass: TMA tiles of W columns as in col_tma.cuh (a partial last box is zero-filled / clipped by the hardware).
#pragma once
#include "gen_kernel.cuh"

namespace fresnel {

// Forward stage order and threads per line of the supported sizes: chosen (by exhaustive search over factorisations into
// radices 2, 3, 4, 5, 7, 8, 16 and over TPL) for the fewest stages, then the fewest idle lanes, under "rounds x radix <= 16"
// in every stage; odd radices first (a first stage of odd radix scatters without bank conflicts), the power of two last.
template <int N> struct MrShape;
#define FR_MR_SHAPE(NN, THREADS, STAGES, ...)                                                                        \
    template <> struct MrShape<NN> {                                                                                 \
        static constexpr int NST = STAGES, TPL = THREADS;                                                            \
        __host__ __device__ static constexpr int radix(int s) { constexpr int r[STAGES] = {__VA_ARGS__}; return r[s]; } \
    };
FR_MR_SHAPE(700, 50, 4, 5, 5, 7, 4)
FR_MR_SHAPE(1000, 125, 4, 5, 5, 5, 8)
FR_MR_SHAPE(1200, 80, 4, 3, 5, 5, 16)
FR_MR_SHAPE(1400, 100, 4, 5, 5, 7, 8)
FR_MR_SHAPE(1500, 150, 5, 3, 5, 5, 5, 4)
FR_MR_SHAPE(2000, 134, 4, 5, 5, 5, 16)
FR_MR_SHAPE(2400, 160, 5, 3, 5, 5, 2, 16)
FR_MR_SHAPE(2800, 200, 4, 5, 5, 7, 16)
FR_MR_SHAPE(3000, 200, 5, 3, 5, 5, 5, 8)
FR_MR_SHAPE(3600, 240, 5, 3, 3, 5, 5, 16)
FR_MR_SHAPE(4000, 286, 5, 5, 5, 5, 2, 16)
FR_MR_SHAPE(5000, 334, 5, 5, 5, 5, 5, 8)
FR_MR_SHAPE(5600, 400, 5, 5, 5, 7, 2, 16)
FR_MR_SHAPE(6000, 400, 5, 3, 5, 5, 5, 16)
#undef FR_MR_SHAPE

template <int N, int ORDER> __host__ __device__ constexpr int mr_radix(int s)
{
    return MrShape<N>::radix(ORDER ? MrShape<N>::NST - 1 - s : s);
}
template <int N, int ORDER> __host__ __device__ constexpr int mr_ns(int s)
{
    int ns = 1;
    for (int i = 0; i < s; ++i) ns *= mr_radix<N, ORDER>(i);
    return ns;
}
template <int N> __host__ __device__ constexpr int mr_rounds(int R) { return (N / R + MrShape<N>::TPL - 1) / MrShape<N>::TPL; }
template <int N> __host__ __device__ constexpr int mr_elems()
{
    int m = 0;
    for (int s = 0; s < MrShape<N>::NST; ++s) {
        const int e = mr_rounds<N>(MrShape<N>::radix(s)) * MrShape<N>::radix(s);
        m = e > m ? e : m;
    }
    return m;
}
template <int N> __host__ __device__ constexpr int mr_line_threads() { return (MrShape<N>::TPL + 31) / 32 * 32; }
// padded position in the exchange buffer: one spare element every 16 (16-byte elements) or every 32 (8-byte elements) --
// the spacing with the fewest shared-memory wavefronts over all scatters and gathers of the 2800-point stage orders
// (counted lane by lane: 1.33x / 1.52x the conflict-free number, against 1.69x / 2.41x unpadded)
#ifndef FR_MR_PADSHIFT_F32
#define FR_MR_PADSHIFT_F32 5
#endif
template <int ES> __host__ __device__ constexpr int mr_pad(int p) { return p + (p >> (ES == 16 ? 4 : FR_MR_PADSHIFT_F32)); }
template <int N> __host__ __device__ constexpr int mr_padlen() { return N + N / 16 + 1; }

// f(e, n) for every element the thread holds in the read pattern of a radix-R stage: register e <-> line index n.
// Threads beyond TPL come in with j = N, so that no butterfly index is ever valid for them.
template <int N, int R, typename F> FR_DEV void mr_for_each(int j, F &&f)
{
    constexpr int NB = N / R, RD = mr_rounds<N>(R), TPL = MrShape<N>::TPL;
#pragma unroll
    for (int i = 0; i < RD; ++i) {
        const int b = j + i * TPL;
        if (b < NB) {
#pragma unroll
            for (int t = 0; t < R; ++t) f(i * R + t, b + t * NB);
        }
    }
}

// u[t] *= w^t, t = 1 .. R-1, w = W_{Ns R}^k: one table load, the powers by short product chains
template <int R, typename C> FR_DEV void mr_twiddle(C (&u)[R], C w)
{
    u[1] = cmul(u[1], w);
    if constexpr (R >= 3) {
        const C p2 = csq(w);
        u[2] = cmul(u[2], p2);
        if constexpr (R >= 4) {
            const C p3 = cmul(p2, w);
            u[3] = cmul(u[3], p3);
            if constexpr (R >= 5) {
                const C p4 = csq(p2);
                C g = p4;                                            // w^(4m)
#pragma unroll
                for (int m = 1; 4 * m < R; ++m) {
                    u[4 * m] = cmul(u[4 * m], g);
                    if (4 * m + 1 < R) u[4 * m + 1] = cmul(u[4 * m + 1], cmul(g, w));
                    if (4 * m + 2 < R) u[4 * m + 2] = cmul(u[4 * m + 2], cmul(g, p2));
                    if (4 * m + 3 < R) u[4 * m + 3] = cmul(u[4 * m + 3], cmul(g, p3));
                    if (4 * (m + 1) < R) g = (m == 1) ? csq(g) : cmul(g, p4);
                }
            }
        }
    }
}

template <int R, typename C> FR_DEV void mr_butterfly(C (&u)[R])
{
    if constexpr (R == 16) dft16<-1>(u);
    else if constexpr (R == 8) dft8<-1>(u[0], u[1], u[2], u[3], u[4], u[5], u[6], u[7]);
    else if constexpr (R == 4) dft4<-1>(u[0], u[1], u[2], u[3]);
    else if constexpr (R == 2) dft2<-1>(u[0], u[1]);
    else dft_odd<R>(u);
}

// v[e] *= exp(2 pi i * opd(n) / lambda) over the elements of the read pattern of radix R: the branch-free polynomial for all of
// them when every phase is small (the common case, as apply_opd16 of pass_kernel.cuh), else the general path one by one
// (row pass with an OPD map at N = 2800: 208 -> 151 us against a per-element branch)
template <typename T, int N, int R, typename Load>
FR_DEV void mr_apply_opd(typename cplx_of<T>::type (&v)[mr_elems<N>()], int j, T inv_lambda, Load &&opd_at)
{
    constexpr int E = mr_elems<N>();
    T u[E];
    bool all_small = true;
    mr_for_each<N, R>(j, [&](int e, int n) {
        u[e] = opd_at(n) * inv_lambda;
        all_small = all_small && phasor_is_small(u[e]);
    });
    if (all_small) mr_for_each<N, R>(j, [&](int e, int) { v[e] = cmul(v[e], phasor_turns_small(u[e])); });
    else mr_for_each<N, R>(j, [&](int e, int) { v[e] = cmul(v[e], phasor_turns_any(u[e])); });
}

// one stage: twiddles + butterflies in registers; unless it is the last, scatter -> barrier -> gather in the read pattern
// of the next stage -> barrier
template <typename T, int N, int ORDER, int S, int GT>
FR_DEV void mr_stage(typename cplx_of<T>::type (&v)[mr_elems<N>()], typename cplx_of<T>::type *buf, int j,
                     const typename cplx_of<T>::type *__restrict__ tw, int bar_id)
{
    using C = typename cplx_of<T>::type;
    constexpr int NST = MrShape<N>::NST, TPL = MrShape<N>::TPL;
    constexpr int R = mr_radix<N, ORDER>(S), NS = mr_ns<N, ORDER>(S), NB = N / R, RD = mr_rounds<N>(R);
#pragma unroll
    for (int i = 0; i < RD; ++i) {
        const int b = j + i * TPL;
        if (b < NB) {
            C u[R];
#pragma unroll
            for (int t = 0; t < R; ++t) u[t] = v[i * R + t];
            if constexpr (NS > 1) mr_twiddle<R>(u, ldg_c(tw + (b % NS) * (N / (NS * R))));
            mr_butterfly<R>(u);
#pragma unroll
            for (int t = 0; t < R; ++t) v[i * R + t] = u[t];
        }
    }
    if constexpr (S + 1 < NST) {
#pragma unroll
        for (int i = 0; i < RD; ++i) {
            const int b = j + i * TPL;
            if (b < NB) {
                const int k = b % NS;
                const int p0 = (b - k) * R + k;
#pragma unroll
                for (int q = 0; q < R; ++q) buf[mr_pad<(int)sizeof(C)>(p0 + q * NS)] = v[i * R + q];
            }
        }
        fr_sync<GT>(bar_id);
        constexpr int R2 = mr_radix<N, ORDER>(S + 1);
        mr_for_each<N, R2>(j, [&](int e, int n) { v[e] = buf[mr_pad<(int)sizeof(C)>(n)]; });
        fr_sync<GT>(bar_id);
    }
}

// forward DFT of the resident line with the stages in forward (ORDER 0) or reversed (ORDER 1) order: in -- read pattern of
// the first radix of that order; out -- read pattern of its last radix
template <typename T, int N, int ORDER, int GT>
FR_DEV void mr_fft(typename cplx_of<T>::type (&v)[mr_elems<N>()], typename cplx_of<T>::type *buf, int j,
                   const typename cplx_of<T>::type *__restrict__ tw, int bar_id)
{
    constexpr int NST = MrShape<N>::NST;
    mr_stage<T, N, ORDER, 0, GT>(v, buf, j, tw, bar_id);
    if constexpr (NST > 1) mr_stage<T, N, ORDER, 1, GT>(v, buf, j, tw, bar_id);
    if constexpr (NST > 2) mr_stage<T, N, ORDER, 2, GT>(v, buf, j, tw, bar_id);
    if constexpr (NST > 3) mr_stage<T, N, ORDER, 3, GT>(v, buf, j, tw, bar_id);
    if constexpr (NST > 4) mr_stage<T, N, ORDER, 4, GT>(v, buf, j, tw, bar_id);
}

// lines per CTA (column pass: columns per TMA tile, at least 16 bytes per tile row) / resident CTAs per SM the launch
// bounds ask for.  Override per build with -DFR_MR_COLW_F64=<W> / -DFR_MR_COLW_F32=<W> (tuning).
template <typename T, int N, bool COL> struct MrGeom {
    static constexpr int ES = (int)sizeof(typename cplx_of<T>::type);
    static constexpr int LT = mr_line_threads<N>();
#ifdef FR_MR_COLW_F64
    static constexpr int WC64 = FR_MR_COLW_F64;
#else
    static constexpr int WC64 = LT <= 128 ? 2 : 1;
#endif
#ifdef FR_MR_COLW_F32
    static constexpr int WC32 = FR_MR_COLW_F32;
#else
    static constexpr int WC32 = LT <= 128 ? 4 : 2;
#endif
    static constexpr int WROW = LT >= 128 ? 1 : 128 / LT;
    static constexpr int W = COL ? (ES == 16 ? WC64 : WC32) : WROW;
    static constexpr int threads = W * LT;
    static constexpr int ROW_BYTES = W * ES;
    static constexpr int tile_rows = (N + kTmaBoxRows - 1) / kTmaBoxRows * kTmaBoxRows;      // whole boxes land
    static constexpr size_t xchg_bytes = (size_t)W * mr_padlen<N>() * ES;
    static constexpr size_t tile_bytes = COL ? (size_t)tile_rows * ROW_BYTES : 0;
    static constexpr size_t smem = (xchg_bytes > tile_bytes ? xchg_bytes : tile_bytes) + (COL ? 1024 : 0);
    static constexpr int regs_goal = ES == 16 ? 128 : 64;
    static constexpr int minb_regs = 65536 / (threads * regs_goal);
    static constexpr int minb_smem = (int)((226 * 1024) / (smem + 1024));
    static constexpr int minb0 = minb_regs < minb_smem ? minb_regs : minb_smem;
    static constexpr int MINB = minb0 < 1 ? 1 : (minb0 > 8 ? 8 : minb0);
};

template <typename T, int N, bool COL, int MODE>
__global__ void __launch_bounds__(MrGeom<T, N, COL>::threads, MrGeom<T, N, COL>::MINB)
mr_pass_kernel(GenArgs<T> a, const __grid_constant__ CUtensorMap tmap)
{
    using C = typename cplx_of<T>::type;
    using G = MrGeom<T, N, COL>;
    constexpr int W = G::W, LT = G::LT, ES = G::ES, ROW_BYTES = G::ROW_BYTES, TPL = MrShape<N>::TPL, NST = MrShape<N>::NST;
    constexpr int E = mr_elems<N>();
    constexpr int GT = W == 1 ? 0 : LT;                       // barrier group: the CTA, or one column's threads
    constexpr int R_IN = mr_radix<N, 0>(0), R_MID = mr_radix<N, 0>(NST - 1);
    constexpr int R_OUT = MODE == MODE_CONV ? R_IN : R_MID;   // pattern the result is held in
    extern __shared__ __align__(1024) unsigned char fr_smem[];
    __shared__ __align__(8) uint64_t full_bar;
    unsigned char *tile = COL ? fr_smem + ((1024u - (smem_u32(fr_smem) & 1023u)) & 1023u) : fr_smem;

    const int tid = threadIdx.x;
    const int g = tid / LT;                                   // line of the CTA
    const int jr = tid - g * LT;
    const int j = jr < TPL ? jr : N;                          // idle lanes of the last warp: no valid butterfly
    const int b = blockIdx.y;
    const int line = blockIdx.x * W + g;                      // row / column of the grid
    C *buf = reinterpret_cast<C *>(tile) + (size_t)g * mr_padlen<N>();
    C *grow = a.wf + (size_t)b * N * N + (size_t)line * N;    // row pass only

    C v[E];
#pragma unroll
    for (int e = 0; e < E; ++e) { v[e].x = (T)0; v[e].y = (T)0; }

    if constexpr (COL) {
        if (tid == 0) mbar_init(&full_bar, 1);
        pdl_launch_dependents();
        __syncthreads();
        pdl_wait();
        if (tid == 0) {
            mbar_expect_tx(&full_bar, (uint32_t)((size_t)G::tile_rows * ROW_BYTES));
#pragma unroll 1
            for (int r0 = 0; r0 < N; r0 += kTmaBoxRows) tma_load_3d(tile + (size_t)r0 * ROW_BYTES, &tmap, &full_bar, blockIdx.x * W * 2, r0, b);
        }
        mbar_wait(&full_bar, 0);
        mr_for_each<N, R_IN>(j, [&](int e, int n) {
            v[e] = *reinterpret_cast<const C *>(tile + tile_swizzle<ROW_BYTES>((uint32_t)(n * ROW_BYTES + g * ES)));
        });
        __syncthreads();                                      // the landing zone becomes exchange space
    } else {
        pdl_launch_dependents();
        pdl_wait();
        mr_for_each<N, R_IN>(j, [&](int e, int n) { v[e] = grow[n]; });
        if (a.opd != nullptr) {
            const T *o = a.opd + (size_t)line * N;
            mr_apply_opd<T, N, R_IN>(v, j, (T)a.inv_lambda[b], [&](int n) { return o[n]; });
        }
        if (a.amp != nullptr) {
            const T *m = a.amp + (size_t)line * N;
            mr_for_each<N, R_IN>(j, [&](int e, int n) { const T s = m[n]; v[e].x *= s; v[e].y *= s; });
        }
    }
    if (a.pre != nullptr) {
        const C *p = a.pre + (size_t)b * N;
        mr_for_each<N, R_IN>(j, [&](int e, int n) { v[e] = cmul(v[e], ldg_c(p + n)); });
    }
    if constexpr (MODE == MODE_INV) {
#pragma unroll
        for (int e = 0; e < E; ++e) v[e].y = -v[e].y;
    }

    mr_fft<T, N, 0, GT>(v, buf, j, a.tw, 1 + g);

    const C *m = a.mid != nullptr ? a.mid + (size_t)b * N : nullptr;
    if constexpr (MODE == MODE_FWD) {
        if (m != nullptr) mr_for_each<N, R_MID>(j, [&](int e, int n) { v[e] = cmul(v[e], ldg_c(m + n)); });
    } else if constexpr (MODE == MODE_INV) {
        if (m != nullptr) mr_for_each<N, R_MID>(j, [&](int e, int n) { v[e] = cmulc(ldg_c(m + n), v[e]); });   // mid * conj(v)
        else {
#pragma unroll
            for (int e = 0; e < E; ++e) v[e].y = -v[e].y;
        }
    } else {
        // x transfer function, conjugated for the inverse transform (reversed stage order) that follows
        if (m != nullptr) {
            mr_for_each<N, R_MID>(j, [&](int e, int n) {
                const C t = cmul(v[e], ldg_c(m + n));
                v[e].x = t.x; v[e].y = -t.y;
            });
        } else {
#pragma unroll
            for (int e = 0; e < E; ++e) v[e].y = -v[e].y;
        }
        mr_fft<T, N, 1, GT>(v, buf, j, a.tw, 1 + g);
#pragma unroll
        for (int e = 0; e < E; ++e) v[e].y = -v[e].y;
    }
    if (a.scale != (T)1) {
#pragma unroll
        for (int e = 0; e < E; ++e) { v[e].x *= a.scale; v[e].y *= a.scale; }
    }

    if constexpr (COL) {
        __syncthreads();                                      // every group is done with its exchange buffer
        mr_for_each<N, R_OUT>(j, [&](int e, int n) {
            *reinterpret_cast<C *>(tile + tile_swizzle<ROW_BYTES>((uint32_t)(n * ROW_BYTES + g * ES))) = v[e];
        });
        fence_async_proxy();
        __syncthreads();
        if (tid == 0) {
#pragma unroll 1
            for (int r0 = 0; r0 < N; r0 += kTmaBoxRows) tma_store_3d(&tmap, tile + (size_t)r0 * ROW_BYTES, blockIdx.x * W * 2, r0, b);
            tma_store_commit_and_wait();
        }
    } else {
        if (a.rowfac != nullptr) {
            const C c = ldg_c(a.rowfac + (size_t)b * N + line);
#pragma unroll
            for (int e = 0; e < E; ++e) v[e] = cmul(v[e], c);
        }
        mr_for_each<N, R_OUT>(j, [&](int e, int n) { grow[n] = v[e]; });
    }
}

template <typename T, int N, bool COL, int MODE>
cudaError_t launch_mr_pass(const GenArgs<T> &a, const CUtensorMap &tmap, int batch, cudaStream_t stream)
{
    using G = MrGeom<T, N, COL>;
    static_assert(mr_elems<N>() <= 16, "a thread holds at most 16 elements");
    static_assert(N % G::W == 0, "whole column tiles");
    auto kern = mr_pass_kernel<T, N, COL, MODE>;
    static std::atomic<unsigned long long> configured{0};
    if (fr_needs_configuring(configured)) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)G::smem);
        if (e != cudaSuccess) return e;
        fr_mark_configured(configured);
    }
    dim3 grid(N / G::W, batch, 1);
    return launch_pdl(kern, grid, dim3(G::threads), G::smem, stream, a.pdl != 0, a, tmap);
}

} // namespace fresnel
