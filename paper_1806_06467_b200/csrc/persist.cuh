// persist.cuh -- persistent pass kernels: ONE CTA per SM for the whole pass.
//
// pass_kernel.cuh / col_tma.cuh launch one CTA per line (or tile).  ncu on the N = 2048 complex128
// row pass shows what that costs (profiles/r01b_*): SMs are idle 17 % of the kernel (2048 CTAs over
// 592 resident slots = 3.46 waves; the last 0.46 wave runs on half-empty SMs), every CTA waits for
// its stores to drain before its slot is handed on (7 % of the stall samples), loads its input cold
// (9 %) and fetches the 32 KB transfer-function table again through a 25 KB L1 (7 %).
//
// Here a CTA owns a contiguous range of lines (all lines / gridDim.x, gridDim.x = number of SMs) and
// its NG line groups (N/16 threads each, private named barrier, private exchange buffer) walk that
// range round-robin, so that an SM works on NG lines at NG different phases until its range is
// empty: no wave quantisation beyond one line per SM, no drain between lines (stores of line i
// overlap line i+1), the next line of every group is prefetched into L2 one line ahead, and the
// 1-D tables (transfer function, lens chirp) are staged in shared memory once per batch element.
#pragma once
#include "col_tma.cuh"

namespace fresnel {

// ---- geometry ----------------------------------------------------------------------------------------------
template <typename T, int N> struct PersistGeom {
    using C = typename cplx_of<T>::type;
    static constexpr int TL = N / 16;
    static constexpr int ES = (int)sizeof(C);
    static constexpr int PL = fr_padded_len(N);
    static constexpr int regs_goal = sizeof(T) == 8 ? 128 : 64;
    static constexpr int ng_regs = 65536 / (regs_goal * TL);
    static constexpr int ng_thr = 1024 / TL;
    static constexpr int ng0 = ng_regs < ng_thr ? ng_regs : ng_thr;
    static constexpr int smem_max = 227 * 1024 - 2048;
    static constexpr int ng_smem = smem_max / (PL * ES);
#ifdef FR_PERSIST_NG
    static constexpr int ng1 = (FR_PERSIST_NG < ng0 ? FR_PERSIST_NG : ng0);
#else
    static constexpr int ng1 = ng0;
#endif
    static constexpr int NG = ng1 < ng_smem ? (ng1 < 1 ? 1 : ng1) : (ng_smem < 1 ? 1 : ng_smem);   // line groups per CTA
    static constexpr int threads = NG * TL;
    static constexpr int exch_bytes = NG * PL * ES;
    // 1-D tables staged in shared memory: 2 = transfer function + input chirp, 1 = transfer function, 0 = none
#ifdef FR_PERSIST_TABS
    static constexpr int TABS = FR_PERSIST_TABS;
#else
    static constexpr int TABS = (exch_bytes + 2 * N * ES <= smem_max) ? 2 : (exch_bytes + N * ES <= smem_max) ? 1 : 0;
#endif
    static constexpr size_t smem = (size_t)exch_bytes + (size_t)TABS * N * ES;
    static constexpr bool supported = TL >= 32 && PL * ES <= smem_max;
};

template <typename T, int N, bool SM>
FR_DEV void persist_mul_table(typename cplx_of<T>::type (&v)[16], const typename cplx_of<T>::type *tab, int j)
{
    constexpr int TL = N / 16;
    if constexpr (SM) {
#pragma unroll
        for (int r = 0; r < 16; ++r) v[r] = cmul(v[r], tab[j + r * TL]);
    } else {
#pragma unroll
        for (int r = 0; r < 16; ++r) v[r] = cmul(v[r], ldg_c(tab + j + r * TL));
    }
}

// ---- row pass ------------------------------------------------------------------------------------------------
template <typename T, int N, int MODE>
__global__ void __launch_bounds__(PersistGeom<T, N>::threads, 1) persist_row_kernel(PassArgs<T> a, int batch)
{
    using G = PersistGeom<T, N>;
    using C = typename cplx_of<T>::type;
    constexpr int TL = G::TL, PL = G::PL, NG = G::NG, TABS = G::TABS;
    constexpr int GT = (NG == 1) ? 0 : TL;
    extern __shared__ __align__(16) unsigned char fr_smem[];
    C *exch = reinterpret_cast<C *>(fr_smem);
    C *tab_mid = exch + (size_t)NG * PL;
    C *tab_pre = tab_mid + N;

    const int tid = threadIdx.x;
    const int grp = tid / TL, j = tid % TL;
    C *buf = exch + (size_t)grp * PL;
    const int bar = 1 + grp;

    const long long total = (long long)N * batch;
    const int lo = (int)(total * blockIdx.x / gridDim.x);
    const int hi = (int)(total * (blockIdx.x + 1) / gridDim.x);

    bool staggered = false;
    for (int seg_lo = lo; seg_lo < hi;) {
        const int b = seg_lo / N;
        const int seg_hi = min(hi, (b + 1) * N);
        const C *gmid = a.mid ? a.mid + (size_t)b * N : nullptr;
        const C *gpre = a.pre ? a.pre + (size_t)b * N : nullptr;
        if constexpr (TABS >= 1) {
            __syncthreads();                         // every group is done with the previous batch element's tables
            if (gmid) for (int i = tid; i < N; i += G::threads) tab_mid[i] = ldg_c(gmid + i);
            if constexpr (TABS >= 2)
                if (gpre) for (int i = tid; i < N; i += G::threads) tab_pre[i] = ldg_c(gpre + i);
            __syncthreads();
        }
        C *wfb = a.wf + (size_t)b * N * N;
        if (!staggered && a.stagger_ns > 0) {
            // the groups of a CTA run identical code on identical amounts of data: started together they
            // stay in lockstep (all loading, then all in the butterflies, then all exchanging) and the
            // three pipes never overlap.  Start them a fraction of a line apart.
            for (int t = grp * a.stagger_ns; t > 0; t -= 1000) __nanosleep(t < 1000 ? t : 1000);
            staggered = true;
        }
        for (int L = seg_lo + grp; L < seg_hi; L += NG) {
            const int row = L - b * N;
            C *g = wfb + (size_t)row * N;
            C v[16];
#pragma unroll
            for (int r = 0; r < 16; ++r) v[r] = g[j + r * TL];
            // ask L2 for the line this group takes next (and its map rows)
            if (j == 0 && a.prefetch_distance != 0 && L + NG < seg_hi) {
                const size_t nrow = (size_t)(row + NG);
                l2_prefetch_bulk(wfb + nrow * N, (uint32_t)(N * sizeof(C)));
                if (a.opd != nullptr) l2_prefetch_bulk(a.opd + nrow * N, (uint32_t)(N * sizeof(T)));
                if (a.amp != nullptr) l2_prefetch_bulk(a.amp + nrow * N, (uint32_t)(N * sizeof(T)));
            }
            if (a.opd != nullptr) {
                const T il = (T)a.inv_lambda[b];
                const T *o = a.opd + (size_t)row * N;
#pragma unroll
                for (int r = 0; r < 16; ++r) v[r] = cmul(v[r], phasor_turns(o[j + r * TL] * il));
            }
            if (a.amp != nullptr) {
                const T *m = a.amp + (size_t)row * N;
#pragma unroll
                for (int r = 0; r < 16; ++r) {
                    T s = m[j + r * TL];
                    v[r].x *= s; v[r].y *= s;
                }
            }
            if (gpre) {
                if constexpr (TABS >= 2) persist_mul_table<T, N, true>(v, tab_pre, j);
                else                     persist_mul_table<T, N, false>(v, gpre, j);
            }
            if constexpr (MODE == MODE_INV) fft_line<T, N, +1, false, 1, GT>(v, buf, 0, j, a.tw, bar);
            else                            fft_line<T, N, -1, false, 1, GT>(v, buf, 0, j, a.tw, bar);
            if (gmid) {
                if constexpr (TABS >= 1) persist_mul_table<T, N, true>(v, tab_mid, j);
                else                     persist_mul_table<T, N, false>(v, gmid, j);
            }
            if constexpr (MODE == MODE_CONV) fft_line<T, N, +1, false, 1, GT>(v, buf, 0, j, a.tw, bar);
            if (a.scale != (T)1) {
#pragma unroll
                for (int r = 0; r < 16; ++r) { v[r].x *= a.scale; v[r].y *= a.scale; }
            }
#pragma unroll
            for (int r = 0; r < 16; ++r) g[j + r * TL] = v[r];
        }
        seg_lo = seg_hi;
    }
}

template <typename T, int N, int MODE>
cudaError_t launch_persist_row(const PassArgs<T> &a, int batch, int sms, cudaStream_t stream)
{
    using G = PersistGeom<T, N>;
    if constexpr (!G::supported) {
        return cudaErrorNotSupported;
    } else {
        auto kern = persist_row_kernel<T, N, MODE>;
        static bool configured = false;
        if (!configured) {
            cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)G::smem);
            if (e != cudaSuccess) return e;
            configured = true;
        }
        const long long total = (long long)N * batch;
        const long long per = (total + G::NG - 1) / G::NG;                 // never more CTAs than rounds of NG lines
        const int grid = (int)(per < sms ? per : sms);
        kern<<<grid, G::threads, G::smem, stream>>>(a, batch);
        return cudaGetLastError();
    }
}

} // namespace fresnel
