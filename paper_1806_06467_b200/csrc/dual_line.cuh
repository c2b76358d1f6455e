// dual_line.cuh -- pass kernels in which every thread carries TWO lines, half a step apart.
//
// The register-resident transform of fft_core.cuh alternates butterflies (FP64/FP32 pipe) with
// exchanges through shared memory (load/store pipe).  Per element and pass the two pipes and HBM
// need about the same number of SM cycles, so whatever time they do not
// overlap is lost.  With one line per thread the only overlap is between co-resident CTAs, and each
// exchange costs two barriers whose latency nothing hides.
//
// Here a thread owns 16 elements of line A and 16 elements of line B (two adjacent rows, or the two
// columns of a TMA tile) and runs them as a two-stage software pipeline.  One half-step is
//
//        barrier;  gather X (16 LDS);  scatter Y (16 STS);  butterflies of X      X, Y = A, B alternating
//
// so the scatter -> gather round trip of one line lies under a whole butterfly block of the other,
// the load/store instructions of a half-step are issued ahead of ~200 independent arithmetic
// instructions of the same warp, and ONE barrier per half-step orders both hazards:
//   RAW  gather X reads what scatter X wrote one half-step (= one barrier) earlier;
//   WAR  scatter Y overwrites what gather Y read one half-step (= one barrier) earlier.
// A line still makes the same number of trips through shared memory; it meets half the barriers.
#pragma once
#include "col_tma.cuh"

namespace fresnel {

template <int N, int MODE> struct DualSched {
    static constexpr int S = fr_num_stages(N);
    static constexpr int NB = (MODE == MODE_CONV) ? 2 * S - 1 : S;          // butterfly blocks per line
    // the stage whose exchange pattern follows block K
    __host__ __device__ static constexpr int xstage(int K) { return (MODE == MODE_CONV && K >= S - 1) ? K - (S - 1) : K; }
};

template <typename T, int N> FR_DEV void dual_mul_table(typename cplx_of<T>::type (&v)[16], const typename cplx_of<T>::type *__restrict__ tab, int j)
{
    constexpr int TL = N / 16;
#pragma unroll
    for (int r = 0; r < 16; ++r) v[r] = cmul(v[r], ldg_c(tab + j + r * TL));
}

// butterfly block K of one line (registers only)
template <typename T, int N, int MODE, int K>
FR_DEV void dual_block(typename cplx_of<T>::type (&v)[16], int j, const PassArgs<T> &a, int b)
{
    using SC = DualSched<N, MODE>;
    constexpr int S = SC::S;
    if constexpr (MODE == MODE_CONV) {
        if constexpr (K < S - 1) {
            fft_stage_compute<T, N, K, -1>(v, j, a.tw);
        } else if constexpr (K == S - 1) {
            fft_stage_compute<T, N, S - 1, -1>(v, j, a.tw);
            if (a.mid != nullptr) dual_mul_table<T, N>(v, a.mid + (size_t)b * N, j);
            fft_stage_compute<T, N, 0, +1>(v, j, a.tw);
        } else {
            fft_stage_compute<T, N, K - (S - 1), +1>(v, j, a.tw);
        }
    } else {
        fft_stage_compute<T, N, K, (MODE == MODE_INV ? +1 : -1)>(v, j, a.tw);
        if constexpr (K == S - 1)
            if (a.mid != nullptr) dual_mul_table<T, N>(v, a.mid + (size_t)b * N, j);
    }
    if constexpr (K == SC::NB - 1) {
        if (a.scale != (T)1) {
#pragma unroll
            for (int r = 0; r < 16; ++r) { v[r].x *= a.scale; v[r].y *= a.scale; }
        }
    }
}

// Half-steps 2K-1 and 2K of the pipeline, K = 1 .. NB-1.  On entry: block K-1 of A is in vA and not yet
// scattered ... no: A's block K-1 has been scattered, B's block K-1 sits in vB.
template <typename T, int N, int MODE, int GT, int K> struct DualLoop {
    using C = typename cplx_of<T>::type;
    using SC = DualSched<N, MODE>;
    static FR_DEV void run(C (&vA)[16], C (&vB)[16], C *bufA, C *bufB, int j, const PassArgs<T> &a, int b, int bar,
                           C *gA /* row pass: where line A goes when it is finished; else nullptr */)
    {
        constexpr int TL = N / 16;
        fr_sync<GT>(bar);
        fft_stage_gather<T, N, false, 1>(vA, bufA, 0, j);
        fft_stage_scatter<T, N, SC::xstage(K - 1), false, 1>(vB, bufB, 0, j);
        dual_block<T, N, MODE, K>(vA, j, a, b);
        fr_sync<GT>(bar);
        fft_stage_gather<T, N, false, 1>(vB, bufB, 0, j);
        if constexpr (K < SC::NB - 1) {
            fft_stage_scatter<T, N, SC::xstage(K), false, 1>(vA, bufA, 0, j);
        } else {
            if (gA != nullptr) {
#pragma unroll
                for (int r = 0; r < 16; ++r) gA[j + r * TL] = vA[r];
            }
        }
        dual_block<T, N, MODE, K>(vB, j, a, b);
        if constexpr (K + 1 < SC::NB) DualLoop<T, N, MODE, GT, K + 1>::run(vA, vB, bufA, bufB, j, a, b, bar, gA);
    }
};

// the whole pipeline for one pair of lines already loaded (and pre-multiplied) into vA, vB
template <typename T, int N, int MODE, int GT>
FR_DEV void dual_pipeline(typename cplx_of<T>::type (&vA)[16], typename cplx_of<T>::type (&vB)[16],
                          typename cplx_of<T>::type *bufA, typename cplx_of<T>::type *bufB, int j, const PassArgs<T> &a, int b,
                          int bar, typename cplx_of<T>::type *gA)
{
    using SC = DualSched<N, MODE>;
    static_assert(SC::NB >= 2, "at least two stages");
    dual_block<T, N, MODE, 0>(vA, j, a, b);
    fft_stage_scatter<T, N, SC::xstage(0), false, 1>(vA, bufA, 0, j);
    dual_block<T, N, MODE, 0>(vB, j, a, b);
    DualLoop<T, N, MODE, GT, 1>::run(vA, vB, bufA, bufB, j, a, b, bar, gA);
}

// optic phasor, amplitude map and input chirp of one row (Eq. 3 and Eq. 2 on the load of the row pass)
template <typename T, int N>
FR_DEV void dual_row_front(typename cplx_of<T>::type (&v)[16], int row, int j, const PassArgs<T> &a, int b)
{
    constexpr int TL = N / 16;
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
    if (a.pre != nullptr) dual_mul_table<T, N>(v, a.pre + (size_t)b * N, j);
}

// ---- row pass: a group of N/16 threads owns rows 2p and 2p+1 ---------------------------------------------
template <typename T, int N, int MODE, int G, int MINB>
__global__ void __launch_bounds__(G *(N / 16), MINB) dual_row_kernel(PassArgs<T> a)
{
    using C = typename cplx_of<T>::type;
    constexpr int TL = N / 16;
    constexpr int PL = fr_padded_len(N);
    constexpr int GT = (G == 1) ? 0 : TL;
    extern __shared__ __align__(16) unsigned char fr_smem[];

    const int tid = threadIdx.x;
    const int grp = tid / TL, j = tid % TL;
    const int b = blockIdx.y;
    const int rowA = (blockIdx.x * G + grp) * 2;
    C *gA = a.wf + (size_t)b * N * N + (size_t)rowA * N;
    C *gB = gA + N;
    C *bufA = reinterpret_cast<C *>(fr_smem) + (size_t)(2 * grp) * PL;
    C *bufB = bufA + PL;

    C vA[16], vB[16];
#pragma unroll
    for (int r = 0; r < 16; ++r) vA[r] = gA[j + r * TL];
#pragma unroll
    for (int r = 0; r < 16; ++r) vB[r] = gB[j + r * TL];

    // L2 prefetch of the two rows (and map rows) that the CTA taking over a resident slot will load
    if (j == 0 && a.prefetch_distance > 0) {
        const int nx = (int)gridDim.x;
        int t = (int)blockIdx.x + a.prefetch_distance, bb = b;
        while (t >= nx) { t -= nx; ++bb; }
        if (bb < (int)gridDim.y) {
            const size_t row = (size_t)(t * G + grp) * 2;
            l2_prefetch_bulk(a.wf + (size_t)bb * N * N + row * N, (uint32_t)(2 * N * sizeof(C)));
            if (a.opd != nullptr) l2_prefetch_bulk(a.opd + row * N, (uint32_t)(2 * N * sizeof(T)));
            if (a.amp != nullptr) l2_prefetch_bulk(a.amp + row * N, (uint32_t)(2 * N * sizeof(T)));
        }
    }
    dual_row_front<T, N>(vA, rowA, j, a, b);
    dual_row_front<T, N>(vB, rowA + 1, j, a, b);
    dual_pipeline<T, N, MODE, GT>(vA, vB, bufA, bufB, j, a, b, 1 + grp, gA);
#pragma unroll
    for (int r = 0; r < 16; ++r) gB[j + r * TL] = vB[r];
}

// ---- column pass: a TMA tile of W = 2G columns; group g owns columns 2g and 2g+1 -----------------------
template <typename T, int N, int MODE, int G, int MINB>
__global__ void __launch_bounds__(G *(N / 16), MINB)
dual_col_kernel(PassArgs<T> a, const __grid_constant__ CUtensorMap tmap)
{
    using C = typename cplx_of<T>::type;
    constexpr int TL = N / 16;
    constexpr int PL = fr_padded_len(N);
    constexpr int W = 2 * G;
    constexpr int ES = (int)sizeof(C);
    constexpr int ROW_BYTES = W * ES;
    constexpr int GT = (G == 1) ? 0 : TL;
    extern __shared__ __align__(1024) unsigned char fr_smem[];
    __shared__ __align__(8) uint64_t full_bar;
    unsigned char *tile = fr_smem + ((1024u - (smem_u32(fr_smem) & 1023u)) & 1023u);

    const int tid = threadIdx.x;
    const int grp = tid / TL, j = tid % TL;
    const int b = blockIdx.y;
    const int col0 = blockIdx.x * W;
    C *bufA = reinterpret_cast<C *>(tile) + (size_t)(2 * grp) * PL;
    C *bufB = bufA + PL;

    if (tid == 0) mbar_init(&full_bar, 1);
    __syncthreads();
    if (tid == 0) {
        mbar_expect_tx(&full_bar, (uint32_t)(N * ROW_BYTES));
#pragma unroll 1
        for (int r0 = 0; r0 < N; r0 += kTmaBoxRows)
            tma_load_3d(tile + (size_t)r0 * ROW_BYTES, &tmap, &full_bar, col0 * 2, r0, b);
    }
    if (tid == 32 && a.prefetch_distance > 0) {
        const int nx = (int)gridDim.x;
        int t = (int)blockIdx.x + a.prefetch_distance, bb = b;
        while (t >= nx) { t -= nx; ++bb; }
        if (bb < (int)gridDim.y) {
#pragma unroll 1
            for (int r0 = 0; r0 < N; r0 += kTmaBoxRows) tma_prefetch_3d(&tmap, t * W * 2, r0, bb);
        }
    }
    mbar_wait(&full_bar, 0);

    C vA[16], vB[16];
#pragma unroll
    for (int r = 0; r < 16; ++r) {
        const uint32_t off = (uint32_t)((j + r * TL) * ROW_BYTES + (2 * grp) * ES);
        vA[r] = *reinterpret_cast<const C *>(tile + tile_swizzle<ROW_BYTES>(off));
        vB[r] = *reinterpret_cast<const C *>(tile + tile_swizzle<ROW_BYTES>(off + ES));
    }
    __syncthreads();                                 // the landing zone becomes exchange space

    if (a.pre != nullptr) {
        dual_mul_table<T, N>(vA, a.pre + (size_t)b * N, j);
        dual_mul_table<T, N>(vB, a.pre + (size_t)b * N, j);
    }
    dual_pipeline<T, N, MODE, GT>(vA, vB, bufA, bufB, j, a, b, 1 + grp, nullptr);

    __syncthreads();                                 // every group is done with its exchange buffers
#pragma unroll
    for (int r = 0; r < 16; ++r) {
        const uint32_t off = (uint32_t)((j + r * TL) * ROW_BYTES + (2 * grp) * ES);
        *reinterpret_cast<C *>(tile + tile_swizzle<ROW_BYTES>(off)) = vA[r];
        *reinterpret_cast<C *>(tile + tile_swizzle<ROW_BYTES>(off + ES)) = vB[r];
    }
    fence_async_proxy();
    __syncthreads();
    if (tid == 0) {
#pragma unroll 1
        for (int r0 = 0; r0 < N; r0 += kTmaBoxRows)
            tma_store_3d(&tmap, tile + (size_t)r0 * ROW_BYTES, col0 * 2, r0, b);
        tma_store_commit_and_wait();
    }
}

// ---- launch geometry -------------------------------------------------------------------------------------
template <typename T, int N> struct DualGeom {
    static constexpr int TL = N / 16;
    static constexpr int ES = (int)sizeof(typename cplx_of<T>::type);
    static constexpr int G = TL >= 128 ? 1 : 128 / TL;                // pairs of lines per CTA
    static constexpr int threads = G * TL;
    static constexpr int W = 2 * G;                                   // columns per TMA tile
    static constexpr size_t smem_row = (size_t)2 * G * fr_padded_len(N) * ES;
    static constexpr size_t smem_col = smem_row + 1024;
    static constexpr bool supported = TL >= 64 && smem_col + 1024 <= 227 * 1024;   // N >= 1024, both exchange buffers on chip
#ifndef FR_DUAL_REGS_F64
#define FR_DUAL_REGS_F64 168
#endif
#ifndef FR_DUAL_REGS_F32
#define FR_DUAL_REGS_F32 96
#endif
    static constexpr int regs_goal = sizeof(T) == 8 ? FR_DUAL_REGS_F64 : FR_DUAL_REGS_F32;
    static constexpr int minb_regs = 65536 / (threads * regs_goal);
    static constexpr int minb_smem = (int)((227 * 1024) / (smem_col + 1024));
    static constexpr int minb0 = minb_regs < minb_smem ? minb_regs : minb_smem;
    static constexpr int MINB = minb0 < 1 ? 1 : (minb0 > 8 ? 8 : minb0);
};

template <typename T, int N, int MODE>
cudaError_t launch_dual_row(const PassArgs<T> &a, int batch, cudaStream_t stream)
{
    using G = DualGeom<T, N>;
    if constexpr (!G::supported) {
        return cudaErrorNotSupported;
    } else {
        auto kern = dual_row_kernel<T, N, MODE, G::G, G::MINB>;
        static bool configured = false;
        if (!configured) {
            cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)G::smem_row);
            if (e != cudaSuccess) return e;
            configured = true;
        }
        dim3 grid(N / (2 * G::G), batch, 1);
        PassArgs<T> b = a;
        if (b.prefetch_distance < 0) b.prefetch_distance = -b.prefetch_distance * G::MINB;
        kern<<<grid, G::threads, G::smem_row, stream>>>(b);
        return cudaGetLastError();
    }
}

template <typename T, int N, int MODE>
cudaError_t launch_dual_col(const PassArgs<T> &a, const CUtensorMap &tmap, int batch, cudaStream_t stream)
{
    using G = DualGeom<T, N>;
    if constexpr (!G::supported) {
        return cudaErrorNotSupported;
    } else {
        auto kern = dual_col_kernel<T, N, MODE, G::G, G::MINB>;
        static bool configured = false;
        if (!configured) {
            cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)G::smem_col);
            if (e != cudaSuccess) return e;
            configured = true;
        }
        dim3 grid(N / G::W, batch, 1);
        PassArgs<T> b = a;
        if (b.prefetch_distance < 0) b.prefetch_distance = -b.prefetch_distance * G::MINB;
        kern<<<grid, G::threads, G::smem_col, stream>>>(b, tmap);
        return cudaGetLastError();
    }
}

} // namespace fresnel
