// col_tma.cuh -- the COLUMN pass with TMA tile movement (sm_100a).
//
// A column tile is [N rows] x [W adjacent columns]: W*sizeof(complex) contiguous bytes per row at a
// pitch of N*sizeof(complex).  Gathered with per-thread loads this costs the load/store pipe one
// wavefront per 128-byte line touched (8..32 per warp instruction instead of 4), which made the
// column pass the slowest kernel.  Here one elected thread asks the TMA unit for the whole tile
// (cp.async.bulk.tensor, boxes of 256 rows x W columns, hardware-swizzled so that a column can be
// read back without bank conflicts); the tile lands in the shared memory that afterwards serves as
// the exchange buffers, and goes back to HBM the same way.  The W columns of a tile are independent
// transforms: each is owned by its own group of N/16 threads that synchronises on a private
// named barrier, so the groups of a CTA drift apart and overlap one another's FP64 and
// shared-memory phases.  Only the tile load and the tile store are CTA-wide events.
#pragma once
#include <cuda.h>
#include <cstdint>
#include "pass_kernel.cuh"

namespace fresnel {

FR_DEV uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

FR_DEV void mbar_init(uint64_t *bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
FR_DEV void mbar_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
FR_DEV void mbar_wait(uint64_t *bar, uint32_t parity)
{
    uint32_t done;
    do {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(done) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    } while (!done);
}
FR_DEV void tma_load_3d(void *dst, const CUtensorMap *map, uint64_t *bar, int x, int y, int z)
{
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
                 ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(bar)), "r"(x), "r"(y), "r"(z) : "memory");
}
FR_DEV void tma_load_2d(void *dst, const CUtensorMap *map, uint64_t *bar, int x, int y)
{
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];"
                 ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(bar)), "r"(x), "r"(y) : "memory");
}
FR_DEV void tma_store_3d(const CUtensorMap *map, const void *src, int x, int y, int z)
{
    asm volatile("cp.async.bulk.tensor.3d.global.shared::cta.bulk_group [%0, {%2, %3, %4}], [%1];"
                 ::"l"(map), "r"(smem_u32(src)), "r"(x), "r"(y), "r"(z) : "memory");
}
FR_DEV void tma_store_commit_and_wait()
{
    asm volatile("cp.async.bulk.commit_group;" ::: "memory");
    asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");   // shared memory may be released
}
// L2 prefetch of a tile box (no shared-memory destination): the tile a later CTA will ask for
FR_DEV void tma_prefetch_3d(const CUtensorMap *map, int x, int y, int z)
{
    asm volatile("cp.async.bulk.prefetch.tensor.3d.L2.global [%0, {%1, %2, %3}];" ::"l"(map), "r"(x), "r"(y), "r"(z) : "memory");
}
FR_DEV void fence_async_proxy() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// byte offset of element (row, col) of a [rows][W] tile written by TMA with the swizzle mode that
// matches the row length (32 / 64 / 128 bytes): XOR of the 16-byte-chunk bits with address bits 7..9
template <int ROW_BYTES> FR_DEV uint32_t tile_swizzle(uint32_t off)
{
    if constexpr (ROW_BYTES == 32) return off ^ ((off >> 3) & 0x10);
    else if constexpr (ROW_BYTES == 64) return off ^ ((off >> 3) & 0x30);
    else if constexpr (ROW_BYTES == 128) return off ^ ((off >> 3) & 0x70);
    else return off;     // 16-byte rows: no swizzle
}

constexpr int kTmaBoxRows = 256;

// Column tile of a REAL [N][N] surface map, fetched in the middle of a fused kernel (MODE_CONV2) into the exchange
// space while it is idle: rows of max(W * sizeof(T), 16) bytes (the TMA minimum), no swizzle.  Every thread then
// picks up its 16 entries (rows j + r*TL of column g).
template <typename T, int W> struct MapTile {
    static constexpr int ROW_BYTES = (W * (int)sizeof(T) < 16) ? 16 : W * (int)sizeof(T);
    static constexpr int BOX_COLS = ROW_BYTES / (int)sizeof(T);
    // A box has to START on a 16-byte boundary of the map row (measured: an 8-byte-aligned start is an illegal
    // instruction), so a tile narrower than the box takes the aligned box around it and reads at an offset.
    static __device__ __forceinline__ int box_x(int col0) { return col0 & ~(BOX_COLS - 1); }
    static __device__ __forceinline__ int col_in_box(int col0, int g) { return (col0 & (BOX_COLS - 1)) + g; }
};

template <typename T, int N, int W>
FR_DEV void fetch_map_tile(unsigned char *tile, const CUtensorMap *mmap, uint64_t *bar, uint32_t &parity, int col0, int tid)
{
    using MT = MapTile<T, W>;
    fence_async_proxy();                             // the exchange traffic (generic proxy) is ordered before the TMA writes
    __syncthreads();                                 // every group is done with the exchange space
    if (tid == 0) {
        mbar_expect_tx(bar, (uint32_t)(N * MT::ROW_BYTES));
#pragma unroll 1
        for (int r0 = 0; r0 < N; r0 += kTmaBoxRows) tma_load_2d(tile + (size_t)r0 * MT::ROW_BYTES, mmap, bar, MT::box_x(col0), r0);
    }
    mbar_wait(bar, parity);
    parity ^= 1u;
}

// Fused column pass: where MINB resident CTAs still fit with it, the FIRST map of the in-between optic gets a
// landing zone of its own behind the tile and is fetched at kernel start (it is an input, not a result of the
// previous pass, so the fetch does not even wait for it): no bubble between the two convolutions.  Elsewhere
// (N >= 2048) the map is fetched into the idle exchange space when it is needed.
template <typename T, int N, int W, int MINB> struct ColMapBuf {
    static constexpr int ES = (int)sizeof(typename cplx_of<T>::type);
    static constexpr size_t tile_bytes = ((size_t)W * fr_padded_len(N) * ES + 127) / 128 * 128;
    static constexpr size_t map_bytes = (size_t)N * MapTile<T, W>::ROW_BYTES;
#ifdef FR_NO_MAPBUF      // tuning / debugging builds only
    static constexpr bool enabled = false;
#else
    static constexpr bool enabled = (size_t)MINB * (tile_bytes + map_bytes + 1024 + 64) <= (size_t)227 * 1024;
#endif
};

template <typename T, int N, int W, int MODE, int MINB>
__global__ void __launch_bounds__(W *(N / 16), MINB)
col_tma_kernel(PassArgs<T> a, const __grid_constant__ CUtensorMap tmap, const __grid_constant__ CUtensorMap tmap_amp2,
               const __grid_constant__ CUtensorMap tmap_opd2)
{
    using C = typename cplx_of<T>::type;
    constexpr int TL = N / 16;                       // threads per column
    constexpr int ES = (int)sizeof(C);
    constexpr int ROW_BYTES = W * ES;
    // Thread <-> (column g, position j).  complex64: adjacent lanes take adjacent columns of the same row, so a warp reads
    // and writes whole tile rows -- 8-byte elements of 16 / 32-byte rows otherwise cost two to four shared-memory wavefronts
    // per access (ncu: ten times the bank conflicts of the row pass) -- at the price of CTA-wide exchange barriers instead of
    // one named barrier per column group (measured: column pass -3..5 % at N = 2048..8192).  complex128 (16-byte elements,
    // swizzled 32-byte rows) gains nothing from it and keeps one thread group per column.  FR_COL_INTERLEAVE: bit 0
    // complex64, bit 1 complex128 (tuning builds).
#ifndef FR_COL_INTERLEAVE
#define FR_COL_INTERLEAVE 1
#endif
    constexpr bool IL = (W > 1) && (sizeof(T) == 4 ? (FR_COL_INTERLEAVE & 1) : (FR_COL_INTERLEAVE & 2)) != 0;
    constexpr int GT = (W == 1 || IL) ? 0 : TL;      // group barrier size (0: the whole CTA)
    extern __shared__ __align__(1024) unsigned char fr_smem[];
    __shared__ __align__(8) uint64_t full_bar;
    __shared__ __align__(8) uint64_t map_bar;
    constexpr bool MAPBUF = MODE == MODE_CONV2 && ColMapBuf<T, N, W, MINB>::enabled;
    // 1024-byte alignment (the TMA swizzle pattern is a function of the shared-memory address)
    unsigned char *tile = fr_smem + ((1024u - (smem_u32(fr_smem) & 1023u)) & 1023u);   // landing zone, later the exchange buffers
    C *buf = reinterpret_cast<C *>(tile);

    const int tid = threadIdx.x;
    const int g = IL ? tid % W : tid / TL;           // column of the tile (== thread group unless interleaved)
    const int j = IL ? tid / W : tid % TL;
    const int b = blockIdx.y;
    const int col0 = blockIdx.x * W;

    if (tid == 0) {
        mbar_init(&full_bar, 1);
        if constexpr (MAPBUF) mbar_init(&map_bar, 1);
    }
    pdl_launch_dependents();
    __syncthreads();
    if constexpr (MAPBUF) {
        if (tid == 0 && (a.opd2 != nullptr || a.amp2 != nullptr)) {
            using MT = MapTile<T, W>;
            unsigned char *mapbuf = tile + ColMapBuf<T, N, W, MINB>::tile_bytes;
            const CUtensorMap *mm = a.opd2 != nullptr ? &tmap_opd2 : &tmap_amp2;
            mbar_expect_tx(&map_bar, (uint32_t)(N * MT::ROW_BYTES));
#pragma unroll 1
            for (int r0 = 0; r0 < N; r0 += kTmaBoxRows) tma_load_2d(mapbuf + (size_t)r0 * MT::ROW_BYTES, mm, &map_bar, MT::box_x(col0), r0);
        }
    }
    pdl_wait();                                      // the row pass has finished: the wavefront may be read
    if (tid == 0) {
        mbar_expect_tx(&full_bar, (uint32_t)(N * ROW_BYTES));
#pragma unroll 1
        for (int r0 = 0; r0 < N; r0 += kTmaBoxRows)
            tma_load_3d(tile + (size_t)r0 * ROW_BYTES, &tmap, &full_bar, col0 * 2, r0, b);
    }
    // Ask L2 for the tile that the CTA taking over one of the currently resident slots will need
    // (CTAs are dispatched in blockIdx order): HBM then streams while this tile is being computed.
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

    C v[16];
#pragma unroll
    for (int r = 0; r < 16; ++r) {
        const uint32_t off = (uint32_t)((j + r * TL) * ROW_BYTES + g * ES);
        v[r] = *reinterpret_cast<const C *>(tile + tile_swizzle<ROW_BYTES>(off));
    }
    __syncthreads();                                 // the landing zone becomes exchange space

    if (a.pre != nullptr) {
        const C *p = a.pre + (size_t)b * N;
#pragma unroll
        for (int r = 0; r < 16; ++r) v[r] = cmul(v[r], ldg_c(p + j + r * TL));
    }
    line_transforms<T, N, MODE, IL, W, GT>(v, buf, g, j, b, a, 1 + g, [&](C (&u)[16]) {
        // MODE_CONV2: the optic of the next surface on the resident tile; its maps arrive by TMA in the exchange
        // space, which is idle between the two convolutions
        using MT = MapTile<T, W>;
        uint32_t parity = 1;                         // phase 0 was the wavefront tile
        const unsigned char *mt = tile;              // where the current map tile is read from
        bool synced = false;                         // a CTA-wide sync is owed before the exchange space is reused
        if (a.opd2 != nullptr) {
            if constexpr (MAPBUF) { mbar_wait(&map_bar, 0); mt = tile + ColMapBuf<T, N, W, MINB>::tile_bytes; }
            else { fetch_map_tile<T, N, W>(tile, &tmap_opd2, &full_bar, parity, col0, tid); synced = true; }
            const T il = (T)a.inv_lambda[b];
            T ph[16];
            bool all_small = true;
#pragma unroll
            for (int r = 0; r < 16; ++r) {
                ph[r] = *reinterpret_cast<const T *>(mt + (size_t)(j + r * TL) * MT::ROW_BYTES + MT::col_in_box(col0, g) * sizeof(T)) * il;
                all_small = all_small && phasor_is_small(ph[r]);
            }
            if (all_small) {
#pragma unroll
                for (int r = 0; r < 16; ++r) u[r] = cmul(u[r], phasor_turns_small(ph[r]));
            } else {
#pragma unroll
                for (int r = 0; r < 16; ++r) u[r] = cmul(u[r], phasor_turns_any(ph[r]));
            }
        }
        if (a.amp2 != nullptr) {
            if (MAPBUF && a.opd2 == nullptr) { mbar_wait(&map_bar, 0); mt = tile + ColMapBuf<T, N, W, MINB>::tile_bytes; }
            else { fetch_map_tile<T, N, W>(tile, &tmap_amp2, &full_bar, parity, col0, tid); mt = tile; synced = true; }
#pragma unroll
            for (int r = 0; r < 16; ++r) {
                const T s = *reinterpret_cast<const T *>(mt + (size_t)(j + r * TL) * MT::ROW_BYTES + MT::col_in_box(col0, g) * sizeof(T));
                u[r].x *= s; u[r].y *= s;
            }
        }
        if (synced) __syncthreads();                 // a map tile was read from the exchange space: release it
        if (a.lens2 != nullptr) {
            const C *l = a.lens2 + (size_t)b * N;
            const C c = ldg_c(l + col0 + g);
#pragma unroll
            for (int r = 0; r < 16; ++r) u[r] = cmul(u[r], cmul(ldg_c(l + j + r * TL), c));
        }
    });
    if (a.scale != (T)1) {
#pragma unroll
        for (int r = 0; r < 16; ++r) { v[r].x *= a.scale; v[r].y *= a.scale; }
    }

    __syncthreads();                                 // every group is done with its exchange buffer
    // (the tile offsets are recomputed from an opaque copy of j: kept from the load they cost nine spilled registers that
    // come back from local memory right here, at the end of the CTA's life)
    int js = j;
    asm volatile("" : "+r"(js));
#pragma unroll
    for (int r = 0; r < 16; ++r) {
        const uint32_t off = (uint32_t)((js + r * TL) * ROW_BYTES + g * ES);
        *reinterpret_cast<C *>(tile + tile_swizzle<ROW_BYTES>(off)) = v[r];
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

// columns per tile for the TMA column pass.  The fused pass (conv2: two convolutions and an optic per tile, i.e. twice the
// arithmetic per byte) at N = 2048 does better with 16-byte-wide tiles and FOUR resident CTAs of one column group each than
// with 32-byte-wide tiles and two CTAs (measured: 93.2 -> 86.2 us complex128, 57.3 -> 52.3 us complex64; the single
// convolution is the other way round, 44.8 vs 48.4 us): the tile load of one CTA hides under three others.
__host__ __device__ constexpr int fr_tma_cols(int N, int elem_bytes, bool conv2 = false)
{
    const int TL = N / 16;
    if (elem_bytes == 16) {
#ifdef FR_TMAW_F64
        if (FR_TMAW_F64 * TL <= 512) return FR_TMAW_F64;
#endif
        if (conv2 && N == 2048) return 1;
        return N <= 1024 ? 4 : (N <= 2048 ? 2 : 1);       // >= 2 resident CTAs per SM wherever the tile allows
    }
#ifdef FR_TMAW_F32
    if (FR_TMAW_F32 * TL <= 1024) return FR_TMAW_F32;
#endif
    if (conv2 && N == 2048) return 2;
    return N <= 1024 ? 8 : (N <= 2048 ? 4 : 2);
}

template <typename T, int N, bool CONV2 = false> struct ColTmaGeom {
    static constexpr int TL = N / 16;
    static constexpr int ES = (int)sizeof(typename cplx_of<T>::type);
    static constexpr int W = fr_tma_cols(N, ES, CONV2);
    static constexpr int threads = W * TL;
    static constexpr size_t smem = (size_t)W * fr_padded_len(N) * ES;
    static constexpr int regs_goal = sizeof(T) == 8 ? FR_REGS_F64 : (N <= 512 && FR_REGS_F32 < 72 ? 72 : FR_REGS_F32);   // as PassGeom
    static constexpr int minb_regs = 65536 / (threads * regs_goal);
    static constexpr int minb_smem = (int)((226 * 1024) / (smem + 1024));
    static constexpr int minb0 = minb_regs < minb_smem ? minb_regs : minb_smem;
    static constexpr int MINB = minb0 < 1 ? 1 : (minb0 > 8 ? 8 : minb0);
    static constexpr bool supported = TL >= 32;      // named barriers work on whole warps
    // dynamic shared memory of the fused (MODE_CONV2) kernel: tile + alignment slack [+ map landing zone]
    static constexpr size_t smem_conv2 = ColMapBuf<T, N, W, MINB>::enabled
        ? ColMapBuf<T, N, W, MINB>::tile_bytes + ColMapBuf<T, N, W, MINB>::map_bytes + 1024 : smem + 1024;
};

// tmap: the wavefront; tmap_amp2 / tmap_opd2: the maps of the in-between optic (MODE_CONV2; read only when
// a.amp2 / a.opd2 are non-null, any valid tensor map otherwise)
template <typename T, int N, int MODE>
cudaError_t launch_col_tma(const PassArgs<T> &a, const CUtensorMap &tmap, const CUtensorMap &tmap_amp2, const CUtensorMap &tmap_opd2,
                           int batch, cudaStream_t stream)
{
    using G = ColTmaGeom<T, N, MODE == MODE_CONV2>;
    if constexpr (!G::supported) {
        return cudaErrorNotSupported;
    } else {
        auto kern = col_tma_kernel<T, N, G::W, MODE, G::MINB>;
        constexpr size_t dyn_smem = MODE == MODE_CONV2 ? G::smem_conv2 : G::smem + 1024;
        static std::atomic<unsigned long long> configured{0};
        if (fr_needs_configuring(configured)) {
            cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn_smem);
            if (e != cudaSuccess) return e;
            fr_mark_configured(configured);
        }
        dim3 grid(N / G::W, batch, 1);
        PassArgs<T> b = a;
        if (b.prefetch_distance < 0) b.prefetch_distance = -b.prefetch_distance * G::MINB;
        return launch_pdl(kern, grid, dim3(G::threads), dyn_smem, stream, b.pdl != 0, b, tmap, tmap_amp2, tmap_opd2);
    }
}

} // namespace fresnel
