// pass_inst.cu -- instantiates the pass kernels for ONE grid size (compile with -DFR_N=<N>).
// One translation unit per N keeps nvcc parallel and each object small.
#include "pass_kernel.cuh"
#include "dispatch.h"

#ifndef FR_N
#error "compile with -DFR_N=<grid size>"
#endif

namespace fresnel {

template <typename T, bool COL>
static cudaError_t by_mode(int mode, const PassArgs<T> &a, int batch, cudaStream_t s)
{
    switch (mode) {
    case MODE_FWD:  return launch_pass<T, FR_N, COL, MODE_FWD>(a, batch, s);
    case MODE_INV:  return launch_pass<T, FR_N, COL, MODE_INV>(a, batch, s);
    case MODE_CONV: return launch_pass<T, FR_N, COL, MODE_CONV>(a, batch, s);
    case MODE_CONV2: return launch_pass<T, FR_N, COL, MODE_CONV2>(a, batch, s);
    }
    return cudaErrorInvalidValue;
}

template <typename T>
static cudaError_t tma_by_mode(int mode, const PassArgs<T> &a, const CUtensorMap &m, const CUtensorMap &ma, const CUtensorMap &mo,
                               int batch, cudaStream_t s)
{
    switch (mode) {
    case MODE_FWD:  return launch_col_tma<T, FR_N, MODE_FWD>(a, m, ma, mo, batch, s);
    case MODE_INV:  return launch_col_tma<T, FR_N, MODE_INV>(a, m, ma, mo, batch, s);
    case MODE_CONV: return launch_col_tma<T, FR_N, MODE_CONV>(a, m, ma, mo, batch, s);
    case MODE_CONV2: return launch_col_tma<T, FR_N, MODE_CONV2>(a, m, ma, mo, batch, s);
    }
    return cudaErrorInvalidValue;
}

#define FR_CAT2(a, b) a##b
#define FR_CAT(a, b) FR_CAT2(a, b)

cudaError_t FR_CAT(launch_pass_f32_, FR_N)(bool col, int mode, const PassArgs<float> &a, int batch, cudaStream_t s)
{
    return col ? by_mode<float, true>(mode, a, batch, s) : by_mode<float, false>(mode, a, batch, s);
}
cudaError_t FR_CAT(launch_pass_f64_, FR_N)(bool col, int mode, const PassArgs<double> &a, int batch, cudaStream_t s)
{
    return col ? by_mode<double, true>(mode, a, batch, s) : by_mode<double, false>(mode, a, batch, s);
}

cudaError_t FR_CAT(launch_col_tma_f32_, FR_N)(int mode, const PassArgs<float> &a, const CUtensorMap &m, const CUtensorMap &ma,
                                              const CUtensorMap &mo, int batch, cudaStream_t s)
{
    return tma_by_mode<float>(mode, a, m, ma, mo, batch, s);
}
cudaError_t FR_CAT(launch_col_tma_f64_, FR_N)(int mode, const PassArgs<double> &a, const CUtensorMap &m, const CUtensorMap &ma,
                                              const CUtensorMap &mo, int batch, cudaStream_t s)
{
    return tma_by_mode<double>(mode, a, m, ma, mo, batch, s);
}
// columns of a surface-map box of the fused column pass (the TMA minimum of 16 bytes may exceed the tile width)
int FR_CAT(col_tma_map_box_f32_, FR_N)() { return MapTile<float, ColTmaGeom<float, FR_N, true>::W>::BOX_COLS; }
int FR_CAT(col_tma_map_box_f64_, FR_N)() { return MapTile<double, ColTmaGeom<double, FR_N, true>::W>::BOX_COLS; }
// columns per TMA tile of the single-transform / single-convolution passes and of the fused pass (0: this N uses the
// per-thread-load column pass)
int FR_CAT(col_tma_width_f32_, FR_N)(bool conv2)
{
    if (!ColTmaGeom<float, FR_N>::supported) return 0;
    return conv2 ? ColTmaGeom<float, FR_N, true>::W : ColTmaGeom<float, FR_N, false>::W;
}
int FR_CAT(col_tma_width_f64_, FR_N)(bool conv2)
{
    if (!ColTmaGeom<double, FR_N>::supported) return 0;
    return conv2 ? ColTmaGeom<double, FR_N, true>::W : ColTmaGeom<double, FR_N, false>::W;
}

} // namespace fresnel
