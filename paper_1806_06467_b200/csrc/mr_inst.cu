// mr_inst.cu -- instantiates the register-resident mixed-radix pass (mr_kernel.cuh) for the grid sizes it supports.
#include "mr_kernel.cuh"
#include "dispatch.h"

namespace fresnel {

template <typename T, int N, bool COL>
static cudaError_t mr_by_mode(int mode, const GenArgs<T> &a, const CUtensorMap &m, int batch, cudaStream_t s)
{
    switch (mode) {
    case MODE_FWD:  return launch_mr_pass<T, N, COL, MODE_FWD>(a, m, batch, s);
    case MODE_INV:  return launch_mr_pass<T, N, COL, MODE_INV>(a, m, batch, s);
    case MODE_CONV: return launch_mr_pass<T, N, COL, MODE_CONV>(a, m, batch, s);
    }
    return cudaErrorInvalidValue;
}

template <typename T>
static cudaError_t mr_by_size(int N, bool col, int mode, const GenArgs<T> &a, const CUtensorMap &m, int batch, cudaStream_t s)
{
    switch (N) {
#define FR_CASE(NN) case NN: return col ? mr_by_mode<T, NN, true>(mode, a, m, batch, s) : mr_by_mode<T, NN, false>(mode, a, m, batch, s);
        FR_MR_SIZES(FR_CASE)
#undef FR_CASE
    }
    return cudaErrorNotSupported;
}

cudaError_t launch_mr_f32(int N, bool col, int mode, const GenArgs<float> &a, const CUtensorMap &m, int batch, cudaStream_t s)
{
    return mr_by_size<float>(N, col, mode, a, m, batch, s);
}
cudaError_t launch_mr_f64(int N, bool col, int mode, const GenArgs<double> &a, const CUtensorMap &m, int batch, cudaStream_t s)
{
    return mr_by_size<double>(N, col, mode, a, m, batch, s);
}

// columns per TMA tile of the column pass (0: this grid size is not taken by the register-resident path)
int mr_col_width(int N, int elem_bytes)
{
    switch (N) {
#define FR_CASE(NN) case NN: return elem_bytes == 16 ? MrGeom<double, NN, true>::W : MrGeom<float, NN, true>::W;
        FR_MR_SIZES(FR_CASE)
#undef FR_CASE
    }
    return 0;
}

} // namespace fresnel
