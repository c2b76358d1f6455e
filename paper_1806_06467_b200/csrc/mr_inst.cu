// mr_inst.cu -- the register-resident mixed-radix pass (mr_kernel.cuh): compiled once per supported grid size with
// -DFR_MR_N=<N> (one object per size keeps nvcc parallel), and once without it for the by-size dispatch.
#include "mr_kernel.cuh"
#include "dispatch.h"

namespace fresnel {

#define FR_CAT2(a, b) a##b
#define FR_CAT(a, b) FR_CAT2(a, b)

#ifdef FR_MR_N

template <typename T, bool COL>
static cudaError_t mr_by_mode(int mode, const GenArgs<T> &a, const CUtensorMap &m, int batch, cudaStream_t s)
{
    switch (mode) {
    case MODE_FWD:  return launch_mr_pass<T, FR_MR_N, COL, MODE_FWD>(a, m, batch, s);
    case MODE_INV:  return launch_mr_pass<T, FR_MR_N, COL, MODE_INV>(a, m, batch, s);
    case MODE_CONV: return launch_mr_pass<T, FR_MR_N, COL, MODE_CONV>(a, m, batch, s);
    }
    return cudaErrorInvalidValue;
}

cudaError_t FR_CAT(launch_mr_f32_, FR_MR_N)(bool col, int mode, const GenArgs<float> &a, const CUtensorMap &m, int batch, cudaStream_t s)
{
    return col ? mr_by_mode<float, true>(mode, a, m, batch, s) : mr_by_mode<float, false>(mode, a, m, batch, s);
}
cudaError_t FR_CAT(launch_mr_f64_, FR_MR_N)(bool col, int mode, const GenArgs<double> &a, const CUtensorMap &m, int batch, cudaStream_t s)
{
    return col ? mr_by_mode<double, true>(mode, a, m, batch, s) : mr_by_mode<double, false>(mode, a, m, batch, s);
}
// columns per TMA tile of the column pass
int FR_CAT(mr_col_width_, FR_MR_N)(int elem_bytes)
{
    return elem_bytes == 16 ? MrGeom<double, FR_MR_N, true>::W : MrGeom<float, FR_MR_N, true>::W;
}

#else

cudaError_t launch_mr_f32(int N, bool col, int mode, const GenArgs<float> &a, const CUtensorMap &m, int batch, cudaStream_t s)
{
    switch (N) {
#define FR_CASE(NN) case NN: return launch_mr_f32_##NN(col, mode, a, m, batch, s);
        FR_MR_SIZES(FR_CASE)
#undef FR_CASE
    }
    return cudaErrorNotSupported;
}
cudaError_t launch_mr_f64(int N, bool col, int mode, const GenArgs<double> &a, const CUtensorMap &m, int batch, cudaStream_t s)
{
    switch (N) {
#define FR_CASE(NN) case NN: return launch_mr_f64_##NN(col, mode, a, m, batch, s);
        FR_MR_SIZES(FR_CASE)
#undef FR_CASE
    }
    return cudaErrorNotSupported;
}
// columns per TMA tile of the column pass (0: this grid size is not taken by the register-resident path)
int mr_col_width(int N, int elem_bytes)
{
    switch (N) {
#define FR_CASE(NN) case NN: return mr_col_width_##NN(elem_bytes);
        FR_MR_SIZES(FR_CASE)
#undef FR_CASE
    }
    return 0;
}

#endif

} // namespace fresnel
