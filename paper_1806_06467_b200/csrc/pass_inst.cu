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

} // namespace fresnel
