// gen_inst.cu -- instantiates the shared-memory pass for grids that are not a power of two (gen_kernel.cuh): compiled with
// -DFR_GEN_F64=<0|1> -DFR_GEN_NT=<256|512> for one (precision, CTA size) each, and once without them for the dispatch.
#include "gen_kernel.cuh"
#include "dispatch.h"

namespace fresnel {

#ifdef FR_GEN_NT
#if FR_GEN_F64
#define FR_GEN_NAME2(nt) launch_gen_pass_f64_##nt
using gen_real = double;
#else
#define FR_GEN_NAME2(nt) launch_gen_pass_f32_##nt
using gen_real = float;
#endif
#define FR_GEN_NAME(nt) FR_GEN_NAME2(nt)
cudaError_t FR_GEN_NAME(FR_GEN_NT)(const GenArgs<gen_real> &a, const CUtensorMap &tmap, int batch, size_t smem, cudaStream_t stream)
{
    return launch_gen_pass_nt<gen_real, FR_GEN_NT>(a, tmap, batch, smem, stream);
}
#else
// two CTAs of kGenThreads per SM where their buffers fit, else one of twice the size
static bool gen_two_ctas(size_t smem) { return 2 * (smem + 1024) <= (size_t)227 * 1024; }
cudaError_t launch_gen_pass_f32(const GenArgs<float> &a, const CUtensorMap &tmap, int batch, size_t smem, cudaStream_t stream)
{
    return gen_two_ctas(smem) ? launch_gen_pass_f32_256(a, tmap, batch, smem, stream) : launch_gen_pass_f32_512(a, tmap, batch, smem, stream);
}
cudaError_t launch_gen_pass_f64(const GenArgs<double> &a, const CUtensorMap &tmap, int batch, size_t smem, cudaStream_t stream)
{
    return gen_two_ctas(smem) ? launch_gen_pass_f64_256(a, tmap, batch, smem, stream) : launch_gen_pass_f64_512(a, tmap, batch, smem, stream);
}
#endif

} // namespace fresnel
