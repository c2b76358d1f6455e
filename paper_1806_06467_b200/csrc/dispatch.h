// dispatch.h -- per-N launchers defined in pass_inst.cu (one object per grid size)
#pragma once
#include <cuda_runtime.h>
#include "pass_kernel.cuh"
#include "col_tma.cuh"

namespace fresnel {
#define FR_DECL(N)                                                                                              \
    cudaError_t launch_pass_f32_##N(bool col, int mode, const PassArgs<float> &a, int batch, cudaStream_t s);  \
    cudaError_t launch_pass_f64_##N(bool col, int mode, const PassArgs<double> &a, int batch, cudaStream_t s);   \
    cudaError_t launch_col_tma_f32_##N(int mode, const PassArgs<float> &a, const CUtensorMap &m, const CUtensorMap &ma,        \
                                       const CUtensorMap &mo, int batch, cudaStream_t s);                                       \
    cudaError_t launch_col_tma_f64_##N(int mode, const PassArgs<double> &a, const CUtensorMap &m, const CUtensorMap &ma,       \
                                       const CUtensorMap &mo, int batch, cudaStream_t s);                                       \
    int col_tma_map_box_f32_##N();                                                                              \
    int col_tma_map_box_f64_##N();                                                                              \
    int col_tma_width_f32_##N(bool conv2);                                                                      \
    int col_tma_width_f64_##N(bool conv2);
FR_DECL(64) FR_DECL(128) FR_DECL(256) FR_DECL(512) FR_DECL(1024) FR_DECL(2048) FR_DECL(4096) FR_DECL(8192)
#undef FR_DECL

// shared-memory pass for any other grid size (gen_kernel.cuh, instantiated in gen_inst.cu)
template <typename T> struct GenArgs;
cudaError_t launch_gen_pass_f32(const GenArgs<float> &a, const CUtensorMap &tmap, int batch, size_t smem, cudaStream_t stream);
cudaError_t launch_gen_pass_f64(const GenArgs<double> &a, const CUtensorMap &tmap, int batch, size_t smem, cudaStream_t stream);
cudaError_t launch_gen_pass_f32_256(const GenArgs<float> &a, const CUtensorMap &tmap, int batch, size_t smem, cudaStream_t stream);
cudaError_t launch_gen_pass_f32_512(const GenArgs<float> &a, const CUtensorMap &tmap, int batch, size_t smem, cudaStream_t stream);
cudaError_t launch_gen_pass_f64_256(const GenArgs<double> &a, const CUtensorMap &tmap, int batch, size_t smem, cudaStream_t stream);
cudaError_t launch_gen_pass_f64_512(const GenArgs<double> &a, const CUtensorMap &tmap, int batch, size_t smem, cudaStream_t stream);

// register-resident mixed-radix pass (mr_kernel.cuh, instantiated in mr_inst.cu) for these grid sizes
#define FR_MR_SIZES(X) X(700) X(1000) X(1200) X(1400) X(1500) X(2000) X(2400) X(2800) X(3000) X(3600) X(4000) X(5000) X(5600) X(6000)
cudaError_t launch_mr_f32(int N, bool col, int mode, const GenArgs<float> &a, const CUtensorMap &m, int batch, cudaStream_t s);
cudaError_t launch_mr_f64(int N, bool col, int mode, const GenArgs<double> &a, const CUtensorMap &m, int batch, cudaStream_t s);
int mr_col_width(int N, int elem_bytes);
#define FR_DECL_MR(N)                                                                                                              \
    cudaError_t launch_mr_f32_##N(bool col, int mode, const GenArgs<float> &a, const CUtensorMap &m, int batch, cudaStream_t s);   \
    cudaError_t launch_mr_f64_##N(bool col, int mode, const GenArgs<double> &a, const CUtensorMap &m, int batch, cudaStream_t s);  \
    int mr_col_width_##N(int elem_bytes);
FR_MR_SIZES(FR_DECL_MR)
#undef FR_DECL_MR
} // namespace fresnel
