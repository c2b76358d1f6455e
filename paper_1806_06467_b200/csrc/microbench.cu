// microbench.cu -- stand-alone measurements behind DESIGN.md's design decisions (not part of libfresnel.so):
//   HBM copy bandwidth, row-tile vs column-tile (strided 16/32/64/128-byte segment) in-place copies with
//   per-thread loads, L2-resident read bandwidth, and the plain-ALU roofs (DFMA / FFMA) that
//   MEASURED_PEAKS.json does not carry; and the IN-SM rates of the transform itself (no HBM): the stage code
//   of fft_core.cuh on registers + shared memory only -- butterflies alone, exchanges alone, both -- in SM
//   cycles per element, next to a synthetic stream that interleaves DFMA with 128-bit shared-memory traffic
//   in every warp (what the two pipes can do when nothing orders them).  These are the numbers bench.py's
//   `roofline.alu.peak_tflops` and DESIGN.md's "balance" paragraph quote (profiles/r01_microbench.txt; the
//   shuffle / tensor-memory lines of that file came from probes that are no longer part of the repository).
//   Build + run:
//     python -m paper_1806_06467_b200.build --microbench && ./paper_1806_06467_b200/microbench
#include <cstdio>
#include <cstdlib>
#include <cuda_runtime.h>
#include "fft_core.cuh"
#define CK(x) do{cudaError_t e=(x); if(e!=cudaSuccess){printf("CUDA error %s at %d\n",cudaGetErrorString(e),__LINE__); exit(1);} }while(0)

__global__ void copy16(const int4* __restrict__ a, int4* __restrict__ b, size_t n){
  size_t i = blockIdx.x*(size_t)blockDim.x+threadIdx.x; size_t st=(size_t)gridDim.x*blockDim.x;
  for(; i<n; i+=st) b[i]=a[i];
}
// column-tile in-place read-modify-write: matrix N x N of 16-byte elements; each CTA takes a tile of SEG bytes wide x N rows.
// thread mapping: lanes cover SEG/16 elements of a row then next row. Each thread handles R=16 rows at stride N/16... emulate pass kernel
template<int SEGE> // elements (16B) per segment
__global__ void coltile(int4* __restrict__ a, int N){
  int TL=N/16; int tid=threadIdx.x; int c=tid%SEGE; int j=tid/SEGE; 
  size_t col=(size_t)blockIdx.x*SEGE+c;
  int4 v[16];
  #pragma unroll
  for(int r=0;r<16;++r) v[r]=a[(size_t)(j+r*TL)*N+col];
  #pragma unroll
  for(int r=0;r<16;++r){ v[r].x^=1; }
  #pragma unroll
  for(int r=0;r<16;++r) a[(size_t)(j+r*TL)*N+col]=v[r];
}
template<int SEGE>
__global__ void rowtile(int4* __restrict__ a, int N){
  int TL=N/16; int tid=threadIdx.x; int j=tid%TL; int line=tid/TL;
  size_t row=(size_t)blockIdx.x*SEGE+line;
  int4 v[16];
  #pragma unroll
  for(int r=0;r<16;++r) v[r]=a[row*N+(j+r*TL)];
  #pragma unroll
  for(int r=0;r<16;++r){ v[r].x^=1; }
  #pragma unroll
  for(int r=0;r<16;++r) a[row*N+(j+r*TL)]=v[r];
}
__global__ void l2read(const int4* __restrict__ a, size_t n, int iters, int* out){
  size_t st=(size_t)gridDim.x*blockDim.x; int acc=0;
  for(int it=0;it<iters;++it){
    for(size_t i=blockIdx.x*(size_t)blockDim.x+threadIdx.x;i<n;i+=st){ int4 v=__ldcg(a+i); acc+=v.x^v.y^v.z^v.w; }
  }
  if(acc==0x12345678) *out=acc;
}
template<typename T> __global__ void fmapeak(T* out, int iters){
  T a0=threadIdx.x, a1=a0+1, a2=a0+2, a3=a0+3, a4=a0+4,a5=a0+5,a6=a0+6,a7=a0+7; T b=(T)1.0000001, c=(T)0.5;
  for(int i=0;i<iters;++i){
    #pragma unroll
    for(int u=0;u<16;++u){ a0=a0*b+c; a1=a1*b+c; a2=a2*b+c; a3=a3*b+c; a4=a4*b+c; a5=a5*b+c; a6=a6*b+c; a7=a7*b+c; }
  }
  out[blockIdx.x*blockDim.x+threadIdx.x]=a0+a1+a2+a3+a4+a5+a6+a7;
}
template<typename F> float timeit(F f, int reps=10){
  cudaEvent_t e0,e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
  f(); f(); cudaDeviceSynchronize();
  float best=1e30;
  for(int i=0;i<reps;++i){ cudaEventRecord(e0); f(); cudaEventRecord(e1); cudaEventSynchronize(e1); float ms; cudaEventElapsedTime(&ms,e0,e1); if(ms<best)best=ms; }
  return best;
}
template<int SEGE> void run_col(int4* a,int N){
  int threads=SEGE*(N/16); if(threads>1024){ printf("  col N=%d seg=%dB: skip (threads %d)\n",N,SEGE*16,threads); return;}
  float ms=timeit([&]{ coltile<SEGE><<<N/SEGE,threads>>>(a,N); });
  CK(cudaGetLastError());
  double bytes=2.0*N*(double)N*16; printf("  col N=%d seg=%3dB threads=%4d: %.3f ms  %.0f GB/s\n",N,SEGE*16,threads,ms,bytes/ms/1e6);
}
template<int SEGE> void run_row(int4* a,int N){
  int threads=SEGE*(N/16); if(threads>1024) return;
  float ms=timeit([&]{ rowtile<SEGE><<<N/SEGE,threads>>>(a,N); });
  CK(cudaGetLastError());
  double bytes=2.0*N*(double)N*16; printf("  row N=%d lines=%d threads=%4d: %.3f ms  %.0f GB/s\n",N,SEGE,threads,ms,bytes/ms/1e6);
}
// ---- in-SM rates ---------------------------------------------------------------------------------------------
// VAR 0: forward + inverse transform of a line (the convolution pass without its table multiplies),
// VAR 1: the butterflies and twiddles of the same stages only, VAR 2: the four exchanges only.
// G groups of N/16 threads per CTA, one CTA per SM; GTX = 32 replaces the group barriers by __syncwarp
// (timing only: the bound a warp-local exchange could reach).
template <typename T, int N, int G, int VAR, int GTX>
__global__ void __launch_bounds__(G * (N / 16), 1) insm(int iters, const typename fresnel::cplx_of<T>::type* tw, typename fresnel::cplx_of<T>::type* out){
  using namespace fresnel; using C = typename cplx_of<T>::type;
  constexpr int TL = N / 16, PL = fr_padded_len(N); constexpr int GT = GTX >= 0 ? GTX : (G == 1 ? 0 : TL);
  extern __shared__ __align__(16) unsigned char smraw[];
  const int tid = threadIdx.x, grp = tid / TL, j = tid % TL;
  C* buf = reinterpret_cast<C*>(smraw) + (size_t)grp * PL;
  C v[16];
  #pragma unroll
  for (int r = 0; r < 16; ++r) { v[r].x = (T)(tid + r) * (T)1e-3; v[r].y = (T)r; }
  for (int it = 0; it < iters; ++it) {
    int jj = j; asm volatile("" : "+r"(jj));            // keep address and twiddle arithmetic inside the loop
    const C* t = tw; asm volatile("" : "+l"(t));
    if (VAR == 0) {
      fft_line<T, N, -1, false, 1, GT>(v, buf, 0, jj, t, 1 + grp);
      asm volatile("" : "+l"(t));
      fft_line<T, N, +1, false, 1, GT>(v, buf, 0, jj, t, 1 + grp);
    } else if (VAR == 1) {
      fft_stage_compute<T, N, 0, -1>(v, jj, t); fft_stage_compute<T, N, 1, -1>(v, jj, t);
      if constexpr (fr_num_stages(N) > 2) fft_stage_compute<T, N, 2, -1>(v, jj, t);
      asm volatile("" : "+l"(t));
      fft_stage_compute<T, N, 0, +1>(v, jj, t); fft_stage_compute<T, N, 1, +1>(v, jj, t);
      if constexpr (fr_num_stages(N) > 2) fft_stage_compute<T, N, 2, +1>(v, jj, t);
    } else {
      #pragma unroll
      for (int rep = 0; rep < 2; ++rep) {
        fft_stage_scatter<T, N, 0, false, 1>(v, buf, 0, jj); fr_sync<GT>(1 + grp);
        fft_stage_gather<T, N, false, 1>(v, buf, 0, jj); fr_sync<GT>(1 + grp);
        fft_stage_scatter<T, N, 1, false, 1>(v, buf, 0, jj); fr_sync<GT>(1 + grp);
        fft_stage_gather<T, N, false, 1>(v, buf, 0, jj); fr_sync<GT>(1 + grp);
      }
    }
    #pragma unroll
    for (int r = 0; r < 16; ++r) { v[r].x *= (T)0.01; v[r].y *= (T)0.01; }
  }
  C s = v[0];
  #pragma unroll
  for (int r = 1; r < 16; ++r) { s.x += v[r].x; s.y += v[r].y; }
  out[blockIdx.x * blockDim.x + tid] = s;
}
template <typename T, int N, int G, int VAR, int GTX = -1> void run_insm(const char* what, double clock_hz){
  using C = typename fresnel::cplx_of<T>::type;
  C *tw, *out; CK(cudaMalloc(&tw, 65536 * sizeof(C))); CK(cudaMemset(tw, 0, 65536 * sizeof(C))); CK(cudaMalloc(&out, 148 * 1024 * sizeof(C)));
  const int smem = G * fresnel::fr_padded_len(N) * sizeof(C);
  CK(cudaFuncSetAttribute(insm<T, N, G, VAR, GTX>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
  const int iters = 400;
  float ms = timeit([&]{ insm<T, N, G, VAR, GTX><<<148, G * (N / 16), smem>>>(iters, tw, out); }, 3);
  CK(cudaGetLastError());
  printf("  in-SM %-22s N=%d %s groups/SM=%d: %.3f clk/element/SM\n", what, N, sizeof(T) == 8 ? "f64" : "f32", G, ms * 1e-3 * clock_hz / iters / ((double)G * N));
  cudaFree(tw); cudaFree(out);
}
// two lines per thread group with ONE register set: a line lives in shared memory between its stages (gather ->
// stage -> scatter per block, lines A and B alternating), so the exchange latency of one line lies under the
// butterflies of the other.  Every transform here ends with one extra (natural-order) exchange that a real pass
// would replace by its global load / store, so compare LINES = 2 with LINES = 1 of this same kernel.
template <typename T, int N, int STAGE, int DIR, int GT>
__device__ __forceinline__ void alt_block(typename fresnel::cplx_of<T>::type* buf, int j, const typename fresnel::cplx_of<T>::type* tw, int bar){
  using namespace fresnel; using C = typename cplx_of<T>::type;
  constexpr bool LAST = STAGE == fr_num_stages(N) - 1; constexpr int TL = N / 16;
  C v[16];
  fr_sync<GT>(bar);
  fft_stage_gather<T, N, false, 1>(v, buf, 0, j);
  fr_sync<GT>(bar);
  fft_stage_compute<T, N, STAGE, DIR>(v, j, tw);
  if constexpr (LAST) {
    #pragma unroll
    for (int r = 0; r < 16; ++r) buf[fr_pad(j + r * TL)] = v[r];
  } else fft_stage_scatter<T, N, STAGE, false, 1>(v, buf, 0, j);
}
template <typename T, int N, int G, int LINES>
__global__ void __launch_bounds__(G * (N / 16), 1) insm_alt(int iters, const typename fresnel::cplx_of<T>::type* tw, typename fresnel::cplx_of<T>::type* out){
  using namespace fresnel; using C = typename cplx_of<T>::type;
  constexpr int TL = N / 16, PL = fr_padded_len(N), S = fr_num_stages(N); constexpr int GT = G == 1 ? 0 : TL;
  extern __shared__ __align__(16) unsigned char smraw[];
  const int tid = threadIdx.x, grp = tid / TL, j = tid % TL;
  C* bufA = reinterpret_cast<C*>(smraw) + (size_t)grp * PL * LINES; C* bufB = bufA + PL;
  for (int r = 0; r < 16; ++r) { C z; z.x = (T)(tid + r) * (T)1e-3; z.y = (T)r; bufA[fr_pad(j + r * TL)] = z; if (LINES == 2) bufB[fr_pad(j + r * TL)] = z; }
  fr_sync<GT>(1 + grp);
  for (int it = 0; it < iters; ++it) {
    int jj = j; asm volatile("" : "+r"(jj));
    const C* t = tw; asm volatile("" : "+l"(t));
#define FR_BOTH(STAGE, DIR) { alt_block<T, N, STAGE, DIR, GT>(bufA, jj, t, 1 + grp); if (LINES == 2) alt_block<T, N, STAGE, DIR, GT>(bufB, jj, t, 1 + grp); }
    FR_BOTH(0, -1) FR_BOTH(1, -1) if constexpr (S > 2) FR_BOTH(2, -1) if constexpr (S > 3) FR_BOTH(3, -1)
    asm volatile("" : "+l"(t));
    FR_BOTH(0, +1) FR_BOTH(1, +1) if constexpr (S > 2) FR_BOTH(2, +1) if constexpr (S > 3) FR_BOTH(3, +1)
#undef FR_BOTH
  }
  fr_sync<GT>(1 + grp);
  C s = bufA[fr_pad(j)]; if (LINES == 2) s.x += bufB[fr_pad(j)].x;
  out[blockIdx.x * blockDim.x + tid] = s;
}
template <typename T, int N, int G, int LINES> void run_alt(double clock_hz){
  using C = typename fresnel::cplx_of<T>::type;
  C *tw, *out; CK(cudaMalloc(&tw, 65536 * sizeof(C))); CK(cudaMemset(tw, 0, 65536 * sizeof(C))); CK(cudaMalloc(&out, 148 * 1024 * sizeof(C)));
  const int smem = G * LINES * fresnel::fr_padded_len(N) * sizeof(C);
  CK(cudaFuncSetAttribute(insm_alt<T, N, G, LINES>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
  const int iters = 300;
  float ms = timeit([&]{ insm_alt<T, N, G, LINES><<<148, G * (N / 16), smem>>>(iters, tw, out); }, 3);
  CK(cudaGetLastError());
  printf("  in-SM lines in shared memory between stages, N=%d %s groups/SM=%d lines/group=%d: %.3f clk/element/SM\n", N, sizeof(T) == 8 ? "f64" : "f32", G, LINES,
         ms * 1e-3 * clock_hz / iters / ((double)G * LINES * N));
  cudaFree(tw); cudaFree(out);
}

// every warp interleaves NM*16 DFMA with NX (STS.128 + LDS.128) pairs per iteration, no barriers, thread-private slots
template <int NM, int NX, int WARPS>
__global__ void __launch_bounds__(WARPS * 32, 1) overlap(int iters, double* out){
  extern __shared__ double2 sm2[];
  const int tid = threadIdx.x;
  double a[16];
  #pragma unroll
  for (int i = 0; i < 16; ++i) a[i] = tid + i;
  const double b = 1.0000001, c = 0.5;
  double2 v[8];
  #pragma unroll
  for (int i = 0; i < 8; ++i) v[i] = make_double2(tid, i);
  const unsigned base = (unsigned)__cvta_generic_to_shared(sm2 + tid);
  for (int it = 0; it < iters; ++it) {
    #pragma unroll
    for (int u = 0; u < (NM > NX ? NM : NX); ++u) {
      if (u < NX) asm volatile("st.shared.v2.f64 [%0], {%1, %2};" ::"r"(base + (u & 7) * WARPS * 32 * 16), "d"(v[u & 7].x), "d"(v[u & 7].y) : "memory");
      if (u < NM) {
        #pragma unroll
        for (int i = 0; i < 16; ++i) a[i] = fma(a[i], b, c);
      }
      if (u < NX) asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v[(u + 3) & 7].x), "=d"(v[(u + 3) & 7].y) : "r"(base + ((u + 5) & 7) * WARPS * 32 * 16) : "memory");
    }
  }
  double s = 0;
  #pragma unroll
  for (int i = 0; i < 16; ++i) s += a[i];
  #pragma unroll
  for (int i = 0; i < 8; ++i) s += v[i].x + v[i].y;
  out[blockIdx.x * WARPS * 32 + tid] = s;
}
template <int NM, int NX, int WARPS> void run_overlap(double clock_hz){
  double* out; CK(cudaMalloc(&out, 148 * 1024 * 8));
  const int smem = WARPS * 32 * 8 * 16;
  CK(cudaFuncSetAttribute(overlap<NM, NX, WARPS>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
  const int iters = 4000;
  float ms = timeit([&]{ overlap<NM, NX, WARPS><<<148, WARPS * 32, smem>>>(iters, out); }, 3);
  CK(cudaGetLastError());
  printf("  overlap warps/SM=%2d dfma=%3d lds+sts=%2d per warp-iteration: %7.1f clk   (fp64 pipe alone %4.0f, shared-memory pipe alone %4.0f)\n",
         WARPS, NM * 16, NX * 2, ms * 1e-3 * clock_hz / iters, WARPS * NM * 16 * 2.0 / 4, WARPS * NX * 2 * 4.0);
  cudaFree(out);
}

int main(){
  cudaDeviceProp p; CK(cudaGetDeviceProperties(&p,0)); printf("%s SMs=%d L2=%d MB clock=%d MHz\n",p.name,p.multiProcessorCount,p.l2CacheSize>>20,p.clockRate/1000);
  size_t n=(size_t)1<<30; // 1 GiB
  int4 *a,*b; CK(cudaMalloc(&a,n)); CK(cudaMalloc(&b,n)); CK(cudaMemset(a,1,n)); CK(cudaMemset(b,0,n));
  { float ms=timeit([&]{ copy16<<<148*16,512>>>(a,b,n/16); }); printf("copy 1GiB kernel: %.3f ms %.0f GB/s\n",ms,2.0*n/ms/1e6); }
  { float ms=timeit([&]{ cudaMemcpyAsync(b,a,n,cudaMemcpyDeviceToDevice); }); printf("copy 1GiB memcpy: %.3f ms %.0f GB/s\n",ms,2.0*n/ms/1e6); }
  for(int N: {2048,4096,8192}){
    printf("N=%d (16B elements, %.0f MiB)\n",N,(double)N*N*16/1048576);
    run_row<1>(a,N); run_row<2>(a,N); run_row<4>(a,N);
    run_col<1>(a,N); run_col<2>(a,N); run_col<4>(a,N); run_col<8>(a,N);
  }
  // L2-resident read
  { size_t m=(size_t)32<<20; int* out; CK(cudaMalloc(&out,4)); int iters=20;
    float ms=timeit([&]{ l2read<<<148*8,512>>>(a,m/16,iters,out); },5); printf("L2 read 32MiB x%d: %.3f ms %.0f GB/s\n",iters,ms,(double)m*iters/ms/1e6); 
    m=(size_t)64<<20; ms=timeit([&]{ l2read<<<148*8,512>>>(a,m/16,iters,out); },5); printf("L2 read 64MiB x%d: %.3f ms %.0f GB/s\n",iters,ms,(double)m*iters/ms/1e6); }
  { double* o; CK(cudaMalloc(&o,148*8*256*8)); int iters=2000; float ms=timeit([&]{ fmapeak<double><<<148*8,256>>>(o,iters); },5);
    double fl=2.0*148*8*256*(double)iters*16*8; printf("DFMA peak: %.3f ms %.2f TFLOP/s\n",ms,fl/ms/1e9); }
  { float* o; CK(cudaMalloc(&o,148*8*256*4)); int iters=4000; float ms=timeit([&]{ fmapeak<float><<<148*8,256>>>(o,iters); },5);
    double fl=2.0*148*8*256*(double)iters*16*8; printf("FFMA peak: %.3f ms %.2f TFLOP/s\n",ms,fl/ms/1e9); }
  // in-SM rates (cycles at the nominal clock printed above)
  { const double hz = p.clockRate * 1e3;
    printf("in-SM (registers + shared memory only; HBM needs %.2f clk/element/SM for complex128, %.2f for complex64 at 6.55 TB/s)\n",
           32.0 / (6.55e12 / 148 / hz), 16.0 / (6.55e12 / 148 / hz));
    run_insm<double, 2048, 1, 1>("butterflies", hz); run_insm<double, 2048, 4, 1>("butterflies", hz);
    run_insm<double, 2048, 1, 2>("exchanges", hz);   run_insm<double, 2048, 4, 2>("exchanges", hz);
    run_insm<double, 2048, 1, 0>("transform pair", hz); run_insm<double, 2048, 2, 0>("transform pair", hz);
    run_insm<double, 2048, 3, 0>("transform pair", hz); run_insm<double, 2048, 4, 0>("transform pair", hz);
    run_insm<double, 2048, 4, 0, 32>("pair, warp-local sync", hz);
    run_insm<double, 4096, 2, 1>("butterflies", hz); run_insm<double, 4096, 2, 2>("exchanges", hz); run_insm<double, 4096, 2, 0>("transform pair", hz);
    run_insm<double, 4096, 2, 0, 32>("pair, warp-local sync", hz);
    run_insm<float, 2048, 4, 1>("butterflies", hz); run_insm<float, 2048, 4, 2>("exchanges", hz);
    run_insm<float, 2048, 4, 0>("transform pair", hz); run_insm<float, 2048, 8, 0>("transform pair", hz);
    run_insm<float, 2048, 8, 0, 32>("pair, warp-local sync", hz);
    run_insm<float, 4096, 4, 1>("butterflies", hz); run_insm<float, 4096, 4, 2>("exchanges", hz); run_insm<float, 4096, 4, 0>("transform pair", hz);
    run_insm<double, 8192, 1, 0>("transform pair", hz); run_insm<float, 8192, 2, 0>("transform pair", hz);
    run_alt<double, 2048, 4, 1>(hz); run_alt<double, 2048, 3, 2>(hz); run_alt<double, 2048, 2, 2>(hz);
    run_alt<double, 4096, 2, 1>(hz); run_alt<double, 4096, 1, 2>(hz);
    run_alt<float, 2048, 8, 1>(hz); run_alt<float, 2048, 4, 2>(hz); run_alt<float, 4096, 4, 1>(hz); run_alt<float, 4096, 2, 2>(hz);
    run_overlap<8, 0, 16>(hz); run_overlap<0, 8, 16>(hz); run_overlap<8, 8, 16>(hz); run_overlap<8, 8, 4>(hz);
  }
  return 0;
}
