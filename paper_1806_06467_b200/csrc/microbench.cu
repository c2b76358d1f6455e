// microbench.cu -- stand-alone measurements behind DESIGN.md's design decisions (not part of libfresnel.so):
//   HBM copy bandwidth, row-tile vs column-tile (strided 16/32/64/128-byte segment) in-place copies with
//   per-thread loads, L2-resident read bandwidth, and the plain-ALU roofs (DFMA / FFMA) that
//   MEASURED_PEAKS.json does not carry.   Build + run:
//     python -m paper_1806_06467_b200.build --microbench && ./paper_1806_06467_b200/microbench
#include <cstdio>
#include <cstdlib>
#include <cuda_runtime.h>
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
  return 0;
}
