// peak_probe_fp64.cu -- standalone microbenchmark: FP64 tensor-core (mma.sync f64 "DMMA") and FP64/FP32 FMA peaks
// with register-resident operands.  Its DMMA figure is the roofline denominator of the FP64 contraction kernel
// (bench.py FP64_DMMA_PEAK_TFLOPS; output kept in profiles/r01_fp64_peak_probe.txt).  Not part of the library.
//   nvcc -O3 -DHAVE_BIG -gencode arch=compute_100a,code=sm_100a -o peak_probe_fp64 paper_1609_08094_b200/csrc/peak_probe_fp64.cu
//   ./peak_probe_fp64
#include <cstdio>
#include <cuda_runtime.h>
#define CK(x) do{cudaError_t e=(x); if(e!=cudaSuccess){printf("ERR %s line %d\n", cudaGetErrorString(e), __LINE__); return 1;}}while(0)

__device__ __forceinline__ void dmma884(double &c0,double &c1,double a,double b){
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n":"+d"(c0),"+d"(c1):"d"(a),"d"(b));
}
#ifdef HAVE_BIG
__device__ __forceinline__ void dmma16816(double *c,const double *a,const double *b){
  asm volatile("mma.sync.aligned.m16n8k16.row.col.f64.f64.f64.f64 {%0,%1,%2,%3}, {%4,%5,%6,%7,%8,%9,%10,%11}, {%12,%13,%14,%15}, {%0,%1,%2,%3};\n"
   :"+d"(c[0]),"+d"(c[1]),"+d"(c[2]),"+d"(c[3])
   :"d"(a[0]),"d"(a[1]),"d"(a[2]),"d"(a[3]),"d"(a[4]),"d"(a[5]),"d"(a[6]),"d"(a[7]),"d"(b[0]),"d"(b[1]),"d"(b[2]),"d"(b[3]));
}
__device__ __forceinline__ void dmma1684(double *c,const double *a,const double *b){
  asm volatile("mma.sync.aligned.m16n8k4.row.col.f64.f64.f64.f64 {%0,%1,%2,%3}, {%4,%5}, {%6}, {%0,%1,%2,%3};\n"
   :"+d"(c[0]),"+d"(c[1]),"+d"(c[2]),"+d"(c[3])
   :"d"(a[0]),"d"(a[1]),"d"(b[0]));
}
#endif

template<int NACC>
__global__ void k_dmma884(double *out, int iters){
  double c[NACC][2];
  for(int i=0;i<NACC;i++){c[i][0]=threadIdx.x*1e-9;c[i][1]=i*1e-9;}
  double a=1.0+threadIdx.x*1e-6, b=1.0-threadIdx.x*1e-6;
  for(int it=0;it<iters;it++){
    #pragma unroll
    for(int i=0;i<NACC;i++) dmma884(c[i][0],c[i][1],a,b);
  }
  double s=0; for(int i=0;i<NACC;i++) s+=c[i][0]+c[i][1];
  out[blockIdx.x*blockDim.x+threadIdx.x]=s;
}
#ifdef HAVE_BIG
template<int NACC>
__global__ void k_dmma16816(double *out, int iters){
  double c[NACC][4]; double a[8],b[4];
  for(int i=0;i<NACC;i++) for(int j=0;j<4;j++) c[i][j]=threadIdx.x*1e-9+j;
  for(int j=0;j<8;j++) a[j]=1.0+threadIdx.x*1e-6*j;
  for(int j=0;j<4;j++) b[j]=1.0-threadIdx.x*1e-6*j;
  for(int it=0;it<iters;it++){
    #pragma unroll
    for(int i=0;i<NACC;i++) dmma16816(c[i],a,b);
  }
  double s=0; for(int i=0;i<NACC;i++) for(int j=0;j<4;j++) s+=c[i][j];
  out[blockIdx.x*blockDim.x+threadIdx.x]=s;
}
template<int NACC>
__global__ void k_dmma1684(double *out, int iters){
  double c[NACC][4]; double a[2],b[1];
  for(int i=0;i<NACC;i++) for(int j=0;j<4;j++) c[i][j]=threadIdx.x*1e-9+j;
  for(int j=0;j<2;j++) a[j]=1.0+threadIdx.x*1e-6*j;
  b[0]=1.0-threadIdx.x*1e-6;
  for(int it=0;it<iters;it++){
    #pragma unroll
    for(int i=0;i<NACC;i++) dmma1684(c[i],a,b);
  }
  double s=0; for(int i=0;i<NACC;i++) for(int j=0;j<4;j++) s+=c[i][j];
  out[blockIdx.x*blockDim.x+threadIdx.x]=s;
}
#endif
template<int NACC>
__global__ void k_dfma(double *out, int iters){
  double c[NACC];
  for(int i=0;i<NACC;i++) c[i]=threadIdx.x*1e-9+i;
  double a=1.0+threadIdx.x*1e-9, b=1e-9*threadIdx.x;
  for(int it=0;it<iters;it++){
    #pragma unroll
    for(int i=0;i<NACC;i++) c[i]=fma(c[i],a,b);
  }
  double s=0; for(int i=0;i<NACC;i++) s+=c[i];
  out[blockIdx.x*blockDim.x+threadIdx.x]=s;
}
template<int NACC>
__global__ void k_ffma(float *out, int iters){
  float c[NACC];
  for(int i=0;i<NACC;i++) c[i]=threadIdx.x*1e-9f+i;
  float a=1.0f+threadIdx.x*1e-9f, b=1e-9f*threadIdx.x;
  for(int it=0;it<iters;it++){
    #pragma unroll
    for(int i=0;i<NACC;i++) c[i]=fmaf(c[i],a,b);
  }
  float s=0; for(int i=0;i<NACC;i++) s+=c[i];
  out[blockIdx.x*blockDim.x+threadIdx.x]=s;
}

int main(){
  cudaDeviceProp p; CK(cudaGetDeviceProperties(&p,0));
  printf("dev %s sm=%d cc=%d.%d clk=%d kHz\n",p.name,p.multiProcessorCount,p.major,p.minor,p.clockRate);
  double *out; CK(cudaMalloc(&out, 148*8*1024*8));
  cudaEvent_t e0,e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
  int nsm=p.multiProcessorCount;
  #define RUN(name, kern, grid, block, iters, flop_per_thread_iter) \
    for(int rep=0;rep<3;rep++){ kern<<<grid,block>>>((decltype(out))out, iters); CK(cudaGetLastError()); CK(cudaDeviceSynchronize()); \
    cudaEventRecord(e0); kern<<<grid,block>>>(out, iters); cudaEventRecord(e1); CK(cudaDeviceSynchronize()); float ms; cudaEventElapsedTime(&ms,e0,e1); \
    double fl=(double)(grid)*(block)*(double)(iters)*(flop_per_thread_iter); if(rep==2) printf("%-28s grid=%d block=%d  %.3f ms  %.2f TFLOP/s\n", name, grid, block, ms, fl/ms*1e-9);}
  // m8n8k4: per warp 8*8*4*2=512 flop -> per thread 16 flop per mma
  for(int wpb: {1,2,4,8}){
    RUN("dmma884 acc8", k_dmma884<8>, nsm, wpb*32, 20000, 16.0*8);
    RUN("dmma884 acc16", k_dmma884<16>, nsm, wpb*32, 20000, 16.0*16);
    RUN("dmma884 acc32", k_dmma884<32>, nsm, wpb*32, 20000, 16.0*32);
  }
  RUN("dmma884 acc32 2cta", k_dmma884<32>, nsm*2, 256, 20000, 16.0*32);
#ifdef HAVE_BIG
  for(int wpb: {4,8}){
    RUN("dmma16816 acc8", k_dmma16816<8>, nsm, wpb*32, 10000, (16.0*8*16*2/32)*8);
    RUN("dmma1684 acc16", k_dmma1684<16>, nsm, wpb*32, 20000, (16.0*8*4*2/32)*16);
  }
#endif
  for(int wpb: {8,16,32}){
    RUN("dfma acc16", k_dfma<16>, nsm, wpb*32, 20000, 2.0*16);
  }
  RUN("dfma acc16 2cta", k_dfma<16>, nsm*2, 512, 20000, 2.0*16);
  float* fo=(float*)out;
  #undef RUN
  #define RUNF(name, kern, grid, block, iters, flop_per_thread_iter) \
    for(int rep=0;rep<3;rep++){ kern<<<grid,block>>>(fo, iters); CK(cudaGetLastError()); CK(cudaDeviceSynchronize()); \
    cudaEventRecord(e0); kern<<<grid,block>>>(fo, iters); cudaEventRecord(e1); CK(cudaDeviceSynchronize()); float ms; cudaEventElapsedTime(&ms,e0,e1); \
    double fl=(double)(grid)*(block)*(double)(iters)*(flop_per_thread_iter); if(rep==2) printf("%-28s grid=%d block=%d  %.3f ms  %.2f TFLOP/s\n", name, grid, block, ms, fl/ms*1e-9);}
  RUNF("ffma acc16", k_ffma<16>, nsm*2, 512, 20000, 2.0*16);
  return 0;
}
