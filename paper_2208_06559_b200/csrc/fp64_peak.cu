// FP64 issue-rate microbenchmark: DFMA vs DMMA (m8n8k4, m16n8k4, m16n8k8, m16n8k16)
#include <cstdio>
#include <cuda_runtime.h>
#define CK(x) do{cudaError_t e=(x); if(e!=cudaSuccess){printf("ERR %s line %d\n",cudaGetErrorString(e),__LINE__);return 1;}}while(0)

template<int ILP>
__global__ void k_dfma(double* out, int iters, double a, double b){
  double acc[ILP];
  #pragma unroll
  for(int i=0;i<ILP;i++) acc[i]=threadIdx.x*1e-3+i;
  for(int it=0;it<iters;it++){
    #pragma unroll
    for(int i=0;i<ILP;i++) acc[i]=fma(acc[i],a,b);
  }
  double s=0;
  #pragma unroll
  for(int i=0;i<ILP;i++) s+=acc[i];
  out[blockIdx.x*blockDim.x+threadIdx.x]=s;
}

template<int ILP>
__global__ void k_dmma884(double* out, int iters, double a, double b){
  double c[ILP][2];
  #pragma unroll
  for(int i=0;i<ILP;i++){c[i][0]=threadIdx.x;c[i][1]=i;}
  for(int it=0;it<iters;it++){
    #pragma unroll
    for(int i=0;i<ILP;i++)
      asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
        : "+d"(c[i][0]), "+d"(c[i][1]) : "d"(a), "d"(b));
  }
  double s=0;
  #pragma unroll
  for(int i=0;i<ILP;i++) s+=c[i][0]+c[i][1];
  out[blockIdx.x*blockDim.x+threadIdx.x]=s;
}
#ifdef BIGSHAPES
template<int ILP>
__global__ void k_dmma1684(double* out, int iters, double a, double b){
  double c[ILP][4];
  #pragma unroll
  for(int i=0;i<ILP;i++){c[i][0]=threadIdx.x;c[i][1]=i;c[i][2]=1;c[i][3]=2;}
  for(int it=0;it<iters;it++){
    #pragma unroll
    for(int i=0;i<ILP;i++)
      asm volatile("mma.sync.aligned.m16n8k4.row.col.f64.f64.f64.f64 {%0,%1,%2,%3}, {%4,%5}, {%6}, {%0,%1,%2,%3};"
        : "+d"(c[i][0]), "+d"(c[i][1]), "+d"(c[i][2]), "+d"(c[i][3]) : "d"(a), "d"(b), "d"(b));
  }
  double s=0;
  #pragma unroll
  for(int i=0;i<ILP;i++) s+=c[i][0]+c[i][1]+c[i][2]+c[i][3];
  out[blockIdx.x*blockDim.x+threadIdx.x]=s;
}
template<int ILP>
__global__ void k_dmma1688(double* out, int iters, double a, double b){
  double c[ILP][4];
  #pragma unroll
  for(int i=0;i<ILP;i++){c[i][0]=threadIdx.x;c[i][1]=i;c[i][2]=1;c[i][3]=2;}
  for(int it=0;it<iters;it++){
    #pragma unroll
    for(int i=0;i<ILP;i++)
      asm volatile("mma.sync.aligned.m16n8k8.row.col.f64.f64.f64.f64 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
        : "+d"(c[i][0]), "+d"(c[i][1]), "+d"(c[i][2]), "+d"(c[i][3]) : "d"(a), "d"(b), "d"(a), "d"(b), "d"(b), "d"(a));
  }
  double s=0;
  #pragma unroll
  for(int i=0;i<ILP;i++) s+=c[i][0]+c[i][1]+c[i][2]+c[i][3];
  out[blockIdx.x*blockDim.x+threadIdx.x]=s;
}
template<int ILP>
__global__ void k_dmma16816(double* out, int iters, double a, double b){
  double c[ILP][4];
  #pragma unroll
  for(int i=0;i<ILP;i++){c[i][0]=threadIdx.x;c[i][1]=i;c[i][2]=1;c[i][3]=2;}
  for(int it=0;it<iters;it++){
    #pragma unroll
    for(int i=0;i<ILP;i++)
      asm volatile("mma.sync.aligned.m16n8k16.row.col.f64.f64.f64.f64 {%0,%1,%2,%3}, {%4,%5,%6,%7,%8,%9,%10,%11}, {%12,%13,%14,%15}, {%0,%1,%2,%3};"
        : "+d"(c[i][0]), "+d"(c[i][1]), "+d"(c[i][2]), "+d"(c[i][3]) : "d"(a), "d"(b), "d"(a), "d"(b), "d"(a), "d"(b), "d"(a), "d"(b), "d"(b), "d"(a), "d"(b), "d"(a));
  }
  double s=0;
  #pragma unroll
  for(int i=0;i<ILP;i++) s+=c[i][0]+c[i][1]+c[i][2]+c[i][3];
  out[blockIdx.x*blockDim.x+threadIdx.x]=s;
}
#endif

template<typename F> float timeit(F f){
  cudaEvent_t e0,e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
  f(); cudaDeviceSynchronize();
  float best=1e30f;
  for(int r=0;r<5;r++){ cudaEventRecord(e0); f(); cudaEventRecord(e1); cudaEventSynchronize(e1); float ms; cudaEventElapsedTime(&ms,e0,e1); if(ms<best)best=ms;}
  return best;
}
int main(){
  cudaDeviceProp p; CK(cudaGetDeviceProperties(&p,0));
  printf("dev %s SMs %d clock %d kHz\n",p.name,p.multiProcessorCount,p.clockRate);
  double* out; CK(cudaMalloc(&out,148*8*1024*8));
  int iters=20000;
  for(int wps=4; wps<=32; wps*=2){ // warps per SM
    int threads = wps*32 > 1024 ? 1024 : wps*32; int blocks=148*(wps*32/threads);
    float ms;
    ms=timeit([&]{k_dfma<8><<<blocks,threads>>>(out,iters,1.0000001,1e-9);});
    printf("DFMA ilp8  wps=%2d: %.3f ms  %.2f TFLOP/s\n",wps,ms, 2.0*8*iters*(double)blocks*threads/ms/1e9);
    ms=timeit([&]{k_dmma884<8><<<blocks,threads>>>(out,iters,1.0000001,1e-9);});
    printf("DMMA m8n8k4 ilp8 wps=%2d: %.3f ms  %.2f TFLOP/s\n",wps,ms, 512.0*8*iters*(double)blocks*threads/32/ms/1e9);
#ifdef BIGSHAPES
    ms=timeit([&]{k_dmma1684<4><<<blocks,threads>>>(out,iters,1.0000001,1e-9);});
    printf("DMMA m16n8k4 ilp4 wps=%2d: %.3f ms  %.2f TFLOP/s\n",wps,ms, 1024.0*4*iters*(double)blocks*threads/32/ms/1e9);
    ms=timeit([&]{k_dmma1688<4><<<blocks,threads>>>(out,iters,1.0000001,1e-9);});
    printf("DMMA m16n8k8 ilp4 wps=%2d: %.3f ms  %.2f TFLOP/s\n",wps,ms, 2048.0*4*iters*(double)blocks*threads/32/ms/1e9);
    ms=timeit([&]{k_dmma16816<4><<<blocks,threads>>>(out,iters,1.0000001,1e-9);});
    printf("DMMA m16n8k16 ilp4 wps=%2d: %.3f ms  %.2f TFLOP/s\n",wps,ms, 4096.0*4*iters*(double)blocks*threads/32/ms/1e9);
#endif
  }
  // latency: single warp dependent chain
  {
    float ms=timeit([&]{k_dfma<1><<<1,32>>>(out,iters*10,1.0000001,1e-9);});
    printf("DFMA dependent chain: %.2f ns per op\n", ms*1e6/(iters*10));
    ms=timeit([&]{k_dmma884<1><<<1,32>>>(out,iters*10,1.0000001,1e-9);});
    printf("DMMA884 dependent chain: %.2f ns per op\n", ms*1e6/(iters*10));
  }
  return 0;
}
