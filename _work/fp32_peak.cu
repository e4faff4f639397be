// fp32_peak.cu -- FFMA-chain microbenchmark: the measured FP32 CUDA-core peak quoted beside the derived
// roofline denominator of bench.py.  Not part of libshwfs.so.
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o fp32_peak fp32_peak.cu && ./fp32_peak
#include <cstdio>
#include <cuda_runtime.h>
__global__ void k(float *o, int iters){
  float a[16]; 
  #pragma unroll
  for(int i=0;i<16;i++) a[i]=threadIdx.x*0.001f+i;
  float b=1.0001f,c=0.5f;
  for(int it=0;it<iters;it++){
    #pragma unroll
    for(int i=0;i<16;i++) a[i]=fmaf(a[i],b,c);
  }
  float s=0; 
  #pragma unroll
  for(int i=0;i<16;i++) s+=a[i];
  o[blockIdx.x*blockDim.x+threadIdx.x]=s;
}
int main(){
  cudaDeviceProp p; cudaGetDeviceProperties(&p,0);
  printf("%s SMs=%d clock=%d kHz\n",p.name,p.multiProcessorCount,p.clockRate);
  float *o; cudaMalloc(&o,148*8*1024*4*4);
  int iters=20000;
  for(int bps=1;bps<=2;bps++) for(int th=256;th<=1024;th*=2){
    cudaEvent_t e0,e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    k<<<p.multiProcessorCount*bps,th>>>(o,iters); cudaDeviceSynchronize();
    float best=1e9;
    for(int r=0;r<5;r++){ cudaEventRecord(e0); k<<<p.multiProcessorCount*bps,th>>>(o,iters); cudaEventRecord(e1); cudaEventSynchronize(e1); float ms; cudaEventElapsedTime(&ms,e0,e1); if(ms<best)best=ms;}
    double fl=2.0*16*iters*(double)th*p.multiProcessorCount*bps;
    printf("blocks/SM=%d threads=%d: %.3f ms  %.2f TFLOP/s\n",bps,th,best,fl/best/1e9);
  }
  // sustained 3 s
  { cudaEvent_t e0,e1; cudaEventCreate(&e0); cudaEventCreate(&e1); cudaEventRecord(e0); int reps=0; 
    for(int r=0;r<300;r++){k<<<p.multiProcessorCount*2,512>>>(o,iters);reps++;} cudaEventRecord(e1); cudaEventSynchronize(e1); float ms; cudaEventElapsedTime(&ms,e0,e1);
    double fl=2.0*16*iters*512.0*p.multiProcessorCount*2*reps; printf("sustained %d launches %.1f ms: %.2f TFLOP/s\n",reps,ms,fl/ms/1e9);}
  return 0;
}
