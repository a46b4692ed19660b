#include <cstdio>
#include <cuda_runtime.h>
// FP64 peak probe: DFMA vs DMMA shapes on sm_100a
__global__ void k_dfma(double* out, int iters){
  double a0=1.0+threadIdx.x*1e-9,a1=a0+1,a2=a0+2,a3=a0+3,a4=a0+4,a5=a0+5,a6=a0+6,a7=a0+7;
  double b=1.0000001,c=1e-9;
  for(int i=0;i<iters;i++){
    a0=fma(a0,b,c);a1=fma(a1,b,c);a2=fma(a2,b,c);a3=fma(a3,b,c);
    a4=fma(a4,b,c);a5=fma(a5,b,c);a6=fma(a6,b,c);a7=fma(a7,b,c);
  }
  out[blockIdx.x*blockDim.x+threadIdx.x]=a0+a1+a2+a3+a4+a5+a6+a7;
}
__global__ void k_m8n8k4(double* out,int iters){
  double a=1.0+threadIdx.x*1e-9,b=1.0000001;
  double c[8][2];
  for(int j=0;j<8;j++){c[j][0]=j;c[j][1]=j+0.5;}
  for(int i=0;i<iters;i++){
    #pragma unroll
    for(int j=0;j<8;j++)
      asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1},{%2},{%3},{%0,%1};":"+d"(c[j][0]),"+d"(c[j][1]):"d"(a),"d"(b));
  }
  double s=0;for(int j=0;j<8;j++)s+=c[j][0]+c[j][1];
  out[blockIdx.x*blockDim.x+threadIdx.x]=s;
}
__global__ void k_m16n8k4(double* out,int iters){
  double a0=1.0+threadIdx.x*1e-9,a1=a0*1.1,b=1.0000001;
  double c[4][4];
  for(int j=0;j<4;j++)for(int q=0;q<4;q++)c[j][q]=j+q;
  for(int i=0;i<iters;i++){
    #pragma unroll
    for(int j=0;j<4;j++)
      asm volatile("mma.sync.aligned.m16n8k4.row.col.f64.f64.f64.f64 {%0,%1,%2,%3},{%4,%5},{%6},{%0,%1,%2,%3};":"+d"(c[j][0]),"+d"(c[j][1]),"+d"(c[j][2]),"+d"(c[j][3]):"d"(a0),"d"(a1),"d"(b));
  }
  double s=0;for(int j=0;j<4;j++)for(int q=0;q<4;q++)s+=c[j][q];
  out[blockIdx.x*blockDim.x+threadIdx.x]=s;
}
__global__ void k_m16n8k8(double* out,int iters){
  double a0=1.0+threadIdx.x*1e-9,a1=a0*1.1,a2=a0*1.2,a3=a0*1.3,b0=1.0000001,b1=1.0000002;
  double c[4][4];
  for(int j=0;j<4;j++)for(int q=0;q<4;q++)c[j][q]=j+q;
  for(int i=0;i<iters;i++){
    #pragma unroll
    for(int j=0;j<4;j++)
      asm volatile("mma.sync.aligned.m16n8k8.row.col.f64.f64.f64.f64 {%0,%1,%2,%3},{%4,%5,%6,%7},{%8,%9},{%0,%1,%2,%3};":"+d"(c[j][0]),"+d"(c[j][1]),"+d"(c[j][2]),"+d"(c[j][3]):"d"(a0),"d"(a1),"d"(a2),"d"(a3),"d"(b0),"d"(b1));
  }
  double s=0;for(int j=0;j<4;j++)for(int q=0;q<4;q++)s+=c[j][q];
  out[blockIdx.x*blockDim.x+threadIdx.x]=s;
}
__global__ void k_m16n8k16(double* out,int iters){
  double a[8],b[4];
  for(int q=0;q<8;q++)a[q]=1.0+threadIdx.x*1e-9*q; for(int q=0;q<4;q++)b[q]=1.0000001+q*1e-9;
  double c[4][4];
  for(int j=0;j<4;j++)for(int q=0;q<4;q++)c[j][q]=j+q;
  for(int i=0;i<iters;i++){
    #pragma unroll
    for(int j=0;j<4;j++)
      asm volatile("mma.sync.aligned.m16n8k16.row.col.f64.f64.f64.f64 {%0,%1,%2,%3},{%4,%5,%6,%7,%8,%9,%10,%11},{%12,%13,%14,%15},{%0,%1,%2,%3};":"+d"(c[j][0]),"+d"(c[j][1]),"+d"(c[j][2]),"+d"(c[j][3]):"d"(a[0]),"d"(a[1]),"d"(a[2]),"d"(a[3]),"d"(a[4]),"d"(a[5]),"d"(a[6]),"d"(a[7]),"d"(b[0]),"d"(b[1]),"d"(b[2]),"d"(b[3]));
  }
  double s=0;for(int j=0;j<4;j++)for(int q=0;q<4;q++)s+=c[j][q];
  out[blockIdx.x*blockDim.x+threadIdx.x]=s;
}
template<class F> void run(const char* name,F f,double flop_per_thread_iter,int threads,int blocks){
  double* out; cudaMalloc(&out,sizeof(double)*threads*blocks);
  int iters=20000;
  f<<<blocks,threads>>>(out,100); cudaDeviceSynchronize();
  cudaEvent_t e0,e1; cudaEventCreate(&e0);cudaEventCreate(&e1);
  float best=1e30;
  for(int r=0;r<3;r++){cudaEventRecord(e0); f<<<blocks,threads>>>(out,iters); cudaEventRecord(e1); cudaEventSynchronize(e1); float ms; cudaEventElapsedTime(&ms,e0,e1); if(ms<best)best=ms;}
  double fl=flop_per_thread_iter*(double)iters*threads*blocks;
  printf("%-12s threads=%4d blocks=%5d  %8.3f ms  %8.2f TFLOP/s  err=%s\n",name,threads,blocks,best,fl/best*1e-9,cudaGetErrorString(cudaGetLastError()));
  cudaFree(out);
}
int main(){
  cudaDeviceProp p; cudaGetDeviceProperties(&p,0); printf("%s SMs=%d clock=%d kHz\n",p.name,p.multiProcessorCount,p.clockRate);
  for(int th: {128,256,512,1024}){
    int blocks=148*(2048/th);
    run("dfma",k_dfma,16.0,th,blocks);
    run("m8n8k4",k_m8n8k4,8.0*2*8*8*4/32,th,blocks);
    run("m16n8k4",k_m16n8k4,4.0*2*16*8*4/32,th,blocks);
    run("m16n8k8",k_m16n8k8,4.0*2*16*8*8/32,th,blocks);
    run("m16n8k16",k_m16n8k16,4.0*2*16*8*16/32,th,blocks);
  }
  return 0;
}
