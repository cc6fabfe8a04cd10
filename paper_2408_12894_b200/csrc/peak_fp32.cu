// FP32-pipe peak of the device the blend kernel's roofline is quoted against: a standalone microbenchmark,
// not part of libflod.so.
//     nvcc -O3 -gencode arch=compute_100a,code=sm_100a -o peak_fp32 paper_2408_12894_b200/csrc/peak_fp32.cu && ./peak_fp32
// Eight independent chains per thread, 8 CTAs of 256 threads per SM, 148 SMs.  Measured on the B200 of this pool (1965 MHz):
//     FFMA 71.9 TFLOP/s, FFMA2 68.5 TFLOP/s (packed instructions halve the issue slots, not the pipe time),
//     8 FFMA + 1 MUFU.EX2 53.8 TFLOP/s, MUFU.EX2 alone 4.63 T/s, FFMA + FMNMX pairs 37.5 T instructions/s (issue bound).
#include <cuda_runtime.h>
#include <stdio.h>
template<int MODE> __global__ void __launch_bounds__(256) k(float* out, int iters, float s){
  float a[8]; float2 b[8];
  for(int i=0;i<8;i++){ a[i]=threadIdx.x*0.001f+i; b[i]=make_float2(a[i],a[i]+1.f);}
  float2 m=make_float2(s,s), c=make_float2(0.5f,0.25f);
  for(int it=0;it<iters;it++){
    if(MODE==0){
#pragma unroll
      for(int i=0;i<8;i++) a[i]=fmaf(a[i],s,0.5f);
    } else if (MODE==1){
#pragma unroll
      for(int i=0;i<8;i++) b[i]=__ffma2_rn(b[i],m,c);
    } else if (MODE==2){
#pragma unroll
      for(int i=0;i<8;i++) a[i]=fmaf(a[i],s,c.y);
    } else if (MODE==3){
#pragma unroll
      for(int i=0;i<8;i++) a[i]=fmaf(a[i],s,c.x);
      float y; asm volatile("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(a[0])); a[0]=y;
    } else if (MODE==4){
#pragma unroll
      for(int i=0;i<8;i++){ float y; asm volatile("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(a[i])); a[i]=y; }
    } else if (MODE==5){   // fmnmx on the alu pipe alongside ffma
#pragma unroll
      for(int i=0;i<8;i++){ a[i]=fmaf(a[i],s,c.x); b[i].x=fminf(b[i].x,a[i]); }
    }
  }
  float r=0; for(int i=0;i<8;i++) r+=a[i]+b[i].x+b[i].y;
  out[blockIdx.x*blockDim.x+threadIdx.x]=r;
}
template<int MODE> void run(const char* name, double ops_per_iter_thread){
  float* out; cudaMalloc(&out, 148*8*256*4);
  int iters=20000; cudaEvent_t e0,e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
  k<MODE><<<148*8,256>>>(out,100,0.999f);
  cudaEventRecord(e0); k<MODE><<<148*8,256>>>(out,iters,0.999f); cudaEventRecord(e1); cudaEventSynchronize(e1);
  float ms; cudaEventElapsedTime(&ms,e0,e1);
  double tot=ops_per_iter_thread*iters*148.0*8*256;
  printf("%s: %.3f ms  %.2f T/s\n", name, ms, tot/(ms*1e-3)/1e12);
  cudaFree(out);
}
int main(){ run<0>("FFMA reg,reg,imm (flops)",16); run<1>("FFMA2 (flops)",32); run<2>("FFMA 3reg (flops)",16); run<3>("8 FFMA+1 ex2 (flops)",16); run<4>("ex2 (ops)",8); run<5>("8 FFMA + 8 FMNMX (instr)",16); return 0; }
