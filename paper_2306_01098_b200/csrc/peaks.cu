// peaks.cu -- stand-alone microbenchmark of this GPU's ceilings used as roofline context: read-only and copy
// HBM bandwidth with 128-bit loads, fp32 / fp64 FMA peaks.  Built and run by `python -m paper_2306_01098_b200.peaks`.
#include <cstdio>
#include <cuda_runtime.h>
__global__ void rd(const double2* __restrict__ p, size_t n, double* out, int reps=1){
  size_t i0 = (size_t)blockIdx.x*blockDim.x+threadIdx.x; size_t st=(size_t)gridDim.x*blockDim.x;
  double s=0; size_t i=i0;
  for(int r=0;r<reps;r++) { i=i0;
  for(; i+3*st<n; i+=4*st){ double2 a=__ldcs(p+i), b=__ldcs(p+i+st), c=__ldcs(p+i+2*st), d=__ldcs(p+i+3*st); s+=a.x+a.y+b.x+b.y+c.x+c.y+d.x+d.y; }
  for(; i<n; i+=st){ double2 a=__ldcs(p+i); s+=a.x+a.y; }
  }
  if(s==1.2345) *out=s;
}
// L2-resident read: n is a power of two (elements of 16 B); every thread streams `iters` 4-load groups, wrapping
// with a mask, so the whole buffer is re-read many times from L2 inside one launch.
__global__ void rd_l2(const double2* __restrict__ p, unsigned mask, int iters, double* out){
  unsigned st=gridDim.x*blockDim.x; unsigned i=blockIdx.x*blockDim.x+threadIdx.x; double s=0;
  for(int k=0;k<iters;k++){
    double2 a=__ldcg(p+(i&mask)), b=__ldcg(p+((i+st)&mask)), c=__ldcg(p+((i+2*st)&mask)), d=__ldcg(p+((i+3*st)&mask));
    s+=a.x+a.y+b.x+b.y+c.x+c.y+d.x+d.y; i+=4*st;
  }
  if(s==1.2345) *out=s;
}
__global__ void cp(const double2* __restrict__ p, double2* __restrict__ q, size_t n){
  size_t i = (size_t)blockIdx.x*blockDim.x+threadIdx.x; size_t st=(size_t)gridDim.x*blockDim.x;
  for(; i<n; i+=st) q[i]=p[i];
}
template<typename T> __global__ void fma_k(T* out, int iters){
  T a[8]; for(int j=0;j<8;j++) a[j]=threadIdx.x*0.001f+j; T b=1.0001f, c=0.0001f;
  for(int i=0;i<iters;i++){
#pragma unroll
    for(int j=0;j<8;j++) a[j]=a[j]*b+c;
  }
  T s=0; for(int j=0;j<8;j++) s+=a[j]; if(s==1.2345f) *out=s;
}
int main(){
  size_t bytes = (size_t)8<<30; size_t n=bytes/16; double2 *p,*q; double* o;
  cudaMalloc(&p,bytes); cudaMalloc(&q,bytes); cudaMalloc(&o,8); cudaMemset(p,0,bytes); cudaMemset(q,0,bytes);
  cudaEvent_t e0,e1; cudaEventCreate(&e0); cudaEventCreate(&e1); float ms;
  for(int blocks: {148*4,148*8,148*16,148*32}) for(int th: {256,512}){
    rd<<<blocks,th>>>(p,n,o); cudaEventRecord(e0); for(int r=0;r<5;r++) rd<<<blocks,th>>>(p,n,o); cudaEventRecord(e1); cudaEventSynchronize(e1); cudaEventElapsedTime(&ms,e0,e1);
    printf("read-only  blocks=%d th=%d : %.1f GB/s\n",blocks,th, 5.0*bytes/ms/1e6);
  }
  for(int blocks: {148*8,148*32}) { cp<<<blocks,512>>>(p,q,n); cudaEventRecord(e0); for(int r=0;r<5;r++) cp<<<blocks,512>>>(p,q,n); cudaEventRecord(e1); cudaEventSynchronize(e1); cudaEventElapsedTime(&ms,e0,e1);
    printf("copy r+w   blocks=%d : %.1f GB/s\n",blocks, 5.0*2*bytes/ms/1e6); }
  // L2-resident read: 32 MB and 64 MB buffers (power-of-two element counts)
  for(size_t mb: {32, 64}) { size_t nn=(mb<<20)/16; int blocks=148*8, th=512; int it=2000;
    rd_l2<<<blocks,th>>>(p,(unsigned)(nn-1),50,o); cudaEventRecord(e0); rd_l2<<<blocks,th>>>(p,(unsigned)(nn-1),it,o); cudaEventRecord(e1); cudaEventSynchronize(e1); cudaEventElapsedTime(&ms,e0,e1);
    printf("L2-resident read %zuMB : %.1f GB/s\n", mb, (double)blocks*th*it*64/ms/1e6); }
  int iters=20000;
  fma_k<float><<<148*8,512>>>((float*)o,iters); cudaEventRecord(e0); fma_k<float><<<148*8,512>>>((float*)o,iters); cudaEventRecord(e1); cudaEventSynchronize(e1); cudaEventElapsedTime(&ms,e0,e1);
  printf("fp32 FMA peak: %.1f TFLOP/s\n", 148.0*8*512*8*2*iters/ms/1e9);
  fma_k<double><<<148*8,512>>>(o,iters); cudaEventRecord(e0); fma_k<double><<<148*8,512>>>(o,iters); cudaEventRecord(e1); cudaEventSynchronize(e1); cudaEventElapsedTime(&ms,e0,e1);
  printf("fp64 FMA peak: %.1f TFLOP/s\n", 148.0*8*512*8*2*iters/ms/1e9);
  return 0;
}
