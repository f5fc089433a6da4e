// bench_pipes.cu -- stand-alone micro-benchmark (not part of libloc_b200.so): issue and pipe cost per warp instruction of FFMA2,
// FFMA, LOP3 and MUFU.EX2 and of their mixes on one SM, 1 / 4 / 8 warps per scheduler.  Justifies the packed arithmetic and the
// pipe figures of the roofline (DESIGN 8.2).  Build: nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o bench_pipes bench_pipes.cu
#include <cstdio>
#include <cuda_runtime.h>
typedef unsigned long long u64;
__device__ __forceinline__ u64 fma2(u64 a, u64 b, u64 c){u64 d; asm volatile("fma.rn.f32x2 %0, %1, %2, %3;":"=l"(d):"l"(a),"l"(b),"l"(c)); return d;}
__device__ __forceinline__ float ex2(float x){float y; asm volatile("ex2.approx.ftz.f32 %0, %1;":"=f"(y):"f"(x)); return y;}
template<int MODE> __global__ void k(float *out, long long *cyc, int iters)
{
    u64 a[8]; float f[8]; unsigned u[8];
    for (int i=0;i<8;i++){a[i]=threadIdx.x+i; f[i]=0.001f*(threadIdx.x+i); u[i]=threadIdx.x*7+i;}
    const u64 c1=0x3f8000013f800001ull, c2=0x3a0000003a000000ull;
    __syncthreads();
    long long t0=clock64();
    for (int it=0; it<iters; it++) {
#pragma unroll
        for (int i=0;i<8;i++) {
            if (MODE==0) { a[i]=fma2(a[i],c1,c2); }                                   // 8 FFMA2
            if (MODE==1) { f[i]=fmaf(f[i],1.0001f,0.5f); }                             // 8 FFMA
            if (MODE==2) { a[i]=fma2(a[i],c1,c2); asm volatile("lop3.b32 %0, %0, 0x55, %1, 0x96;" : "+r"(u[i]) : "r"(u[(i+1)&7])); }   // FFMA2 + LOP3
            if (MODE==3) { a[i]=fma2(a[i],c1,c2); f[i]=fmaf(f[i],1.0001f,0.5f); }      // FFMA2 + FFMA
            if (MODE==4) { f[i]=ex2(f[i]); }                                           // MUFU
            if (MODE==5) { a[i]=fma2(a[i],c1,c2); if (i&1) f[i]=ex2(f[i]); }           // 8 FFMA2 + 4 MUFU
            if (MODE==6) { asm volatile("lop3.b32 %0, %0, 0x55, %1, 0x96;" : "+r"(u[i]) : "r"(u[(i+1)&7])); }   // LOP3 only
            if (MODE==7) { a[i]=fma2(a[i],c1,c2); asm volatile("lop3.b32 %0, %0, 0x55, %1, 0x96;" : "+r"(u[i]) : "r"(u[(i+1)&7])); if (i&1) f[i]=ex2(f[i]); }
        }
    }
    long long t1=clock64();
    float s=0; for(int i=0;i<8;i++) s+=f[i]+(float)a[i]+(float)u[i];
    out[blockIdx.x*blockDim.x+threadIdx.x]=s;
    if (threadIdx.x==0) cyc[blockIdx.x]=t1-t0;
}
template<int MODE> void run(const char*name,int ninstr,int threads){
    float*o; long long*c; cudaMalloc(&o,4*1024*4); cudaMalloc(&c,64);
    int iters=20000; k<MODE><<<1,threads>>>(o,c,iters); k<MODE><<<1,threads>>>(o,c,iters);
    long long h; cudaMemcpy(&h,c,8,cudaMemcpyDeviceToHost);
    int wps=threads/128; if(wps<1)wps=1;
    printf("%-28s threads %4d: %.3f cycles per warp-instruction per scheduler (%.2f cyc/iter/warp)\n",name,threads,(double)h/((double)iters*ninstr*wps),(double)h/iters);
    cudaFree(o);cudaFree(c);
}
int main(){
    for (int th : {128, 512, 1024}) {
        run<0>("FFMA2",8,th); run<1>("FFMA",8,th); run<6>("LOP3",8,th); run<4>("MUFU.EX2",8,th);
        run<2>("FFMA2+LOP3 (1:1)",16,th); run<3>("FFMA2+FFMA (1:1)",16,th); run<5>("FFMA2+MUFU (2:1)",12,th); run<7>("FFMA2+LOP3+MUFU (2:2:1)",20,th);
    }
    return 0;
}
