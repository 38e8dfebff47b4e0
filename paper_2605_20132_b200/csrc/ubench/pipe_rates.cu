// pipe_rates.cu -- micro-benchmark behind DESIGN.md 6: FP32 FMA throughput on B200 for scalar FFMA
// with reusable / immediate operands, scalar FFMA with three distinct register operands, FFMA2
// (fma.rn.f32x2), and FFMA mixed with SHFL or MUFU.RCP; prints lane-FMA/s (peak 37.2 T/s).
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o pipe_rates pipe_rates.cu && ./pipe_rates
#include <cstdio>
#include <cuda_runtime.h>
#define CHECK(x) do{cudaError_t e=(x); if(e!=cudaSuccess){printf("err %s line %d\n",cudaGetErrorString(e),__LINE__);return 1;}}while(0)

template<int CH> __global__ void k_ffma(float* out, float a, float b, int iters){
    float v[CH];
    #pragma unroll
    for(int i=0;i<CH;i++) v[i]=threadIdx.x*0.001f+i;
    for(int it=0;it<iters;it++){
        #pragma unroll
        for(int r=0;r<8;r++){
            #pragma unroll
            for(int i=0;i<CH;i++) v[i]=fmaf(v[i],a,b);
        }
    }
    float s=0; 
    #pragma unroll
    for(int i=0;i<CH;i++) s+=v[i];
    out[blockIdx.x*blockDim.x+threadIdx.x]=s;
}
// 3 distinct register operands: v = v*w[i] + u[i]
template<int CH> __global__ void k_ffma3(float* out, const float* in, int iters){
    float v[CH], w[CH], u[CH];
    #pragma unroll
    for(int i=0;i<CH;i++){ v[i]=threadIdx.x*0.001f+i; w[i]=in[i]; u[i]=in[i+CH]; }
    for(int it=0;it<iters;it++){
        #pragma unroll
        for(int r=0;r<8;r++){
            #pragma unroll
            for(int i=0;i<CH;i++) v[i]=fmaf(v[i],w[i],u[(i+r)%CH]);
        }
    }
    float s=0; 
    #pragma unroll
    for(int i=0;i<CH;i++) s+=v[i];
    out[blockIdx.x*blockDim.x+threadIdx.x]=s;
}
__device__ __forceinline__ unsigned long long pk(float x,float y){ unsigned long long r; asm("mov.b64 %0,{%1,%2};":"=l"(r):"f"(x),"f"(y)); return r;}
template<int CH> __global__ void k_ffma2(float* out, float a, float b, int iters){
    unsigned long long v[CH]; unsigned long long A=pk(a,a), B=pk(b,b);
    #pragma unroll
    for(int i=0;i<CH;i++) v[i]=pk(threadIdx.x*0.001f+i, i*0.5f);
    for(int it=0;it<iters;it++){
        #pragma unroll
        for(int r=0;r<8;r++){
            #pragma unroll
            for(int i=0;i<CH;i++) asm volatile("fma.rn.f32x2 %0,%0,%1,%2;":"+l"(v[i]):"l"(A),"l"(B));
        }
    }
    float s=0;
    #pragma unroll
    for(int i=0;i<CH;i++){ float x,y; asm("mov.b64 {%0,%1},%2;":"=f"(x),"=f"(y):"l"(v[i])); s+=x+y; }
    out[blockIdx.x*blockDim.x+threadIdx.x]=s;
}
// mix: per 4 FFMA one SHFL
template<int CH> __global__ void k_mix_shfl(float* out, float a, float b, int iters){
    float v[CH];
    #pragma unroll
    for(int i=0;i<CH;i++) v[i]=threadIdx.x*0.001f+i;
    for(int it=0;it<iters;it++){
        #pragma unroll
        for(int r=0;r<8;r++){
            #pragma unroll
            for(int i=0;i<CH;i++) v[i]=fmaf(v[i],a,b);
            v[r%CH]+=__shfl_up_sync(0xffffffffu,v[(r+1)%CH],1);
        }
    }
    float s=0; 
    #pragma unroll
    for(int i=0;i<CH;i++) s+=v[i];
    out[blockIdx.x*blockDim.x+threadIdx.x]=s;
}
// MUFU rcp mix: per 8 FFMA one rcp
template<int CH> __global__ void k_mix_rcp(float* out, float a, float b, int iters){
    float v[CH];
    #pragma unroll
    for(int i=0;i<CH;i++) v[i]=threadIdx.x*0.001f+i+1.f;
    for(int it=0;it<iters;it++){
        #pragma unroll
        for(int r=0;r<8;r++){
            #pragma unroll
            for(int i=0;i<CH;i++) v[i]=fmaf(v[i],a,b);
            float q; asm volatile("rcp.approx.ftz.f32 %0,%1;":"=f"(q):"f"(v[r%CH])); v[(r+1)%CH]+=q;
        }
    }
    float s=0; 
    #pragma unroll
    for(int i=0;i<CH;i++) s+=v[i];
    out[blockIdx.x*blockDim.x+threadIdx.x]=s;
}
template<typename F> float timeit(F f){
    cudaEvent_t e0,e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    f(); cudaDeviceSynchronize();
    cudaEventRecord(e0); f(); cudaEventRecord(e1); cudaEventSynchronize(e1);
    float ms; cudaEventElapsedTime(&ms,e0,e1); return ms;
}
int main(){
    float* out; CHECK(cudaMalloc(&out, 148*1024*4*4)); float* in; CHECK(cudaMalloc(&in, 4096)); cudaMemset(in,0,4096);
    int iters=20000; 
    int clk; cudaDeviceGetAttribute(&clk, cudaDevAttrClockRate, 0);
    printf("clock attr kHz %d\n", clk);
    for(int warps: {4,8,16,32}){
        int thr=warps*32; int grid=148;
        double ops = (double)grid*thr*iters*8.0;
        #define RUN(name, kern, CH, mult, ...) { float ms=timeit([&]{kern<CH><<<grid,thr>>>(__VA_ARGS__);}); \
            printf("%-12s warps/SM=%2d chains=%d : %.3f ms  %.2f Tfma-lane/s  (%.1f lane-fma/clk/SM at 1965 MHz)\n", name, warps, CH, ms, ops*CH*mult/ms/1e9, ops*CH*mult/ms/1e6/148/1.965e6);}
        RUN("ffma_imm", k_ffma, 4, 1, out, 1.0001f, 0.5f, iters)
        RUN("ffma_imm", k_ffma, 8, 1, out, 1.0001f, 0.5f, iters)
        RUN("ffma_3reg", k_ffma3, 4, 1, out, in, iters)
        RUN("ffma_3reg", k_ffma3, 8, 1, out, in, iters)
        RUN("ffma2", k_ffma2, 4, 2, out, 1.0001f, 0.5f, iters)
        RUN("ffma2", k_ffma2, 8, 2, out, 1.0001f, 0.5f, iters)
        RUN("mix_shfl", k_mix_shfl, 4, 1, out, 1.0001f, 0.5f, iters)
        RUN("mix_rcp", k_mix_rcp, 8, 1, out, 1.0001f, 0.5f, iters)
    }
    return 0;
}
