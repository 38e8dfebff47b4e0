// fma_operands.cu -- micro-benchmark behind DESIGN.md 6 ("uniform operands"): the per-section inner
// loops of the stream kernel (zero-state DF2 recurrence + fix-up, L = 24, 8 sections, data in
// registers) in three operand forms: scalar FFMA on two chains with table values in registers,
// packed FFMA2 with table values in registers, packed FFMA2 with table values read from the
// kernel-parameter constant bank (uniform-register operands).  Prints lane-samples/s through 8
// sections and the share of the FMA-pipe peak (148 SMs x 128 lanes x 1.965 GHz).
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o fma_operands fma_operands.cu && ./fma_operands
#include <cstdio>
#include <cuda_runtime.h>
constexpr int L=24, NSEC=8;
extern __shared__ __align__(16) float sm[];
// table per section: [0..7] coef dup pairs, [8..8+4L) g rows (g1,g1,g2,g2)
constexpr int STR = 8 + 4*L;

__global__ void __launch_bounds__(512,1) k_scalar(float* out, const float* tab, int reps){
    for(int i=threadIdx.x;i<NSEC*STR;i+=blockDim.x) sm[i]=tab[i];
    __syncthreads();
    float lo[L], hi[L];
    #pragma unroll
    for(int i=0;i<L;i++){ lo[i]=threadIdx.x*1e-3f+i; hi[i]=lo[i]*0.5f; }
    for(int r=0;r<reps;r++){
        for(int k=0;k<NSEC;k++){
            const float* T=&sm[k*STR];
            const float c0=T[0],c1=T[2],c2=T[4],c3=T[6];
            float a1=0,a2=0,b1=0,b2=0;
            #pragma unroll
            for(int i=0;i<L;i++){
                const float wa=fmaf(c0,a1,fmaf(c1,a2,lo[i]));
                const float wb=fmaf(c0,b1,fmaf(c1,b2,hi[i]));
                lo[i]=fmaf(c2,a1,fmaf(c3,a2,wa));
                hi[i]=fmaf(c2,b1,fmaf(c3,b2,wb));
                a2=a1;a1=wa;b2=b1;b1=wb;
            }
            // fake "scan": one shuffle each
            float E1=__shfl_up_sync(~0u,a1,1),E2=__shfl_up_sync(~0u,a2,1),o1=__shfl_up_sync(~0u,b1,1),o2=__shfl_up_sync(~0u,b2,1);
            const float4* G=reinterpret_cast<const float4*>(T+8);
            #pragma unroll
            for(int i=0;i<L;i++){
                const float4 g=G[i];
                lo[i]=fmaf(g.x,E1,fmaf(g.z,E2,lo[i]));
                hi[i]=fmaf(g.x,o1,fmaf(g.z,o2,hi[i]));
            }
        }
    }
    float s=0;
    #pragma unroll
    for(int i=0;i<L;i++) s+=lo[i]+hi[i];
    out[blockIdx.x*blockDim.x+threadIdx.x]=s;
}
__global__ void __launch_bounds__(512,1) k_packed(float* out, const float* tab, int reps){
    for(int i=threadIdx.x;i<NSEC*STR;i+=blockDim.x) sm[i]=tab[i];
    __syncthreads();
    float2 x[L];
    #pragma unroll
    for(int i=0;i<L;i++){ x[i].x=threadIdx.x*1e-3f+i; x[i].y=x[i].x*0.5f; }
    for(int r=0;r<reps;r++){
        for(int k=0;k<NSEC;k++){
            const float* T=&sm[k*STR];
            const float4 ca=*reinterpret_cast<const float4*>(T), cb=*reinterpret_cast<const float4*>(T+4);
            const float2 c0=make_float2(ca.x,ca.y),c1=make_float2(ca.z,ca.w),c2=make_float2(cb.x,cb.y),c3=make_float2(cb.z,cb.w);
            float2 s1=make_float2(0,0),s2=s1;
            #pragma unroll
            for(int i=0;i<L;i++){
                const float2 w=__ffma2_rn(c0,s1,__ffma2_rn(c1,s2,x[i]));
                x[i]=__ffma2_rn(c2,s1,__ffma2_rn(c3,s2,w));
                s2=s1;s1=w;
            }
            float2 E1,E2;
            E1.x=__shfl_up_sync(~0u,s1.x,1);E2.x=__shfl_up_sync(~0u,s2.x,1);E1.y=__shfl_up_sync(~0u,s1.y,1);E2.y=__shfl_up_sync(~0u,s2.y,1);
            const float4* G=reinterpret_cast<const float4*>(T+8);
            #pragma unroll
            for(int i=0;i<L;i++){
                const float4 g=G[i];
                x[i]=__ffma2_rn(make_float2(g.x,g.y),E1,__ffma2_rn(make_float2(g.z,g.w),E2,x[i]));
            }
        }
    }
    float s=0;
    #pragma unroll
    for(int i=0;i<L;i++) s+=x[i].x+x[i].y;
    out[blockIdx.x*blockDim.x+threadIdx.x]=s;
}
struct Sec { float c[4]; float pad[4]; float g[L][2]; };
struct P { Sec s[NSEC]; int n_sec; int reps; };
__global__ void __launch_bounds__(512,1) k_ur(float* out, const __grid_constant__ P p){
    float2 x[L];
    #pragma unroll
    for(int i=0;i<L;i++){ x[i].x=threadIdx.x*1e-3f+i; x[i].y=x[i].x*0.5f; }
    for(int r=0;r<p.reps;r++){
        for(int k=0;k<p.n_sec;k++){
            const Sec& T=p.s[k];
            const float c0=T.c[0],c1=T.c[1],c2=T.c[2],c3=T.c[3];
            float2 s1=make_float2(0,0),s2=s1;
            #pragma unroll
            for(int i=0;i<L;i++){
                const float2 w=__ffma2_rn(make_float2(c0,c0),s1,__ffma2_rn(make_float2(c1,c1),s2,x[i]));
                x[i]=__ffma2_rn(make_float2(c2,c2),s1,__ffma2_rn(make_float2(c3,c3),s2,w));
                s2=s1;s1=w;
            }
            float2 E1,E2;
            E1.x=__shfl_up_sync(~0u,s1.x,1);E2.x=__shfl_up_sync(~0u,s2.x,1);E1.y=__shfl_up_sync(~0u,s1.y,1);E2.y=__shfl_up_sync(~0u,s2.y,1);
            #pragma unroll
            for(int i=0;i<L;i++){
                const float g1=T.g[i][0], g2=T.g[i][1];
                x[i]=__ffma2_rn(make_float2(g1,g1),E1,__ffma2_rn(make_float2(g2,g2),E2,x[i]));
            }
        }
    }
    float s=0;
    #pragma unroll
    for(int i=0;i<L;i++) s+=x[i].x+x[i].y;
    out[blockIdx.x*blockDim.x+threadIdx.x]=s;
}
template<typename F> float timeit(F f){
    cudaEvent_t e0,e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    f(); cudaDeviceSynchronize();
    cudaEventRecord(e0); f(); cudaEventRecord(e1); cudaEventSynchronize(e1);
    float ms; cudaEventElapsedTime(&ms,e0,e1); return ms;
}
int main(){
    float* out; cudaMalloc(&out,148*512*4); float* tab; cudaMalloc(&tab,NSEC*STR*4);
    float h[NSEC*STR]; for(int i=0;i<NSEC*STR;i++) h[i]=((i%STR)<8)?0.3f:1e-3f;
    cudaMemcpy(tab,h,sizeof(h),cudaMemcpyHostToDevice);
    P p; for(int k=0;k<NSEC;k++){ for(int j=0;j<4;j++) p.s[k].c[j]=0.3f; for(int i=0;i<L;i++){p.s[k].g[i][0]=1e-3f;p.s[k].g[i][1]=2e-3f;} }
    p.n_sec=NSEC; p.reps=2000;
    const int reps=2000;
    for(int warps: {4,8,12,16}){
        double samples=(double)148*warps*32*2*L*reps;
        float ms=timeit([&]{k_scalar<<<148,warps*32,NSEC*STR*4>>>(out,tab,reps);});
        printf("scalar FFMA, table in registers   warps/SM=%2d: %7.1f Gsamples/s  fma-pipe %.1f%%\n",warps,samples/ms/1e6, samples*48/ms/1e6/37200*100);
        ms=timeit([&]{k_packed<<<148,warps*32,NSEC*STR*4>>>(out,tab,reps);});
        printf("FFMA2, table in registers         warps/SM=%2d: %7.1f Gsamples/s  fma-pipe %.1f%%\n",warps,samples/ms/1e6, samples*48/ms/1e6/37200*100);
        ms=timeit([&]{k_ur<<<148,warps*32>>>(out,p);});
        printf("FFMA2, table in uniform registers warps/SM=%2d: %7.1f Gsamples/s  fma-pipe %.1f%%\n",warps,samples/ms/1e6, samples*48/ms/1e6/37200*100);
    }
    return 0;
}
