// microbenchmark: throughput of cp.async.bulk global->shared as a function of request size
#include <cstdio>
#include <cstdint>
#include <cuda_runtime.h>
__device__ __forceinline__ uint32_t s32(const void* p){return (uint32_t)__cvta_generic_to_shared(p);}
__global__ void __launch_bounds__(64,1) k(const unsigned char* src, size_t span, uint32_t bytes, uint32_t per_stage, int stages, int iters, int one_lane, unsigned long long* sink)
{
    extern __shared__ __align__(128) unsigned char sm[];
    uint64_t* bar = (uint64_t*)sm;            // [stages]
    unsigned char* buf = sm + 1024;
    if (threadIdx.x==0){ for(int s=0;s<stages;++s) asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;"::"r"(s32(bar+s))); asm volatile("fence.mbarrier_init.release.cluster;"); }
    __syncthreads();
    if (threadIdx.x >= 32) return;
    const uint32_t lane = threadIdx.x;
    size_t off = ((size_t)blockIdx.x * 7919u * 4096u) % span;
    const uint32_t stage_bytes = bytes*per_stage;
    for (int it=0; it<iters; ++it) {
        int s = it % stages; uint32_t ph = (it/stages)&1;
        if (it >= stages) { // wait for the previous use of this slot to land
            uint32_t ok=0; while(!ok) asm volatile("{.reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0,1,0,p;}":"=r"(ok):"r"(s32(bar+s)),"r"(ph^1):"memory");
        }
        if (lane==0) asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;"::"r"(s32(bar+s)),"r"(stage_bytes):"memory");
        __syncwarp();
        for (uint32_t id = one_lane ? 0 : lane; id < per_stage; id += one_lane ? 1 : 32) {
            if (one_lane && lane) break;
            const unsigned char* g = src + (off + (size_t)id * 65536u) % span;   // scattered runs like the link chunks
            asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"::"r"(s32(buf + (size_t)s*stage_bytes + id*bytes)),"l"(g),"r"(bytes),"r"(s32(bar+s)):"memory");
        }
        off = (off + bytes) % (span - 32*65536u);
        __syncwarp();
    }
    // drain
    for (int it=iters; it<iters+stages; ++it){ int s=it%stages; uint32_t ph=(it/stages)&1; if (it>=stages){uint32_t ok=0; while(!ok) asm volatile("{.reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0,1,0,p;}":"=r"(ok):"r"(s32(bar+s)),"r"(ph^1):"memory");} }
    if (lane==0) sink[blockIdx.x] = buf[0];
}
int main(){
    size_t span = (size_t)64<<20;   // 64 MB: L2 resident after the first pass
    unsigned char* src; cudaMalloc(&src, span + (64<<20)); cudaMemset(src,1,span + (64<<20));
    unsigned long long* sink; cudaMalloc(&sink, 8*1024);
    cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, 200*1024);
    int sizes[] = {256,512,1024,2048,4096,8192,16384};
    for (int one=0; one<2; ++one)
    for (int bi=0; bi<7; ++bi){
        uint32_t bytes=sizes[bi];
        uint32_t per_stage = 32768/bytes; if (per_stage<1) per_stage=1; if (per_stage>72) per_stage=72;
        int stages = (180*1024)/(bytes*per_stage); if (stages>8) stages=8;
        int iters = (int)((size_t)(64<<20)/(bytes*per_stage)); if (iters>4000) iters=4000;
        size_t smem = 1024 + (size_t)stages*bytes*per_stage;
        cudaEvent_t a,b; cudaEventCreate(&a); cudaEventCreate(&b);
        k<<<148,64,smem>>>(src,span,bytes,per_stage,stages,iters/4,one,sink); cudaDeviceSynchronize();
        cudaEventRecord(a); k<<<148,64,smem>>>(src,span,bytes,per_stage,stages,iters,one,sink); cudaEventRecord(b); cudaDeviceSynchronize();
        float ms; cudaEventElapsedTime(&ms,a,b);
        double total = 148.0*iters*bytes*per_stage;
        printf("%s bytes/req %5u  req/stage %2u stages %d: %.1f GB/s total, %.1f ns per request per SM, err %s\n", one?"one lane ":"all lanes", bytes, per_stage, stages, total/ms/1e6, ms*1e6/(double)(iters*per_stage), cudaGetErrorString(cudaGetLastError()));
    }
    return 0;
}
