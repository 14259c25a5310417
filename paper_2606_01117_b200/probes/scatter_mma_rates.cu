// probe4: cost of tf32 A-from-TMEM scatter MMAs (N=64) and of switching kinds between f16 and tf32 MMAs
#include <cstdio>
#include <cstdint>
#include <cuda_runtime.h>
#define CK(x) do{cudaError_t e=(x); if(e!=cudaSuccess){printf("ERR %s line %d\n",cudaGetErrorString(e),__LINE__);exit(1);} }while(0)
__device__ __forceinline__ uint32_t smem_u32(const void* p){return (uint32_t)__cvta_generic_to_shared(p);}
__device__ __forceinline__ uint64_t sdesc(uint32_t saddr, uint32_t lbo, uint32_t sbo, uint32_t type){
  uint64_t d=0; d|=(uint64_t)((saddr>>4)&0x3FFF); d|=(uint64_t)((lbo>>4)&0x3FFF)<<16; d|=(uint64_t)((sbo>>4)&0x3FFF)<<32; d|=(uint64_t)1<<46; d|=(uint64_t)type<<61; return d;}
__device__ __forceinline__ void mma_f16(uint32_t d, uint64_t a, uint64_t b, uint32_t idesc){
  asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, 1, 0;\n\ttcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"::"r"(d),"l"(a),"l"(b),"r"(idesc):"memory"); }
__device__ __forceinline__ void mma_tf32_ts(uint32_t d, uint32_t a, uint64_t b, uint32_t idesc){
  asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, 1, 0;\n\ttcgen05.mma.cta_group::1.kind::tf32 [%0], [%1], %2, %3, p;\n\t}"::"r"(d),"r"(a),"l"(b),"r"(idesc):"memory"); }
__device__ __forceinline__ void mma_f16_ts(uint32_t d, uint32_t a, uint64_t b, uint32_t idesc){
  asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, 1, 0;\n\ttcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t}"::"r"(d),"r"(a),"l"(b),"r"(idesc):"memory"); }
// mode 0: reps x (nf f16 SS MMAs N=64), mode 1: reps x (nt tf32 TS MMAs N=64), mode 2: reps x (nf f16 then nt tf32), mode 3: reps x (nf f16 SS then nt f16 TS N=64 K=16)
__global__ void __launch_bounds__(128,1) k(int mode, int nf, int nt, int reps, long long* out){
  extern __shared__ __align__(1024) uint8_t sm[];
  __shared__ uint32_t slot; __shared__ uint64_t bar;
  const int tid=threadIdx.x, warp=tid>>5;
  if(warp==0){ asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;"::"r"(smem_u32(&slot)):"memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;":::"memory"); }
  if(tid==0){ asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;"::"r"(smem_u32(&bar)):"memory"); asm volatile("fence.mbarrier_init.release.cluster;":::"memory"); }
  for(int i=tid;i<65536/4;i+=128) ((uint32_t*)sm)[i]=0;
  asm volatile("fence.proxy.async.shared::cta;":::"memory");
  asm volatile("tcgen05.fence::before_thread_sync;":::"memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;":::"memory");
  if(warp==0){
    uint32_t e; asm volatile("{\n\t.reg .pred p;\n\telect.sync _|p, 0xffffffff;\n\tselp.u32 %0,1,0,p;\n\t}":"=r"(e));
    if(e){
      const uint32_t id_f16 = (1u<<4)|(1u<<7)|(1u<<10)|(0u<<15)|(1u<<16)|((64u>>3)<<17)|((128u>>4)<<24);   // bf16, A K-major, B MN-major, N=64
      const uint32_t id_tf = (1u<<4)|(2u<<7)|(2u<<10)|((64u>>3)<<17)|((128u>>4)<<24);
      const uint32_t id_f16ts = (1u<<4)|(0u<<7)|(0u<<10)|((64u>>3)<<17)|((128u>>4)<<24);                  // f16 x f16, K-major B no swizzle
      const uint64_t ad = sdesc(smem_u32(sm), 16, 1024, 2), bd = sdesc(smem_u32(sm)+16384, 8192, 1024, 2), sd = sdesc(smem_u32(sm)+32768, 128, 256, 0);
      long long t0=clock64();
      for(int r=0;r<reps;++r){
        if(mode==0){        // 8 tf32 TS, same D window
#pragma unroll
          for(int j=0;j<8;++j) mma_tf32_ts(slot + 128, slot + j*8, sd, id_tf);
        } else if(mode==1){ // 8 tf32 TS, D windows rotate over 4 disjoint windows
#pragma unroll
          for(int j=0;j<8;++j) mma_tf32_ts(slot + 128 + (j&3)*64, slot + j*8, sd, id_tf);
        } else if(mode==2){ // 8 tf32 TS, overlapping windows shifted by 48 columns
#pragma unroll
          for(int j=0;j<8;++j) mma_tf32_ts(slot + 128 + j*40, slot + j*8, sd, id_tf);
        } else if(mode==3){ // 8 f16 SS same D (a k-loop)
#pragma unroll
          for(int j=0;j<8;++j) mma_f16(slot, ad + (j&3)*2, bd + (j&3)*128, id_f16);
        } else if(mode==4){ // 8 f16 SS alternating D
#pragma unroll
          for(int j=0;j<8;++j) mma_f16(slot + (j&1)*64, ad + (j&3)*2, bd + (j&3)*128, id_f16);
        } else {            // 4 f16 same D then 8 tf32 rotating
#pragma unroll
          for(int j=0;j<4;++j) mma_f16(slot, ad + (j&3)*2, bd + (j&3)*128, id_f16);
#pragma unroll
          for(int j=0;j<8;++j) mma_tf32_ts(slot + 128 + (j&3)*64, slot + j*8, sd, id_tf);
        }
      }
      asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];"::"r"(smem_u32(&bar)):"memory");
      uint32_t ok=0; while(!ok){ asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], 0;\n\tselp.u32 %0,1,0,p;\n\t}":"=r"(ok):"r"(smem_u32(&bar)):"memory"); }
      long long t1=clock64();
      out[0]=t1-t0;
    }
    __syncwarp();
  }
  asm volatile("tcgen05.fence::before_thread_sync;":::"memory");
  __syncthreads();
  if(warp==0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;"::"r"(slot):"memory");
}
int main(){
  long long* out; CK(cudaMalloc(&out,8));
  CK(cudaFuncSetAttribute(k,cudaFuncAttributeMaxDynamicSharedMemorySize,65536));
  struct { int mode,nf,nt; const char* name; } cs[] = {
    {0,8,0,"8 tf32 TS same D"}, {1,8,0,"8 tf32 TS, 4 disjoint D windows"}, {2,8,0,"8 tf32 TS, D shifted by 40 cols (overlap)"},
    {3,8,0,"8 f16 SS same D"}, {4,8,0,"8 f16 SS alternating D"}, {5,12,0,"4 f16 same D + 8 tf32 rotating"} };
  for(auto& c: cs){
    const int reps=2000; long long h=0;
    for(int it=0;it<2;++it){ k<<<1,128,65536>>>(c.mode,c.nf,c.nt,reps,out); cudaError_t e=cudaDeviceSynchronize(); if(e!=cudaSuccess){printf("%s: CUDA error %s\n",c.name,cudaGetErrorString(e)); return 0;} }
    CK(cudaMemcpy(&h,out,8,cudaMemcpyDeviceToHost));
    printf("%-45s : %.1f cycles per rep (%.1f per MMA)\n", c.name, (double)h/reps, (double)h/reps/(c.nf+c.nt));
  }
  return 0;
}
