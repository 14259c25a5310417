// probe2: on-chip scatter-add rates for the dX kernel design.
#include <cstdio>
#include <cstdint>
#include <cuda_runtime.h>
#include <vector>
#define CK(x) do{cudaError_t e=(x); if(e!=cudaSuccess){printf("ERR %s line %d\n",cudaGetErrorString(e),__LINE__);exit(1);} }while(0)
__device__ __forceinline__ uint32_t smem_u32(const void* p){return (uint32_t)__cvta_generic_to_shared(p);}

// ---- SMEM RMW: acc[F][128] fp32, thread = column b, NW warps (multiple of 4 -> warps w and w+4 own the same b? no: separate halves of the slots)
// each warp-group of 4 warps (128 threads = 128 b) processes a stream of "slots" (feature byte offsets read from smem, LDS.128 broadcast)
template<int NWG>
__global__ void __launch_bounds__(128*NWG,1) k_smem_rmw(const int* offs, int nslots, int iters, float* out, int F){
  extern __shared__ __align__(16) uint8_t sm[];
  float* acc = (float*)sm;                       // F*128 floats
  int* soff = (int*)(sm + (size_t)F*512);        // nslots ints (byte offsets, multiples of 512); NWG disjoint lists
  for(int i=threadIdx.x;i<F*128;i+=blockDim.x) acc[i]=0.f;
  for(int i=threadIdx.x;i<nslots*NWG;i+=blockDim.x) soff[i]=offs[i];
  __syncthreads();
  const int wg = threadIdx.x>>7, b = threadIdx.x&127;
  const uint32_t base = smem_u32(acc) + b*4;
  const uint32_t sidx = smem_u32(soff + wg*nslots);
  float v = 1.0f + b;
  for(int it=0; it<iters; ++it){
    #pragma unroll 1
    for(int j=0;j<nslots;j+=8){
      int4 o0,o1;
      asm volatile("ld.shared.v4.b32 {%0,%1,%2,%3}, [%4];":"=r"(o0.x),"=r"(o0.y),"=r"(o0.z),"=r"(o0.w):"r"(sidx+j*4));
      asm volatile("ld.shared.v4.b32 {%0,%1,%2,%3}, [%4];":"=r"(o1.x),"=r"(o1.y),"=r"(o1.z),"=r"(o1.w):"r"(sidx+j*4+16));
      int o[8]={o0.x,o0.y,o0.z,o0.w,o1.x,o1.y,o1.z,o1.w};
      float a[8];
      #pragma unroll
      for(int u=0;u<8;++u) asm volatile("ld.shared.f32 %0, [%1];":"=f"(a[u]):"r"(base+o[u]));
      #pragma unroll
      for(int u=0;u<8;++u){ a[u]+=v; asm volatile("st.shared.f32 [%0], %1;"::"r"(base+o[u]),"f"(a[u]):"memory"); }
    }
  }
  __syncthreads();
  float s=0; for(int i=threadIdx.x;i<F*128;i+=blockDim.x) s+=acc[i];
  if(s==123.f) out[0]=s;
}

// ---- TMEM RMW: acc in TMEM columns [0,NC), thread = lane; tcgen05.ld x1 + add + tcgen05.st x1 with dynamic columns
__device__ __forceinline__ uint32_t tld1(uint32_t a){uint32_t v; asm volatile("tcgen05.ld.sync.aligned.32x32b.x1.b32 {%0}, [%1];":"=r"(v):"r"(a):"memory"); return v;}
__device__ __forceinline__ void tst1(uint32_t a, uint32_t v){asm volatile("tcgen05.st.sync.aligned.32x32b.x1.b32 [%0], {%1};"::"r"(a),"r"(v):"memory");}
__device__ __forceinline__ void twait_ld(){asm volatile("tcgen05.wait::ld.sync.aligned;":::"memory");}
__device__ __forceinline__ void twait_st(){asm volatile("tcgen05.wait::st.sync.aligned;":::"memory");}
template<int U>
__global__ void __launch_bounds__(128,1) k_tmem_rmw(const int* cols, int nslots, int iters, float* out){
  __shared__ uint32_t slot; __shared__ int scol[4096];
  if(threadIdx.x<32){ asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;"::"r"(smem_u32(&slot)):"memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;":::"memory"); }
  for(int i=threadIdx.x;i<nslots;i+=blockDim.x) scol[i]=cols[i];
  asm volatile("tcgen05.fence::before_thread_sync;":::"memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;":::"memory");
  const uint32_t tb = slot + ((uint32_t)((threadIdx.x>>5)*32)<<16);
  for(int c=0;c<512;++c) tst1(tb+c,0u);
  twait_st();
  float v = 1.0f;
  for(int it=0;it<iters;++it){
    #pragma unroll 1
    for(int j=0;j<nslots;j+=U){
      uint32_t a[U]; int c[U];
      #pragma unroll
      for(int u=0;u<U;++u){ c[u]=scol[j+u]; a[u]=tld1(tb+c[u]); }
      twait_ld();
      #pragma unroll
      for(int u=0;u<U;++u){ float f=__uint_as_float(a[u])+v; tst1(tb+c[u],__float_as_uint(f)); }
      twait_st();   // conservative: order next iteration's loads after these stores
    }
  }
  uint32_t r=tld1(tb+5); twait_ld();
  if(__uint_as_float(r)==-1.f) out[0]=1;
  asm volatile("tcgen05.fence::before_thread_sync;":::"memory");
  __syncthreads();
  if(threadIdx.x<32) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;"::"r"(slot):"memory");
}
// TMEM read-only bandwidth: x32 loads
__global__ void __launch_bounds__(128,1) k_tmem_ld(int iters, float* out){
  __shared__ uint32_t slot;
  if(threadIdx.x<32){ asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;"::"r"(smem_u32(&slot)):"memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;":::"memory"); }
  asm volatile("tcgen05.fence::before_thread_sync;":::"memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;":::"memory");
  const uint32_t tb = slot + ((uint32_t)((threadIdx.x>>5)*32)<<16);
  uint32_t acc=0;
  for(int it=0;it<iters;++it){
    #pragma unroll 1
    for(int c=0;c<512;c+=32){
      uint32_t v[32];
      asm volatile("tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
        :"=r"(v[0]),"=r"(v[1]),"=r"(v[2]),"=r"(v[3]),"=r"(v[4]),"=r"(v[5]),"=r"(v[6]),"=r"(v[7]),"=r"(v[8]),"=r"(v[9]),"=r"(v[10]),"=r"(v[11]),"=r"(v[12]),"=r"(v[13]),"=r"(v[14]),"=r"(v[15]),"=r"(v[16]),"=r"(v[17]),"=r"(v[18]),"=r"(v[19]),"=r"(v[20]),"=r"(v[21]),"=r"(v[22]),"=r"(v[23]),"=r"(v[24]),"=r"(v[25]),"=r"(v[26]),"=r"(v[27]),"=r"(v[28]),"=r"(v[29]),"=r"(v[30]),"=r"(v[31]):"r"(tb+c):"memory");
      twait_ld();
      #pragma unroll
      for(int i=0;i<32;++i) acc^=v[i];
    }
  }
  if(acc==12345u) out[0]=1;
  asm volatile("tcgen05.fence::before_thread_sync;":::"memory");
  __syncthreads();
  if(threadIdx.x<32) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;"::"r"(slot):"memory");
}

int main(){
  cudaDeviceProp pr; CK(cudaGetDeviceProperties(&pr,0));
  int clk_khz; cudaDeviceGetAttribute(&clk_khz, cudaDevAttrClockRate, 0);
  printf("device %s SMs %d clock %d kHz\n", pr.name, pr.multiProcessorCount, clk_khz);
  float* out; CK(cudaMalloc(&out,4));
  cudaEvent_t e0,e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
  const int nslots=2048;
  const int nsm=pr.multiProcessorCount;
  // SMEM RMW
  for(int F : {128, 384}){
    std::vector<int> h(nslots*2);
    uint32_t s=12345; for(auto& x:h){ s=s*1664525u+1013904223u; x=(int)((s>>8)%F)*512; }
    int* d; CK(cudaMalloc(&d,h.size()*4)); CK(cudaMemcpy(d,h.data(),h.size()*4,cudaMemcpyHostToDevice));
    size_t smem=(size_t)F*512+nslots*2*4;
    CK(cudaFuncSetAttribute(k_smem_rmw<1>,cudaFuncAttributeMaxDynamicSharedMemorySize,(int)smem));
    CK(cudaFuncSetAttribute(k_smem_rmw<2>,cudaFuncAttributeMaxDynamicSharedMemorySize,(int)smem));
    for(int nwg=1;nwg<=2;++nwg){
      int iters=40;
      for(int rep=0;rep<2;++rep){
        cudaEventRecord(e0);
        if(nwg==1) k_smem_rmw<1><<<nsm,128,smem>>>(d,nslots,iters,out,F); else k_smem_rmw<2><<<nsm,256,smem>>>(d,nslots,iters,out,F);
        cudaEventRecord(e1); CK(cudaDeviceSynchronize());
      }
      float ms; cudaEventElapsedTime(&ms,e0,e1);
      double adds=(double)nsm*128*nwg*nslots*iters;
      printf("SMEM RMW F=%d warps=%d: %.3f ms  %.1f Gadd/s  = %.2f adds/clk/SM @%.3f GHz\n",F,4*nwg,ms,adds/ms/1e6,adds/ms/1e6/nsm/(clk_khz/1e6),clk_khz/1e6);
    }
    cudaFree(d);
  }
  // TMEM RMW
  {
    std::vector<int> h(nslots);
    // distinct columns within every aligned block of 16 (no in-flight hazards): random permutation blocks of 256 columns
    uint32_t s=777; for(int i=0;i<nslots;i+=16){ int base=(int)((s=s*1664525u+1013904223u)>>8)%240; for(int u=0;u<16;++u) h[i+u]=base+u; for(int u=15;u>0;--u){ s=s*1664525u+1013904223u; int k=(s>>8)%(u+1); std::swap(h[i+u],h[i+k]); } }
    int* d; CK(cudaMalloc(&d,h.size()*4)); CK(cudaMemcpy(d,h.data(),h.size()*4,cudaMemcpyHostToDevice));
    int iters=40;
    for(int U : {4,8,16}){
      for(int rep=0;rep<2;++rep){
        cudaEventRecord(e0);
        if(U==4) k_tmem_rmw<4><<<nsm,128>>>(d,nslots,iters,out); else if(U==8) k_tmem_rmw<8><<<nsm,128>>>(d,nslots,iters,out); else k_tmem_rmw<16><<<nsm,128>>>(d,nslots,iters,out);
        cudaEventRecord(e1); CK(cudaDeviceSynchronize());
      }
      float ms; cudaEventElapsedTime(&ms,e0,e1);
      double adds=(double)nsm*128*nslots*iters;
      printf("TMEM RMW x1 U=%d warps=4: %.3f ms  %.1f Gadd/s  = %.2f adds/clk/SM\n",U,ms,adds/ms/1e6,adds/ms/1e6/nsm/(clk_khz/1e6));
    }
    for(int rep=0;rep<2;++rep){ cudaEventRecord(e0); k_tmem_ld<<<nsm,128>>>(2000,out); cudaEventRecord(e1); CK(cudaDeviceSynchronize()); }
    float ms; cudaEventElapsedTime(&ms,e0,e1);
    double bytes=(double)nsm*128*512*4*2000;
    printf("TMEM ld x32, 4 warps: %.3f ms  %.1f GB/s = %.1f B/clk/SM\n",ms,bytes/ms/1e6,bytes/ms/1e6/nsm/(clk_khz/1e6));
  }
  printf("done\n");
  return 0;
}
