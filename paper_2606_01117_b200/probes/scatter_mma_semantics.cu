// probe3: tf32 MMA with A taken from TMEM (fp32 P as is) and a one-hot B in shared memory: D[i][n] += sum_k P[i][k] * S[n][k]
#include <cstdio>
#include <cstdint>
#include <cstring>
#include <cuda_runtime.h>
#include <vector>
#define CK(x) do{cudaError_t e=(x); if(e!=cudaSuccess){printf("ERR %s line %d\n",cudaGetErrorString(e),__LINE__);exit(1);} }while(0)
__device__ __forceinline__ uint32_t smem_u32(const void* p){return (uint32_t)__cvta_generic_to_shared(p);}
__device__ __forceinline__ uint32_t tld1(uint32_t a){uint32_t v; asm volatile("tcgen05.ld.sync.aligned.32x32b.x1.b32 {%0}, [%1];":"=r"(v):"r"(a):"memory"); return v;}
__device__ __forceinline__ void tst1(uint32_t a, uint32_t v){asm volatile("tcgen05.st.sync.aligned.32x32b.x1.b32 [%0], {%1};"::"r"(a),"r"(v):"memory");}
__device__ __forceinline__ uint64_t sdesc(uint32_t saddr, uint32_t lbo, uint32_t sbo, uint32_t type){
  uint64_t d=0; d|=(uint64_t)((saddr>>4)&0x3FFF); d|=(uint64_t)((lbo>>4)&0x3FFF)<<16; d|=(uint64_t)((sbo>>4)&0x3FFF)<<32; d|=(uint64_t)1<<46; d|=(uint64_t)type<<61; return d;}
// variant: 0: K-major no-swizzle LBO=128 (K), SBO=256 (N) ; 1: swapped ; N = 64, K = 8 tf32
// P at TMEM cols [pcol, pcol+8), D at cols [dcol, dcol+64)
__global__ void __launch_bounds__(128,1) k(int variant, int pcol, int dcol, const int* feat /*8: n index of slot k, or -1*/, float* out /*[128][64]*/, float* pin /*[128][8]*/){
  __shared__ uint32_t slot; __shared__ __align__(1024) float S[64*8*2]; __shared__ uint64_t bar;
  const int tid=threadIdx.x, warp=tid>>5;
  if(warp==0){ asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;"::"r"(smem_u32(&slot)):"memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;":::"memory"); }
  if(tid==0){ asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;"::"r"(smem_u32(&bar)):"memory"); asm volatile("fence.mbarrier_init.release.cluster;":::"memory"); }
  for(int i=tid;i<64*8*2;i+=128) S[i]=0.f;
  __syncthreads();
  // one-hot: element (n,k) of K-major no-swizzle: core (n/8, k/4) of 8 rows x 16 B
  const uint32_t lboK = 128, sboN = 256;
  if(tid<8 && feat[tid]>=0){ int n=feat[tid], kk=tid; S[( (n/8)*sboN + (kk/4)*lboK + (n%8)*16 + (kk%4)*4 )/4] = 1.0f; }
  asm volatile("fence.proxy.async.shared::cta;":::"memory");
  asm volatile("tcgen05.fence::before_thread_sync;":::"memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;":::"memory");
  const uint32_t tb = slot + ((uint32_t)(warp*32)<<16);
  for(int c=0;c<8;++c) tst1(tb+pcol+c, __float_as_uint(pin[tid*8+c]));
  for(int c=0;c<64;++c) tst1(tb+dcol+c, __float_as_uint(1000.f));      // D starts at 1000: accumulate must keep it
  asm volatile("tcgen05.wait::st.sync.aligned;":::"memory");
  asm volatile("tcgen05.fence::before_thread_sync;":::"memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;":::"memory");
  if(warp==0){
    uint32_t e; asm volatile("{\n\t.reg .pred p;\n\telect.sync _|p, 0xffffffff;\n\tselp.u32 %0,1,0,p;\n\t}":"=r"(e));
    if(e){
      const uint32_t idesc = (1u<<4)|(2u<<7)|(2u<<10)|(0u<<15)|(0u<<16)|((64u>>3)<<17)|((128u>>4)<<24);
      uint64_t bd = variant==0 ? sdesc(smem_u32(S), lboK, sboN, 0) : sdesc(smem_u32(S), sboN, lboK, 0);
      uint32_t d = slot + dcol, a = slot + pcol;
      asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, 1, 0;\n\ttcgen05.mma.cta_group::1.kind::tf32 [%0], [%1], %2, %3, p;\n\t}"::"r"(d),"r"(a),"l"(bd),"r"(idesc):"memory");
      asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];"::"r"(smem_u32(&bar)):"memory");
    }
    __syncwarp();
  }
  { uint32_t ok=0; while(!ok){ asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], 0;\n\tselp.u32 %0,1,0,p;\n\t}":"=r"(ok):"r"(smem_u32(&bar)):"memory"); } }
  asm volatile("tcgen05.fence::after_thread_sync;":::"memory");
  for(int c=0;c<64;++c){ uint32_t v=tld1(tb+dcol+c); asm volatile("tcgen05.wait::ld.sync.aligned;":::"memory"); out[tid*64+c]=__uint_as_float(v); }
  asm volatile("tcgen05.fence::before_thread_sync;":::"memory");
  __syncthreads();
  if(warp==0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;"::"r"(slot):"memory");
}
int main(){
  float *out,*pin; int* feat; CK(cudaMalloc(&out,128*64*4)); CK(cudaMalloc(&pin,128*8*4)); CK(cudaMalloc(&feat,32));
  std::vector<float> hp(128*8); for(int i=0;i<128;++i) for(int c=0;c<8;++c) hp[i*8+c]= (float)(i*8+c) + 0.000123f*(c+1);   // not exactly tf32-representable
  CK(cudaMemcpy(pin,hp.data(),hp.size()*4,cudaMemcpyHostToDevice));
  int hf[8]={3,17,17,40,63,-1,0,9};  // duplicates (17 twice) and an empty slot
  CK(cudaMemcpy(feat,hf,32,cudaMemcpyHostToDevice));
  for(int variant=0;variant<2;++variant) for(int pc : {0, 8, 40, 3}) for(int dc : {256, 272, 300}){
    k<<<1,128>>>(variant,pc,dc,feat,out,pin); cudaError_t e=cudaDeviceSynchronize();
    if(e!=cudaSuccess){ printf("variant %d pcol %d dcol %d: CUDA error %s\n",variant,pc,dc,cudaGetErrorString(e)); return 0; }
    std::vector<float> ho(128*64); CK(cudaMemcpy(ho.data(),out,ho.size()*4,cudaMemcpyDeviceToHost));
    double maxerr=0, maxrel=0; int bad=0;
    for(int i=0;i<128;++i) for(int n=0;n<64;++n){ double ref=1000.0; for(int c=0;c<8;++c) if(hf[c]==n) ref+=hp[i*8+c]; double err=fabs(ho[i*64+n]-ref); if(err>maxerr) maxerr=err; if(err>0.6) ++bad; }
    printf("variant %d pcol %d dcol %d: max abs err %.4f  bad %d   sample row5: n3=%.4f (ref %.4f) n17=%.4f (ref %.4f) n1=%.1f\n",variant,pc,dc,maxerr,bad,ho[5*64+3],1000+hp[5*8+0],ho[5*64+17],1000+hp[5*8+1]+hp[5*8+2],ho[5*64+1]);
  }
  return 0;
}
