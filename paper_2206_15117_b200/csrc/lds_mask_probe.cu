// probe: cost of shared-memory loads on sm_100a versus width, lane mask and address pattern (profiles/r1_lds_mask_probe.md)
#include <cstdio>
#include <cstdint>
#include <cuda_runtime.h>
#define CK(x) do{cudaError_t e=(x); if(e!=cudaSuccess){printf("CUDA error %s at %d\n",cudaGetErrorString(e),__LINE__); return 1;}}while(0)
constexpr int kThreads=512, kIters=4096;
__device__ __forceinline__ float2 lds64p(uint32_t a,bool p){ float2 v=make_float2(0.f,0.f); asm volatile("{.reg .pred q; setp.ne.b32 q,%3,0; @q ld.shared.v2.f32 {%0,%1}, [%2];}":"+f"(v.x),"+f"(v.y):"r"(a),"r"((int)p)); return v; }
__device__ __forceinline__ float lds32p(uint32_t a,bool p){ float v=0.f; asm volatile("{.reg .pred q; setp.ne.b32 q,%2,0; @q ld.shared.f32 %0, [%1];}":"+f"(v):"r"(a),"r"((int)p)); return v; }
__device__ __forceinline__ float4 lds128p(uint32_t a,bool p){ float4 v=make_float4(0,0,0,0); asm volatile("{.reg .pred q; setp.ne.b32 q,%5,0; @q ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];}":"+f"(v.x),"+f"(v.y),"+f"(v.z),"+f"(v.w):"r"(a),"r"((int)p)); return v; }
// MODE: lane mask pattern; W: 0 = LDS.64, 1 = LDS.32, 2 = LDS.128 ; BC: broadcast (all lanes same address)
template<int W>
__global__ void __launch_bounds__(kThreads,1) k(uint32_t mask,int bc,float* out,long long* cyc){
  extern __shared__ float2 sm[];
  for(int i=threadIdx.x;i<8192;i+=blockDim.x) sm[i]=make_float2(i*1e-9f,1e-9f);
  __syncthreads();
  const int lane=threadIdx.x&31, warp=threadIdx.x>>5;
  const bool p=(mask>>lane)&1;
  const int esz=(W==0)?8:(W==1)?4:16;
  const uint32_t sbase=(uint32_t)__cvta_generic_to_shared(sm)+(bc==0?lane*esz:bc==2?(lane>>4)*272:bc==3?(lane>>3)*272:0)+warp*512;
  float acc=0.f;
  long long t0=clock64();
  #pragma unroll 1
  for(int it=0;it<kIters;++it){
    const uint32_t off=(uint32_t)((it&7)*4096);
    #pragma unroll
    for(int j=0;j<8;++j){
      if(W==0){ float2 t=lds64p(sbase+off+j*512*(bc?0:1)+(bc?j*16:0),p); acc+=t.x+t.y; }
      if(W==1){ acc+=lds32p(sbase+off+j*256*(bc?0:1)+(bc?j*16:0),p); }
      if(W==2){ float4 t=lds128p(sbase+off+(j&3)*1024*(bc?0:1)+(bc?j*16:0),p); acc+=t.x+t.w; }
    }
  }
  long long t1=clock64();
  out[blockIdx.x*blockDim.x+threadIdx.x]=acc;
  if(threadIdx.x==0) cyc[blockIdx.x]=t1-t0;
}
int main(){
  float* out; long long* cyc; CK(cudaMalloc(&out,148*kThreads*4)); CK(cudaMalloc(&cyc,148*8));
  const int smem=65536;
  CK(cudaFuncSetAttribute(k<0>,cudaFuncAttributeMaxDynamicSharedMemorySize,smem));
  CK(cudaFuncSetAttribute(k<1>,cudaFuncAttributeMaxDynamicSharedMemorySize,smem));
  CK(cudaFuncSetAttribute(k<2>,cudaFuncAttributeMaxDynamicSharedMemorySize,smem));
  struct {const char* n; uint32_t m;} masks[]={{"all",0xffffffffu},{"lanes0-15",0x0000ffffu},{"lanes16-31",0xffff0000u},{"even",0x55555555u},{"lanes0-7",0xffu},{"0-7,16-23",0x00ff00ffu},{"0-3 of each 8",0x0f0f0f0fu},{"lanes0-23",0x00ffffffu},{"lane0",1u}};
  for(int w=0;w<3;++w) for(int bc=0;bc<4;++bc) for(auto& mk:masks){
    if(bc>=2 && mk.m!=0xffffffffu) continue;
    auto launch=[&]{ if(w==0) k<0><<<148,kThreads,smem>>>(mk.m,bc,out,cyc); else if(w==1) k<1><<<148,kThreads,smem>>>(mk.m,bc,out,cyc); else k<2><<<148,kThreads,smem>>>(mk.m,bc,out,cyc); };
    launch(); CK(cudaDeviceSynchronize()); launch(); CK(cudaDeviceSynchronize());
    long long h[148]; CK(cudaMemcpy(h,cyc,sizeof(h),cudaMemcpyDeviceToHost));
    double avg=0; for(int i=0;i<148;++i) avg+=h[i]; avg/=148;
    printf("%s %s mask %-14s: %.3f clk/warp-instr/SM\n",w==0?"LDS.64 ":w==1?"LDS.32 ":"LDS.128",bc==0?"linear":bc==1?"bcast ":bc==2?"2 addr":"4 addr",mk.n,avg/(kIters*8.0*16));
  }
  return 0;
}
