// probe: do SHFL, REDUX and STS share the LSU pipe with LDS on sm_100a? (profiles/r1_lsu_mix_probe.md)
#include <cstdio>
#include <cstdint>
#include <cuda_runtime.h>
#define CK(x) do{cudaError_t e=(x); if(e!=cudaSuccess){printf("CUDA error %s at %d\n",cudaGetErrorString(e),__LINE__); return 1;}}while(0)
constexpr int kThreads=512, kIters=4096;
__device__ __forceinline__ float2 lds64(uint32_t a){ float2 v; asm volatile("ld.shared.v2.f32 {%0,%1}, [%2];":"=f"(v.x),"=f"(v.y):"r"(a)); return v; }
// MODE bit0: 8 LDS.64, bit1: 8 SHFL.BFLY, bit2: 8 REDUX.OR, bit3: 8 STS.64
template<int MODE>
__global__ void __launch_bounds__(kThreads,1) k(float* out,long long* cyc){
  extern __shared__ float2 sm[];
  for(int i=threadIdx.x;i<8192;i+=blockDim.x) sm[i]=make_float2(i*1e-9f,1e-9f);
  __syncthreads();
  const int lane=threadIdx.x&31, warp=threadIdx.x>>5;
  const uint32_t sbase=(uint32_t)__cvta_generic_to_shared(sm)+lane*8+warp*512;
  float acc=lane*1e-3f; uint32_t u=lane;
  long long t0=clock64();
  #pragma unroll 1
  for(int it=0;it<kIters;++it){
    const uint32_t off=(uint32_t)((it&7)*4096);
    if(MODE&1){
      #pragma unroll
      for(int j=0;j<8;++j){ float2 t=lds64(sbase+off+j*256); acc+=t.x; }
    }
    if(MODE&2){
      #pragma unroll
      for(int j=0;j<8;++j) acc+=__shfl_xor_sync(0xffffffffu,acc,1<<(j&3));
    }
    if(MODE&4){
      #pragma unroll
      for(int j=0;j<8;++j) u+=__reduce_or_sync(0xffffffffu,u+j);
    }
    if(MODE&8){
      #pragma unroll
      for(int j=0;j<8;++j) asm volatile("st.shared.v2.f32 [%0], {%1,%2};"::"r"(sbase+off+j*256),"f"(acc),"f"(acc+1.f):"memory");
    }
  }
  long long t1=clock64();
  out[blockIdx.x*blockDim.x+threadIdx.x]=acc+u;
  if(threadIdx.x==0) cyc[blockIdx.x]=t1-t0;
}
template<int MODE> int run(const char* name,float* out,long long* cyc,int ninstr){
  CK(cudaFuncSetAttribute(k<MODE>,cudaFuncAttributeMaxDynamicSharedMemorySize,65536));
  k<MODE><<<148,kThreads,65536>>>(out,cyc); CK(cudaDeviceSynchronize());
  k<MODE><<<148,kThreads,65536>>>(out,cyc); CK(cudaDeviceSynchronize());
  long long h[148]; CK(cudaMemcpy(h,cyc,sizeof(h),cudaMemcpyDeviceToHost));
  double avg=0; for(int i=0;i<148;++i) avg+=h[i]; avg/=148;
  printf("%-28s %.3f clk per warp-instr per SM (%d instr/iter)\n",name,avg/(kIters*(double)ninstr*16),ninstr);
  return 0;
}
int main(){
  float* out; long long* cyc; CK(cudaMalloc(&out,148*kThreads*4)); CK(cudaMalloc(&cyc,148*8));
  run<1>("LDS.64 x8",out,cyc,8);
  run<2>("SHFL.BFLY x8",out,cyc,8);
  run<3>("LDS.64 x8 + SHFL x8",out,cyc,16);
  run<4>("REDUX.OR x8",out,cyc,8);
  run<5>("LDS.64 x8 + REDUX x8",out,cyc,16);
  run<8>("STS.64 x8",out,cyc,8);
  run<9>("LDS.64 x8 + STS.64 x8",out,cyc,16);
  return 0;
}
