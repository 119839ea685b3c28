// micro-benchmarks: operand-delivery ports of one SM (B200).  Build: nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o probe probe.cu
#include <cstdio>
#include <cstdint>
#include <cuda_runtime.h>
#define CK(x) do{cudaError_t e=(x); if(e!=cudaSuccess){printf("CUDA error %s at %d\n",cudaGetErrorString(e),__LINE__); return 1;}}while(0)

constexpr int kThreads = 512;
constexpr int kIters = 4096;

__device__ __forceinline__ float2 lds64(uint32_t a){ float2 v; asm volatile("ld.shared.v2.f32 {%0,%1}, [%2];":"=f"(v.x),"=f"(v.y):"r"(a)); return v; }
__device__ __forceinline__ void ffma2(float2& d, float2 a, float2 b){
  unsigned long long dd=*reinterpret_cast<unsigned long long*>(&d);
  asm volatile("fma.rn.f32x2 %0, %1, %2, %0;":"+l"(dd):"l"(*reinterpret_cast<unsigned long long*>(&a)),"l"(*reinterpret_cast<unsigned long long*>(&b)));
  d=*reinterpret_cast<float2*>(&dd);
}

// MODE bit0: LDS.64 x8 per iter, bit1: LDG.64 (L1 hit) x8 per iter, bit2: 16 FFMA2 per iter, bit3: tex x8
template<int MODE>
__global__ void __launch_bounds__(kThreads,1) k_mix(const float2* __restrict__ gtab, cudaTextureObject_t tex, float* out, long long* cyc){
  extern __shared__ float2 sm[];
  for(int i=threadIdx.x;i<8192;i+=blockDim.x) sm[i]=make_float2(i*1e-9f,1e-9f);
  __syncthreads();
  const int lane=threadIdx.x&31, warp=threadIdx.x>>5;
  const uint32_t sbase=(uint32_t)__cvta_generic_to_shared(sm)+lane*8+warp*256;
  const float2* g=gtab+lane+warp*32;
  float2 A[8],B[8];
  for(int j=0;j<8;++j){A[j]=make_float2(0,0);B[j]=make_float2(0,0);}
  float2 v=make_float2(1.0f+lane*1e-6f,0.5f);
  long long t0=clock64();
  #pragma unroll 1
  for(int it=0;it<kIters;++it){
    const uint32_t off=(uint32_t)((it&7)*4096);
    float2 t[8];
    #pragma unroll
    for(int j=0;j<8;++j) t[j]=make_float2(1e-9f,1e-9f);
    if(MODE&1){
      #pragma unroll
      for(int j=0;j<8;++j) t[j]=lds64(sbase+off+j*512*0+ ((j*4352)&0xffff)%32768 );
    }
    float2 u[8];
    if(MODE&2){
      #pragma unroll
      for(int j=0;j<8;++j) u[j]=__ldg(g+(((it&3)*8+j)*512));
    }
    if(MODE&8){
      #pragma unroll
      for(int j=0;j<8;++j) u[j]=tex1Dfetch<float2>(tex,(int)(lane+warp*32+(((it&3)*8+j)*512)));
    }
    if(MODE&4){
      #pragma unroll
      for(int j=0;j<8;++j){ ffma2(A[j],t[j],v); ffma2(B[j],t[j],make_float2(v.y,v.y)); }
      if(MODE&10){
        #pragma unroll
        for(int j=0;j<8;++j){ ffma2(A[j],u[j],v); }
      }
    } else {
      #pragma unroll
      for(int j=0;j<8;++j){ A[j].x+=t[j].x; if(MODE&10) A[j].y+=u[j].x; }
    }
  }
  long long t1=clock64();
  float s=0; for(int j=0;j<8;++j) s+=A[j].x+A[j].y+B[j].x+B[j].y;
  out[blockIdx.x*blockDim.x+threadIdx.x]=s;
  if(threadIdx.x==0) cyc[blockIdx.x]=t1-t0;
}

// tcgen05.ld throughput: each warp reads NCOL 32-bit columns per instruction from its quadrant; MIXLDS adds 8 LDS.64 per iter
template<int NREG,int MIXLDS>
__global__ void __launch_bounds__(kThreads,1) k_tmem(float* out,long long* cyc){
  extern __shared__ float2 sm[];
  __shared__ uint32_t tbase_s;
  for(int i=threadIdx.x;i<8192;i+=blockDim.x) sm[i]=make_float2(i*1e-9f,1e-9f);
  const int lane=threadIdx.x&31, warp=threadIdx.x>>5;
  if(warp==0){
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;"::"r"((uint32_t)__cvta_generic_to_shared(&tbase_s)));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
  }
  asm volatile("tcgen05.fence::before_thread_sync;");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;");
  const uint32_t tb=tbase_s+(((uint32_t)(warp&3)*32u)<<16);
  // initialise my quadrant's columns (only warps 0-3 write)
  if(warp<4){
    for(int c=0;c<512;c+=4){
      asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1,%2,%3,%4};"::"r"(tb+c),"r"(__float_as_uint(1e-9f*c)),"r"(__float_as_uint(1e-9f)),"r"(__float_as_uint(2e-9f)),"r"(__float_as_uint(3e-9f)));
    }
    asm volatile("tcgen05.wait::st.sync.aligned;");
  }
  asm volatile("tcgen05.fence::before_thread_sync;");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;");
  const uint32_t sbase=(uint32_t)__cvta_generic_to_shared(sm)+lane*8+warp*256;
  float acc=0.f;
  long long t0=clock64();
  #pragma unroll 1
  for(int it=0;it<kIters;++it){
    const uint32_t col=(uint32_t)((it*16)&255);
    uint32_t r[16];
    if(NREG==16){
      asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
        :"=r"(r[0]),"=r"(r[1]),"=r"(r[2]),"=r"(r[3]),"=r"(r[4]),"=r"(r[5]),"=r"(r[6]),"=r"(r[7]),"=r"(r[8]),"=r"(r[9]),"=r"(r[10]),"=r"(r[11]),"=r"(r[12]),"=r"(r[13]),"=r"(r[14]),"=r"(r[15]):"r"(tb+col));
    } else {
      #pragma unroll
      for(int q=0;q<8;++q)
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x2.b32 {%0,%1}, [%2];":"=r"(r[2*q]),"=r"(r[2*q+1]):"r"(tb+col+2*q+((q*34)&254)));
    }
    float2 t[8];
    if(MIXLDS){
      const uint32_t off=(uint32_t)((it&7)*4096);
      #pragma unroll
      for(int j=0;j<8;++j) t[j]=lds64(sbase+off+(((j*4352)&0xffff)%32768));
    }
    asm volatile("tcgen05.wait::ld.sync.aligned;");
    #pragma unroll
    for(int q=0;q<16;++q) acc+=__uint_as_float(r[q]);
    if(MIXLDS){
      #pragma unroll
      for(int j=0;j<8;++j) acc+=t[j].x;
    }
  }
  long long t1=clock64();
  out[blockIdx.x*blockDim.x+threadIdx.x]=acc;
  if(threadIdx.x==0) cyc[blockIdx.x]=t1-t0;
  asm volatile("tcgen05.fence::before_thread_sync;");
  __syncthreads();
  if(warp==0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;"::"r"(tbase_s));
}

// REDG.v2 flush rate: each warp adds float2 to spread addresses (16 per lane per "flush")
__global__ void __launch_bounds__(kThreads,1) k_red(float2* grid,int N,long long* cyc,int iters){
  const int lane=threadIdx.x&31, warp=threadIdx.x>>5, lx=lane&7, ly=lane>>3;
  long long t0=clock64();
  for(int it=0;it<iters;++it){
    const int strip=(blockIdx.x*16+warp+it*2368)%( (N/16)*(N/32) );
    const int sy=strip/(N/16), sx=strip%(N/16);
    float2* gp=grid+(size_t)(sy*32+ly)*N+sx*16+lx;
    #pragma unroll
    for(int j=0;j<8;++j){ atomicAdd(gp+(size_t)(4*j)*N,make_float2(1.f,1.f)); atomicAdd(gp+(size_t)(4*j)*N+8,make_float2(1.f,1.f)); }
  }
  long long t1=clock64();
  if(threadIdx.x==0) cyc[blockIdx.x]=t1-t0;
}

template<typename F> int run(const char* name,F launch,long long* d_cyc,double ops_per_iter_per_thread,double bytes_per_op,int iters=kIters){
  launch(); CK(cudaDeviceSynchronize());
  cudaEvent_t a,b; cudaEventCreate(&a); cudaEventCreate(&b);
  cudaEventRecord(a); launch(); cudaEventRecord(b); CK(cudaDeviceSynchronize());
  float ms; cudaEventElapsedTime(&ms,a,b);
  long long h[148]; CK(cudaMemcpy(h,d_cyc,sizeof(h),cudaMemcpyDeviceToHost));
  double avg=0; for(int i=0;i<148;++i) avg+=h[i]; avg/=148;
  double ops=ops_per_iter_per_thread*iters*(kThreads/32.0);   // warp-instructions per SM
  printf("%-34s %8.3f ms  %10.0f cyc  %6.3f clk/warp-instr/SM  %7.1f B/clk/SM  (%.0f MHz)\n",name,ms,avg,avg/ops,ops*32*bytes_per_op/avg,avg/ms/1e3);
  return 0;
}

int main(){
  float2* gtab; float* out; long long* cyc; float2* grid;
  CK(cudaMalloc(&gtab,1<<20)); CK(cudaMemset(gtab,0,1<<20));
  CK(cudaMalloc(&out,148*kThreads*4)); CK(cudaMalloc(&cyc,148*8));
  const int N=2048; CK(cudaMalloc(&grid,(size_t)N*N*8)); CK(cudaMemset(grid,0,(size_t)N*N*8));
  cudaResourceDesc rd={}; rd.resType=cudaResourceTypeLinear; rd.res.linear.devPtr=gtab; rd.res.linear.desc=cudaCreateChannelDesc<float2>(); rd.res.linear.sizeInBytes=1<<20;
  cudaTextureDesc td={}; td.readMode=cudaReadModeElementType; cudaTextureObject_t tex; CK(cudaCreateTextureObject(&tex,&rd,&td,nullptr));
  const int smem=65536;
  #define SETSM(k) CK(cudaFuncSetAttribute(k,cudaFuncAttributeMaxDynamicSharedMemorySize,smem))
  SETSM(k_mix<1>); SETSM(k_mix<2>); SETSM(k_mix<3>); SETSM(k_mix<4>); SETSM(k_mix<5>); SETSM(k_mix<7>); SETSM(k_mix<8>); SETSM(k_mix<9>); SETSM(k_mix<13>); SETSM(k_mix<6>);
  run("LDS.64 x8",[&]{k_mix<1><<<148,kThreads,smem>>>(gtab,tex,out,cyc);},cyc,8,8);
  run("LDG.64(L1) x8",[&]{k_mix<2><<<148,kThreads,smem>>>(gtab,tex,out,cyc);},cyc,8,8);
  run("LDS.64 x8 + LDG.64 x8",[&]{k_mix<3><<<148,kThreads,smem>>>(gtab,tex,out,cyc);},cyc,16,8);
  run("FFMA2 x16",[&]{k_mix<4><<<148,kThreads,smem>>>(gtab,tex,out,cyc);},cyc,16,0);
  run("LDS.64 x8 + FFMA2 x16",[&]{k_mix<5><<<148,kThreads,smem>>>(gtab,tex,out,cyc);},cyc,8,8);
  run("LDG x8 + FFMA2 x24",[&]{k_mix<6><<<148,kThreads,smem>>>(gtab,tex,out,cyc);},cyc,8,8);
  run("LDS x8 + LDG x8 + FFMA2 x24",[&]{k_mix<7><<<148,kThreads,smem>>>(gtab,tex,out,cyc);},cyc,16,8);
  run("TEX.64 x8",[&]{k_mix<8><<<148,kThreads,smem>>>(gtab,tex,out,cyc);},cyc,8,8);
  run("LDS.64 x8 + TEX x8",[&]{k_mix<9><<<148,kThreads,smem>>>(gtab,tex,out,cyc);},cyc,16,8);
  run("LDS x8 + TEX x8 + FFMA2 x24",[&]{k_mix<13><<<148,kThreads,smem>>>(gtab,tex,out,cyc);},cyc,16,8);
  SETSM((k_tmem<16,0>)); SETSM((k_tmem<16,1>)); SETSM((k_tmem<2,0>)); SETSM((k_tmem<2,1>));
  run("LDTM 32x32b.x16",[&]{k_tmem<16,0><<<148,kThreads,smem>>>(out,cyc);},cyc,1,64);
  run("LDTM x16 + LDS.64 x8 (bytes both)",[&]{k_tmem<16,1><<<148,kThreads,smem>>>(out,cyc);},cyc,1,128);
  run("LDTM 32x32b.x2 x8",[&]{k_tmem<2,0><<<148,kThreads,smem>>>(out,cyc);},cyc,8,8);
  run("LDTM x2 x8 + LDS.64 x8",[&]{k_tmem<2,1><<<148,kThreads,smem>>>(out,cyc);},cyc,16,8);
  run("REDG.v2 flush (16/lane)",[&]{k_red<<<148,kThreads>>>(grid,N,cyc,256);},cyc,16,8,256);
  printf("done\n");
  return 0;
}
