// probe: tcgen05.ld shapes (thread <-> TMEM lane / column mapping), base-lane alignment, throughput (profiles/r1_tmem_shape_probe.md)
#include <cstdio>
#include <cstdint>
#include <cuda_runtime.h>
#define CK(x) do{cudaError_t e=(x); if(e!=cudaSuccess){printf("CUDA error %s at %d\n",cudaGetErrorString(e),__LINE__); return 1;}}while(0)
constexpr int kThreads=512;
__device__ uint32_t tmem_alloc(uint32_t* slot){
  if((threadIdx.x>>5)==0){
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;"::"r"((uint32_t)__cvta_generic_to_shared(slot)));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
  }
  asm volatile("tcgen05.fence::before_thread_sync;");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;");
  return *slot;
}
__device__ void tmem_free(uint32_t base){
  asm volatile("tcgen05.fence::before_thread_sync;");
  __syncthreads();
  if((threadIdx.x>>5)==0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;"::"r"(base));
}
__device__ void fill(uint32_t tbase){
  const int warp=threadIdx.x>>5, lane=threadIdx.x&31;
  if(warp<4){
    const uint32_t row=tbase+(((uint32_t)warp*32u)<<16);
    const uint32_t m=warp*32+lane;
    for(int c=0;c<512;c+=2)
      asm volatile("tcgen05.st.sync.aligned.32x32b.x2.b32 [%0], {%1,%2};"::"r"(row+c),"r"(m*1000u+c),"r"(m*1000u+c+1));
    asm volatile("tcgen05.wait::st.sync.aligned;");
  }
  asm volatile("tcgen05.fence::before_thread_sync;");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;");
}
// SHAPE 0: 16x256b.x1 (4 regs)  1: 16x128b.x1 (2 regs)  2: 16x64b.x1 (1 reg) 3: 32x32b.x2
template<int SHAPE>
__global__ void k_map(int base_lane,int col,uint32_t* out){
  __shared__ uint32_t slot;
  const uint32_t tb=tmem_alloc(&slot);
  fill(tb);
  const int warp=threadIdx.x>>5, lane=threadIdx.x&31;
  uint32_t r[4]={0xdeadu,0xdeadu,0xdeadu,0xdeadu};
  const uint32_t addr=tb+(((uint32_t)(warp&3)*32u+base_lane)<<16)+col;
  if(SHAPE==0) asm volatile("tcgen05.ld.sync.aligned.16x256b.x1.b32 {%0,%1,%2,%3}, [%4];":"=r"(r[0]),"=r"(r[1]),"=r"(r[2]),"=r"(r[3]):"r"(addr));
  if(SHAPE==1) asm volatile("tcgen05.ld.sync.aligned.16x128b.x1.b32 {%0,%1}, [%2];":"=r"(r[0]),"=r"(r[1]):"r"(addr));
  if(SHAPE==2) asm volatile("tcgen05.ld.sync.aligned.16x64b.x1.b32 {%0}, [%1];":"=r"(r[0]):"r"(addr));
  if(SHAPE==3) asm volatile("tcgen05.ld.sync.aligned.32x32b.x2.b32 {%0,%1}, [%2];":"=r"(r[0]),"=r"(r[1]):"r"(addr));
  asm volatile("tcgen05.wait::ld.sync.aligned;":::"memory");
  if(warp<4) for(int q=0;q<4;++q) out[(warp*32+lane)*4+q]=r[q];
  tmem_free(tb);
}
// throughput: 16x256b.x4 (16 regs), base lane = (it*step)&15 style variation
template<int SHAPE>
__global__ void __launch_bounds__(kThreads,1) k_tp(int lane_step,float* out,long long* cyc,int iters){
  __shared__ uint32_t slot;
  const uint32_t tb=tmem_alloc(&slot);
  fill(tb);
  const int warp=threadIdx.x>>5;
  const uint32_t q0=tb+(((uint32_t)(warp&3)*32u)<<16);
  float acc=0.f;
  long long t0=clock64();
  #pragma unroll 1
  for(int it=0;it<iters;++it){
    const uint32_t col=(uint32_t)((it*32)&255);
    const uint32_t bl=(uint32_t)((it*lane_step)&15);
    const uint32_t addr=q0+(bl<<16)+col;
    uint32_t r[16];
    if(SHAPE==0)
      asm volatile("tcgen05.ld.sync.aligned.16x256b.x4.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
        :"=r"(r[0]),"=r"(r[1]),"=r"(r[2]),"=r"(r[3]),"=r"(r[4]),"=r"(r[5]),"=r"(r[6]),"=r"(r[7]),"=r"(r[8]),"=r"(r[9]),"=r"(r[10]),"=r"(r[11]),"=r"(r[12]),"=r"(r[13]),"=r"(r[14]),"=r"(r[15]):"r"(addr));
    else
      asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
        :"=r"(r[0]),"=r"(r[1]),"=r"(r[2]),"=r"(r[3]),"=r"(r[4]),"=r"(r[5]),"=r"(r[6]),"=r"(r[7]),"=r"(r[8]),"=r"(r[9]),"=r"(r[10]),"=r"(r[11]),"=r"(r[12]),"=r"(r[13]),"=r"(r[14]),"=r"(r[15]):"r"(q0+col));
    asm volatile("tcgen05.wait::ld.sync.aligned;":::"memory");
    #pragma unroll
    for(int q=0;q<16;++q) acc+=__uint_as_float(r[q]);
  }
  long long t1=clock64();
  out[blockIdx.x*blockDim.x+threadIdx.x]=acc;
  if(threadIdx.x==0) cyc[blockIdx.x]=t1-t0;
  tmem_free(tb);
}
template<int SHAPE> int map_test(const char* name,int base_lane,int col,uint32_t* d_out){
  CK(cudaMemset(d_out,0xff,128*4*4));
  k_map<SHAPE><<<1,kThreads>>>(base_lane,col,d_out);
  cudaError_t e=cudaDeviceSynchronize();
  if(e!=cudaSuccess){printf("%s base_lane %d col %d: ERROR %s\n",name,base_lane,col,cudaGetErrorString(e)); return 1;}
  uint32_t h[128*4]; CK(cudaMemcpy(h,d_out,sizeof(h),cudaMemcpyDeviceToHost));
  printf("%s base_lane %d col %d (warp 1: thread -> lane.col per reg):\n",name,base_lane,col);
  for(int t=32;t<64;++t){ printf(" t%02d:",t-32); for(int q=0;q<4;++q){ uint32_t v=h[t*4+q]; if(v==0xdeadu) printf(" ----"); else printf(" %3u.%-3u",v/1000,v%1000);} if((t&3)==3) printf("\n"); }
  return 0;
}
int main(){
  uint32_t* d_out; float* out; long long* cyc;
  CK(cudaMalloc(&d_out,128*4*4)); CK(cudaMalloc(&out,148*kThreads*4)); CK(cudaMalloc(&cyc,148*8));
  // throughput first (legal bases only)
  for(int shape=0;shape<2;++shape){
    for(int step: {0,16}){
      if(shape==1&&step) continue;
      cudaEvent_t a,b; cudaEventCreate(&a); cudaEventCreate(&b);
      const int iters=4096;
      if(shape==0) k_tp<0><<<148,kThreads>>>(step,out,cyc,iters); else k_tp<1><<<148,kThreads>>>(step,out,cyc,iters);
      CK(cudaDeviceSynchronize());
      cudaEventRecord(a);
      if(shape==0) k_tp<0><<<148,kThreads>>>(step,out,cyc,iters); else k_tp<1><<<148,kThreads>>>(step,out,cyc,iters);
      cudaEventRecord(b); CK(cudaDeviceSynchronize());
      float ms; cudaEventElapsedTime(&ms,a,b);
      long long h[148]; CK(cudaMemcpy(h,cyc,sizeof(h),cudaMemcpyDeviceToHost));
      double avg=0; for(int i=0;i<148;++i) avg+=h[i]; avg/=148;
      printf("%s lane_step %d: %.3f ms %.0f cyc  %.1f B/clk/SM\n",shape==0?"16x256b.x4":"32x32b.x16",step,ms,avg,(double)iters*16*32*16*4/avg);
    }
  }
  map_test<3>("32x32b.x2",0,0,d_out);
  map_test<0>("16x256b.x1",0,0,d_out);
  map_test<0>("16x256b.x1",16,8,d_out);
  map_test<1>("16x128b.x1",0,0,d_out);
  map_test<2>("16x64b.x1",0,0,d_out);
  // possibly illegal: unaligned base lanes (each may kill the context; run last)
  if(map_test<0>("16x256b.x1",1,0,d_out)) return 0;
  if(map_test<0>("16x256b.x1",5,2,d_out)) return 0;
  if(map_test<0>("16x256b.x1",13,0,d_out)) return 0;
  if(map_test<0>("16x256b.x1",0,3,d_out)) return 0;
  if(map_test<3>("32x32b.x2",3,0,d_out)) return 0;
  // throughput with rotating base lanes
  {
    k_tp<0><<<148,kThreads>>>(5,out,cyc,4096); CK(cudaDeviceSynchronize());
    long long h[148]; CK(cudaMemcpy(h,cyc,sizeof(h),cudaMemcpyDeviceToHost));
    double avg=0; for(int i=0;i<148;++i) avg+=h[i]; avg/=148;
    printf("16x256b.x4 lane_step 5: %.0f cyc %.1f B/clk/SM\n",avg,(double)4096*16*32*16*4/avg);
  }
  printf("done\n");
  return 0;
}
