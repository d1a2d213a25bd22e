// ubench_peaks.cu -- measured denominators that MEASURED_PEAKS.json does not hold: the FP32 FFMA /
// packed FFMA2 issue rate, HBM read / copy / memset bandwidth, and the L2 hit bandwidth (a buffer that fits the 126 MB
// L2 read / written repeatedly) which bounds the row->column ring of the Fresnel stage.  Standalone binary; its output
// is kept under profiles/.   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o ubench_peaks ubench_peaks.cu
#include <cstdio>
#include <cuda_runtime.h>
#include <cstdint>
#include <cuda.h>
#define CK(x) do{cudaError_t e=(x); if(e!=cudaSuccess){printf("ERR %s line %d\n",cudaGetErrorString(e),__LINE__); return 1;}}while(0)
#define LAUNCH_OK() CK(cudaGetLastError())     /* a launch that failed must not be timed as a success */
template<int NACC>
__global__ void k_ffma(float* out, float a, float b, int iters){
  float acc[NACC];
  #pragma unroll
  for(int i=0;i<NACC;i++) acc[i]=threadIdx.x*0.001f+i;
  for(int it=0; it<iters; ++it){
    #pragma unroll
    for(int i=0;i<NACC;i++) acc[i]=fmaf(acc[i],a,b);
  }
  float s=0; 
  #pragma unroll
  for(int i=0;i<NACC;i++) s+=acc[i];
  out[blockIdx.x*blockDim.x+threadIdx.x]=s;
}
// outer-product style: 8x8 acc, 8 a + 8 b regs (3 distinct regs per FFMA)
__global__ void k_ffma_outer(float* out, const float* in, int iters){
  float acc[8][8]; float a[8], b[8];
  #pragma unroll
  for(int i=0;i<8;i++){a[i]=in[threadIdx.x+i*32]; b[i]=in[threadIdx.x+i*32+256];}
  #pragma unroll
  for(int i=0;i<8;i++)
  #pragma unroll
  for(int j=0;j<8;j++) acc[i][j]=0;
  for(int it=0; it<iters; ++it){
    #pragma unroll
    for(int i=0;i<8;i++)
    #pragma unroll
    for(int j=0;j<8;j++) acc[i][j]=fmaf(a[i],b[j],acc[i][j]);
    #pragma unroll
    for(int i=0;i<8;i++){a[i]+=1e-9f;}
  }
  float s=0;
  #pragma unroll
  for(int i=0;i<8;i++)
  #pragma unroll
  for(int j=0;j<8;j++) s+=acc[i][j];
  out[blockIdx.x*blockDim.x+threadIdx.x]=s;
}
template<int NACC>
__global__ void k_ffma2(float* out, float a, float b, int iters){
  unsigned long long acc[NACC];
  unsigned long long A, B;
  asm("mov.b64 %0, {%1,%2};":"=l"(A):"f"(a),"f"(a));
  asm("mov.b64 %0, {%1,%2};":"=l"(B):"f"(b),"f"(b));
  #pragma unroll
  for(int i=0;i<NACC;i++){ float x=threadIdx.x*0.001f+i; asm("mov.b64 %0, {%1,%2};":"=l"(acc[i]):"f"(x),"f"(x+0.5f)); }
  for(int it=0; it<iters; ++it){
    #pragma unroll
    for(int i=0;i<NACC;i++) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;":"+l"(acc[i]):"l"(A),"l"(B));
  }
  float s=0;
  #pragma unroll
  for(int i=0;i<NACC;i++){ float x,y; asm("mov.b64 {%0,%1}, %2;":"=f"(x),"=f"(y):"l"(acc[i])); s+=x+y; }
  out[blockIdx.x*blockDim.x+threadIdx.x]=s;
}
__global__ void k_read(const uint4* __restrict__ in, size_t n, uint4* out){
  size_t i=(size_t)blockIdx.x*blockDim.x+threadIdx.x; size_t stride=(size_t)gridDim.x*blockDim.x;
  uint4 s=make_uint4(0,0,0,0);
  for(; i+3*stride<n; i+=4*stride){ uint4 a=in[i],b=in[i+stride],c=in[i+2*stride],d=in[i+3*stride]; s.x^=a.x^b.x^c.x^d.x; s.y^=a.y^b.y^c.y^d.y; s.z^=a.z^b.z^c.z^d.z; s.w^=a.w^b.w^c.w^d.w;}
  if(s.x==0x12345678u) out[0]=s;
}
__global__ void k_copy(const uint4* __restrict__ in, uint4* __restrict__ out, size_t n){
  size_t i=(size_t)blockIdx.x*blockDim.x+threadIdx.x; size_t stride=(size_t)gridDim.x*blockDim.x;
  for(; i<n; i+=stride) out[i]=in[i];
}
// the same buffer streamed `reps` times inside ONE launch (no launch gaps): L2 hit bandwidth when it fits L2
__global__ void k_read_loop(const uint4* __restrict__ in, size_t n, int reps, uint4* out){
  size_t stride=(size_t)gridDim.x*blockDim.x;
  uint4 s=make_uint4(0,0,0,0);
  for(int r=0;r<reps;r++){
    size_t i=(size_t)blockIdx.x*blockDim.x+threadIdx.x;
    for(; i+3*stride<n; i+=4*stride){
      uint4 a,b,c,d;
      asm volatile("ld.global.cg.v4.u32 {%0,%1,%2,%3}, [%4];":"=r"(a.x),"=r"(a.y),"=r"(a.z),"=r"(a.w):"l"(in+i));
      asm volatile("ld.global.cg.v4.u32 {%0,%1,%2,%3}, [%4];":"=r"(b.x),"=r"(b.y),"=r"(b.z),"=r"(b.w):"l"(in+i+stride));
      asm volatile("ld.global.cg.v4.u32 {%0,%1,%2,%3}, [%4];":"=r"(c.x),"=r"(c.y),"=r"(c.z),"=r"(c.w):"l"(in+i+2*stride));
      asm volatile("ld.global.cg.v4.u32 {%0,%1,%2,%3}, [%4];":"=r"(d.x),"=r"(d.y),"=r"(d.z),"=r"(d.w):"l"(in+i+3*stride));
      s.x^=a.x^b.x^c.x^d.x; s.y^=a.y^b.y^c.y^d.y; s.z^=a.z^b.z^c.z^d.z; s.w^=a.w^b.w^c.w^d.w;}
  }
  if(s.x==0x12345678u) out[0]=s;
}
__global__ void k_copy_loop(const uint4* __restrict__ in, uint4* __restrict__ out, size_t n, int reps){
  size_t stride=(size_t)gridDim.x*blockDim.x;
  for(int r=0;r<reps;r++)
    for(size_t i=(size_t)blockIdx.x*blockDim.x+threadIdx.x; i<n; i+=stride){
      uint4 a; asm volatile("ld.global.cg.v4.u32 {%0,%1,%2,%3}, [%4];":"=r"(a.x),"=r"(a.y),"=r"(a.z),"=r"(a.w):"l"(in+i));
      a.x+=r; out[i]=a; }
}
// ---- TMA throughput versus box row width: every CTA streams [rows x rowbytes] boxes (16 KB each, 4 in flight) of an
// L2-resident tensor into shared memory (and back out with TMA stores when `store` is set)
__device__ __forceinline__ uint32_t s_u32(const void* p){ return (uint32_t)__cvta_generic_to_shared(p); }
__global__ void k_tma_rows(const __grid_constant__ CUtensorMap tm, int box_rows, int cols_boxes, int rows_boxes, int iters, int store){
  extern __shared__ __align__(1024) unsigned char sm[];
  uint64_t* bar = reinterpret_cast<uint64_t*>(sm + 4*16384);
  if(threadIdx.x==0){ for(int s=0;s<4;s++){ asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;"::"r"(s_u32(bar+s))); } asm volatile("fence.mbarrier_init.release.cluster;":::"memory"); }
  __syncthreads();
  if(threadIdx.x!=0) return;
  const int nboxes = cols_boxes*rows_boxes;
  uint32_t ph[4]={0,0,0,0};
  int issued=0, done=0; const int total=iters;
  int b = blockIdx.x*37 % nboxes;
  auto issue=[&](int s){
    const int cb=b%cols_boxes, rb=b/cols_boxes; b+=gridDim.x; if(b>=nboxes) b-=nboxes;
    if(store){ asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.bulk_group [%0, {%1, %2}], [%3];"::"l"(&tm),"r"(cb*(16384/box_rows/4)),"r"(rb*box_rows),"r"(s_u32(sm+s*16384)):"memory"); asm volatile("cp.async.bulk.commit_group;":::"memory"); }
    else { asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;"::"r"(s_u32(bar+s)),"r"(16384):"memory");
      asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"::"r"(s_u32(sm+s*16384)),"l"(&tm),"r"(cb*(16384/box_rows/4)),"r"(rb*box_rows),"r"(s_u32(bar+s)):"memory"); }
  };
  for(;issued<4 && issued<total;issued++) issue(issued);
  while(done<total){
    const int s=done&3;
    if(store){ asm volatile("cp.async.bulk.wait_group.read 3;":::"memory"); }
    else { uint32_t ok; do{ asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}":"=r"(ok):"r"(s_u32(bar+s)),"r"(ph[s]):"memory"); }while(!ok); ph[s]^=1; }
    done++;
    if(issued<total){ issue(s); issued++; }
  }
  if(store) asm volatile("cp.async.bulk.wait_group 0;":::"memory");
}
typedef CUresult (*EncFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
int main(){
  int sms; cudaDeviceGetAttribute(&sms,cudaDevAttrMultiProcessorCount,0);
  float* out; CK(cudaMalloc(&out, 148*8*1024*4)); float* in; CK(cudaMalloc(&in,4096*4)); CK(cudaMemset(in,0,4096*4));
  cudaEvent_t e0,e1; cudaEventCreate(&e0); cudaEventCreate(&e1); float ms;
  int iters=20000;
  for(int thr: {256,512,1024}) for(int bps: {1,2,4}){
    if(thr*bps>2048) continue;
    k_ffma<16><<<sms*bps,thr>>>(out,1.0001f,0.5f,100); LAUNCH_OK(); cudaDeviceSynchronize();
    cudaEventRecord(e0); k_ffma<16><<<sms*bps,thr>>>(out,1.0001f,0.5f,iters); LAUNCH_OK(); cudaEventRecord(e1); CK(cudaEventSynchronize(e1)); cudaEventElapsedTime(&ms,e0,e1);
    printf("FFMA  thr=%4d bps=%d: %.2f TFLOPS\n",thr,bps, 2.0*16*iters*(double)sms*bps*thr/ms/1e9);
    if(thr>512) continue;      // k_ffma2<16> holds 34 register pairs: more than 64 registers per thread, no 1024-thread launch
    k_ffma2<16><<<sms*bps,thr>>>(out,1.0001f,0.5f,100); LAUNCH_OK(); cudaDeviceSynchronize();
    cudaEventRecord(e0); k_ffma2<16><<<sms*bps,thr>>>(out,1.0001f,0.5f,iters); LAUNCH_OK(); cudaEventRecord(e1); CK(cudaEventSynchronize(e1)); cudaEventElapsedTime(&ms,e0,e1);
    printf("FFMA2 thr=%4d bps=%d: %.2f TFLOPS\n",thr,bps, 4.0*16*iters*(double)sms*bps*thr/ms/1e9);
  }
  for(int thr: {128,256,320}){
    k_ffma_outer<<<sms,thr>>>(out,in,100); LAUNCH_OK(); cudaDeviceSynchronize();
    cudaEventRecord(e0); k_ffma_outer<<<sms,thr>>>(out,in,iters); LAUNCH_OK(); cudaEventRecord(e1); CK(cudaEventSynchronize(e1)); cudaEventElapsedTime(&ms,e0,e1);
    printf("FFMA outer8x8 thr=%d: %.2f TFLOPS\n",thr, 2.0*64*iters*(double)sms*thr/ms/1e9);
  }
  size_t bytes=(size_t)4<<30; uint4 *a,*b; CK(cudaMalloc(&a,bytes)); CK(cudaMalloc(&b,bytes)); CK(cudaMemset(a,1,bytes)); CK(cudaMemset(b,0,bytes));
  size_t n=bytes/16;
  for(int rep=0;rep<3;rep++){
    cudaEventRecord(e0); k_read<<<sms*8,512>>>(a,n,b); cudaEventRecord(e1); CK(cudaEventSynchronize(e1)); cudaEventElapsedTime(&ms,e0,e1);
    printf("read  4GiB: %.1f GB/s\n", bytes/ms/1e6);
    cudaEventRecord(e0); k_copy<<<sms*8,512>>>(a,b,n); cudaEventRecord(e1); CK(cudaEventSynchronize(e1)); cudaEventElapsedTime(&ms,e0,e1);
    printf("copy  4GiB: %.1f GB/s (r+w)\n", 2.0*bytes/ms/1e6);
    cudaEventRecord(e0); cudaMemsetAsync(b,0,bytes); cudaEventRecord(e1); CK(cudaEventSynchronize(e1)); cudaEventElapsedTime(&ms,e0,e1);
    printf("memset 4GiB: %.1f GB/s\n", bytes/ms/1e6);
  }
  // ---- L2 hit bandwidth: a 32 MiB / 64 MiB buffer (fits the 126 MB L2) streamed repeatedly
  for(size_t mb: {32, 64}){
    size_t nb=mb<<20, m=nb/16; int reps=40;
    k_read<<<sms*8,512>>>(a,m,b); LAUNCH_OK(); cudaDeviceSynchronize();
    cudaEventRecord(e0); for(int r=0;r<reps;r++) k_read<<<sms*8,512>>>(a,m,b); LAUNCH_OK(); cudaEventRecord(e1); CK(cudaEventSynchronize(e1)); cudaEventElapsedTime(&ms,e0,e1);
    printf("L2 read  %zu MiB x%d: %.1f GB/s\n", mb, reps, (double)nb*reps/ms/1e6);
    k_copy<<<sms*8,512>>>(a,a+m,m); LAUNCH_OK(); cudaDeviceSynchronize();
    cudaEventRecord(e0); for(int r=0;r<reps;r++) k_copy<<<sms*8,512>>>(a,a+m,m); LAUNCH_OK(); cudaEventRecord(e1); CK(cudaEventSynchronize(e1)); cudaEventElapsedTime(&ms,e0,e1);
    printf("L2 copy  %zu MiB -> %zu MiB x%d: %.1f GB/s (r+w)\n", mb, mb, reps, 2.0*nb*reps/ms/1e6);
  }
  for(size_t mb: {16, 32, 48}){
    size_t nb=mb<<20, m=nb/16; int reps=100;
    k_read_loop<<<sms*4,512>>>(a,m,2,b); LAUNCH_OK(); cudaDeviceSynchronize();
    cudaEventRecord(e0); k_read_loop<<<sms*4,512>>>(a,m,reps,b); LAUNCH_OK(); cudaEventRecord(e1); CK(cudaEventSynchronize(e1)); cudaEventElapsedTime(&ms,e0,e1);
    printf("L2 read loop  %zu MiB x%d in one launch: %.1f GB/s\n", mb, reps, (double)nb*reps/ms/1e6);
    k_copy_loop<<<sms*4,512>>>(a,a+m,m,2); LAUNCH_OK(); cudaDeviceSynchronize();
    cudaEventRecord(e0); k_copy_loop<<<sms*4,512>>>(a,a+m,m,reps); LAUNCH_OK(); cudaEventRecord(e1); CK(cudaEventSynchronize(e1)); cudaEventElapsedTime(&ms,e0,e1);
    printf("L2 copy loop  %zu MiB -> %zu MiB x%d in one launch: %.1f GB/s (r+w)\n", mb, mb, reps, 2.0*nb*reps/ms/1e6);
  }
  {
    void* fn=nullptr; cudaDriverEntryPointQueryResult q; CK(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled",&fn,cudaEnableDefault,&q)); EncFn enc=(EncFn)fn;
    CK(cudaFuncSetAttribute(k_tma_rows, cudaFuncAttributeMaxDynamicSharedMemorySize, 4*16384+64));
    const int W=2048;                          // floats per tensor row (8 KB), 6144 rows = 48 MiB: fits L2
    const int ROWS=6144;
    for(int store=0; store<2; store++) for(int rowbytes: {32,64,128,256,1024}){
      const int box_rows=16384/rowbytes; if(box_rows>256) continue;
      alignas(64) CUtensorMap tm; cuuint64_t gd[2]={(cuuint64_t)W,(cuuint64_t)ROWS}, gs[1]={(cuuint64_t)W*4}; cuuint32_t bx[2]={(cuuint32_t)(rowbytes/4),(cuuint32_t)box_rows}, es[2]={1,1};
      if(enc(&tm,CU_TENSOR_MAP_DATA_TYPE_FLOAT32,2,a,gd,gs,bx,es,CU_TENSOR_MAP_INTERLEAVE_NONE,CU_TENSOR_MAP_SWIZZLE_NONE,CU_TENSOR_MAP_L2_PROMOTION_NONE,CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE)!=CUDA_SUCCESS){ printf("encode failed\n"); continue; }
      const int iters=2000;
      k_tma_rows<<<sms,32,4*16384+64>>>(tm,box_rows,W*4/rowbytes,ROWS/box_rows,200,store); LAUNCH_OK(); CK(cudaDeviceSynchronize());
      cudaEventRecord(e0); k_tma_rows<<<sms,32,4*16384+64>>>(tm,box_rows,W*4/rowbytes,ROWS/box_rows,iters,store); LAUNCH_OK(); cudaEventRecord(e1); CK(cudaEventSynchronize(e1)); cudaEventElapsedTime(&ms,e0,e1);
      printf("TMA %s box [%3d rows x %4d B] (16 KB, 4 in flight per SM, L2-resident 48 MiB): %.1f GB/s, %.0f ns per box per SM\n", store?"store":"load ", box_rows, rowbytes, 16384.0*iters*sms/ms/1e6, ms*1e6/iters);
    }
  }
  return 0;
}
