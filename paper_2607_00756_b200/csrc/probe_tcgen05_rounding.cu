// Probe: how does tcgen05.mma kind::tf32 round when accumulating into an fp32 TMEM accumulator?
#include <cstdio>
#include <cstdint>
#include <cmath>
#include <cuda_runtime.h>
constexpr int TM=128, TN=256;
__device__ __forceinline__ uint32_t smem_u32(const void* p){ return (uint32_t)__cvta_generic_to_shared(p);}
__device__ __forceinline__ uint64_t umma_desc(uint32_t saddr){ uint64_t d=0; d|=(uint64_t)((saddr&0x3FFFF)>>4); d|=(uint64_t)1<<16; d|=(uint64_t)(512>>4)<<32; d|=(uint64_t)1<<46; d|=(uint64_t)4<<61; return d;}
__device__ __forceinline__ void umma_tf32(uint32_t t, uint64_t da, uint64_t db, uint32_t idesc, uint32_t acc){
  asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\ttcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t}"::"r"(t),"l"(da),"l"(db),"r"(idesc),"r"(acc):"memory");}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity){ uint32_t done=0; while(!done){ asm volatile("{\n\t.reg .pred P1;\n\tmbarrier.try_wait.parity.shared::cta.b64 P1, [%1], %2;\n\tselp.b32 %0, 1, 0, P1;\n\t}":"=r"(done):"r"(smem_u32(bar)),"r"(parity):"memory");}}
// element (row r, k) byte offset in a K-major SWIZZLE_64B tile (64-byte rows)
__device__ __forceinline__ int sw64(int r, int k){ int chunk=(k*4)/16; int phys=chunk ^ ((r>>1)&3); return r*64 + phys*16 + (k*4)%16; }
// out[step][col] = accumulator of row 0 after each step
__global__ void probe(const float* __restrict__ bvals, int nsteps, float* out){
  extern __shared__ uint8_t raw[];
  uint8_t* sm=(uint8_t*)(((uintptr_t)raw+1023)&~(uintptr_t)1023);
  uint8_t* A=sm; uint8_t* B=sm+8192; uint64_t* bar=(uint64_t*)(sm+8192+16384); uint32_t* slot=(uint32_t*)(bar+1);
  int warp=threadIdx.x>>5, lane=threadIdx.x&31;
  if(threadIdx.x==0){ asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;"::"r"(smem_u32(bar))); asm volatile("fence.mbarrier_init.release.cluster;":::"memory"); }
  if(warp==0){ asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;"::"r"(smem_u32(slot)):"memory"); asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;":::"memory"); }
  asm volatile("tcgen05.fence::before_thread_sync;":::"memory"); __syncthreads(); asm volatile("tcgen05.fence::after_thread_sync;":::"memory");
  uint32_t tm=*slot;
  uint32_t idesc=(1u<<4)|(2u<<7)|(2u<<10)|((uint32_t)(TN>>3)<<17)|((uint32_t)(TM>>4)<<24);
  for(int step=0; step<nsteps; ++step){
    // A: every row = [1,1,0,0,0,0,0,0 ...]; B[n][k] = bvals[step][n][k] for k<8
    for(int i=threadIdx.x;i<8192/4;i+=blockDim.x) ((float*)A)[i]=0.f;
    for(int i=threadIdx.x;i<16384/4;i+=blockDim.x) ((float*)B)[i]=0.f;
    __syncthreads();
    for(int r=threadIdx.x;r<TM;r+=blockDim.x){ for(int k=0;k<8;++k) *(float*)(A+sw64(r,k))=1.f; }
    for(int n=threadIdx.x;n<TN;n+=blockDim.x){ for(int k=0;k<8;++k) *(float*)(B+sw64(n,k))=bvals[(step*TN+n)*8+k]; }
    asm volatile("fence.proxy.async.shared::cta;":::"memory");
    __syncthreads();
    if(threadIdx.x==0){
      asm volatile("tcgen05.fence::after_thread_sync;":::"memory");
      umma_tf32(tm, umma_desc(smem_u32(A)), umma_desc(smem_u32(B)), idesc, step?1u:0u);
      asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];"::"r"(smem_u32(bar)):"memory");
    }
    mbar_wait(bar, step&1);
    asm volatile("tcgen05.fence::after_thread_sync;":::"memory");
    if(warp==0){
      for(int c0=0;c0<TN;c0+=32){
        uint32_t v[32];
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
          : "=r"(v[0]),"=r"(v[1]),"=r"(v[2]),"=r"(v[3]),"=r"(v[4]),"=r"(v[5]),"=r"(v[6]),"=r"(v[7]),"=r"(v[8]),"=r"(v[9]),"=r"(v[10]),"=r"(v[11]),"=r"(v[12]),"=r"(v[13]),"=r"(v[14]),"=r"(v[15]),"=r"(v[16]),"=r"(v[17]),"=r"(v[18]),"=r"(v[19]),"=r"(v[20]),"=r"(v[21]),"=r"(v[22]),"=r"(v[23]),"=r"(v[24]),"=r"(v[25]),"=r"(v[26]),"=r"(v[27]),"=r"(v[28]),"=r"(v[29]),"=r"(v[30]),"=r"(v[31]) : "r"(tm+c0));
        asm volatile("tcgen05.wait::ld.sync.aligned;":::"memory");
        if(lane==0) for(int j=0;j<32;++j) out[step*TN+c0+j]=__uint_as_float(v[j]);
      }
    }
    asm volatile("tcgen05.fence::before_thread_sync;":::"memory");
    __syncthreads();
  }
  if(warp==0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;"::"r"(tm):"memory");
}
int main(){
  const int nsteps=3;
  float* h=(float*)calloc(nsteps*TN*8,sizeof(float));
  const float ulp=ldexpf(1.f,-23);   // ulp of values in [1,2)
  // step 0: acc = base (col-dependent sign): base=+1.5 for cols<128, -1.5 for cols>=128
  for(int n=0;n<TN;++n) h[(0*TN+n)*8+0]= n<128? 1.5f:-1.5f;
  // step 1: single addend x in slot 0 = f*ulp, f from list (exact in tf32: small mantissa)
  const float fr[16]={0.25f,0.5f,0.75f,1.25f,-0.25f,-0.5f,-0.75f,-1.25f, 1.5f,-1.5f,0.125f,-0.125f,0.375f,-0.375f, 1.75f,-1.75f};
  for(int n=0;n<TN;++n){ int t=n%128;
    if(t<16) h[(1*TN+n)*8+0]=fr[t]*ulp;
    else if(t<32){ // two addends in slots 0,1 each f*ulp  (sum 2f ulp)
      h[(1*TN+n)*8+0]=fr[t-16]*ulp; h[(1*TN+n)*8+1]=fr[t-16]*ulp; }
    else if(t<48){ // eight addends each f/4 ulp (sum 2f ulp)
      for(int k=0;k<8;++k) h[(1*TN+n)*8+k]=fr[t-32]*0.25f*ulp; }
    else if(t<64){ // cancelling pair: +1 and -1 plus f ulp  (tests internal width)
      h[(1*TN+n)*8+0]=1.0f; h[(1*TN+n)*8+1]=-1.0f; h[(1*TN+n)*8+2]=fr[t-48]*ulp; }
  }
  // step 2: repeat step-1 pattern of case 0 (accumulate again)
  for(int n=0;n<TN;++n){ int t=n%128; if(t<16) h[(2*TN+n)*8+0]=fr[t]*ulp; }
  float *d,*o; cudaMalloc(&d,nsteps*TN*8*4); cudaMalloc(&o,nsteps*TN*4); cudaMemcpy(d,h,nsteps*TN*8*4,cudaMemcpyHostToDevice);
  cudaFuncSetAttribute(probe,cudaFuncAttributeMaxDynamicSharedMemorySize,40000);
  probe<<<1,128,40000>>>(d,nsteps,o); cudaError_t e=cudaDeviceSynchronize(); printf("status %s\n",cudaGetErrorString(e));
  float* r=(float*)malloc(nsteps*TN*4); cudaMemcpy(r,o,nsteps*TN*4,cudaMemcpyDeviceToHost);
  const char* names[4]={"1 addend f","2 addends f each","8 addends f/4 each","(+1,-1,f)"};
  for(int half=0;half<2;++half){ float base=half?-1.5f:1.5f; printf("== base %+.1f ==\n",base);
    for(int c=0;c<4;++c){ printf("%s:\n",names[c]); for(int t=0;t<16;++t){ int n=half*128+c*16+t; float exact=(c==0?fr[t]:c==3?fr[t]:2*fr[t]);
      printf("  f=%+.3f exact %+.3f ulp -> got %+.2f ulp (step2: %+.2f)\n",fr[t],exact,(r[1*TN+n]-base)/ulp,(r[2*TN+n]-base)/ulp);} } }
  return 0; }
