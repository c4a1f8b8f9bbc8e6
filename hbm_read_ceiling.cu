// =============================================================================
// hbm_read_ceiling.cu -- standalone probe: the READ-ONLY HBM ceiling of this GPU for the access
// patterns a tile-wise streaming reduction can use (build step 5).  No arithmetic:
// one thread per CTA issues TMA loads into a ring of shared-memory boxes, a second thread waits for
// each box and hands it straight back.  Sweeps the box shape (2-D 128x32, 256x16, 256x32, 128x16,
// 64x64, 256x8 fp32 boxes of an 8192-wide image; 1-D 16 KiB bulk copies), the ring depth and the
// CTAs per SM, i.e. the bytes in flight per SM, and prints one line per point plus "best".
// Result on B200 (profiles/r01f_read_ceiling.md): 7.30-7.34 TB/s for EVERY shape once 96-128 KiB
// are in flight per SM; 64 KiB gives 6.9, 192 KiB 7.16.  Not part of libiqa_tiles.so.
// Usage: hbm_read_ceiling [image width, default 8192]
// Build: nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o hbm_read_ceiling hbm_read_ceiling.cu
// =============================================================================
#include <cuda.h>
#include <cuda_runtime.h>
#include <cstdio>
#include <cstdlib>
#include <cstdint>
__device__ __forceinline__ uint32_t sa(const void* p){return (uint32_t)__cvta_generic_to_shared(p);}
__device__ __forceinline__ void mwait(uint32_t bar, uint32_t par){
  asm volatile("{\n.reg .pred p;\nW_%=:\nmbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1, %2;\n@p bra D_%=;\nbra W_%=;\nD_%=:\n}\n"::"r"(bar),"r"(par),"r"(0x989680u):"memory");}
struct P { CUtensorMap map; const float* src; int N; int units_x; long long n_items; int bw, bh; int mode; int nb; };
__global__ void __launch_bounds__(64) k(const __grid_constant__ P p){
  extern __shared__ unsigned char sm[];
  unsigned char* base = sm + ((1024u - (sa(sm)&1023u))&1023u);
  const uint32_t box_bytes = p.bw*p.bh*4;
  uint32_t full = sa(base + (size_t)p.nb*box_bytes), empty = full + 8*p.nb;
  if(threadIdx.x==0){ for(int i=0;i<p.nb;i++){ asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;"::"r"(full+8*i)); asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;"::"r"(empty+8*i)); }
    asm volatile("fence.mbarrier_init.release.cluster;":::"memory"); }
  __syncthreads();
  int w = threadIdx.x>>5, lane = threadIdx.x&31;
  if(lane) return;
  int slot=0; uint32_t ph=0;
  if(w==0){
    for(long long it=blockIdx.x; it<p.n_items; it+=gridDim.x){
      mwait(empty+8*slot, ph^1);
      asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;"::"r"(full+8*slot),"r"(box_bytes):"memory");
      uint32_t dst = sa(base)+slot*box_bytes;
      if(p.mode==2){
        const char* s = (const char*)p.src + it*(long long)box_bytes;
        asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"::"r"(dst),"l"(s),"r"(box_bytes),"r"(full+8*slot):"memory");
      } else {
        int ux = (int)(it % p.units_x), uy = (int)(it / p.units_x);
        asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"::"r"(dst),"l"(&p.map),"r"(ux*p.bw),"r"(uy*p.bh),"r"(full+8*slot):"memory");
      }
      if(++slot==p.nb){slot=0;ph^=1;}
    }
  } else {
    for(long long it=blockIdx.x; it<p.n_items; it+=gridDim.x){
      mwait(full+8*slot, ph);
      asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];"::"r"(empty+8*slot):"memory");
      if(++slot==p.nb){slot=0;ph^=1;}
    }
  }
}
typedef CUresult (*Enc)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
int main(int argc, char** argv){
  // image width N (default 8192; argv[1]) and as many rows as make 2 GiB
  int N = argc > 1 ? atoi(argv[1]) : 8192; if (N < 256 || N % 256) { printf("N must be a multiple of 256\n"); return 1; }
  int rows_total = (int)((2ll << 30) / 4 / N);
  float* d; cudaMalloc(&d, (size_t)N*rows_total*4); cudaMemset(d, 0, (size_t)N*rows_total*4);
  void* f; cudaDriverEntryPointQueryResult q; cudaGetDriverEntryPoint("cuTensorMapEncodeTiled",&f,cudaEnableDefault,&q); Enc enc=(Enc)f;
  int modes[][3] = {{0,128,32},{1,256,16},{2,128,32},{3,256,32},{4,128,16},{5,64,64},{6,256,8}};
  double best=0; char best_desc[256]="";
  for(int promo=0;promo<1;promo+=3) for(auto& m: modes) for(int nb: {2,3,4,6}) for(int cps: {1,2,3,4}){
    P p; p.src=d; p.N=N; p.bw=m[1]; p.bh=m[2]; p.mode = m[0]==2?2:0; p.nb=nb;
    if (p.mode==2 && promo) continue;
    cuuint64_t dims[2]={(cuuint64_t)N,(cuuint64_t)rows_total}; cuuint64_t str[1]={(cuuint64_t)N*4}; cuuint32_t box[2]={(cuuint32_t)p.bw,(cuuint32_t)p.bh}; cuuint32_t es[2]={1,1};
    if(enc(&p.map,CU_TENSOR_MAP_DATA_TYPE_FLOAT32,2,d,dims,str,box,es,CU_TENSOR_MAP_INTERLEAVE_NONE,CU_TENSOR_MAP_SWIZZLE_NONE,(CUtensorMapL2promotion)promo,CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE)!=CUDA_SUCCESS){printf("enc fail\n");continue;}
    p.units_x = N/p.bw; p.n_items = (long long)p.units_x*(rows_total/p.bh);
    size_t smem = 1024 + (size_t)nb*p.bw*p.bh*4 + 16*nb;
    if (smem*cps > 220*1024) continue;
    cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    int grid = 148*cps;
    cudaEvent_t e0,e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    k<<<grid,64,smem>>>(p); cudaDeviceSynchronize();
    cudaEventRecord(e0); for(int i=0;i<5;i++) k<<<grid,64,smem>>>(p); cudaEventRecord(e1); cudaDeviceSynchronize();
    float ms; cudaEventElapsedTime(&ms,e0,e1); 
    double tb = (double)N*rows_total*4*5/ (ms*1e-3)/1e12;
    char desc[256]; snprintf(desc, sizeof desc, "%s box=%dx%d ring=%d ctas/sm=%d inflight/SM=%dKiB", p.mode==2?"1-D bulk":"2-D tensor", p.bw,p.bh,nb,cps, nb*cps*p.bw*p.bh*4/1024);
    printf("%-70s %.3f TB/s  %s\n", desc, tb, cudaGetErrorString(cudaGetLastError()));
    if (tb > best) { best = tb; snprintf(best_desc, sizeof best_desc, "%s", desc); }
  }
  printf("best %.3f TB/s %s\n", best, best_desc);
  return 0;
}
