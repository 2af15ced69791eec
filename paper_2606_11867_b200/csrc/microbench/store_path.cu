// Micro-benchmark of the dispatch store path (evidence for DESIGN.md sec. 6; not part of the library).
// Pattern of foremoe_dispatch at config-2 shape: per token one 4 KB row read, K = 8 rows of 4 KB written
// to 8 separate streams.  Variants: store-only vs load+store, CTA-per-token vs warp-per-token.
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -std=c++17 -o /tmp/store_path \
//        paper_2606_11867_b200/csrc/microbench/store_path.cu && /tmp/store_path 16384 && /tmp/store_path 65536
#include <cstdio>
#include <cstdlib>
#include <cuda_runtime.h>
#include <vector>
#define CK(x) do{cudaError_t e=(x); if(e!=cudaSuccess){printf("err %s line %d\n", cudaGetErrorString(e), __LINE__); exit(1);} }while(0)
__device__ __forceinline__ void st16(void*p,int4 v){ asm volatile("st.global.cs.v4.s32 [%0], {%1,%2,%3,%4};"::"l"(p),"r"(v.x),"r"(v.y),"r"(v.z),"r"(v.w):"memory"); }
__device__ __forceinline__ int4 ld16(const void*p){ int4 r; asm volatile("ld.global.nc.L1::no_allocate.v4.s32 {%0,%1,%2,%3}, [%4];":"=r"(r.x),"=r"(r.y),"=r"(r.z),"=r"(r.w):"l"(p)); return r; }
// token per CTA: blockDim*VPT == 256 vectors; thread loads VPT vecs, stores K*VPT
template<int VPT, bool LOAD>
__global__ void tok_cta(const int* __restrict__ inv, const int4* __restrict__ x, int4* buf, int n_tok, int K, int tpc){
  __shared__ int sd[32];
  for(int q=0;q<tpc;q++){
    int t = blockIdx.x*tpc+q; if(t>=n_tok) return;
    if(threadIdx.x<K) sd[threadIdx.x]=__ldg(inv+t*K+threadIdx.x);
    int4 r[VPT];
    #pragma unroll
    for(int u=0;u<VPT;u++){ int v=u*blockDim.x+threadIdx.x; r[u]= LOAD? ld16(x+(size_t)t*256+v) : make_int4(t,v,u,0); }
    __syncthreads();
    for(int k=0;k<K;k++){ int4* dst=buf+(size_t)sd[k]*256;
      #pragma unroll
      for(int u=0;u<VPT;u++) st16(dst+u*blockDim.x+threadIdx.x, r[u]); }
    __syncthreads();
  }
}
// warp per token, WPC warps per CTA, one token per warp (non persistent)
template<bool LOAD>
__global__ void tok_warp(const int* __restrict__ inv, const int4* __restrict__ x, int4* buf, int n_tok, int K){
  int lane=threadIdx.x&31; int t=blockIdx.x*(blockDim.x>>5)+(threadIdx.x>>5); if(t>=n_tok) return;
  int d = lane<K ? __ldg(inv+t*K+lane):0; int4 r[8];
  #pragma unroll
  for(int u=0;u<8;u++) r[u]= LOAD? ld16(x+(size_t)t*256+u*32+lane): make_int4(t,u,lane,0);
  for(int k=0;k<K;k++){ int dk=__shfl_sync(0xffffffffu,d,k); int4* dst=buf+(size_t)dk*256;
    #pragma unroll
    for(int u=0;u<8;u++) st16(dst+u*32+lane,r[u]); }
}
int main(int argc,char**argv){
  int n_tok = argc>1?atoi(argv[1]):16384; int K=8; int reps=20;
  size_t nvec=(size_t)n_tok*K*256; int4 *buf,*x; int*inv;
  CK(cudaMalloc(&buf,nvec*16*2)); CK(cudaMalloc(&x,(size_t)n_tok*256*16*4)); CK(cudaMalloc(&inv,(size_t)n_tok*K*4));
  std::vector<int> h(n_tok*K); 
  // slot-major scatter like the real thing: pair (t,k) -> row k*n_tok + t  (8 streams) 
  for(int t=0;t<n_tok;t++) for(int k=0;k<K;k++) h[t*K+k]=k*n_tok+t;
  CK(cudaMemcpy(inv,h.data(),h.size()*4,cudaMemcpyHostToDevice));
  CK(cudaMemset(x,1,(size_t)n_tok*256*16*4));
  cudaEvent_t a,b; cudaEventCreate(&a); cudaEventCreate(&b);
  auto run=[&](const char*name, auto launch, double bytes){ float best=1e9,sum=0; for(int r=0;r<reps+3;r++){ int4* bb = buf + (r&1)*nvec; const int4* xx = x + (size_t)(r&3)*n_tok*256; cudaEventRecord(a); launch(bb,xx); cudaEventRecord(b); CK(cudaEventSynchronize(b)); float ms; cudaEventElapsedTime(&ms,a,b); if(r>=3){sum+=ms; if(ms<best)best=ms;} } printf("%-40s avg %7.1f us %6.0f GB/s  best %7.1f us %6.0f GB/s\n",name,sum/reps*1e3,bytes/(sum/reps)/1e6,best*1e3,bytes/best/1e6); };
  double wb=(double)nvec*16, rb=(double)n_tok*256*16;
  run("cta256/token store-only",[&](int4*bb,const int4*xx){tok_cta<1,false><<<n_tok,256>>>(inv,xx,bb,n_tok,K,1);},wb);
  run("cta256/token load+store",[&](int4*bb,const int4*xx){tok_cta<1,true><<<n_tok,256>>>(inv,xx,bb,n_tok,K,1);},wb+rb);
  run("cta128/token load+store",[&](int4*bb,const int4*xx){tok_cta<2,true><<<n_tok,128>>>(inv,xx,bb,n_tok,K,1);},wb+rb);
  run("cta64/token load+store",[&](int4*bb,const int4*xx){tok_cta<4,true><<<n_tok,64>>>(inv,xx,bb,n_tok,K,1);},wb+rb);
  run("cta256 x2 tokens load+store",[&](int4*bb,const int4*xx){tok_cta<1,true><<<n_tok/2,256>>>(inv,xx,bb,n_tok,K,2);},wb+rb);
  run("cta256 x4 tokens load+store",[&](int4*bb,const int4*xx){tok_cta<1,true><<<n_tok/4,256>>>(inv,xx,bb,n_tok,K,4);},wb+rb);
  run("cta128 x4 tokens load+store",[&](int4*bb,const int4*xx){tok_cta<2,true><<<n_tok/4,128>>>(inv,xx,bb,n_tok,K,4);},wb+rb);
  for(int wpc: {1,2,4,8}){ char nm[64]; sprintf(nm,"warp/token %d warps/cta store-only",wpc); run(nm,[&](int4*bb,const int4*xx){tok_warp<false><<<n_tok/wpc,wpc*32>>>(inv,xx,bb,n_tok,K);},wb);
    sprintf(nm,"warp/token %d warps/cta load+store",wpc); run(nm,[&](int4*bb,const int4*xx){tok_warp<true><<<n_tok/wpc,wpc*32>>>(inv,xx,bb,n_tok,K);},wb+rb); }
  return 0; }
