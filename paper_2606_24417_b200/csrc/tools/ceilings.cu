// ceilings.cu — box ceilings the rooflines in DESIGN.md §6 are quoted against (SURVEY.md §8(d) asks for them):
//   random-sector RED.OR / 256-bit loads over a filter-sized array (512 MiB and 32 MiB), and integer pipe rates.
// Stand-alone: no part of the library's hot path.  Built by paper_2606_24417_b200/build.py:build_tools() into
// paper_2606_24417_b200/sbf_ceilings;  usage: sbf_ceilings [l2_fetch_granularity_bytes]
#include <cstdio>
#include <cstdint>
#include <cstdlib>
#include <cuda_runtime.h>
#define CK(x) do{cudaError_t e=(x); if(e!=cudaSuccess){printf("ERR %s line %d\n",cudaGetErrorString(e),__LINE__); exit(1);} }while(0)
__device__ __forceinline__ uint64_t mix(uint64_t x){ x^=x>>33; x*=0xff51afd7ed558ccdULL; x^=x>>33; x*=0xc4ceb9fe1a85ec53ULL; x^=x>>33; return x; }

template<int NRED, int WIDTH64>
__global__ void k_red(uint64_t* f, uint64_t nshards_mask, uint64_t n_per_thread){
  uint64_t t = (uint64_t)blockIdx.x*blockDim.x+threadIdx.x;
  for(uint64_t i=0;i<n_per_thread;i++){
    uint64_t h = mix(t*n_per_thread+i+1);
    uint64_t* p = f + (h & nshards_mask)*4;
    uint64_t v = 1ull<<(h>>58);
    if (WIDTH64){
#pragma unroll
      for(int q=0;q<NRED;q++) asm volatile("red.global.or.b64 [%0], %1;"::"l"(p+q),"l"(v):"memory");
    } else {
#pragma unroll
      for(int q=0;q<NRED;q++) asm volatile("red.global.or.b32 [%0], %1;"::"l"((uint32_t*)p+q),"r"((uint32_t)v|1u):"memory");
    }
  }
}
// MODE 0: ld.global.nc.v4.u64 ; 1: two ld.global.nc.v2.u64; 2: ld.global.nc.L2::64B? ; 3: plain ld.global.v4.u64 ; 4: ld.global.nc.v2.u64 only (16B)
template<int MODE, int MLP>
__global__ void k_ld(const uint64_t* f, uint64_t nshards_mask, uint64_t n_per_thread, uint64_t* out){
  uint64_t t = (uint64_t)blockIdx.x*blockDim.x+threadIdx.x;
  uint64_t acc=0;
  for(uint64_t i=0;i<n_per_thread;i+=MLP){
    uint64_t w[MLP][4];
#pragma unroll
    for(int u=0;u<MLP;u++){
      uint64_t h = mix(t*n_per_thread+i+u+1);
      const uint64_t* p = f + (h & nshards_mask)*4;
      if (MODE==0) asm volatile("ld.global.nc.v4.u64 {%0,%1,%2,%3}, [%4];":"=l"(w[u][0]),"=l"(w[u][1]),"=l"(w[u][2]),"=l"(w[u][3]):"l"(p));
      else if (MODE==1){ asm volatile("ld.global.nc.v2.u64 {%0,%1}, [%2];":"=l"(w[u][0]),"=l"(w[u][1]):"l"(p)); asm volatile("ld.global.nc.v2.u64 {%0,%1}, [%2];":"=l"(w[u][2]),"=l"(w[u][3]):"l"(p+2)); }
      else if (MODE==2) asm volatile("ld.global.nc.L2::64B.v4.u64 {%0,%1,%2,%3}, [%4];":"=l"(w[u][0]),"=l"(w[u][1]),"=l"(w[u][2]),"=l"(w[u][3]):"l"(p));
      else if (MODE==3) asm volatile("ld.global.v4.u64 {%0,%1,%2,%3}, [%4];":"=l"(w[u][0]),"=l"(w[u][1]),"=l"(w[u][2]),"=l"(w[u][3]):"l"(p));
      else if (MODE==4){ asm volatile("ld.global.nc.v2.u64 {%0,%1}, [%2];":"=l"(w[u][0]),"=l"(w[u][1]):"l"(p)); w[u][2]=w[u][3]=0; }
      else if (MODE==5) asm volatile("ld.global.L1::no_allocate.v4.u64 {%0,%1,%2,%3}, [%4];":"=l"(w[u][0]),"=l"(w[u][1]),"=l"(w[u][2]),"=l"(w[u][3]):"l"(p));
    }
#pragma unroll
    for(int u=0;u<MLP;u++) acc += w[u][0]^w[u][1]^w[u][2]^w[u][3];
  }
  if(acc==0x1234567) out[0]=acc;
}
// integer pipe rates: 0 LOP3, 1 IMAD, 2 SHF(funnel), 3 mix LOP3+IMAD 1:1, 4 IADD3, 5 LOP3+SHF, 6 VIMNMX3
template<int OP>
__global__ void k_alu(uint32_t* out, int iters, uint32_t s){
  uint32_t a=threadIdx.x, b=blockIdx.x+s, c=s*3+1, d=s^0x55, e=a+7,f=b+9,g=c+11,h=d+13;
  for(int i=0;i<iters;i++){
#pragma unroll
    for(int u=0;u<16;u++){
      if(OP==0){ a=(a&b)^c; d=(d&e)^f; g=(g&h)^a; b=(b&c)^d; }
      if(OP==1){ a=a*b+c; d=d*e+f; g=g*h+a; b=b*c+d; }
      if(OP==2){ a=__funnelshift_r(a,b,7)+0; d=__funnelshift_r(d,e,9); g=__funnelshift_r(g,h,11); b=__funnelshift_r(b,c,13); }
      if(OP==3){ a=(a&b)^c; d=d*e+f; g=(g&h)^a; b=b*c+d; }
      if(OP==4){ a=a+b+c; d=d+e+f; g=g+h+a; b=b+c+d; }
      if(OP==5){ a=(a&b)^c; d=__funnelshift_r(d,e,9); g=(g&h)^a; b=__funnelshift_r(b,c,13); }
      if(OP==6){ a=min(min(a,b),c)+1; d=min(min(d,e),f)+1; g=min(min(g,h),a)+1; b=min(min(b,c),d)+1; }
      if(OP==7){ a=(a&b)^c; d=d*e+f; g=__funnelshift_r(g,h,11); b=(b&c)^d; e=e*f+g; h=__funnelshift_r(h,a,5);}
    }
  }
  if((a^b^c^d^e^f^g^h)==0x12345) out[0]=a;
}
template<class F> float timeit(F f, int rep=5){ cudaEvent_t a,b; cudaEventCreate(&a); cudaEventCreate(&b); f(); float best=1e30f; for(int i=0;i<rep;i++){ cudaEventRecord(a); f(); cudaEventRecord(b); cudaEventSynchronize(b); float ms; cudaEventElapsedTime(&ms,a,b); if(ms<best)best=ms;} return best; }

int main(int argc,char**argv){
  int fetch = argc>1? atoi(argv[1]):0;
  if(fetch){ CK(cudaDeviceSetLimit(cudaLimitMaxL2FetchGranularity, fetch)); }
  size_t g=0; cudaDeviceGetLimit(&g,cudaLimitMaxL2FetchGranularity); printf("L2 fetch granularity limit: %zu\n", g);
  uint64_t* f; uint64_t* out; CK(cudaMalloc(&out,64));
  for (int P : {24, 20}) {
    uint64_t nsh = 1ull<<P; CK(cudaMalloc(&f, nsh*32)); CK(cudaMemset(f,0,nsh*32));
    printf("== filter %llu MiB\n", (unsigned long long)(nsh*32>>20));
    for (int tpb : {128, 256}) for (int bps : {2, 4, 8, 16}) {
      int blocks = 148*bps; uint64_t npt = 2048; double n = (double)blocks*tpb*npt;
      float ms = timeit([&]{ k_red<4,1><<<blocks,tpb>>>(f, nsh-1, npt); });
      float ms1 = timeit([&]{ k_red<1,1><<<blocks,tpb>>>(f, nsh-1, npt); });
      float ms8 = timeit([&]{ k_red<8,0><<<blocks,tpb>>>(f, nsh-1, npt); });
      printf("RED tpb %d blocks/SM %d : 4xb64 %.2f Gshard/s | 1xb64 %.2f | 8xb32 %.2f\n", tpb, bps, n/ms/1e6, n/ms1/1e6, n/ms8/1e6);
    }
    for (int bps : {4, 8, 16}) {
      int tpb=128; int blocks=148*bps; uint64_t npt=2048; double n=(double)blocks*tpb*npt;
      float a0 = timeit([&]{ k_ld<0,1><<<blocks,tpb>>>(f,nsh-1,npt,out); });
      float a4 = timeit([&]{ k_ld<0,4><<<blocks,tpb>>>(f,nsh-1,npt,out); });
      float b4 = timeit([&]{ k_ld<1,4><<<blocks,tpb>>>(f,nsh-1,npt,out); });
      float c4 = timeit([&]{ k_ld<2,4><<<blocks,tpb>>>(f,nsh-1,npt,out); });
      float d4 = timeit([&]{ k_ld<3,4><<<blocks,tpb>>>(f,nsh-1,npt,out); });
      float e4 = timeit([&]{ k_ld<4,4><<<blocks,tpb>>>(f,nsh-1,npt,out); });
      float f4 = timeit([&]{ k_ld<5,4><<<blocks,tpb>>>(f,nsh-1,npt,out); });
      printf("LD blocks/SM %d : nc.v4 mlp1 %.2f Gshard/s | nc.v4 mlp4 %.2f | 2x nc.v2 %.2f | L2::64B %.2f | plain v4 %.2f | 16B only %.2f | no_alloc %.2f\n", bps, n/a0/1e6, n/a4/1e6, n/b4/1e6, n/c4/1e6, n/d4/1e6, n/e4/1e6, n/f4/1e6);
    }
    CK(cudaFree(f));
  }
  uint32_t* o32; CK(cudaMalloc(&o32,64));
  const char* names[]={"LOP3","IMAD","SHF","LOP3+IMAD","IADD3","LOP3+SHF","VIMNMX3+IADD","LOP3:IMAD:SHF 3:2:2(ish)"};
  int iters=4096; 
  auto run=[&](int op){ int blocks=148*8, tpb=256; float ms=0;
    switch(op){case 0: ms=timeit([&]{k_alu<0><<<blocks,tpb>>>(o32,iters,1);});break; case 1: ms=timeit([&]{k_alu<1><<<blocks,tpb>>>(o32,iters,1);});break;
    case 2: ms=timeit([&]{k_alu<2><<<blocks,tpb>>>(o32,iters,1);});break; case 3: ms=timeit([&]{k_alu<3><<<blocks,tpb>>>(o32,iters,1);});break;
    case 4: ms=timeit([&]{k_alu<4><<<blocks,tpb>>>(o32,iters,1);});break; case 5: ms=timeit([&]{k_alu<5><<<blocks,tpb>>>(o32,iters,1);});break;
    case 6: ms=timeit([&]{k_alu<6><<<blocks,tpb>>>(o32,iters,1);});break; case 7: ms=timeit([&]{k_alu<7><<<blocks,tpb>>>(o32,iters,1);});break;}
    double nops = (double)blocks*tpb*iters*16*(op==7?6:(op==6?8:4)); // source-level ops (op 6: min3+add = 2 each)
    printf("ALU %-28s %.2f T source-ops/s  (%.1f lane-ops/clk/SM at 1.965 GHz)\n", names[op], nops/ms/1e9, nops/(ms*1e-3)/148/1.965e9);
  };
  for(int op=0;op<8;op++) if (op != 4) run(op); // 4 (IADD3 chain) folds at compile time
  return 0;
}
