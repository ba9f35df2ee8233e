// Microbenchmark behind DESIGN.md section 7: dispatch cost (clocks per warp instruction per SM sub-partition, 4 warps each)
// of the instruction types and mixes the PairHMM engine is made of, on sm_100a.  Not part of the library.
// Build + run:  nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o /tmp/ubench_dispatch paper_2606_25738_b200/csrc/ubench_dispatch.cu && /tmp/ubench_dispatch
#include <cstdio>
#include <cuda_runtime.h>
#define ITERS 2048
#define R16(X) X(0) X(1) X(2) X(3) X(4) X(5) X(6) X(7) X(8) X(9) X(10) X(11) X(12) X(13) X(14) X(15)
template<int MODE> __global__ void __launch_bounds__(128) k(float* out, float a, float b, unsigned sel) {
  float f[16]; unsigned u[16]; float g[16]; unsigned long long p2[16], a2, b2; a2=((unsigned long long)__float_as_uint(a)<<32)|__float_as_uint(a); b2=((unsigned long long)__float_as_uint(b)<<32)|__float_as_uint(b); for (int i=0;i<16;i++) p2[i]=a2+i*threadIdx.x;
  for (int i=0;i<16;i++){f[i]=threadIdx.x+i; u[i]=threadIdx.x*i+sel; g[i]=i*a;}
  unsigned m = sel*threadIdx.x+1;
  _Pragma("unroll 1") for (int it=0; it<ITERS; it++) {
    asm volatile("{.reg .pred p,q;\n setp.ne.u32 p, %0, 7;\n setp.ne.u32 q, %0, 9;" :: "r"(m));
#define FSEL1(i) asm volatile("selp.f32 %0, %0, %1, p;" : "+f"(f[i]) : "f"(g[i]));
#define FSEL2(i) asm volatile("selp.f32 %0, %0, %1, q;" : "+f"(g[i]) : "f"(f[i]));
#define LOP1(i) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(u[i]) : "r"(m), "r"(u[(i+1)&15]));
#define FMUL1(i) asm volatile("mul.f32 %0, %0, %1;" : "+f"(f[i]) : "f"(a));
#define FMUL2(i) asm volatile("mul.f32 %0, %0, %1;" : "+f"(g[i]) : "f"(b));
#define FFMA1(i) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(f[i]) : "f"(a), "f"(b));
#define IMAD1(i) asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(u[i]) : "r"(m), "r"(sel));
#define HSET1(i) asm volatile("{.reg .pred r,s; setp.eq.f16x2 r|s, %1, %2; @r mul.f32 %0, %0, %3;}" : "+f"(f[i]) : "r"(u[i]), "r"(m), "f"(a));
#define PMUL1(i) asm volatile("@p mul.f32 %0, %0, %1;\n @!p mul.f32 %0, %0, %2;" : "+f"(f[i]) : "f"(a), "f"(b));
#define ISETP1(i) asm volatile("{.reg .pred r; setp.lt.u32 r, %1, %2; @r mul.f32 %0, %0, %3;}" : "+f"(f[i]) : "r"(u[i]), "r"(m), "f"(a));
#define F2A(i) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(p2[i]) : "l"(a2), "l"(b2));
#define F2B(i) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(p2[(i+8)&15]) : "l"(b2), "l"(a2));
#define CELLP(i) LOP1(i) F2A(i) FSEL1(i) F2B(i) LOP1(i) F2A(i) FSEL2(i) F2B(i) F2A(i)
#define CELLS(i) LOP1(i) FFMA1(i) FFMA1(i) FSEL1(i) FFMA1(i) FFMA1(i) FFMA1(i) LOP1(i) FFMA1(i) FFMA1(i) FSEL2(i) FFMA1(i) FFMA1(i) FFMA1(i)
#define ALT1(i) LOP1(i) FMUL2(i)
#define ALT2(i) LOP1(i) FMUL2(i) FMUL1(i)
#define SHF1(i) asm volatile("shr.u32 %0, %0, %1;" : "+r"(u[i]) : "r"(sel));
#define MOV1(i) asm volatile("mov.b32 %0, %1;" : "=r"(u[i]) : "r"(u[(i+3)&15]));
#define PRMT1(i) asm volatile("prmt.b32 %0, %0, %1, %2;" : "+r"(u[i]) : "r"(m), "r"(sel));
    if (MODE==0) { R16(FSEL1) R16(FSEL2) R16(FSEL1) R16(FSEL2) }
    if (MODE==1) { R16(LOP1) R16(LOP1) R16(LOP1) R16(LOP1) }
    if (MODE==2) { R16(FMUL1) R16(FMUL2) R16(FMUL1) R16(FMUL2) }
    if (MODE==3) { R16(FSEL1) R16(FMUL2) R16(FSEL1) R16(FMUL2) }   // 32 FSEL + 32 FMUL (blocks of 16)
    if (MODE==4) { R16(LOP1) R16(FMUL2) R16(LOP1) R16(FMUL2) }
    if (MODE==5) { R16(IMAD1) R16(IMAD1) R16(IMAD1) R16(IMAD1) }
    if (MODE==6) { R16(HSET1) R16(HSET1) }                           // 32 HSETP2 + 32 @FMUL
    if (MODE==7) { R16(PMUL1) R16(PMUL1) }                           // 64 predicated FMUL
    if (MODE==8) { R16(ISETP1) R16(ISETP1) }                         // 32 ISETP + 32 @FMUL
    if (MODE==9) { R16(FFMA1) R16(FFMA1) R16(FFMA1) R16(FFMA1) }
    if (MODE==10) { R16(SHF1) R16(SHF1) R16(SHF1) R16(SHF1) }
    if (MODE==11) { R16(PRMT1) R16(PRMT1) R16(PRMT1) R16(PRMT1) }
    if (MODE==12) { R16(FSEL1) R16(LOP1) R16(FSEL2) R16(LOP1) }     // both ALU?
    if (MODE==13) { R16(IMAD1) R16(FMUL1) R16(IMAD1) R16(FMUL2) }
    if (MODE==14) { R16(CELLP) }   // 16 x [2 LOP3 + 2 FSEL + 5 FFMA2]
    if (MODE==15) { R16(CELLS) }   // 16 x [2 LOP3 + 2 FSEL + 10 FFMA]
    if (MODE==16) { R16(ALT1) R16(ALT1) }   // 32 x [LOP3, FMUL] alternating
    if (MODE==17) { R16(ALT2) R16(ALT2) }   // 32 x [LOP3, FMUL, FMUL]
    if (MODE==18) { R16(F2A) R16(F2B) R16(F2A) R16(F2B) }  // 64 FFMA2
    if (MODE==19) { R16(F2A) R16(LOP1) R16(F2B) R16(LOP1) }  // 32 FFMA2 + 32 LOP3 blocks
    asm volatile("}");
    m = m*5+1;
  }
  float s=0; for(int i=0;i<16;i++) s+=f[i]+g[i]+u[i]+(float)(p2[i]>>7);
  if (s==123.456f) out[0]=s+m;
}
template<int MODE> void run(const char* name) {
  float* out; cudaMalloc(&out,4); int nsm=148, tpb=128, w=4; cudaEvent_t e0,e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
  k<MODE><<<nsm*w,tpb>>>(out,0.999f,0.998f,1); cudaDeviceSynchronize();
  cudaEventRecord(e0); k<MODE><<<nsm*w,tpb>>>(out,0.999f,0.998f,1); cudaEventRecord(e1); cudaEventSynchronize(e1);
  float ms; cudaEventElapsedTime(&ms,e0,e1);
  printf("%-36s clk/iter=%.1f  err=%s\n", name, ms*1e-3*1.965e9/ITERS/w, cudaGetErrorString(cudaGetLastError()));
}
int main(){
  run<0>("64 FSEL"); run<1>("64 LOP3"); run<2>("64 FMUL"); run<3>("32 FSEL + 32 FMUL"); run<4>("32 LOP3 + 32 FMUL"); run<5>("64 IMAD");
  run<6>("32 HSETP2 + 32 @FMUL"); run<7>("64 pred FMUL"); run<8>("32 ISETP + 32 @FMUL"); run<9>("64 FFMA"); run<10>("64 SHF"); run<11>("64 PRMT");
  run<12>("32 FSEL + 32 LOP3"); run<13>("32 IMAD + 32 FMUL");
  run<14>("16x[2 LOP3+2 FSEL+5 FFMA2]"); run<15>("16x[2 LOP3+2 FSEL+10 FFMA]"); run<16>("32x[LOP3,FMUL] alternating"); run<17>("32x[LOP3,FMUL,FMUL]"); run<18>("64 FFMA2"); run<19>("32 FFMA2 + 32 LOP3 blocks");
  return 0; }
