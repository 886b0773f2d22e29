// probe_issue_cost.cu — stand-alone micro-benchmark behind DESIGN.md §7's issue-cost table (not part of the library).
//
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o /tmp/probe_issue_cost paper_2512_10520_b200/csrc/probe_issue_cost.cu
//   /tmp/probe_issue_cost
//
// One CTA of 1024 threads per SM (8 warps per scheduler), 8 independent dependency chains per thread, 2000 iterations
// of a 32-instruction body; prints the cycles one warp slot of a scheduler spends per body.  The cost of an instruction
// class X mixed into an FP32 stream is (cycles(24 FFMA + 8 X) - 24 * cycles(32 FFMA) / 32) / 8.
#include <cstdio>
#include <cuda_runtime.h>
#define ITER 2000
#define OP_FFMA(i)  asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(f[i]) : "f"(ca), "f"(cb));
#define OP_FADDRM(i) asm volatile("add.rm.f32 %0, %0, %1;" : "+f"(f[i]) : "f"(cb));
#define OP_LOP3(i)  asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(u[i]) : "r"(ka), "r"(kb));
#define OP_IMAD(i)  asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(u[i]) : "r"(ka), "r"(kb));
#define OP_IMADW(i) { unsigned long long t; asm volatile("mul.wide.u32 %0, %1, %2;" : "=l"(t) : "r"(u[i]), "r"(ka)); asm volatile("mov.b64 {%0, %1}, %2;" : "=r"(u[i]), "=r"(v[i]) : "l"(t)); }
#define OP_FMNMX(i) asm volatile("min.f32 %0, %0, %1;" : "+f"(f[i]) : "f"(ca));
#define OP_FSETSEL(i) asm volatile("{.reg .pred p; setp.lt.f32 p, %0, %1; selp.f32 %0, %2, %0, p;}" : "+f"(f[i]) : "f"(ca), "f"(cb));
#define OP_F2I(i)   asm volatile("{.reg .s32 t; cvt.rmi.s32.f32 t, %0; mov.b32 %0, t;}" : "+f"(f[i]));
#define OP_FRND(i)  asm volatile("cvt.rmi.f32.f32 %0, %0;" : "+f"(f[i]));
#define OP_MUFU(i)  asm volatile("rcp.approx.ftz.f32 %0, %0;" : "+f"(f[i]));
#define OP_SHF(i)   asm volatile("shf.l.wrap.b32 %0, %0, %1, 7;" : "+r"(u[i]) : "r"(ka));
#define OP_PRMT(i)  asm volatile("prmt.b32 %0, %0, %1, 0x5410;" : "+r"(u[i]) : "r"(ka));
#define OP_IMNMX(i) asm volatile("min.s32 %0, %0, %1;" : "+r"(u[i]) : "r"(ka));
#define OP_FFMA2(i) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(p[i]) : "l"(pa), "l"(pb));
#define REP8(M) M(0) M(1) M(2) M(3) M(4) M(5) M(6) M(7)
#define A REP8(OP_FFMA)

template <int KIND> __global__ void __launch_bounds__(1024) probe(float* out, float ca, float cb, unsigned ka, unsigned kb, long long* cyc) {
  float f[8]; unsigned u[8], v[8]; unsigned long long p[8];
  const unsigned long long pa = ((unsigned long long)__float_as_uint(ca) << 32) | __float_as_uint(ca);
  const unsigned long long pb = ((unsigned long long)__float_as_uint(cb) << 32) | __float_as_uint(cb);
  for (int i = 0; i < 8; ++i) {
    f[i] = threadIdx.x * 0.001f + i; u[i] = threadIdx.x * 77u + i; v[i] = 0;
    p[i] = ((unsigned long long)__float_as_uint(f[i]) << 32) | __float_as_uint(f[i] + 1.0f);
  }
  const long long t0 = clock64();
#pragma unroll 1
  for (int it = 0; it < ITER; ++it) {
    if (KIND == 0) { A A A A }
    if (KIND == 1) { REP8(OP_LOP3) REP8(OP_LOP3) REP8(OP_LOP3) REP8(OP_LOP3) }
    if (KIND == 2) { A REP8(OP_LOP3) A REP8(OP_LOP3) }
    if (KIND == 3) { A A A REP8(OP_LOP3) }
    if (KIND == 4) { A REP8(OP_IMAD) A REP8(OP_IMAD) }
    if (KIND == 5) { REP8(OP_IMADW) REP8(OP_IMADW) REP8(OP_IMADW) REP8(OP_IMADW) }
    if (KIND == 6) { A REP8(OP_IMADW) A REP8(OP_IMADW) }
    if (KIND == 7) { A REP8(OP_FMNMX) A REP8(OP_FMNMX) }
    if (KIND == 8) { A A REP8(OP_FSETSEL) }
    if (KIND == 9) { A A A REP8(OP_F2I) }
    if (KIND == 10) { A A A REP8(OP_FRND) }
    if (KIND == 11) { A A A REP8(OP_MUFU) }
    if (KIND == 12) { A REP8(OP_FADDRM) A REP8(OP_FADDRM) }
    if (KIND == 13) { A REP8(OP_SHF) A REP8(OP_SHF) }
    if (KIND == 14) { A REP8(OP_PRMT) A REP8(OP_PRMT) }
    if (KIND == 15) { A REP8(OP_IMNMX) A REP8(OP_IMNMX) }
    if (KIND == 16) { REP8(OP_F2I) REP8(OP_F2I) REP8(OP_F2I) REP8(OP_F2I) }
    if (KIND == 17) { REP8(OP_LOP3) REP8(OP_IMADW) REP8(OP_LOP3) REP8(OP_IMADW) }
    if (KIND == 18) { REP8(OP_FFMA2) REP8(OP_FFMA2) REP8(OP_FFMA2) REP8(OP_FFMA2) }
    if (KIND == 19) { REP8(OP_FFMA2) REP8(OP_LOP3) REP8(OP_FFMA2) REP8(OP_LOP3) }
  }
  const long long t1 = clock64();
  float s = 0; unsigned w = 0;
  for (int i = 0; i < 8; ++i) { s += f[i] + __uint_as_float((unsigned)p[i]) + __uint_as_float((unsigned)(p[i] >> 32)); w ^= u[i] ^ v[i]; }
  out[blockIdx.x * blockDim.x + threadIdx.x] = s + (float)w;
  if (threadIdx.x == 0 && blockIdx.x == 0) *cyc = t1 - t0;
}

template <int KIND> void run(const char* name, float* out, long long* cyc) {
  for (int r = 0; r < 2; ++r) { probe<KIND><<<148, 1024>>>(out, 0.999f, 0.5f, 0x9E3779B9u, 0x85EBCA6Bu, cyc); cudaDeviceSynchronize(); }
  long long c = 0; cudaMemcpy(&c, cyc, 8, cudaMemcpyDeviceToHost);
  printf("%-44s %7.2f cycles per 32-instruction body per warp slot\n", name, (double)c / ITER / 8.0);
}

int main() {
  float* out; long long* cyc;
  cudaMalloc(&out, 148 * 1024 * 4); cudaMalloc(&cyc, 8);
  run<0>("32 FFMA", out, cyc);
  run<1>("32 LOP3 (3 register inputs)", out, cyc);
  run<2>("16 FFMA + 16 LOP3", out, cyc);
  run<3>("24 FFMA + 8 LOP3", out, cyc);
  run<4>("16 FFMA + 16 IMAD", out, cyc);
  run<5>("32 IMAD.WIDE.U32", out, cyc);
  run<6>("16 FFMA + 16 IMAD.WIDE.U32", out, cyc);
  run<7>("16 FFMA + 16 FMNMX", out, cyc);
  run<8>("16 FFMA + 8 FSETP + 8 FSEL", out, cyc);
  run<9>("24 FFMA + 8 F2I.FLOOR", out, cyc);
  run<10>("24 FFMA + 8 FRND.FLOOR", out, cyc);
  run<11>("24 FFMA + 8 MUFU.RCP", out, cyc);
  run<12>("16 FFMA + 16 FADD.RM", out, cyc);
  run<13>("16 FFMA + 16 SHF", out, cyc);
  run<14>("16 FFMA + 16 PRMT", out, cyc);
  run<15>("16 FFMA + 16 IMNMX", out, cyc);
  run<16>("32 F2I.FLOOR", out, cyc);
  run<17>("16 LOP3 + 16 IMAD.WIDE.U32", out, cyc);
  run<18>("32 FFMA2 (fma.rn.f32x2)", out, cyc);
  run<19>("16 FFMA2 + 16 LOP3", out, cyc);
  printf("%s\n", cudaGetErrorString(cudaGetLastError()));
  return 0;
}
