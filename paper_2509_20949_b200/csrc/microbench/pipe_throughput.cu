// Measurement aid, not part of libsmcx.so: integer-pipe throughputs on sm_100a that the thread-per-cell
// kernel design rests on (profiles/r1_pipe_microbench.md).  Build and run:
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o /tmp/pipe_throughput paper_2509_20949_b200/csrc/microbench/pipe_throughput.cu && /tmp/pipe_throughput
// Pipe-throughput microbenchmarks: each kernel runs a long chain of one instruction type with 8 independent
// accumulators per thread; reports warp-instructions per clock per SM.
#include <cstdio>
#include <cstdint>
#include <cuda_runtime.h>
#define N_ITER 4096
template <int OP>
__global__ void k(uint32_t* out, uint32_t seed, uint32_t m) {
  uint32_t a[8];
  for (int i = 0; i < 8; ++i) a[i] = seed + threadIdx.x * 7 + i;
  uint32_t c = m;
  long long t0 = clock64();
  for (int it = 0; it < N_ITER; ++it) {
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      if (OP == 0) asm volatile("mul.hi.u32 %0, %0, %1;" : "+r"(a[i]) : "r"(c));
      if (OP == 1) { uint64_t p; asm volatile("mul.wide.u32 %0, %1, %2;" : "=l"(p) : "r"(a[i]), "r"(c)); a[i] = (uint32_t)p ^ (uint32_t)(p >> 32); }
      if (OP == 2) asm volatile("shr.u32 %0, %0, %1;" : "+r"(a[i]) : "r"(c & 3));
      if (OP == 3) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a[i]) : "r"(c), "r"(seed));
      if (OP == 4) asm volatile("popc.b32 %0, %0;" : "+r"(a[i]));
      if (OP == 5) asm volatile("prmt.b32 %0, %0, %1, 0x5410;" : "+r"(a[i]) : "r"(c));
      if (OP == 6) asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(a[i]) : "r"(c), "r"(seed));
      if (OP == 7) asm volatile("add.u32 %0, %0, %1;" : "+r"(a[i]) : "r"(c));
      if (OP == 8) asm volatile("shf.r.wrap.b32 %0, %0, %0, %1;" : "+r"(a[i]) : "r"(c));
      if (OP == 9) { asm volatile("mul.hi.u32 %0, %0, %1;" : "+r"(a[i]) : "r"(c)); asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a[i]) : "r"(c), "r"(seed)); }
      if (OP == 10) { asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(a[i]) : "r"(c), "r"(seed)); asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a[i]) : "r"(c), "r"(seed)); }
      if (OP == 11) { asm volatile("popc.b32 %0, %0;" : "+r"(a[i])); asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a[i]) : "r"(c), "r"(seed)); asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a[i]) : "r"(c), "r"(seed)); asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a[i]) : "r"(c), "r"(seed));}
      if (OP == 13) asm volatile("dp2a.lo.s32.u32 %0, %0, %1, %2;" : "+r"(a[i]) : "r"(c), "r"(seed));
      if (OP == 14) asm volatile("dp4a.s32.u32 %0, %0, %1, %2;" : "+r"(a[i]) : "r"(c), "r"(seed));
      if (OP == 15) { asm volatile("dp2a.hi.s32.u32 %0, %0, %1, %2;" : "+r"(a[i]) : "r"(c), "r"(seed)); asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a[i]) : "r"(c), "r"(seed)); }
      if (OP == 16) { asm volatile("dp2a.lo.s32.u32 %0, %0, %1, %2;" : "+r"(a[i]) : "r"(c), "r"(seed)); asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(a[i]) : "r"(c), "r"(seed)); }
      if (OP == 12) { int p; asm volatile("{.reg .pred q; setp.lt.u32 q, %1, %2; selp.u32 %0, 1, 0, q;}" : "=r"(p) : "r"(a[i]), "r"(c)); a[i] += p; }
    }
  }
  long long t1 = clock64();
  uint32_t s = 0;
  for (int i = 0; i < 8; ++i) s ^= a[i];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s + (uint32_t)(t1 - t0);
  if (threadIdx.x == 0 && blockIdx.x == 0) out[gridDim.x * blockDim.x] = (uint32_t)(t1 - t0);
}
template <int OP> void run(const char* name, int per) {
  uint32_t* d; cudaMalloc(&d, (148 * 1024 + 1) * 4);
  for (int warps = 4; warps <= 32; warps *= 2) {
    k<OP><<<148, warps * 32>>>(d, 12345u, 0x9E3779B1u);
    cudaDeviceSynchronize();
    uint32_t cyc; cudaMemcpy(&cyc, d + 148 * warps * 32, 4, cudaMemcpyDeviceToHost);
    double winst = (double)N_ITER * 8 * per * warps;
    printf("%-22s warps/SM=%2d  cycles=%8u  warp-inst/clk/SM=%.3f\n", name, warps, cyc, winst / cyc);
  }
  cudaFree(d);
}
int main() {
  run<0>("mul.hi.u32", 1); run<1>("mul.wide.u32(+xor)", 2); run<2>("shr.u32", 1); run<3>("lop3", 1); run<4>("popc", 1);
  run<5>("prmt", 1); run<6>("mad.lo", 1); run<7>("add", 1); run<8>("shf.wrap", 1); run<9>("mul.hi+lop3", 2); run<10>("mad.lo+lop3", 2);
  run<11>("popc+3lop3", 4); run<12>("setp+selp+add", 3);
  run<13>("dp2a.lo", 1); run<14>("dp4a", 1); run<15>("dp2a.hi+lop3", 2); run<16>("dp2a.lo+mad.lo", 2);
  return 0;
}
