// Measurement aid, not part of libsmcx.so: how the instruction types of the trial loop share the issue port
// and the integer pipes of an SM sub-partition on sm_100a (profiles/r1_pipe_microbench.md).  Every kernel runs a
// loop whose body holds the named instructions on independent registers; the figure is cycles per loop
// iteration per sub-partition with 8 warps per sub-partition (the loop itself adds about 3 issue slots).
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o /tmp/pipe_pairs paper_2509_20949_b200/csrc/microbench/pipe_pairs.cu && /tmp/pipe_pairs
#include <cstdio>
#include <cstdint>
#include <cuda_runtime.h>
#define N_ITER 2048
#define LOP(i)  asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a[i]) : "r"(c), "r"(seed));
#define PRM(i)  asm volatile("prmt.b32 %0, %0, %1, 0x5410;" : "+r"(a[i]) : "r"(c));
#define MAD(i)  asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(a[i]) : "r"(c), "r"(seed));
#define WID(i)  asm volatile("mul.wide.u32 %0, %1, %2;" : "=l"(w[i]) : "r"((uint32_t)w[i]), "r"(c));
#define HI(i)   asm volatile("mul.hi.u32 %0, %0, %1;" : "+r"(a[i]) : "r"(c));
#define POP(i)  asm volatile("popc.b32 %0, %0;" : "+r"(a[i]));
#define LDS(i)  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(a[i]) : "r"(sbase + ((a[i] & 31u) << 9)));
#define SHR(i)  asm volatile("shr.u32 %0, %0, %1;" : "+r"(a[i]) : "r"(c & 3));
#define ADD(i)  asm volatile("add.u32 %0, %0, %1;" : "+r"(a[i]) : "r"(c));
#define SETP(i) asm volatile("{.reg .pred q; setp.lt.u32 q, %0, %1; selp.u32 %0, %1, %2, q;}" : "+r"(a[i]) : "r"(c), "r"(seed));
#define MNMX(i) asm volatile("min.u32 %0, %0, %1;" : "+r"(a[i]) : "r"(c));
template <int OP>
__global__ void k(uint32_t* out, uint32_t seed, uint32_t m) {
  __shared__ uint32_t sm[32 * 128];
  uint32_t a[16]; uint64_t w[4];
  for (int i = 0; i < 16; ++i) a[i] = seed + threadIdx.x * 7 + i;
  for (int i = 0; i < 4; ++i) w[i] = seed * 3 + threadIdx.x + i;
  for (int i = threadIdx.x; i < 32 * 128; i += blockDim.x) sm[i] = i * 2654435761u;
  __syncthreads();
  const uint32_t sbase = (uint32_t)__cvta_generic_to_shared(sm) + (threadIdx.x & 127) * 4;
  uint32_t c = m;
  long long t0 = clock64();
#pragma unroll 1
  for (int it = 0; it < N_ITER; ++it) {
    if (OP == 0) { LOP(0) LOP(1) LOP(2) LOP(3) }
    if (OP == 1) { LOP(0) MAD(4) LOP(1) MAD(5) LOP(2) MAD(6) LOP(3) MAD(7) }
    if (OP == 2) { LOP(0) LOP(1) WID(0) LOP(2) LOP(3) }
    if (OP == 3) { LOP(0) WID(0) LOP(1) LOP(2) WID(1) LOP(3) }
    if (OP == 4) { LOP(0) LOP(1) POP(4) LOP(2) LOP(3) }
    if (OP == 5) { LOP(0) LOP(1) HI(4) LOP(2) LOP(3) }
    if (OP == 6) { LOP(0) LOP(1) LDS(4) LOP(2) LOP(3) }
    if (OP == 7) { MAD(0) MAD(1) WID(0) MAD(2) MAD(3) }
    if (OP == 8) { MAD(0) MAD(1) POP(4) MAD(2) MAD(3) }
    if (OP == 9) { PRM(0) MAD(4) PRM(1) MAD(5) PRM(2) MAD(6) PRM(3) MAD(7) }
    if (OP == 10) { LOP(0) MAD(4) LOP(1) MAD(5) POP(8) LOP(2) MAD(6) LOP(3) MAD(7) }
    if (OP == 11) { LOP(0) MAD(4) LOP(1) MAD(5) WID(0) LOP(2) MAD(6) LOP(3) MAD(7) }
    if (OP == 12) { WID(0) WID(1) WID(2) WID(3) }
    if (OP == 13) { LOP(0) MAD(4) LOP(1) HI(5) LOP(2) LOP(3) }   // mul.lo + mul.hi instead of wide
    if (OP == 14) { POP(0) POP(1) MAD(4) MAD(5) MAD(6) MAD(7) MAD(8) MAD(9) MAD(10) MAD(11) }
    if (OP == 15) { POP(0) LOP(4) LOP(5) LOP(6) LOP(7) LOP(8) LOP(9) LOP(10) LOP(11) }
    if (OP == 16) { SHR(0) SHR(1) SHR(2) SHR(3) MAD(4) MAD(5) MAD(6) MAD(7) }
    if (OP == 17) { ADD(0) ADD(1) ADD(2) ADD(3) LOP(4) LOP(5) LOP(6) LOP(7) }
    if (OP == 18) { SETP(0) SETP(1) MAD(4) MAD(5) MAD(6) MAD(7) }
    if (OP == 19) { MNMX(0) MNMX(1) MNMX(2) MNMX(3) MAD(4) MAD(5) MAD(6) MAD(7) }
    if (OP == 20) { LDS(0) LDS(1) LDS(2) LDS(3) MAD(4) MAD(5) LOP(6) LOP(7) }
  }
  long long t1 = clock64();
  uint32_t s = 0;
  for (int i = 0; i < 16; ++i) s ^= a[i];
  for (int i = 0; i < 4; ++i) s ^= (uint32_t)w[i] ^ (uint32_t)(w[i] >> 32);
  out[blockIdx.x * blockDim.x + threadIdx.x] = s + (uint32_t)(t1 - t0);
  if (threadIdx.x == 0 && blockIdx.x == 0) out[gridDim.x * blockDim.x] = (uint32_t)(t1 - t0);
}
template <int OP> void run(const char* name) {
  uint32_t* d; cudaMalloc(&d, (148 * 1024 + 1) * 4);
  for (int warps = 16; warps <= 32; warps *= 2) {
    k<OP><<<148, warps * 32>>>(d, 12345u, 0x9E3779B1u);
    cudaDeviceSynchronize();
    uint32_t cyc; cudaMemcpy(&cyc, d + 148 * warps * 32, 4, cudaMemcpyDeviceToHost);
    printf("%-34s warps/SM=%2d cycles/iter/SMSP=%.2f\n", name, warps, (double)cyc / N_ITER / (warps / 4.0));
  }
  cudaFree(d);
}
int main() {
  run<0>("4lop3"); run<1>("4lop3+4mad"); run<2>("4lop3+1wide"); run<3>("4lop3+2wide"); run<4>("4lop3+1popc"); run<5>("4lop3+1hi");
  run<6>("4lop3+1lds"); run<7>("4mad+1wide"); run<8>("4mad+1popc"); run<9>("4prmt+4mad"); run<10>("4lop3+4mad+1popc");
  run<11>("4lop3+4mad+1wide"); run<12>("4wide"); run<13>("4lop3+mad+hi"); run<14>("2popc+8mad"); run<15>("1popc+8lop3");
  run<16>("4shr+4mad"); run<17>("4add+4lop3"); run<18>("2(setp+selp)+4mad"); run<19>("4min+4mad"); run<20>("4lds+2mad+2lop3");
  return 0;
}
