// mb_pipes.cu - issue-rate micro-benchmarks for the roofline of the voting kernel ("first micro-benchmark
// pure IADD3, pure IMAD, pure IMAD.WIDE and the kernel's own mix; the roofline for the reported fraction is the
// measured peak of that mix").  A standalone measurement program, not part of libemu4pi.so:
//
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o mb_pipes paper_1311_5334_b200/microbench/mb_pipes.cu && ./mb_pipes
//
// Every kernel runs one instruction (or the instruction mix of the tube test) on 8 independent registers per
// thread in a long unrolled loop, 2 blocks of 1 024 threads per SM (all 64 warps resident), and reports
// lane-operations per clock and SM = instructions x threads / (elapsed x SM clock x SMs).  The SM clock is read with
// cudaDevAttrClockRate (the bench samples the real clock with nvidia-smi; both read 1 965 MHz on the B200s used).
#include <cstdio>
#include <cuda_runtime.h>

#define REP8(X) X(0) X(1) X(2) X(3) X(4) X(5) X(6) X(7)

constexpr int kIters = 4096;

template <int kOp>
__global__ void __launch_bounds__(1024, 2) k_pipe(unsigned* out, unsigned a, unsigned b, float fa, float fb) {
  unsigned r[8];
  float f[8];
  unsigned long long w[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) { r[i] = threadIdx.x * 8u + i; f[i] = (float)(threadIdx.x + i) * 1e-3f; w[i] = r[i]; }
  for (int it = 0; it < kIters; ++it) {
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      if (kOp == 0) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(f[i]) : "f"(fa), "f"(fb));
      // (the second operand of the next three is the NEIGHBOURING register, which changes every iteration: with a loop
      //  constant there ptxas folds two adds into one IADD3, drops the idempotent max and shortens the mad.wide chain)
      if (kOp == 1) asm volatile("add.s32 %0, %0, %1;" : "+r"(r[i]) : "r"(r[(i + 1) & 7]));
      if (kOp == 2) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(r[i]) : "r"(a), "r"(b));
      if (kOp == 3) asm volatile("prmt.b32 %0, %0, %1, %2;" : "+r"(r[i]) : "r"(a), "r"(b));
      if (kOp == 4) asm volatile("mad.lo.s32 %0, %0, %1, %2;" : "+r"(r[i]) : "r"(a), "r"(b));
      if (kOp == 5) asm volatile("mad.wide.u32 %0, %1, %2, %0;" : "+l"(w[i]) : "r"(a), "r"((unsigned)(w[(i + 1) & 7] >> 32)));   // the HIGH half: all 64 bits of the chain stay live
      if (kOp == 6) asm volatile("max.f32 %0, %0, %1;" : "+f"(f[i]) : "f"(f[(i + 1) & 7]));
      if (kOp == 7) asm volatile("{ .reg .pred p; setp.gt.f32 p, %0, %1; selp.f32 %0, %0, %2, p; }" : "+f"(f[i]) : "f"(fa), "f"(fb));
    }
  }
  unsigned acc = 0;
#pragma unroll
  for (int i = 0; i < 8; ++i) acc += r[i] + __float_as_uint(f[i]) + (unsigned)w[i] + (unsigned)(w[i] >> 32);
  if (acc == 0x12345678u) out[0] = acc;
}

// the instruction mix of one pair of tube tests as k_brick<kVote> issues it (profiles/r2_sass_counts.md):
// 2 LDS stand-ins (shared loads), 6 PRMT, 8 FADD, 6 FMUL, 12 FFMA, 1 FMNMX, 3 FSETP / ISETP, 6 integer (IADD3 / LEA /
// VIMNMX) - run here without the branches and the stores, on register operands and one shared-memory table
__global__ void __launch_bounds__(1024, 2) k_mix(unsigned* out, unsigned a, float fa, float fb, float fc) {
  __shared__ unsigned tab[1024];
  tab[threadIdx.x] = threadIdx.x * 2654435761u;
  __syncthreads();
  float dx = fa, dy = fb, dz = fc, ox = 8388608.f + fa, oy = 8388608.f + fb, oz = 8388608.f + fc, T = 1e9f, band = 1e3f;
  unsigned j = threadIdx.x, cnt = 0;
  for (int it = 0; it < kIters; ++it) {
    unsigned g0, g1;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(g0) : "r"((unsigned)__cvta_generic_to_shared(tab + (j & 1023u))));
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(g1) : "r"((unsigned)__cvta_generic_to_shared(tab + ((j + 1u) & 1023u))));
    float s[2];
#pragma unroll
    for (int k = 0; k < 2; ++k) {
      const unsigned g = k ? g1 : g0;
      const float vx = __uint_as_float(__byte_perm(g, 0x4B000000u, 0x7410)) - ox;
      const float vy = __uint_as_float(__byte_perm(g, 0x4B000000u, 0x7442)) - oy;
      const float vz = __uint_as_float(__byte_perm(g, 0x4B000000u, 0x7443)) - oz;
      const float cx = __fmaf_rn(vy, dz, -__fmul_rn(vz, dy));
      const float cy = __fmaf_rn(vz, dx, -__fmul_rn(vx, dz));
      const float cz = __fmaf_rn(vx, dy, -__fmul_rn(vy, dx));
      s[k] = __fmaf_rn(cx, cx, __fmaf_rn(cy, cy, __fmul_rn(cz, cz)));
    }
    const bool clear = fminf(fabsf(s[0] - T), fabsf(s[1] - T)) > band;
    cnt += (unsigned)(clear && s[0] <= T) + (unsigned)(clear && s[1] <= T);
    j = j * a + cnt + 8u;
    ox += 1.0f; oy -= 1.0f;
  }
  if (cnt == 0x12345678u) out[0] = cnt + j;
}

template <class F>
static double time_ms(F launch) {
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  launch();
  cudaDeviceSynchronize();
  cudaEventRecord(e0);
  for (int r = 0; r < 5; ++r) launch();
  cudaEventRecord(e1);
  cudaEventSynchronize(e1);
  float ms = 0.f;
  cudaEventElapsedTime(&ms, e0, e1);
  return ms / 5.0;
}

int main() {
  int sm = 0, khz = 0;
  cudaDeviceGetAttribute(&sm, cudaDevAttrMultiProcessorCount, 0);
  cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, 0);
  unsigned* out = nullptr;
  cudaMalloc(&out, 256);
  const int blocks = sm * 2, threads = 1024;
  const double clk = (double)khz * 1e3;
  const char* names[8] = {"FFMA", "add.s32 (IADD3|IMAD.IADD)", "LOP3", "PRMT", "IMAD (mad.lo)", "mad.wide.u32 + 64-bit acc", "FMNMX", "FSETP+FSEL"};
  const double per_iter[8] = {8, 8, 8, 8, 8, 8, 8, 16};
  printf("device: %d SMs, %.0f MHz\n", sm, clk / 1e6);
  printf("%-28s %12s %22s\n", "instruction", "ms", "lane-ops / clk / SM");
  double ms[8];
  ms[0] = time_ms([&] { k_pipe<0><<<blocks, threads>>>(out, 3u, 5u, 1.0001f, 0.5f); });
  ms[1] = time_ms([&] { k_pipe<1><<<blocks, threads>>>(out, 3u, 5u, 1.0001f, 0.5f); });
  ms[2] = time_ms([&] { k_pipe<2><<<blocks, threads>>>(out, 3u, 5u, 1.0001f, 0.5f); });
  ms[3] = time_ms([&] { k_pipe<3><<<blocks, threads>>>(out, 3u, 0x3210u, 1.0001f, 0.5f); });
  ms[4] = time_ms([&] { k_pipe<4><<<blocks, threads>>>(out, 3u, 5u, 1.0001f, 0.5f); });
  ms[5] = time_ms([&] { k_pipe<5><<<blocks, threads>>>(out, 3u, 5u, 1.0001f, 0.5f); });
  ms[6] = time_ms([&] { k_pipe<6><<<blocks, threads>>>(out, 3u, 5u, 1.0001f, 0.5f); });
  ms[7] = time_ms([&] { k_pipe<7><<<blocks, threads>>>(out, 3u, 5u, 1.0001f, 0.5f); });
  for (int k = 0; k < 8; ++k)
    printf("%-28s %12.4f %22.1f\n", names[k], ms[k], per_iter[k] * kIters * (double)blocks * threads / (ms[k] * 1e-3 * clk * sm));
  const double mix_ms = time_ms([&] { k_mix<<<blocks, threads>>>(out, 1664525u, 3.f, 5.f, 7.f); });
  // instructions of one iteration of k_mix are counted from its SASS (cuobjdump -sass mb_pipes | the loop of k_mix):
  // the figure printed is per SOURCE iteration; multiply by the SASS count to get lane-instructions per clock
  printf("%-28s %12.4f %22s\n", "tube-test mix", mix_ms, "(see iterations/clk)");
  printf("tube-test mix: %.3f pair-iterations / clk / SM per lane-group of 32 = %.2f lane-pairs / clk / SM\n",
         (double)kIters * blocks * threads / 32.0 / (mix_ms * 1e-3 * clk * sm), (double)kIters * blocks * threads / (mix_ms * 1e-3 * clk * sm));
  cudaFree(out);
  return 0;
}
