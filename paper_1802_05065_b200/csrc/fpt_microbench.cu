// fpt_microbench.cu -- issue-rate microbenchmark behind DESIGN.md section 9: how many clocks per SM sub-partition a DFMA
// costs on sm_100a when other instruction classes of the hot loop (LOP3 / IADD / SEL, IMAD, IMAD.WIDE of Philox, FFMA, MUFU)
// are interleaved with it.  Stand-alone executable (python -m paper_1802_05065_b200.build --microbench); not part of the library.
// Every thread runs 8 independent chains per class; 8 warps per sub-partition; "group" = one DFMA plus the listed extras.
#include <cstdio>
#include <cuda_runtime.h>

#define DF(a) asm volatile("fma.rn.f64 %0, %0, %1, %2;" : "+d"(a) : "d"(m), "d"(c))
#define LO(x) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(x) : "r"(y), "r"(z))
#define FF(f) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(f) : "f"(fm), "f"(fc))
#define IW(w, x) asm volatile("mul.wide.u32 %0, %1, 0xD2511F53;" : "=l"(w) : "r"(x))
#define IH(h, x) asm volatile("mul.hi.u32 %0, %1, 0xD2511F53;" : "=r"(h) : "r"(x))
#define IM(h, x) asm volatile("mad.lo.u32 %0, %1, 0xD2511F53, %2;" : "=r"(h) : "r"(x), "r"(y))
#define SE(x) asm volatile("{.reg .pred p; setp.ne.b32 p, %2, 0; selp.b32 %0, %0, %1, p;}" : "+r"(x) : "r"(y), "r"(pp))
#define MU(f) asm volatile("rcp.approx.ftz.f32 %0, %0;" : "+f"(f))

enum { D = 1, L = 2, F = 4, W = 8, H = 16, M = 32, S = 64, U = 128, F2 = 256, F3 = 512, D2 = 1024, D3 = 2048, L2 = 4096 };

template <int MODE>
__global__ void __launch_bounds__(256) mix_kernel(double* sink, int iters, double m, double c, unsigned y, unsigned z,
                                                  float fm, float fc) {
  double a[8];
  unsigned x[8], h[8];
  float f[8];
  unsigned long long w[8];
  const int pp = (int)(y & 1);
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    a[i] = threadIdx.x * 1e-3 + i; x[i] = threadIdx.x + i; f[i] = threadIdx.x + i; w[i] = 0; h[i] = i;
  }
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int u = 0; u < 4; ++u) {
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        if (MODE & D) DF(a[i]);
        if (MODE & D2) DF(a[(i + 1) & 7]);
        if (MODE & D3) { DF(a[(i + 1) & 7]); DF(a[(i + 2) & 7]); }
        if (MODE & L) LO(x[i]);
        if (MODE & L2) LO(x[(i + 2) & 7]);
        if (MODE & F) FF(f[i]);
        if (MODE & F2) { FF(f[i]); FF(f[(i + 1) & 7]); }
        if (MODE & F3) { FF(f[i]); FF(f[(i + 1) & 7]); FF(f[(i + 2) & 7]); }
        if (MODE & W) { IW(w[i], x[i]); x[i] = (unsigned)(w[i] >> 32); }
        if (MODE & H) { IH(h[i], x[i]); x[i] = h[i]; }
        if (MODE & M) { IM(h[i], x[i]); x[i] = h[i]; }
        if (MODE & S) SE(x[i]);
        if (MODE & U) MU(f[i]);
      }
    }
  }
  double s = 0; unsigned xs = 0; float fs = 0;
#pragma unroll
  for (int i = 0; i < 8; ++i) { s += a[i]; xs += x[i] + h[i] + (unsigned)w[i]; fs += f[i]; }
  if (s == 123.456 && xs == 77 && fs == 1.5f) sink[0] = s;
}

template <int MODE>
void run(const char* name, double sm_clock_hz, int block = 256, int per_sm = 4) {
  double* sink = nullptr;
  cudaMalloc(&sink, 8);
  const int iters = 2000;
  int sms = 0;
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, 0);
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  mix_kernel<MODE><<<sms * per_sm, block>>>(sink, iters, 0.999, 1e-3, 0x1234567u, 0x89abcdefu, 0.999f, 1e-3f);
  if (cudaDeviceSynchronize() != cudaSuccess) { printf("%s: launch failed\n", name); return; }
  float best = 1e9f;
  for (int r = 0; r < 5; ++r) {
    cudaEventRecord(e0);
    mix_kernel<MODE><<<sms * per_sm, block>>>(sink, iters, 0.999, 1e-3, 0x1234567u, 0x89abcdefu, 0.999f, 1e-3f);
    cudaEventRecord(e1);
    cudaEventSynchronize(e1);
    float ms;
    cudaEventElapsedTime(&ms, e0, e1);
    if (ms < best) best = ms;
  }
  const double groups_per_warp = (double)iters * 32, warps_per_subpartition = (double)per_sm * block / 32 / 4;
  printf("| %-28s (%2d warps/sub-partition) | %8.3f | %6.2f |\n", name, per_sm * block / 128, best, best * 1e-3 * sm_clock_hz / (groups_per_warp * warps_per_subpartition));
  cudaFree(sink);
}

int main(int argc, char** argv) {
  const double clk = argc > 1 ? atof(argv[1]) * 1e6 : 1.95e9;       // SM clock in MHz (bench.py reports the one it sees)
  printf("| group (per warp, x64000)       | best ms  | clk per group per sub-partition at %.0f MHz |\n|---|---|---|\n", clk / 1e6);
  run<D>("DFMA", clk);
  run<L>("LOP3", clk);
  run<S>("SEL", clk);
  run<M>("IMAD (mad.lo)", clk);
  run<W>("IMAD.WIDE.U32", clk);
  run<H>("IMAD.HI.U32", clk);
  run<F>("FFMA", clk);
  run<D | L>("DFMA + LOP3", clk);
  run<D | S>("DFMA + SEL", clk);
  run<D | M>("DFMA + IMAD", clk);
  run<D | W>("DFMA + IMAD.WIDE", clk);
  run<D | F>("DFMA + FFMA", clk);
  run<D | F2>("DFMA + 2 FFMA", clk);
  run<D | F3>("DFMA + 3 FFMA", clk);
  run<D | U>("DFMA + MUFU", clk);
  run<D | L | F>("DFMA + LOP3 + FFMA", clk);
  run<D | L | M | L2>("DFMA + 2 LOP3 + IMAD", clk);
  run<D | W | L>("DFMA + IMAD.WIDE + LOP3", clk);
  run<D | D2 | L>("2 DFMA + LOP3", clk);
  run<D | D3 | L>("3 DFMA + LOP3", clk);
  // how many warps the FP64 pipe needs: DFMA only (8 independent chains per thread) at 1 .. 16 warps per sub-partition
  run<D>("DFMA", clk, 128, 1);
  run<D>("DFMA", clk, 128, 2);
  run<D>("DFMA", clk, 128, 3);
  run<D>("DFMA", clk, 128, 4);
  run<D>("DFMA", clk, 256, 4);
  run<D>("DFMA", clk, 256, 8);
  run<D | L>("DFMA + LOP3", clk, 128, 1);
  run<D | L>("DFMA + LOP3", clk, 128, 4);
  run<D | L>("DFMA + LOP3", clk, 256, 8);
  // fp32 variant: FFMA next to the integer classes
  run<F | L>("FFMA + LOP3", clk);
  run<F2 | L>("2 FFMA + LOP3", clk);
  run<F3 | L>("3 FFMA + LOP3", clk);
  run<F | W>("FFMA + IMAD.WIDE", clk);
  run<F3 | W>("3 FFMA + IMAD.WIDE", clk);
  run<F3 | F2 | F | W | L>("6 FFMA + IMAD.WIDE + LOP3", clk);
  run<F3 | F2 | F | L | L2>("6 FFMA + 2 LOP3", clk);
  return 0;
}
