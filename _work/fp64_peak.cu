// fp64_peak.cu -- stand-alone microbenchmark behind the FP64 roofline denominator of DESIGN.md section 8:
// register-resident DFMA and DMMA (mma.sync m8n8k4 / m16n8k8 f64) loops at several occupancies, then a
// 200 ms sustained loop of each.  Not linked into libdftb200.so.
// Build + run:  nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o fp64_peak fp64_peak.cu && ./fp64_peak
#include <cstdio>
#include <cuda_runtime.h>
__global__ void k_dfma(double *out, int iters) {
  double a[16]; double x = threadIdx.x * 1e-3, y = 1.0000001;
#pragma unroll
  for (int i = 0; i < 16; i++) a[i] = i;
  for (int it = 0; it < iters; it++) {
#pragma unroll
    for (int i = 0; i < 16; i++) a[i] = fma(a[i], y, x);
  }
  double s = 0;
#pragma unroll
  for (int i = 0; i < 16; i++) s += a[i];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}
template <int NACC>
__global__ void k_dmma(double *out, int iters) {
  double c[NACC][2]; double a = threadIdx.x * 1e-3, b = 1.0000001;
#pragma unroll
  for (int i = 0; i < NACC; i++) { c[i][0] = i; c[i][1] = -i; }
  for (int it = 0; it < iters; it++) {
#pragma unroll
    for (int i = 0; i < NACC; i++)
      asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                   : "+d"(c[i][0]), "+d"(c[i][1]) : "d"(a), "d"(b));
  }
  double s = 0;
#pragma unroll
  for (int i = 0; i < NACC; i++) s += c[i][0] + c[i][1];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}
template <int NACC>
__global__ void k_dmma16(double *out, int iters) {  // m16n8k8 PTX shape... 
  double c[NACC][4]; double a[4], b[2];
  for (int i = 0; i < 4; i++) a[i] = threadIdx.x * 1e-3 + i;
  b[0] = 1.0000001; b[1] = 0.999999;
#pragma unroll
  for (int i = 0; i < NACC; i++) { c[i][0] = i; c[i][1] = -i; c[i][2] = 1; c[i][3] = 2; }
  for (int it = 0; it < iters; it++) {
#pragma unroll
    for (int i = 0; i < NACC; i++)
      asm volatile("mma.sync.aligned.m16n8k8.row.col.f64.f64.f64.f64 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                   : "+d"(c[i][0]), "+d"(c[i][1]), "+d"(c[i][2]), "+d"(c[i][3])
                   : "d"(a[0]), "d"(a[1]), "d"(a[2]), "d"(a[3]), "d"(b[0]), "d"(b[1]));
  }
  double s = 0;
#pragma unroll
  for (int i = 0; i < NACC; i++) s += c[i][0] + c[i][1] + c[i][2] + c[i][3];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}
template <typename F> float timeit(F f) {
  cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
  f(); cudaDeviceSynchronize();
  cudaEventRecord(e0); f(); cudaEventRecord(e1); cudaEventSynchronize(e1);
  float ms; cudaEventElapsedTime(&ms, e0, e1); return ms;
}
int main() {
  double *out; cudaMalloc(&out, 148 * 32 * 1024 * 8);
  int iters = 20000;
  for (int warps : {4, 8, 16, 32}) {
    int thr = warps * 32;
    for (int bps : {1, 2}) {
      int grid = 148 * bps;
      if (thr * bps > 2048) continue;
      float ms = timeit([&] { k_dfma<<<grid, thr>>>(out, iters); });
      double fl = 2.0 * 16 * iters * (double)grid * thr;
      printf("DFMA  warps/cta %2d cta/sm %d : %8.3f ms  %7.2f TF\n", warps, bps, ms, fl / ms * 1e-9);
      ms = timeit([&] { k_dmma<16><<<grid, thr>>>(out, iters / 4); });
      fl = 512.0 * 16 * (iters / 4) * (double)grid * warps;
      printf("DMMA884 x16acc warps %2d cta/sm %d : %8.3f ms  %7.2f TF\n", warps, bps, ms, fl / ms * 1e-9);
      ms = timeit([&] { k_dmma<4><<<grid, thr>>>(out, iters / 4); });
      fl = 512.0 * 4 * (iters / 4) * (double)grid * warps;
      printf("DMMA884 x4acc  warps %2d cta/sm %d : %8.3f ms  %7.2f TF\n", warps, bps, ms, fl / ms * 1e-9);
      ms = timeit([&] { k_dmma16<8><<<grid, thr>>>(out, iters / 4); });
      fl = 2.0 * 16 * 8 * 8 * 8 * (iters / 4) * (double)grid * warps;
      printf("DMMA1688 x8acc warps %2d cta/sm %d : %8.3f ms  %7.2f TF\n", warps, bps, ms, fl / ms * 1e-9);
    }
  }
  // sustained: 3 s of DMMA, print clock
  cudaDeviceProp p; cudaGetDeviceProperties(&p, 0);
  printf("SMs %d clock %d kHz L2 %d smem/blk optin %zu\n", p.multiProcessorCount, p.clockRate, p.l2CacheSize, p.sharedMemPerBlockOptin);
  for (int rep = 0; rep < 6; rep++) {
    float ms = timeit([&] { k_dmma<16><<<148 * 2, 256>>>(out, 400000); });
    double fl = 512.0 * 16 * 400000 * 296.0 * 8;
    printf("sustained DMMA rep %d: %8.3f ms %7.2f TF\n", rep, ms, fl / ms * 1e-9);
  }
  for (int rep = 0; rep < 3; rep++) {
    float ms = timeit([&] { k_dfma<<<148 * 2, 512>>>(out, 400000); });
    double fl = 2.0 * 16 * 400000 * 296.0 * 512;
    printf("sustained DFMA rep %d: %8.3f ms %7.2f TF\n", rep, ms, fl / ms * 1e-9);
  }
  return 0;
}
