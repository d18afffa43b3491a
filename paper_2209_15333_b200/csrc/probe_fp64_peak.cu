// fp64 DFMA peak, fp64 divide / sqrt rate and HBM copy bandwidth probe: the "alu" roofline denominator of DESIGN.md section 8.
// Build + run: nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o probe_fp64_peak paper_2209_15333_b200/csrc/probe_fp64_peak.cu && ./probe_fp64_peak
#include <cstdio>
#include <cuda_runtime.h>
__global__ void dfma_kernel(double* out, int iters, double a, double b) {
  double x0 = threadIdx.x, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0+4, x5=x0+5, x6=x0+6, x7=x0+7;
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
      x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
    }
  }
  out[blockIdx.x * blockDim.x + threadIdx.x] = x0 + x1 + x2 + x3 + x4 + x5 + x6 + x7;
}
__global__ void copy_kernel(const double2* __restrict__ a, double2* __restrict__ b, size_t n) {
  size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x;
  size_t stride = (size_t)gridDim.x * blockDim.x;
  for (; i < n; i += stride) b[i] = a[i];
}
__global__ void ddiv_kernel(double* out, int iters, double a) {
  double x0 = threadIdx.x + 1.5, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3;
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int u = 0; u < 8; ++u) { x0 = a / x0 + 1.0; x1 = a / x1 + 1.0; x2 = a / x2 + 1.0; x3 = a / x3 + 1.0; }
  }
  out[blockIdx.x * blockDim.x + threadIdx.x] = x0 + x1 + x2 + x3;
}
__global__ void dsqrt_kernel(double* out, int iters, double a) {
  double x0 = threadIdx.x + 1.5, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3;
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int u = 0; u < 8; ++u) { x0 = sqrt(x0) + a; x1 = sqrt(x1) + a; x2 = sqrt(x2) + a; x3 = sqrt(x3) + a; }
  }
  out[blockIdx.x * blockDim.x + threadIdx.x] = x0 + x1 + x2 + x3;
}
int main() {
  cudaDeviceProp p; cudaGetDeviceProperties(&p, 0);
  printf("dev %s SMs %d clock %d kHz smem/blk optin %zu\n", p.name, p.multiProcessorCount, p.clockRate, p.sharedMemPerBlockOptin);
  double* out; cudaMalloc(&out, 148 * 32 * 1024 * 8);
  cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
  for (int tpb : {128, 256, 512, 1024}) for (int bps : {1, 2, 4}) {
    if (tpb * bps > 2048) continue;
    int iters = 20000;
    dfma_kernel<<<148 * bps, tpb>>>(out, 1000, 1.0000001, 1e-9);
    cudaEventRecord(e0);
    dfma_kernel<<<148 * bps, tpb>>>(out, iters, 1.0000001, 1e-9);
    cudaEventRecord(e1); cudaEventSynchronize(e1);
    float ms; cudaEventElapsedTime(&ms, e0, e1);
    double flops = 2.0 * 64 * iters * 148.0 * bps * tpb;
    printf("dfma tpb %4d bps %d : %.3f ms  %.2f TFLOP/s\n", tpb, bps, ms, flops / ms * 1e-9);
  }
  { // sustained 3 s
    cudaEventRecord(e0);
    int n = 0; float ms = 0;
    while (ms < 3000) { dfma_kernel<<<148 * 2, 512>>>(out, 100000, 1.0000001, 1e-9); ++n; cudaEventRecord(e1); cudaEventSynchronize(e1); cudaEventElapsedTime(&ms, e0, e1); }
    double flops = 2.0 * 64 * 100000 * 148.0 * 2 * 512 * n;
    printf("dfma sustained %d launches %.1f ms: %.2f TFLOP/s\n", n, ms, flops / ms * 1e-9);
  }
  {
    int iters = 2000;
    cudaEventRecord(e0); ddiv_kernel<<<148 * 2, 512>>>(out, iters, 3.7); cudaEventRecord(e1); cudaEventSynchronize(e1);
    float ms; cudaEventElapsedTime(&ms, e0, e1);
    double ndiv = 32.0 * iters * 148 * 2 * 512;
    printf("ddiv: %.3f ms  %.3f Tdiv/s (=> %.1f dfma-equiv per div+add at 37 TF)\n", ms, ndiv / ms * 1e-9, 18.5e12 / (ndiv / ms * 1e3));
    cudaEventRecord(e0); dsqrt_kernel<<<148 * 2, 512>>>(out, iters, 3.7); cudaEventRecord(e1); cudaEventSynchronize(e1);
    cudaEventElapsedTime(&ms, e0, e1);
    printf("dsqrt: %.3f ms  %.3f Tsqrt/s\n", ms, ndiv / ms * 1e-9);
  }
  size_t n = (size_t)1 << 30;  // 1 GiB each
  double2 *a, *b; cudaMalloc(&a, n); cudaMalloc(&b, n); cudaMemset(a, 1, n);
  for (int g : {148 * 4, 148 * 8, 148 * 16, 148 * 32}) {
    copy_kernel<<<g, 512>>>(a, b, n / 16);
    cudaEventRecord(e0);
    for (int r = 0; r < 5; ++r) copy_kernel<<<g, 512>>>(a, b, n / 16);
    cudaEventRecord(e1); cudaEventSynchronize(e1);
    float ms; cudaEventElapsedTime(&ms, e0, e1);
    printf("copy grid %d: %.1f GB/s\n", g, 5 * 2.0 * n / ms * 1e-6);
  }
  cudaEventRecord(e0);
  for (int r = 0; r < 5; ++r) cudaMemcpyAsync(b, a, n, cudaMemcpyDeviceToDevice);
  cudaEventRecord(e1); cudaEventSynchronize(e1);
  float ms; cudaEventElapsedTime(&ms, e0, e1);
  printf("cudaMemcpy D2D: %.1f GB/s\n", 5 * 2.0 * n / ms * 1e-6);
  printf("err %s\n", cudaGetErrorString(cudaGetLastError()));
  return 0;
}
