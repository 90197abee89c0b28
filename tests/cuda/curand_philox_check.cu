// curand_philox_check.cu -- test-only: the CUDA toolkit's own Philox4x32-10 (curand_philox4x32_x.h,
// curand_Philox4x32_10(counter, key)) on n (ctr[4], key[2]) pairs, as an INDEPENDENT third implementation
// for pin P8(i) of SURVEY.md 8(c): the product's device Philox and the oracle's are both compared with it.
// Not part of the product library and not part of the oracle; built by tests/helpers.py.
#include <cuda_runtime.h>
#include <curand_philox4x32_x.h>
#include <stdint.h>

__global__ void toolkit_philox_kernel(const uint4 *ctr, const uint2 *key, uint4 *out, long long n) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) out[i] = curand_Philox4x32_10(ctr[i], key[i]);
}

extern "C" int toolkit_philox4x32_10(int device, const uint32_t *ctr, const uint32_t *key, uint32_t *out, uint64_t n) {
  if (cudaSetDevice(device) != cudaSuccess) return -4;
  uint4 *dc = nullptr, *dout = nullptr;
  uint2 *dk = nullptr;
  int rc = 0;
  if (cudaMalloc(&dc, n * 16) != cudaSuccess || cudaMalloc(&dk, n * 8) != cudaSuccess || cudaMalloc(&dout, n * 16) != cudaSuccess) rc = -5;
  if (rc == 0) {
    cudaMemcpy(dc, ctr, n * 16, cudaMemcpyHostToDevice);
    cudaMemcpy(dk, key, n * 8, cudaMemcpyHostToDevice);
    toolkit_philox_kernel<<<(unsigned)((n + 255) / 256), 256>>>(dc, dk, dout, (long long)n);
    if (cudaMemcpy(out, dout, n * 16, cudaMemcpyDeviceToHost) != cudaSuccess) rc = -4;
  }
  cudaFree(dc); cudaFree(dk); cudaFree(dout);
  return rc;
}
