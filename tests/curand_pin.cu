// curand_pin.cu — TEST ONLY (built by tests/test_gpu_curand_pin.py with nvcc on the GPU box; not part of the library and
// not of the oracle).  SURVEY.md §8(c) pin P-1: cuRAND's CURAND_RNG_PSEUDO_PHILOX4_32_10 is the independent implementation
// of Philox4x32-10 that is available on the box.  curand_init(seed, subsequence, offset) sets key = (seed lo, seed hi) and
// the 128-bit counter to (offset / 4) + (subsequence << 64), so subsequence = step and offset = 4 * id is exactly the
// counter (id lo, id hi, step, 0) of DESIGN.md §3.0, and curand4() returns the four words of that block.
#include <curand_kernel.h>
#include <stdint.h>

__global__ void curand_blocks_kernel(unsigned long long seed, unsigned long long id_base, unsigned step,
                                     unsigned long long n, uint4* out) {
  const unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  curandStatePhilox4_32_10_t st;
  curand_init(seed, (unsigned long long)step, 4ull * (id_base + i), &st);
  out[i] = curand4(&st);
}

extern "C" int curand_philox_blocks(unsigned long long seed, unsigned long long id_base, unsigned step,
                                    unsigned long long n, void* d_out) {
  if (n == 0) return 0;
  curand_blocks_kernel<<<(unsigned)((n + 255) / 256), 256>>>(seed, id_base, step, n, (uint4*)d_out);
  return (int)cudaDeviceSynchronize();
}
