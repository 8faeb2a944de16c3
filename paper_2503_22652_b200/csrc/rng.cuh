// Counter-based N(0,1): splitmix64 of (base + index), Box-Muller.  The same map is implemented by
// workloads/noise.py (random numbers are INPUTS of the method, reading S11): used by the debug noise hook
// (elementwise.cu) and for the Lanczos start vector of rchfsi_estimate_bounds (bounds.cu).
#pragma once
#include <stdint.h>

namespace rchfsi {

__host__ __device__ __forceinline__ uint64_t splitmix64(uint64_t x) {
  x += 0x9E3779B97F4A7C15ull;
  uint64_t z = x;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}
__device__ __forceinline__ double counter_gauss(uint64_t base, uint64_t idx) {
  const uint64_t k1 = splitmix64(base + idx);
  const uint64_t k2 = splitmix64(k1);
  const double u1 = ((double)(k1 >> 11) + 0.5) * (1.0 / 9007199254740992.0);
  const double u2 = ((double)(k2 >> 11) + 0.5) * (1.0 / 9007199254740992.0);
  return sqrt(-2.0 * log(u1)) * cos(2.0 * 3.14159265358979323846 * u2);
}

}  // namespace rchfsi
