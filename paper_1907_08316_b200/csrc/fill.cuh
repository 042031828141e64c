// fill.cuh -- device side of the counter-based uniform generator of the config-4 sweep
// microbenchmark.  The recipe (restated, not shared code):
//   x = g + 0x9E3779B97F4A7C15*(tag+1) + 0xD1B54A32D192ED03*seed   (mod 2^64)
//   x ^= x>>30; x *= 0xBF58476D1CE4E5B9; x ^= x>>27; x *= 0x94D049BB133111EB; x ^= x>>31
//   U = (x >> 11) * 2^-53  in [0,1), then rounded to T.
// It draws inputs; it is not part of the method's arithmetic.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace sldg {

template <typename T>
__global__ void fill_uniform_kernel(T *__restrict__ f, long ndof, unsigned long long seed,
                                    unsigned tag) {
    const unsigned long long off =
        0x9E3779B97F4A7C15ull * (unsigned long long)(tag + 1u) + 0xD1B54A32D192ED03ull * seed;
    for (long g = (long)blockIdx.x * blockDim.x + threadIdx.x; g < ndof;
         g += (long)gridDim.x * blockDim.x) {
        unsigned long long x = (unsigned long long)g + off;
        x ^= x >> 30; x *= 0xBF58476D1CE4E5B9ull;
        x ^= x >> 27; x *= 0x94D049BB133111EBull;
        x ^= x >> 31;
        double u = (double)(x >> 11) * 0x1.0p-53;
        f[g] = (T)u;
    }
}

}  // namespace sldg
