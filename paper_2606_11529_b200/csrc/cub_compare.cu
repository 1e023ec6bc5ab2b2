// cub_compare.cu -- NOT part of libxpr.so and never on the product path: a separate library (libxpr_cubcmp.so,
// built by build.py --cub-compare, loaded only by `bench.py --sort-compare`) that runs the library radix sort
// cub::DeviceRadixSort::SortPairs on the same (key, value) pairs, as the comparison BASELINE.json:north_star asks for
// ("the onesweep-style radix sort ... CUB is timed only as a comparison").
#include <cub/device/device_radix_sort.cuh>
#include <cuda_runtime.h>
#include <stdint.h>

// temp == NULL: *temp_bytes receives the scratch size.  Sorts bits [begin_bit, end_bit) of the 64-bit keys, stable.
extern "C" int32_t xpr_cubcmp_sort_pairs(int64_t n, const uint64_t* keys_in, const uint32_t* vals_in, uint64_t* keys_out,
                                         uint32_t* vals_out, void* temp, size_t* temp_bytes, int32_t begin_bit,
                                         int32_t end_bit, void* stream) {
    if (n < 0 || n > 0x7fffffffLL || !temp_bytes) return 1;
    size_t bytes = *temp_bytes;
    const cudaError_t e = cub::DeviceRadixSort::SortPairs(temp, bytes, keys_in, keys_out, vals_in, vals_out, (int)n, begin_bit,
                                                          end_bit, (cudaStream_t)stream);
    if (!temp) *temp_bytes = bytes;
    return e == cudaSuccess ? 0 : 3;
}
