// cub_sort_compare.cu — COMPARISON ONLY (north_star: "a hand-written device radix sort ... (CUB only as a comparison)").
// Built into its own library (libfdgs_cubcmp.so), loaded only by `python -m paper_2412_20720_b200.sweep --sort-compare`;
// nothing in libfdgs.so or in the product path links or calls it.
// Sorts (64-bit tile|depth key, 32-bit primitive id) pairs on key bits [0, end_bit) with cub::DeviceRadixSort — the
// single 64-bit sort of the tile rasterizer of [23] that the two-level sort of DESIGN.md section 1 replaces.
#include <cstddef>
#include <cstdint>

#include <cub/device/device_radix_sort.cuh>

extern "C" {

// temp == NULL: writes the required temporary storage size to *temp_bytes.  Returns the cudaError_t as int.
int fdgs_cmp_cub_sort_pairs(const unsigned long long* keys_in, unsigned long long* keys_out, const unsigned int* vals_in,
                            unsigned int* vals_out, int64_t n, int end_bit, void* temp, size_t* temp_bytes, void* stream) {
  if (!temp_bytes) return (int)cudaErrorInvalidValue;
  return (int)cub::DeviceRadixSort::SortPairs(temp, *temp_bytes, keys_in, keys_out, vals_in, vals_out, n, 0, end_bit, (cudaStream_t)stream);
}

}  // extern "C"
