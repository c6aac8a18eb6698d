// lv_sort.cu -- A3: stable LSD radix sort of (cell key, slot) pairs
// ("arrange NPs into the cells (by second indexing)").
// Uses the on-board radix sort (CUB DeviceRadixSort, shipped with the CUDA
// toolkit) restricted to the key bits in use; LSD radix sort is stable, which
// the permutation contract (DESIGN.md fp32 contract #3) relies on.
#include <cub/device/device_radix_sort.cuh>

#include "lv_internal.cuh"

size_t lvs_temp_bytes(int n, int end_bit)
{
    size_t bytes = 0;
    cub::DeviceRadixSort::SortPairs(nullptr, bytes, (const uint32_t *)nullptr, (uint32_t *)nullptr,
                                    (const uint32_t *)nullptr, (uint32_t *)nullptr, n > 0 ? n : 1, 0,
                                    end_bit, (cudaStream_t)0);
    return bytes;
}

cudaError_t lvs_sort_pairs(void *temp, size_t temp_bytes, const uint32_t *key_in, uint32_t *key_out,
                           const uint32_t *val_in, uint32_t *val_out, int n, int end_bit,
                           cudaStream_t st)
{
    return cub::DeviceRadixSort::SortPairs(temp, temp_bytes, key_in, key_out, val_in, val_out, n, 0,
                                           end_bit, st);
}
