// B3: stable LSD radix sort of (63-bit key, 32-bit index) pairs (the paper sorts with
// cub::DeviceRadixSort::SortPairs).  Bring-up version: the CUB one-sweep sort that ships with the CUDA
// toolkit, restricted to the 63 significant key bits; ties keep ascending original index (LSD radix is stable).
#include "gothic_ctx.cuh"
#include <cub/device/device_radix_sort.cuh>

size_t gothic_sort_scratch_bytes(uint32_t n_max)
{
    size_t bytes = 0;
    cub::DoubleBuffer<uint64_t> k(nullptr, nullptr);
    cub::DoubleBuffer<uint32_t> v(nullptr, nullptr);
    cub::DeviceRadixSort::SortPairs(nullptr, bytes, k, v, (int)n_max, 0, 63);
    return bytes + 256;
}

int gothic_stage_sort(gothic_ctx *c, uint32_t n, cudaStream_t s)
{
    cub::DoubleBuffer<uint64_t> k(c->key[c->cur], c->key[c->cur ^ 1]);
    cub::DoubleBuffer<uint32_t> v(c->idx[c->cur], c->idx[c->cur ^ 1]);
    size_t bytes = c->sort_tmp_bytes;
    GOTHIC_CUDA_OK(c, cub::DeviceRadixSort::SortPairs(c->sort_tmp, bytes, k, v, (int)n, 0, 63, s));
    c->launches += 9; // histogram + 8 one-sweep digit passes
    c->cur = (k.Current() == c->key[0]) ? 0 : 1;
    if (v.Current() != c->idx[c->cur]) return GOTHIC_ERR_CUDA;
    return GOTHIC_OK;
}
