// afs_bits.cuh -- bit-word helpers shared by the kernels: restarts are packed 32 to a word (bit r = restart r of a tile).
#pragma once
#include <stdint.h>

namespace afs {

constexpr unsigned FULL = 0xffffffffu;

// Column sums of a 32 x 32 bit matrix held one row per lane: returns, in lane r, the number of lanes whose word has
// bit r set.  Five butterfly steps; after step s a lane keeps the 32 >> s columns whose low s bits match its own lane
// index, as packed (s+1)-bit counters.
__device__ __forceinline__ int bit_column_sums(uint32_t w, int lane)
{
    uint32_t o;
    o = __shfl_xor_sync(FULL, w, 1);
    w = (lane & 1) ? ((w >> 1) & 0x55555555u) + ((o >> 1) & 0x55555555u) : (w & 0x55555555u) + (o & 0x55555555u);
    o = __shfl_xor_sync(FULL, w, 2);
    w = (lane & 2) ? ((w >> 2) & 0x33333333u) + ((o >> 2) & 0x33333333u) : (w & 0x33333333u) + (o & 0x33333333u);
    o = __shfl_xor_sync(FULL, w, 4);
    w = (lane & 4) ? ((w >> 4) & 0x0f0f0f0fu) + ((o >> 4) & 0x0f0f0f0fu) : (w & 0x0f0f0f0fu) + (o & 0x0f0f0f0fu);
    o = __shfl_xor_sync(FULL, w, 8);
    w = (lane & 8) ? ((w >> 8) & 0x00ff00ffu) + ((o >> 8) & 0x00ff00ffu) : (w & 0x00ff00ffu) + (o & 0x00ff00ffu);
    o = __shfl_xor_sync(FULL, w, 16);
    w = (lane & 16) ? (w >> 16) + (o >> 16) : (w & 0xffffu) + (o & 0xffffu);
    return (int)w;
}

// Transpose of a 32 x 32 bit matrix held one row per lane (bit j of lane i  ->  bit i of lane j): five butterfly steps.
__device__ __forceinline__ uint32_t transpose32(uint32_t x, int lane)
{
    uint32_t y;
    y = __shfl_xor_sync(FULL, x, 16);
    x = (lane & 16) ? ((x & 0xffff0000u) | (y >> 16)) : ((x & 0x0000ffffu) | (y << 16));
    y = __shfl_xor_sync(FULL, x, 8);
    x = (lane & 8) ? ((x & 0xff00ff00u) | ((y >> 8) & 0x00ff00ffu)) : ((x & 0x00ff00ffu) | ((y << 8) & 0xff00ff00u));
    y = __shfl_xor_sync(FULL, x, 4);
    x = (lane & 4) ? ((x & 0xf0f0f0f0u) | ((y >> 4) & 0x0f0f0f0fu)) : ((x & 0x0f0f0f0fu) | ((y << 4) & 0xf0f0f0f0u));
    y = __shfl_xor_sync(FULL, x, 2);
    x = (lane & 2) ? ((x & 0xccccccccu) | ((y >> 2) & 0x33333333u)) : ((x & 0x33333333u) | ((y << 2) & 0xccccccccu));
    y = __shfl_xor_sync(FULL, x, 1);
    x = (lane & 1) ? ((x & 0xaaaaaaaau) | ((y >> 1) & 0x55555555u)) : ((x & 0x55555555u) | ((y << 1) & 0xaaaaaaaau));
    return x;
}

}  // namespace afs
