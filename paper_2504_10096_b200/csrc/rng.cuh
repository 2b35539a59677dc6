// Counter-based generator shared by the device-side input generators and the solver's start block.
#pragma once
#include "bse_common.cuh"

namespace bse {

// ---- counter-based generator: identical integer arithmetic to bse_inputs/__init__.py -------------------
__device__ __forceinline__ uint64_t mix64(uint64_t z)
{
    z ^= z >> 30; z *= 0xBF58476D1CE4E5B9ull;
    z ^= z >> 27; z *= 0x94D049BB133111EBull;
    z ^= z >> 31;
    return z;
}
__device__ __forceinline__ void hash2(uint64_t h0, uint64_t i, uint64_t j, uint64_t &h2, uint64_t &h3)
{
    uint64_t h1 = mix64(h0 + i * 0xD1B54A32D192ED03ull);
    h2 = mix64(h1 ^ (j * 0x8CB92BA72F3D8DD7ull));
    h3 = mix64(h2 + 0x9E3779B97F4A7C15ull);
}
__host__ __device__ __forceinline__ uint64_t stream_key(uint64_t seed, uint64_t stream)
{
    uint64_t z = seed ^ (stream * 0x9E3779B97F4A7C15ull);
    z ^= z >> 30; z *= 0xBF58476D1CE4E5B9ull;
    z ^= z >> 27; z *= 0x94D049BB133111EBull;
    z ^= z >> 31;
    return z;
}
__device__ __forceinline__ double u01(uint64_t h) { return ((double)(h >> 12) + 0.5) * 0x1.0p-52; }
__device__ __forceinline__ double2 normal_pair(uint64_t h0, uint64_t i, uint64_t j)
{
    uint64_t h2, h3;
    hash2(h0, i, j, h2, h3);
    double r = sqrt(-2.0 * log(u01(h2)));
    double th = 6.283185307179586 * u01(h3);
    double s, c;
    sincos(th, &s, &c);
    return make_double2(r * c, r * s);
}

}  // namespace bse
