// Common device helpers for the BSE hot-path kernels (sm_100a).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace bse {

constexpr int TB = 64;                 // tile edge (complex elements)
constexpr int TILE_BYTES = TB * TB * 16;
constexpr int PATCH_BYTES = 8 * 8 * 16;

// Slot (16-byte unit) of entry (a, b), 0 <= a, b < 8, inside an 8 x 8 patch.  Chosen so that both
// DMMA fragment reads of the apply kernel -- lanes (g, t) reading (a = g, b = 4s + t) and
// (a = 4s + t, b = g) -- touch 8 distinct 16-byte bank groups per quarter-warp (see include/bse.h).
__host__ __device__ __forceinline__ int patch_slot(int a, int b)
{
    int r = ((a >> 2) << 2) | ((b >> 2) << 1) | ((a >> 1) & 1);
    int c = ((a & 1) << 2) | ((b & 1) << 1) | (((a >> 1) ^ (b >> 1)) & 1);
    return r * 8 + c;
}
// Byte offset of entry (il, jl), 0 <= il, jl < 64, inside a tile.
__host__ __device__ __forceinline__ int tile_offset(int il, int jl)
{
    return ((jl >> 3) * 8 + (il >> 3)) * PATCH_BYTES + patch_slot(il & 7, jl & 7) * 16;
}
__host__ __device__ __forceinline__ int64_t tile_index(int64_t I, int64_t J) { return I * (I + 1) / 2 + J; }

// Storage type of the tile store: ES = bytes per complex entry, 16 (complex128) or 8 (complex64: the paper's
// matrices are single precision; converted to FP64 when a fragment is loaded, all arithmetic
// stays FP64).  Same tile order, same patch order, same slot function: only the slot size changes, and with 8-byte
// slots both fragment reads touch 16 distinct 8-byte bank pairs per half-warp (slot mod 16 is a bijection of the
// four lane bits of a half-warp for both offP1 and offP2), i.e. LDS.64 without bank conflicts.
constexpr int ES_C128 = 16, ES_C64 = 8;
__host__ __device__ __forceinline__ int64_t tile_bytes_es(int es) { return (int64_t)TB * TB * es; }
__host__ __device__ __forceinline__ int tile_offset_es(int il, int jl, int es) { return (tile_offset(il, jl) >> 4) * es; }

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t *b, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *b, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(b)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t *b)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(b)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *b, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}" ::"r"(smem_u32(b)), "r"(parity) : "memory");
}
// TMA bulk copy global -> shared, completion signalled on an mbarrier (SASS: UBLKCP).
__device__ __forceinline__ void bulk_g2s(void *dst_smem, const void *src_gmem, uint32_t bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst_smem)),
                 "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
// Same, with an L2 eviction-priority hint (createpolicy): the operand stream is read once and must not push the
// L2-resident X and Y blocks out (measured at N = 98304: 1.7 GB of DRAM writes for a 6 MB Y without the hint).
__device__ __forceinline__ uint64_t l2_policy_evict_first()
{
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
__device__ __forceinline__ void bulk_g2s_hint(void *dst_smem, const void *src_gmem, uint32_t bytes, uint64_t *bar,
                                              uint64_t policy)
{
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(
            smem_u32(dst_smem)),
        "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar)), "l"(policy)
        : "memory");
}
__device__ __forceinline__ void fence_barrier_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

__device__ __forceinline__ void cp_async16(void *dst, const void *src, bool valid)
{
    int sz = valid ? 16 : 0;
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(smem_u32(dst)), "l"(src), "r"(sz) : "memory");
}
__device__ __forceinline__ void cp_async8(void *dst, const void *src, bool valid)
{
    int sz = valid ? 8 : 0;
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;" ::"r"(smem_u32(dst)), "l"(src), "r"(sz) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

__device__ __forceinline__ double2 lds128(uint32_t addr)
{
    double2 v;
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(addr));
    return v;
}
// One fragment entry (re, im) as doubles from a tile in shared memory.
template <int ES> __device__ __forceinline__ double2 load_frag(const char *p);
template <> __device__ __forceinline__ double2 load_frag<16>(const char *p) { return *reinterpret_cast<const double2 *>(p); }
// F2F.F64.F32 runs at 16 results/clk/SM (measured); re-biasing the exponent with integer ops instead was measured
// slower in both kernels (9.3 vs 8.6 ms at k = 1, 12.2 vs 11.0 ms at k = 4, N = 98304), so the conversion stays.
template <> __device__ __forceinline__ double2 load_frag<8>(const char *p)
{
    const float2 f = *reinterpret_cast<const float2 *>(p);
    return make_double2((double)f.x, (double)f.y);
}
// FP64 tensor-core MMA, D(8x8) += A(8x4, row) * B(4x8, col).  SASS: DMMA.8x8x4.
// Fragments: lane = 4 g + t;  a = A[g][t];  b = B[t][g];  c[0..1] = C[g][2t .. 2t+1].
__device__ __forceinline__ void dmma(double (&c)[2], double a, double b)
{
    // volatile: keeps the hand-interleaved order of independent accumulator chains (ptxas otherwise schedules
    // dependent DMMAs back to back, paying the 26-cycle latency instead of the 16-cycle issue interval)
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};"
                 : "+d"(c[0]), "+d"(c[1])
                 : "d"(a), "d"(b));
}
// v or -v (mask = SIGN_BIT) without touching the FP64 pipe, whose instructions share the issue port of the DMMAs
constexpr unsigned long long SIGN_BIT = 0x8000000000000000ull;
__device__ __forceinline__ double neg_if(double v, unsigned long long mask)
{
    return __longlong_as_double(__double_as_longlong(v) ^ (long long)mask);
}
__device__ __forceinline__ void red_add(double *p, double v) { atomicAdd(p, v); }

}  // namespace bse
