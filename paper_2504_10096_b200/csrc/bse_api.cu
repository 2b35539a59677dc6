// C-ABI entry points: layout, pack / generators, handle, apply.  (orth: bse_orth.cu, solve: bse_solve.cu)
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <new>

#include "bse_common.cuh"
#include "bse_internal.h"
#include "tile_layout.cuh"

namespace bse {

std::atomic<int64_t> g_launches{0};

static bse_status_t grow(void **p, size_t *have, size_t want)
{
    if (*have >= want) return BSE_OK;
    if (*have && want < *have + *have / 2) want = *have + *have / 2;      // geometric growth: no realloc per step
    if (*p) cudaFree(*p);
    *p = nullptr;
    *have = 0;
    if (cudaMalloc(p, want) != cudaSuccess) { cudaGetLastError(); return BSE_ERR_ALLOC; }
    *have = want;
    return BSE_OK;
}
bse_status_t ensure_ws(bse_handle_s *h, size_t bytes) { return grow(&h->ws, &h->ws_bytes, bytes); }
bse_status_t ensure_ws2(bse_handle_s *h, size_t bytes) { return grow(&h->ws2, &h->ws2_bytes, bytes); }
bse_status_t ensure_pin(bse_handle_s *h, size_t bytes)
{
    if (h->hpin_bytes >= bytes) return BSE_OK;
    if (h->hpin_bytes && bytes < 2 * h->hpin_bytes) bytes = 2 * h->hpin_bytes;
    if (h->hpin) cudaFreeHost(h->hpin);
    h->hpin = nullptr;
    h->hpin_bytes = 0;
    if (cudaMallocHost(&h->hpin, bytes) != cudaSuccess) { cudaGetLastError(); return BSE_ERR_ALLOC; }
    h->hpin_bytes = bytes;
    return BSE_OK;
}

static void tile_grid(int64_t n_tiles, dim3 &grid)
{
    int64_t gy = n_tiles < 32768 ? n_tiles : 32768;
    int64_t gz = (n_tiles + gy - 1) / gy;
    grid = dim3(TB * TB / 256, (unsigned)gy, (unsigned)gz);
}

bse_status_t zero_block(bse_handle_s *h, void *dY, int64_t ldy, int64_t rows, int32_t k)
{
    BSE_CUDA(cudaMemset2DAsync(dY, (size_t)ldy * 16, 0, (size_t)rows * 16, (size_t)k, h->stream));
    return BSE_OK;
}

bse_status_t comm_sum_block(bse_handle_s *h, void *dY, int64_t ld, int64_t rows, int k)
{
    if (!h->comm) return BSE_OK;
    if (ld == rows) return h->comm(h->comm_user, BSE_COMM_SUM, dY, 2 * rows * k) ? BSE_ERR_INTERNAL : BSE_OK;
    for (int c = 0; c < k; ++c)
        if (h->comm(h->comm_user, BSE_COMM_SUM, (char *)dY + (size_t)c * ld * 16, 2 * rows)) return BSE_ERR_INTERNAL;
    return BSE_OK;
}
bse_status_t comm_bcast_dev(bse_handle_s *h, void *dBuf, int64_t n_doubles)
{
    if (!h->comm || n_doubles <= 0) return BSE_OK;
    return h->comm(h->comm_user, BSE_COMM_BCAST, dBuf, n_doubles) ? BSE_ERR_INTERNAL : BSE_OK;
}
bse_status_t comm_sum_dev(bse_handle_s *h, void *dBuf, int64_t n_doubles)
{
    if (!h->comm || n_doubles <= 0) return BSE_OK;
    return h->comm(h->comm_user, BSE_COMM_SUM, dBuf, n_doubles) ? BSE_ERR_INTERNAL : BSE_OK;
}
bse_status_t comm_bcast_host(bse_handle_s *h, void *hBuf, size_t bytes)
{
    if (!h->comm || bytes == 0) return BSE_OK;
    const size_t padded = (bytes + 7) / 8 * 8;
    if (h->comm_buf_bytes < padded) {
        if (h->comm_buf) cudaFree(h->comm_buf);
        h->comm_buf = nullptr;
        h->comm_buf_bytes = 0;
        if (cudaMalloc(&h->comm_buf, padded) != cudaSuccess) { cudaGetLastError(); return BSE_ERR_ALLOC; }
        h->comm_buf_bytes = padded;
    }
    BSE_CUDA(cudaMemsetAsync((char *)h->comm_buf + (padded - 8), 0, 8, h->stream));
    BSE_CUDA(cudaMemcpyAsync(h->comm_buf, hBuf, bytes, cudaMemcpyHostToDevice, h->stream));
    if (h->comm(h->comm_user, BSE_COMM_BCAST, h->comm_buf, (int64_t)(padded / 8))) return BSE_ERR_INTERNAL;
    BSE_CUDA(cudaMemcpyAsync(hBuf, h->comm_buf, bytes, cudaMemcpyDeviceToHost, h->stream));
    BSE_CUDA(cudaStreamSynchronize(h->stream));
    return BSE_OK;
}

}  // namespace bse

using namespace bse;

extern "C" {

const char *bse_status_string(bse_status_t s)
{
    switch (s) {
        case BSE_OK: return "ok";
        case BSE_ERR_INVALID_ARG: return "invalid argument";
        case BSE_ERR_CUDA: return "CUDA error";
        case BSE_ERR_ALLOC: return "allocation failed";
        case BSE_ERR_NOT_CONVERGED: return "not converged";
        case BSE_ERR_NOT_POSITIVE_DEFINITE: return "operator not positive definite";
        case BSE_ERR_STATIC_LIMIT: return "size exceeds the static scratch limit";
        default: return "internal error";
    }
}

int64_t bse_launch_count(void) { return g_launches.load(); }

bse_status_t bse_host_heev(int32_t m, void *hA, int32_t lda, double *hW, void *hZ, int32_t ldz, int32_t nz)
{
    if (m < 1 || !hA || !hW || lda < m || (nz > 0 && (!hZ || ldz < m))) return BSE_ERR_INVALID_ARG;
    return host_heev(m, hA, lda, hW, hZ, ldz, nz) ? BSE_ERR_INTERNAL : BSE_OK;
}

bse_status_t bse_host_syev(int32_t m, double *hA, int32_t lda, double *hW, double *hZ, int32_t ldz, int32_t nz)
{
    if (m < 1 || !hA || lda < m || !hW || nz < 0 || (nz > 0 && (!hZ || ldz < m))) return BSE_ERR_INVALID_ARG;
    return host_syev(m, hA, lda, hW, hZ, ldz, nz) ? BSE_ERR_INTERNAL : BSE_OK;
}

bse_status_t bse_host_stev(int32_t m, const double *hD, const double *hE, double *hW, double *hZ, int32_t ldz, int32_t nz)
{
    if (m < 1 || !hD || (m > 1 && !hE) || !hW || nz < 0 || (nz > 0 && (!hZ || ldz < m))) return BSE_ERR_INVALID_ARG;
    return host_stev(m, const_cast<double *>(hD), const_cast<double *>(hE), hW, hZ, ldz, nz) ? BSE_ERR_INTERNAL : BSE_OK;
}

bse_status_t bse_host_stev_lowest(int32_t m, const double *hD, const double *hE, int32_t nz, double *hW, double *hZ, int32_t ldz)
{
    if (m < 1 || !hD || (m > 1 && !hE) || !hW || nz < 1 || nz > m || (hZ && ldz < m)) return BSE_ERR_INVALID_ARG;
    return host_stev_lowest(m, const_cast<double *>(hD), const_cast<double *>(hE), nz, hW, hZ, ldz) ? BSE_ERR_INTERNAL : BSE_OK;
}

static inline bool storage_ok(int32_t storage) { return storage == BSE_STORE_C128 || storage == BSE_STORE_C64; }
static inline bool storage_real_form(int32_t storage) { return storage == BSE_STORE_REAL_FORM || storage == BSE_STORE_REAL_FORM_C64; }
static inline int storage_es(int32_t storage)
{
    return (storage == BSE_STORE_C64 || storage == BSE_STORE_REAL_FORM_C64) ? ES_C64 : ES_C128;
}

bse_status_t bse_layout(int64_t N, int32_t storage, int32_t *tile, int64_t *n_tiles, int64_t *bytes_per_matrix)
{
    if (N < 1 || !(storage_ok(storage) || storage_real_form(storage))) return BSE_ERR_INVALID_ARG;
    int64_t nt = (N + TB - 1) / TB;
    if (tile) *tile = TB;
    if (n_tiles) *n_tiles = nt * (nt + 1) / 2;
    if (bytes_per_matrix) *bytes_per_matrix = nt * (nt + 1) / 2 * tile_bytes_es(storage_es(storage));
    return BSE_OK;
}

bse_status_t bse_pack_from_dense(const void *dDense, int64_t ld, int64_t N, int32_t which, void *dTiles,
                                 int32_t storage, void *stream)
{
    if (!dDense || !dTiles || N < 1 || ld < N || (which != 0 && which != 1) || !storage_ok(storage))
        return BSE_ERR_INVALID_ARG;
    int64_t n_tiles;
    bse_layout(N, storage, nullptr, &n_tiles, nullptr);
    dim3 grid;
    tile_grid(n_tiles, grid);
    pack_from_dense_kernel<<<grid, 256, 0, (cudaStream_t)stream>>>((const double2 *)dDense, ld, N, which,
                                                                   (char *)dTiles, storage_es(storage), n_tiles);
    count_launch();
    BSE_CUDA(cudaGetLastError());
    return BSE_OK;
}

bse_status_t bse_unpack_to_dense(const void *dTiles, int32_t storage, int64_t N, int32_t which, void *dDense,
                                 int64_t ld, void *stream)
{
    if (!dDense || !dTiles || N < 1 || ld < N || (which != 0 && which != 1) || !storage_ok(storage))
        return BSE_ERR_INVALID_ARG;
    int64_t n_tiles;
    bse_layout(N, storage, nullptr, &n_tiles, nullptr);
    dim3 grid;
    tile_grid(n_tiles, grid);
    unpack_to_dense_kernel<<<grid, 256, 0, (cudaStream_t)stream>>>((const char *)dTiles, storage_es(storage), N, which,
                                                                   (double2 *)dDense, ld, n_tiles);
    count_launch();
    BSE_CUDA(cudaGetLastError());
    return BSE_OK;
}

bse_status_t bse_fill_synthetic(void *dTiles, int32_t storage, int64_t N, int32_t which, uint64_t seed, double sigma,
                                int32_t group, void *stream)
{
    return bse_fill_synthetic_shard(dTiles, storage, N, which, seed, sigma, group, 0, (int32_t)((N + TB - 1) / TB), stream);
}

bse_status_t bse_fill_synthetic_shard(void *dTiles, int32_t storage, int64_t N, int32_t which, uint64_t seed, double sigma,
                                      int32_t group, int32_t tile_row_begin, int32_t tile_row_end, void *stream)
{
    if (!dTiles || N < 1 || (which != 0 && which != 1) || !storage_ok(storage)) return BSE_ERR_INVALID_ARG;
    if (tile_row_begin < 0 || tile_row_end < tile_row_begin || tile_row_end > (N + TB - 1) / TB) return BSE_ERR_INVALID_ARG;
    cudaStream_t s = (cudaStream_t)stream;
    double *deps = nullptr;
    if (which == 0) {
        if (group < 1 || group > 64 || N % group) return BSE_ERR_INVALID_ARG;
        if (cudaMallocAsync(&deps, sizeof(double) * N, s) != cudaSuccess) { cudaGetLastError(); return BSE_ERR_ALLOC; }
        int64_t ngroups = N / group;
        transition_energies_kernel<<<(unsigned)((ngroups + 127) / 128), 128, 0, s>>>(deps, N, group,
                                                                                    stream_key(seed, 1));
        count_launch();
    }
    const int64_t tile0 = tile_index(tile_row_begin, 0), tile1 = tile_index(tile_row_end, 0);
    if (tile1 > tile0) {
        dim3 grid;
        tile_grid(tile1 - tile0, grid);
        // the kernel addresses tiles by their global number: pass the virtual base of the whole packed store
        fill_synthetic_kernel<<<grid, 256, 0, s>>>((char *)dTiles - tile0 * tile_bytes_es(storage_es(storage)), storage_es(storage), N,
                                                   which, stream_key(seed, which == 0 ? 2 : 3), sigma, deps, tile0, tile1);
        count_launch();
    }
    if (deps) cudaFreeAsync(deps, s);
    BSE_CUDA(cudaGetLastError());
    return BSE_OK;
}

bse_status_t bse_fill_closed_form_tda(void *dTiles, int32_t storage, int64_t N, const double *dLam, const void *dU,
                                      double s, void *stream)
{
    if (!dTiles || !dLam || !dU || N < 1 || !storage_ok(storage)) return BSE_ERR_INVALID_ARG;
    int64_t n_tiles;
    bse_layout(N, storage, nullptr, &n_tiles, nullptr);
    dim3 grid;
    tile_grid(n_tiles, grid);
    fill_closed_tda_kernel<<<grid, 256, 0, (cudaStream_t)stream>>>((char *)dTiles, storage_es(storage), N, dLam, (const double2 *)dU, s,
                                                                   n_tiles);
    count_launch();
    BSE_CUDA(cudaGetLastError());
    return BSE_OK;
}

bse_status_t bse_fill_closed_form_full(void *dRTiles, void *dCTiles, int32_t storage, int64_t N, const double *dD1,
                                       const double *dD2, const double *dUr, const double *dPhi, double s1, double s2,
                                       void *stream)
{
    if (!dRTiles || !dCTiles || !dD1 || !dD2 || !dUr || !dPhi || N < 1 || !storage_ok(storage))
        return BSE_ERR_INVALID_ARG;
    int64_t n_tiles;
    bse_layout(N, storage, nullptr, &n_tiles, nullptr);
    dim3 grid;
    tile_grid(n_tiles, grid);
    fill_closed_full_kernel<<<grid, 256, 0, (cudaStream_t)stream>>>((char *)dRTiles, storage_es(storage), N, 0, dD1, dD2, dUr, dPhi, s1,
                                                                    s2,
                                                                    n_tiles);
    fill_closed_full_kernel<<<grid, 256, 0, (cudaStream_t)stream>>>((char *)dCTiles, storage_es(storage), N, 1, dD1, dD2, dUr, dPhi, s1,
                                                                    s2,
                                                                    n_tiles);
    count_launch(2);
    BSE_CUDA(cudaGetLastError());
    return BSE_OK;
}

bse_status_t bse_create(bse_handle_t *out, int32_t mode, int32_t storage, int64_t N, const void *dRTiles,
                        const void *dCTiles, void *stream)
{
    const bool real_form = storage_real_form(storage);
    if (!out || !dRTiles || N < 1 || (mode != BSE_MODE_TDA && mode != BSE_MODE_FULL) || !(storage_ok(storage) || real_form))
        return BSE_ERR_INVALID_ARG;
    if (mode == BSE_MODE_FULL && !dCTiles) return BSE_ERR_INVALID_ARG;
    if (real_form && mode != BSE_MODE_FULL) return BSE_ERR_INVALID_ARG;     // S = R + C, D = R - C need both matrices
    int dev = 0;
    BSE_CUDA(cudaGetDevice(&dev));
    int sms = 0;
    BSE_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    bse_handle_s *h = new (std::nothrow) bse_handle_s();
    if (!h) return BSE_ERR_ALLOC;
    h->mode = mode;
    h->N = N;
    h->nt = (int)((N + TB - 1) / TB);
    h->es = storage_es(storage);
    h->real_form = real_form ? 1 : 0;
    h->row_begin = 0;
    h->row_end = h->nt;
    h->comm = nullptr;
    h->comm_user = nullptr;
    h->comm_buf = nullptr;
    h->comm_buf_bytes = 0;
    h->vr_begin = 0;
    h->vr_end = N;
    h->rp_buf = nullptr;
    h->rp_buf_bytes = 0;
    h->R = (const char *)dRTiles;
    h->C = (mode == BSE_MODE_FULL) ? (const char *)dCTiles : nullptr;
    h->stream = (cudaStream_t)stream;
    h->num_sms = sms;
    bse_status_t st = handle_finalize(h);
    if (st) { bse_destroy(h); return st; }
    *out = h;
    return BSE_OK;
}

// (r, c) <- (r + c, r - c) on every stored double of the two tile stores
__global__ void __launch_bounds__(256) to_real_form_kernel(double2 *__restrict__ r, double2 *__restrict__ c, int64_t n)
{
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const double2 a = r[i], b = c[i];
        r[i] = make_double2(a.x + b.x, a.y + b.y);
        c[i] = make_double2(a.x - b.x, a.y - b.y);
    }
}

// the same on binary32 planes: the sum and difference are formed exactly in FP64 and rounded to nearest-even once
__global__ void __launch_bounds__(256) to_real_form_c64_kernel(float2 *__restrict__ r, float2 *__restrict__ c, int64_t n)
{
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const float2 a = r[i], b = c[i];
        r[i] = make_float2(__double2float_rn((double)a.x + (double)b.x), __double2float_rn((double)a.y + (double)b.y));
        c[i] = make_float2(__double2float_rn((double)a.x - (double)b.x), __double2float_rn((double)a.y - (double)b.y));
    }
}

bse_status_t bse_to_real_form(void *dRTiles, void *dCTiles, int32_t storage, int64_t n_tiles, void *stream)
{
    if (!dRTiles || !dCTiles || n_tiles < 0 || !storage_ok(storage)) return BSE_ERR_INVALID_ARG;
    if (n_tiles == 0) return BSE_OK;
    const int64_t n = n_tiles * TB * TB;
    if (storage == BSE_STORE_C64)
        to_real_form_c64_kernel<<<148 * 8, 256, 0, (cudaStream_t)stream>>>((float2 *)dRTiles, (float2 *)dCTiles, n);
    else
        to_real_form_kernel<<<148 * 8, 256, 0, (cudaStream_t)stream>>>((double2 *)dRTiles, (double2 *)dCTiles, n);
    count_launch();
    BSE_CUDA(cudaGetLastError());
    return BSE_OK;
}

bse_status_t bse_shard_layout(int64_t N, int32_t storage, int32_t n_shards, int32_t shard, int32_t *tile_row_begin,
                              int32_t *tile_row_end, int64_t *first_tile, int64_t *n_tiles, int64_t *bytes)
{
    if (N < 1 || !(storage_ok(storage) || storage_real_form(storage)) || n_shards < 1 || shard < 0 || shard >= n_shards)
        return BSE_ERR_INVALID_ARG;
    const int64_t nt = (N + TB - 1) / TB, total = nt * (nt + 1) / 2;
    // boundary r: the smallest tile row I with I (I + 1) / 2 >= r * total / n_shards (equal tile counts to within one row)
    auto bound = [&](int64_t r) -> int64_t {
        if (r <= 0) return 0;
        if (r >= n_shards) return nt;
        const double target = (double)total * (double)r / (double)n_shards;
        int64_t I = (int64_t)((std::sqrt(8.0 * target + 1.0) - 1.0) * 0.5);
        while (I > 0 && (double)(I * (I + 1) / 2) >= target) --I;
        while (I < nt && (double)(I * (I + 1) / 2) < target) ++I;
        return I;
    };
    const int64_t b0 = bound(shard), b1 = bound(shard + 1);
    if (tile_row_begin) *tile_row_begin = (int32_t)b0;
    if (tile_row_end) *tile_row_end = (int32_t)b1;
    if (first_tile) *first_tile = b0 * (b0 + 1) / 2;
    if (n_tiles) *n_tiles = b1 * (b1 + 1) / 2 - b0 * (b0 + 1) / 2;
    if (bytes) *bytes = (b1 * (b1 + 1) / 2 - b0 * (b0 + 1) / 2) * tile_bytes_es(storage_es(storage));
    return BSE_OK;
}

bse_status_t bse_create_shard(bse_handle_t *out, int32_t mode, int32_t storage, int64_t N, int32_t tile_row_begin,
                              int32_t tile_row_end, const void *dRSlice, const void *dCSlice, void *stream)
{
    if (N < 1) return BSE_ERR_INVALID_ARG;
    const int64_t nt = (N + TB - 1) / TB;
    if (tile_row_begin < 0 || tile_row_end < tile_row_begin || tile_row_end > nt) return BSE_ERR_INVALID_ARG;
    bse_status_t st = bse_create(out, mode, storage, N, dRSlice, dCSlice, stream);
    if (st) return st;
    (*out)->row_begin = tile_row_begin;
    (*out)->row_end = tile_row_end;
    return handle_finalize(*out);                            // the unit range of this slice
}

bse_status_t bse_set_comm(bse_handle_t h, bse_comm_fn fn, void *user)
{
    if (!h) return BSE_ERR_INVALID_ARG;
    h->comm = fn;
    h->comm_user = fn ? user : nullptr;
    return BSE_OK;
}

bse_status_t bse_set_row_partition(bse_handle_t h, int64_t row_begin, int64_t row_end)
{
    if (!h || row_begin < 0 || row_end <= row_begin || row_end > h->N) return BSE_ERR_INVALID_ARG;
    h->vr_begin = row_begin;
    h->vr_end = row_end;
    return BSE_OK;
}

bse_status_t bse_destroy(bse_handle_t h)
{
    if (!h) return BSE_ERR_INVALID_ARG;
    if (h->ws) cudaFree(h->ws);
    if (h->ws2) cudaFree(h->ws2);
    if (h->ws_op) cudaFree(h->ws_op);
    if (h->hpin) cudaFreeHost(h->hpin);
    if (h->comm_buf) cudaFree(h->comm_buf);
    if (h->rp_buf) cudaFree(h->rp_buf);
    delete h;
    return BSE_OK;
}

}  // extern "C"
