// Internal declarations shared by the translation units of libbse_b200.so (not part of the ABI).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <atomic>

#include "../../include/bse.h"

struct bse_handle_s {
    int32_t mode;
    int64_t N;
    int nt;
    const char *R;
    const char *C;
    cudaStream_t stream;
    int num_sms;
    // lazily grown scratch (device)
    void *ws;
    size_t ws_bytes;
    // second scratch used by the solver / orth (device)
    void *ws2;
    size_t ws2_bytes;
    // pinned host staging for small results
    void *hpin;
    size_t hpin_bytes;
};

namespace bse {

extern std::atomic<int64_t> g_launches;
inline void count_launch(int n = 1) { g_launches.fetch_add(n, std::memory_order_relaxed); }

#define BSE_CUDA(call)                                   \
    do {                                                 \
        cudaError_t e__ = (call);                        \
        if (e__ != cudaSuccess) return BSE_ERR_CUDA;     \
    } while (0)

bse_status_t ensure_ws(bse_handle_s *h, size_t bytes);
bse_status_t ensure_ws2(bse_handle_s *h, size_t bytes);
bse_status_t ensure_pin(bse_handle_s *h, size_t bytes);

// One pass over one matrix: Y += sign * (R X)  or  Y += sign * (C conj X), k columns (chunked by 4).
bse_status_t launch_apply_pass(bse_handle_s *h, const char *tiles, int pass, double sign, const void *dX,
                               int64_t ldx, void *dY, int64_t ldy, int32_t k);
bse_status_t zero_block(bse_handle_s *h, void *dY, int64_t ldy, int64_t rows, int32_t k);

}  // namespace bse
