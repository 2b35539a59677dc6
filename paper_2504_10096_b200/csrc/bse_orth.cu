// placeholder until the orthogonalisation kernels land
#include "bse_internal.h"
extern "C" bse_status_t bse_orth(bse_handle_t, const void *, int64_t, int32_t, const void *, int64_t, void *, int64_t,
                                 int32_t, void *, int64_t, void *, void *, int32_t *)
{
    return BSE_ERR_INTERNAL;
}
