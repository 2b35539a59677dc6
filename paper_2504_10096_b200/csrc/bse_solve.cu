// placeholder until the solver lands
#include "bse_internal.h"
extern "C" bse_status_t bse_solve(bse_handle_t, int32_t, int32_t, int32_t, double, int32_t, uint64_t, double *, void *,
                                  int64_t, double *, bse_info_t *)
{
    return BSE_ERR_INTERNAL;
}
