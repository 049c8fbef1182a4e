// Brick-tiled kernel (placeholder until the tiled kernel lands: never selected).
#include "rs_internal.h"

bool rs_brick_supported(const rs_mesh *, int, int) { return false; }
rs_status rs_brick_prepare(rs_mesh *) { return RS_OK; }
rs_status rs_launch_brick(const rs_mesh *, int, const rs_weights &, const double *, const double *, double *, int,
                          cudaStream_t)
{
    return rs_fail(RS_ERR_UNSUPPORTED, "brick kernel not built");
}
int64_t rs_brick_table_bytes(const rs_mesh *m) { return m->nbricks * 12; }
