// dfr_kernels_tiled.cu — tiled fast path (placeholder: routes to the exact path
// until the tile kernels land; stats report every tile as "exact").
#include "dfr_tiled.h"

namespace dfr {

cudaError_t launch_tiled_reproject(const float *src, int n, int sny, int snx,
                                   const TargetDev &tgt, const SourceDev *srcdev,
                                   int ony, int onx, int order, float *out, cudaStream_t st,
                                   TiledStats *stats)
{
    stats->tiles_fast = 0;
    stats->tiles_exact = -1;
    stats->tiles_empty = 0;
    stats->kernels = 1;
    return launch_exact_reproject(src, n, sny, snx, tgt, srcdev, ony, onx, order, out, st);
}

cudaError_t launch_tiled_coords(int n, int, int, const TargetDev &tgt, const SourceDev *srcdev,
                                int ony, int onx, int, double *x, double *y, cudaStream_t st)
{
    return launch_exact_coords(n, tgt, srcdev, ony, onx, x, y, st);
}

}  // namespace dfr
