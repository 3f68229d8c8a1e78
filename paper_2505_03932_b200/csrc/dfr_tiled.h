// dfr_tiled.h — launchers of the tiled fast path (dfr_kernels_tiled.cu).
#pragma once
#include "dfr_internal.h"

namespace dfr {

struct TiledStats {
    int64_t tiles_fast, tiles_exact, tiles_empty, kernels;
};

cudaError_t launch_tiled_reproject(const float *src, int n, int sny, int snx,
                                   const TargetDev &tgt, const SourceDev *srcdev,
                                   int ony, int onx, int order, float *out, cudaStream_t st,
                                   TiledStats *stats);
cudaError_t launch_tiled_coords(int n, int sny, int snx, const TargetDev &tgt,
                                const SourceDev *srcdev, int ony, int onx, int order,
                                double *x, double *y, cudaStream_t st);

}  // namespace dfr
