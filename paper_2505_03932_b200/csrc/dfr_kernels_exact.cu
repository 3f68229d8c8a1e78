// dfr_kernels_exact.cu — the exact per-pixel path: every output pixel runs the
// whole fp64 map (a1-a6) and gathers straight from global memory (a7-a9).
// It is the reference GPU path (DFR_PATH_EXACT), the fallback of the tiled
// path, and what dfr_src_coords reports for path = EXACT.
#include "dfr_device.cuh"

namespace dfr {

constexpr int EX_BX = 64, EX_BY = 4;

template <int ORDER>
__global__ void __launch_bounds__(EX_BX *EX_BY)
exact_reproject_kernel(const float *__restrict__ src, int sny, int snx,
                       const __grid_constant__ TargetDev tgt,
                       const SourceDev *__restrict__ srcdev,
                       int ony, int onx, float *__restrict__ out, int edge, float *__restrict__ foot)
{
    // blockIdx.x enumerates the EX_BX x EX_BY output tiles row-major (no 65535 limit)
    const int tiles_x = (onx + EX_BX - 1) / EX_BX;
    const int i = (blockIdx.x % tiles_x) * EX_BX + threadIdx.x;
    const int j = (blockIdx.x / tiles_x) * EX_BY + threadIdx.y;
    const int e = blockIdx.y;
    if (i >= onx || j >= ony) return;
    double U, V, x, y;
    target_uv(tgt, (double)i, (double)j, U, V);
    source_xy(srcdev[e], U, V, x, y);
    float val = qnanf();
    if (in_footprint(x, y, sny, snx, edge))
        val = sample_global<ORDER>(src + (size_t)e * sny * snx, sny, snx, x, y);
    out[((size_t)e * ony + j) * onx + i] = val;
    if (foot) foot[((size_t)e * ony + j) * onx + i] = footprint_value(x, y, sny, snx, ORDER, edge);
}

__global__ void __launch_bounds__(EX_BX *EX_BY)
exact_coords_kernel(const __grid_constant__ TargetDev tgt, const SourceDev *__restrict__ srcdev,
                    int ony, int onx, double *__restrict__ xo, double *__restrict__ yo)
{
    // blockIdx.x enumerates the EX_BX x EX_BY output tiles row-major (no 65535 limit)
    const int tiles_x = (onx + EX_BX - 1) / EX_BX;
    const int i = (blockIdx.x % tiles_x) * EX_BX + threadIdx.x;
    const int j = (blockIdx.x / tiles_x) * EX_BY + threadIdx.y;
    const int e = blockIdx.y;
    if (i >= onx || j >= ony) return;
    double U, V, x, y;
    target_uv(tgt, (double)i, (double)j, U, V);
    source_xy(srcdev[e], U, V, x, y);
    const size_t k = ((size_t)e * ony + j) * onx + i;
    xo[k] = x;
    yo[k] = y;
}

static dim3 exact_grid(int n, int ony, int onx)
{
    return dim3(((onx + EX_BX - 1) / EX_BX) * ((ony + EX_BY - 1) / EX_BY), n, 1);
}

cudaError_t launch_exact_reproject(const float *src, int n, int sny, int snx,
                                   const TargetDev &tgt, const SourceDev *srcdev,
                                   int ony, int onx, int order, float *out, cudaStream_t st, int edge, float *foot)
{
    const dim3 block(EX_BX, EX_BY);
    // grid.y is limited to 65535 exposures per launch
    for (int e0 = 0; e0 < n; e0 += 65535) {
        const int ne = (n - e0 < 65535) ? n - e0 : 65535;
        const dim3 grid = exact_grid(ne, ony, onx);
        const float *s = src + (size_t)e0 * sny * snx;
        float *o = out + (size_t)e0 * ony * onx;
        float *f = foot ? foot + (size_t)e0 * ony * onx : nullptr;
        if (order == DFR_NEAREST)
            exact_reproject_kernel<DFR_NEAREST><<<grid, block, 0, st>>>(s, sny, snx, tgt, srcdev + e0, ony, onx, o, edge, f);
        else if (order == DFR_BILINEAR)
            exact_reproject_kernel<DFR_BILINEAR><<<grid, block, 0, st>>>(s, sny, snx, tgt, srcdev + e0, ony, onx, o, edge, f);
        else
            exact_reproject_kernel<DFR_BICUBIC><<<grid, block, 0, st>>>(s, sny, snx, tgt, srcdev + e0, ony, onx, o, edge, f);
        cudaError_t err = cudaGetLastError();
        if (err != cudaSuccess) return err;
    }
    return cudaSuccess;
}

cudaError_t launch_exact_coords(int n, const TargetDev &tgt, const SourceDev *srcdev,
                                int ony, int onx, double *x, double *y, cudaStream_t st)
{
    const dim3 block(EX_BX, EX_BY);
    for (int e0 = 0; e0 < n; e0 += 65535) {
        const int ne = (n - e0 < 65535) ? n - e0 : 65535;
        exact_coords_kernel<<<exact_grid(ne, ony, onx), block, 0, st>>>(
            tgt, srcdev + e0, ony, onx, x + (size_t)e0 * ony * onx, y + (size_t)e0 * ony * onx);
        cudaError_t err = cudaGetLastError();
        if (err != cudaSuccess) return err;
    }
    return cudaSuccess;
}

}  // namespace dfr
