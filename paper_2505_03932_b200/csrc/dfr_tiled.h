// dfr_tiled.h — the tiled fast path (dfr_tiled_setup.cu, dfr_tiled_main.cu, dfr_tiled_stack.cu): data layout of the
// per-(exposure, tile) records and the launchers. DESIGN.md §6 describes it.
#pragma once
#include <cuda.h>

#include "dfr_internal.h"

namespace dfr {

constexpr int TS = 32;              // polynomial tile edge in output pixels (one warp wide)
constexpr int CTA_T = 2;            // a CTA covers CTA_T x CTA_T polynomial tiles (64 x 64 px)
constexpr int NPTS = 25;            // 16 interpolation nodes + 9 check points per tile
constexpr float FIT_TOL = 2e-6f;    // px: max |cubic fit - exact map| at the check points

enum { TILE_FAST = 0, TILE_EXACT = 1, TILE_EMPTY = 2 };

// Per (exposure, tile) record written by tile_setup_kernel, read by the main kernels.
// Source pixel of target pixel (tx0 + 15.5 + di, ty0 + 15.5 + dj), |di|,|dj| <= 15.5:
//   x = ix0 + sum_{p,q<=3} cx[4q+p] di^p dj^q     (fp32 evaluation, |x - ix0| small)
struct __align__(16) TileRec {
    float   cx[16];
    float   cy[16];
    int32_t ix0, iy0;               // integer base (floor of the tile-centre source pixel)
    int32_t bx0, by0, bx1, by1;     // inclusive range of floor(x), floor(y) over the tile
    int32_t flag;                   // TILE_*
    int32_t deg;                    // degree in dj the main kernel must keep (1..3)
};
static_assert(sizeof(TileRec) == 160, "TileRec layout");

struct TiledStats {
    int64_t tiles_fast, tiles_exact, tiles_empty, kernels;
};

// Timing hooks (dfr_profile_*): events recorded around the main kernel only.
struct ProfileEvents {
    cudaEvent_t setup_begin, main_begin, main_end;
    bool enabled;
};

// Per-call constants (SourceDev x n, then float weights x nweights) reach device scratch through the
// first setup kernel, never through the copy engine (a copy in front of the kernels is a
// cross-engine dependency: measured +8 us per C2 step). Two routes:
//   packed  : a compact form (only the polynomial coefficients the batch's highest order needs) rides
//             in the kernel's PARAMETERS and is expanded on the device — up to kPackedMaxBytes;
//   mapped  : the full-size block sits in pinned, device-mapped host memory and is read from there.
struct ConstsCopy {
    const void *packed = nullptr;       // HOST: packed form (see pack_consts in dfr_api.cu), or
    const void *mapped = nullptr;       // device-visible address of the full-size block in the pinned ring
    void *dst = nullptr;                // device scratch, `bytes` long
    size_t bytes = 0;                   // full size, multiple of 16
    int packed_bytes = 0, n = 0, T = 0, nweights = 0;      // packed: exposures, coefficients per polynomial, weights
    bool any() const { return packed || mapped; }
};
constexpr int kPackedSmallBytes = 3 * 1024;      // single frames: keeps the parameter block of the common launch small
constexpr int kPackedMaxBytes = 28 * 1024;       // kernel parameters hold 32 764 bytes in all
constexpr int kPackedHead = 12;                  // doubles per exposure before the coefficients: m[9], c1, c2, header
template <int BYTES> struct PackedConsts {
    uint4 q[BYTES / 16];
};

struct TiledParams {
    const float *src;
    float *out;
    const TileRec *recs;
    const int2 *cta_box;                           // [n][ctas_y][ctas_x] box origin (kNoBox: none)
    const SourceDev *srcdev;
    int n, e0, sny, snx, ony, onx;                 // e0: first exposure of this launch
    int tiles_x, tiles_y, ctas_x, ctas_y;
    int BW, BH;                                    // staged box (STAGE) in source pixels
    int prefetch_dist;                             // L2 prefetch distance in CTA tiles (0: off)
    int stage_bytes, rec_off;                      // stack kernel: bytes per stage, offset of its records
};

constexpr int kNoBox = 0x7fffffff;            // cta_box entry of a CTA tile without FAST tiles
constexpr int kMaxBoxBytes = 36 * 1024;       // staged box limit: keeps >= 6 CTAs (24 warps) per SM

// ---- host side shared by the launchers (dfr_tiled_setup.cu) ----------------
struct Scratch {
    void *block = nullptr;                          // one stream-ordered allocation holding all four
    double2 *uv = nullptr;
    TileRec *recs = nullptr;
    int2 *cta_box = nullptr;
    int32_t *counters = nullptr;                    // fast, exact, empty, ticket
};
cudaError_t scratch_alloc(void **p, size_t bytes, cudaStream_t st);     // dfr_context.cu: the library's own pool

// Setup kernels + staging decision shared by the per-exposure and the stacking launchers.
struct Prepared {
    TiledParams P;
    Scratch sc;
    CUtensorMap tmap;
    bool stage = false;
    size_t box_bytes = 0;
};

cudaError_t run_setup(int n, int sny, int snx, const TargetDev &tgt, const SourceDev *srcdev,
                      const SourceDev *srchost, int ony, int onx, cudaStream_t st,
                      int32_t *host_stats, int stats_add, Scratch &sc, TiledParams &P, const ConstsCopy &cc);
void free_scratch(Scratch &sc, cudaStream_t st);
cudaError_t prepare_tiled(const float *src, int n, int sny, int snx, const TargetDev &tgt,
                          const SourceDev *srcdev, const SourceDev *srchost, int ony, int onx,
                          int order, cudaStream_t st, int32_t *host_stats, int stats_add, Prepared &R,
                          const ConstsCopy &cc, int span_tiles = CTA_T /* the staged box serves span_tiles x span_tiles tiles */,
                          size_t max_box_bytes = kMaxBoxBytes);

cudaError_t launch_tiled_reproject(const float *src, int n, int sny, int snx,
                                   const TargetDev &tgt, const SourceDev *srcdev,
                                   const SourceDev *srchost,
                                   int ony, int onx, int order, float *out, cudaStream_t st,
                                   int32_t *host_stats /* 3 ints the setup kernel can write (mapped host or device memory), or NULL */,
                                   int stats_add /* 0: store the totals, 1: atomically add them (streaming) */,
                                   TiledStats *stats, ProfileEvents *prof, const ConstsCopy &cc, int edge = DFR_EDGE_AREA,
                                   float *foot = nullptr /* DEVICE [n][ony][onx] footprint array, or NULL */);
// dfr_reproject_stack: sum / wsum accumulated over the n exposures in one kernel.
cudaError_t launch_tiled_stack(const float *src, int n, int sny, int snx, const TargetDev &tgt,
                               const SourceDev *srcdev, const SourceDev *srchost, int ony, int onx, int order,
                               const float *dev_weights, float *sum, float *wsum, int accumulate,
                               cudaStream_t st, int32_t *host_stats, int stats_add, TiledStats *stats, ProfileEvents *prof,
                               const ConstsCopy &cc);
cudaError_t launch_stack_add(float *a, const float *b, long long n, cudaStream_t st);
cudaError_t launch_stack_finalize(const float *sum, const float *wsum, long long npix, float *mean, cudaStream_t st);
cudaError_t launch_tiled_coords(int n, int sny, int snx, const TargetDev &tgt,
                                const SourceDev *srcdev, const SourceDev *srchost, int ony, int onx, int order,
                                double *x, double *y, cudaStream_t st, const ConstsCopy &cc);

}  // namespace dfr
