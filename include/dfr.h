/*
 * dfr.h — C ABI of libdfr: B200-native reprojection hot path of dfreproject
 *         (arXiv 2505.03932; PAPER.md = /root/reference/PAPER.md).
 *
 * What the library computes (PAPER.md:55-69, §3.1; :71-121, §3.2):
 *   for every pixel (i, j) of a target grid with WCS t and every source
 *   exposure e with WCS s_e
 *     1. target pixel -> sky      shift, SIP_A/SIP_B, CD, gnomonic (TAN)
 *                                  deprojection + rotation
 *     2. sky -> source pixel      inverse rotation + TAN projection, CD^-1,
 *                                  SIP_INV_A/SIP_INV_B, shift
 *     3. interpolate src[e] there nearest / bilinear / bicubic
 *     4. NaN outside the source footprint
 *     5. batched over exposures
 *
 * Conventions (DESIGN.md lists the readings of the paper they rest on):
 *   - pixel indices are 0-based, x = column (fastest varying), y = row;
 *     integer index = pixel centre; CRPIX is FITS 1-based.
 *   - images are C-contiguous float32 [n][ny][nx].
 *   - angles in dfr_wcs are DEGREES; CD is degrees per pixel.
 *   - SIP sign: u <- u + A(u,v) (Shupe 2005); both polynomials
 *     are evaluated at the pre-update (u,v).
 *   - footprint: valid <=> -0.5 <= x < nx-0.5 and -0.5 <= y < ny-0.5;
 *     interpolation taps are edge-replicated; bicubic = Keys, a = -0.75.
 *
 * Ownership: the caller owns every buffer named in a signature. The library
 * allocates only private, stream-ordered scratch and frees it itself. WCS
 * structs are read during the call and may be freed on return.
 *
 * Asynchrony: functions taking DEVICE pointers enqueue work on `stream`
 * (a cudaStream_t passed as void*, NULL = legacy default stream) and return
 * after enqueue; results are valid once the caller synchronises the stream.
 * dfr_reproject_host is synchronous: it returns when `out` is complete.
 *
 * Errors: every function returns DFR_OK (0) or a negative dfr_status, never
 * throws, never aborts; on a validation error nothing is written to outputs.
 * dfr_last_error() returns thread-local text for the last failure.
 *
 * There is no CPU fallback: without a CUDA device every compute entry point
 * returns DFR_ERR_CUDA.
 */
#ifndef DFR_H
#define DFR_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define DFR_SIP_MAX_ORDER 9                     /* SIP convention limit (Shupe 2005) */
#define DFR_SIP_DIM (DFR_SIP_MAX_ORDER + 1)
/* ap_order = bp_order = DFR_SIP_INVERSE_EXACT: the WCS carries no inverse polynomials and the
 * library inverts the forward distortion itself (PAPER.md:51 assumes SIP_INV_A / SIP_INV_B exist;
 * SURVEY.md §8(f) f4): wherever SIP_INV_A / SIP_INV_B would be applied it solves
 *   u + A(u, v) = U,  v + B(u, v) = V
 * for (u, v) in fp64 by fixed-point iteration to 1e-11 px (at most 32 steps: distortions whose
 * gradient exceeds ~0.4 do not converge and give NaN). Exact where a fitted AP/BP is only as good
 * as its order allows. On the tiled path the solve runs at the sample points of the per-tile fit
 * (16 nodes + 16 check points per 128 x 128 output pixels, or 25 per tile), not per pixel. */
#define DFR_SIP_INVERSE_EXACT (-1)

/* Packed WCS parameter set. POD, no pointers,
 * 3280 bytes, no padding. Polynomial coefficient of u^p v^q is stored at
 * [p*DFR_SIP_DIM + q]; entries with p+q > order are ignored; order 0 means
 * "polynomial absent". */
typedef struct dfr_wcs {
    double  crpix[2];          /* CRPIX1, CRPIX2 — FITS 1-based */
    double  crval[2];          /* ra0, dec0 in degrees              */
    double  cd[4];             /* CD1_1, CD1_2, CD2_1, CD2_2, deg/pixel */
    int32_t a_order, b_order, ap_order, bp_order;   /* 0..9; ap = bp = DFR_SIP_INVERSE_EXACT allowed */
    double  a [DFR_SIP_DIM * DFR_SIP_DIM];     /* SIP_A   */
    double  b [DFR_SIP_DIM * DFR_SIP_DIM];     /* SIP_B                          */
    double  ap[DFR_SIP_DIM * DFR_SIP_DIM];     /* SIP_INV_A      */
    double  bp[DFR_SIP_DIM * DFR_SIP_DIM];     /* SIP_INV_B      */
} dfr_wcs;

/* Interpolation order (PAPER.md:35 `order=`, :135 "three interpolation schemes"). */
enum { DFR_NEAREST = 0, DFR_BILINEAR = 1, DFR_BICUBIC = 3 };

typedef enum dfr_status {
    DFR_OK = 0,
    DFR_ERR_NULL = -1,           /* a required pointer is NULL                    */
    DFR_ERR_SHAPE = -2,          /* n < 1, a dimension < 1, or ny*nx >= 2^31      */
    DFR_ERR_ORDER = -3,          /* order not in {0, 1, 3}                        */
    DFR_ERR_SIP_ORDER = -4,      /* a SIP order outside [0, DFR_SIP_MAX_ORDER] (or a lone DFR_SIP_INVERSE_EXACT) */
    DFR_ERR_SINGULAR_CD = -5,    /* det(CD) == 0 or not finite                    */
    DFR_ERR_NONFINITE_WCS = -6,  /* NaN/Inf in crpix, crval, cd or used SIP terms */
    DFR_ERR_ALIAS = -7,          /* out overlaps src_batch                        */
    DFR_ERR_CUDA = -8,           /* CUDA runtime/driver failure (see dfr_last_error) */
    DFR_ERR_WEIGHT = -9          /* NaN/Inf in the stacking weights               */
} dfr_status;

/* Path selection for dfr_reproject_ex / dfr_src_coords_ex.
 *   AUTO  : tiled fast path where its per-tile cubic fit passes a spot check against the exact
 *           map (16 check points per 128 x 128 output pixels; 9 per tile on the refit level),
 *           exact per-pixel path elsewhere (what dfr_reproject uses).
 *   EXACT : every pixel through the per-pixel fp64 map, direct gathers.
 *   TILED : as AUTO (kept distinct so tests can assert the fast path ran). */
enum { DFR_PATH_AUTO = 0, DFR_PATH_EXACT = 1, DFR_PATH_TILED = 2 };

/* Footprint rule of dfr_reproject_edge.
 *   AREA  : a pixel is valid where its source coordinate lies in the union of the source
 *           pixel areas, -0.5 <= x < n - 0.5 (what every other entry point uses).
 *   PAPER : the paper's literal rule: the image and an identity ("footprint")
 *           image are interpolated with zero padding and divided; for bilinear this is
 *           valid on the open square -1 < x < n and equals the AREA result wherever both
 *           are valid (the half-pixel band it adds takes the edge pixel's value). Nearest:
 *           identical to AREA. Bicubic: not defined (the projected identity changes sign
 *           near the rim) -> DFR_ERR_ORDER. */
enum { DFR_EDGE_AREA = 0, DFR_EDGE_PAPER = 1 };

/* ---- the hot path (calculate_reprojection) -------------- */

/* Reproject n source exposures onto one target grid.
 *   src_batch : DEVICE float32 [n][src_ny][src_nx], contiguous
 *   src_wcs   : HOST, n entries (exposure e uses src_wcs[e])
 *   tgt_wcs   : HOST, 1 entry
 *   out_ny/nx : shape_out
 *   order     : DFR_NEAREST | DFR_BILINEAR | DFR_BICUBIC
 *   out       : DEVICE float32 [n][out_ny][out_nx]; every element is written
 *               (value, or NaN outside the footprint of exposure e)
 * Steps a1–a10 of SURVEY.md §8(a) all run inside the library's kernels. */
int dfr_reproject(const float *src_batch, int32_t n, int32_t src_ny, int32_t src_nx,
                  const dfr_wcs *src_wcs, const dfr_wcs *tgt_wcs,
                  int32_t out_ny, int32_t out_nx, int32_t order,
                  float *out, void *stream);

/* Same, with an explicit footprint rule (DFR_EDGE_*) and, optionally, the footprint array
 * (PAPER.md:69: "simultaneously projecting an identity tensor called the footprint"; :27: a drop-in
 * for reproject_interp, which returns (array, footprint)).
 *   footprint : DEVICE float32 [n][out_ny][out_nx], or NULL. Must not overlap src_batch or out.
 *               DFR_EDGE_PAPER with bilinear: the projected identity itself — the zero-padded
 *               bilinear interpolation of an all-ones image at the pixel's source coordinate:
 *               1 on [0, n-1]^2, falling linearly to 0 at -1 and at n on each axis (product of
 *               the two); `out` is valid exactly where it is > 0. Every other mode (AREA; PAPER
 *               with nearest): 1 where the source coordinate lies in the footprint, else 0.
 *               NaN pixels of the source do not change it: it describes geometry only.
 * `out` is bit-identical with and without a footprint array (the footprint is written by a
 * separate pass over the same per-tile coordinates). Errors as dfr_reproject. */
int dfr_reproject_fp(const float *src_batch, int32_t n, int32_t src_ny, int32_t src_nx,
                     const dfr_wcs *src_wcs, const dfr_wcs *tgt_wcs,
                     int32_t out_ny, int32_t out_nx, int32_t order, int32_t edge_mode,
                     float *out, float *footprint, void *stream);

/* dfr_reproject_fp without a footprint array. */
int dfr_reproject_edge(const float *src_batch, int32_t n, int32_t src_ny, int32_t src_nx,
                       const dfr_wcs *src_wcs, const dfr_wcs *tgt_wcs,
                       int32_t out_ny, int32_t out_nx, int32_t order, int32_t edge_mode,
                       float *out, void *stream);

/* Same, with an explicit path (DFR_PATH_*). */
int dfr_reproject_ex(const float *src_batch, int32_t n, int32_t src_ny, int32_t src_nx,
                     const dfr_wcs *src_wcs, const dfr_wcs *tgt_wcs,
                     int32_t out_ny, int32_t out_nx, int32_t order,
                     float *out, void *stream, int32_t path);

/* dfr_reproject for callers that must not trigger a device allocation.
 *
 * Every other entry point draws per-call scratch from a CUDA memory pool and keeps events and
 * pinned staging memory per host thread. Two kinds of caller cannot live with that: code that
 * shares the GPU with something that already owns all of its memory (a framework's caching
 * allocator grown to the whole card, a reduction pipeline that reserved HBM for the night's
 * frames), where the library's first allocation may simply fail; and real-time loops (quick-look
 * reduction between read-outs) that cannot risk the device-wide synchronisation cudaMalloc /
 * cudaFree may imply. This entry point calls no cudaMalloc, cudaFree, cudaMallocAsync, pool,
 * event, stream or pinned-memory routine. The only scratch its kernel needs, the table of
 * per-exposure constants, is a fixed array inside the library image:
 *   limit : n <= DFR_NOALLOC_MAX_EXPOSURES per call (more -> DFR_ERR_SHAPE, nothing written);
 *   cost  : DFR_NOALLOC_MAX_EXPOSURES x 992 B = 63 488 B on every GPU that loads libdfr, held
 *           from load until the process exits, used or not.
 * What it computes: steps a1-a9 of SURVEY.md §8(a) through the exact
 * per-pixel fp64 map with direct gathers — the same arithmetic as dfr_reproject_ex(...,
 * DFR_PATH_EXACT), bit for bit, area footprint rule. It is slower than the tiled path of
 * dfr_reproject (that path's scratch grows with the output size and does not fit a fixed array).
 * Arguments, layouts, asynchrony and validation errors are those of dfr_reproject; the caller
 * owns and passes src_batch and out as usual.
 * First call per device: the first call made with a given device current looks up the array's
 * device address (cudaGetSymbolAddress, which also makes the runtime load the library's device
 * code there) and remembers it. Make that first call during set-up, outside any stream capture.
 * Sharing: all calls on a device use the same array, which keeps the previous call's contents;
 * each call overwrites the n entries it reads before reading them, so nothing needs clearing and
 * calls issued on ONE stream are safe back to back. Two calls that can overlap on the GPU
 * (different streams, or different host threads, same device) race on the array: the later
 * call's constants may replace the earlier call's while its kernel still runs. Serialise them. */
#define DFR_NOALLOC_MAX_EXPOSURES 64
int dfr_reproject_noalloc(const float *src_batch, int32_t n, int32_t src_ny, int32_t src_nx,
                          const dfr_wcs *src_wcs, const dfr_wcs *tgt_wcs,
                          int32_t out_ny, int32_t out_nx, int32_t order,
                          float *out, void *stream);

/* End-to-end form with HOST buffers (">1000 exposures"; SURVEY.md
 * §8(a) a10): src_host [n][src_ny][src_nx] and out_host [n][out_ny][out_nx]
 * are HOST float32 arrays (pinned memory gives full PCIe rate, pageable
 * works). Exposures are processed in batches of `batch` (<=0 selects 32); the
 * upload of batch k+1 and the download of batch k-1 overlap the kernels of
 * batch k on private CUDA streams. Synchronous. */
int dfr_reproject_host(const float *src_host, int32_t n, int32_t src_ny, int32_t src_nx,
                       const dfr_wcs *src_wcs, const dfr_wcs *tgt_wcs,
                       int32_t out_ny, int32_t out_nx, int32_t order,
                       float *out_host, int32_t batch);

/* The same over several devices of this node (exposures are
 * independent). The n exposures are cut into ndev contiguous shards (dfr_shard_range); shard k
 * runs the pipeline above on device devices[k] from its own host thread; there is no collective.
 * A device may be listed more than once (two pipelines on it). Every listed device must be
 * visible to the process. The calling thread's current device is left unchanged. */
int dfr_reproject_host_multi(const float *src_host, int32_t n, int32_t src_ny, int32_t src_nx,
                             const dfr_wcs *src_wcs, const dfr_wcs *tgt_wcs,
                             int32_t out_ny, int32_t out_nx, int32_t order,
                             float *out_host, int32_t batch, const int32_t *devices, int32_t ndev);

/* The partition rule of the *_multi entry points: shard k of `parts` over n units is
 * [*lo, *hi), contiguous, sizes differing by at most one (the first n % parts shards are the
 * longer ones). HOST only. */
int dfr_shard_range(int32_t n, int32_t parts, int32_t k, int32_t *lo, int32_t *hi);

/* ---- fused reproject-and-stack --------- */

/* The paper's stated purpose of reprojection is that images "can be combined to
 * produce a single, deeper image". This entry point does both in
 * one kernel, so the n per-exposure frames never reach HBM:
 *   sum [j][i] (+)= sum over e of weights[e] * v_e(i, j)
 *   wsum[j][i] (+)= sum over the same e of weights[e]
 * where v_e is what dfr_reproject would store for exposure e, and exposure e
 * contributes to a pixel only where v_e is not NaN (inside its footprint and no
 * NaN under the taps). Accumulation is float32, in exposure order within one kernel pass;
 * every output pixel has one owner (small outputs are cut into exposure chunks whose partial
 * sums are added in chunk order), so the same call gives the same bits on every run. `wsum` is
 * exact whenever the weights' partial sums are (it is the sum of a per-tile and a per-pixel part).
 * With accumulate = 1 the batch is added by plain read-modify-write: do not run two such calls on
 * the same sum / wsum concurrently on different streams.
 *   src_batch, src_wcs, tgt_wcs, out_ny/nx, order : as dfr_reproject
 *   weights    : HOST float32[n], or NULL for 1.0 each (must be finite: DFR_ERR_WEIGHT)
 *   sum, wsum  : DEVICE float32 [out_ny][out_nx] each; must not overlap src_batch
 *                or each other
 *   accumulate : 0 = both arrays are overwritten; 1 = the batch is added to their
 *                current contents (co-adding a stream of batches)
 * The mean image is sum / wsum (dfr_stack_finalize). Errors as dfr_reproject. */
int dfr_reproject_stack(const float *src_batch, int32_t n, int32_t src_ny, int32_t src_nx,
                        const dfr_wcs *src_wcs, const dfr_wcs *tgt_wcs,
                        int32_t out_ny, int32_t out_nx, int32_t order,
                        const float *weights, float *sum, float *wsum, int32_t accumulate,
                        void *stream);

/* End-to-end form of the stack with HOST buffers (the ">1000 exposures" case of
 * PAPER.md:25 co-added instead of returned one by one): src_host [n][src_ny][src_nx]
 * is uploaded in batches of `batch` (<= 0 selects 32) on private streams, every batch is
 * added into one device-resident sum / wsum pair while the next uploads, and only the two
 * [out_ny][out_nx] frames come back. weights: HOST float32[n] or NULL. Synchronous. */
int dfr_stack_host(const float *src_host, int32_t n, int32_t src_ny, int32_t src_nx,
                   const dfr_wcs *src_wcs, const dfr_wcs *tgt_wcs,
                   int32_t out_ny, int32_t out_nx, int32_t order, const float *weights,
                   float *sum_host, float *wsum_host, int32_t batch);

/* dfr_stack_host over several devices: every shard (as dfr_reproject_host_multi) co-adds its
 * exposures into a sum / wsum pair on its own device; the one exchange step of the path follows:
 * the partial pairs are copied to the first shard's device (peer copy) and added there in shard
 * order, so the result does not depend on timing between devices. */
int dfr_stack_host_multi(const float *src_host, int32_t n, int32_t src_ny, int32_t src_nx,
                         const dfr_wcs *src_wcs, const dfr_wcs *tgt_wcs,
                         int32_t out_ny, int32_t out_nx, int32_t order, const float *weights,
                         float *sum_host, float *wsum_host, int32_t batch,
                         const int32_t *devices, int32_t ndev);

/* mean[k] = sum[k] / wsum[k], NaN where wsum[k] == 0. DEVICE float32[npix] each;
 * mean may be the same array as sum. */
int dfr_stack_finalize(const float *sum, const float *wsum, int64_t npix, float *mean, void *stream);

/* ---- coordinate entry points, for testing (§3.2.1 / §3.2.2) ---- */

/* Pixel -> sky with WCS *w (HOST). x, y, ra_deg, dec_deg: DEVICE double[npts].
 * Literal formulas of PAPER.md:87-95 in fp64. RA is reduced to [0,360),
 * Dec is in [-90,90]. */
int dfr_pix2world(const dfr_wcs *w, const double *x, const double *y, int64_t npts,
                  double *ra_deg, double *dec_deg, void *stream);

/* Sky -> pixel with WCS *w (HOST). Literal formulas of PAPER.md:101-121 in
 * fp64; uses AP/BP (absent AP/BP => no inverse distortion; DFR_SIP_INVERSE_EXACT =>
 * the forward distortion inverted by iteration). Points >= 90 degrees from CRVAL give NaN. */
int dfr_world2pix(const dfr_wcs *w, const double *ra_deg, const double *dec_deg, int64_t npts,
                  double *x, double *y, void *stream);

/* Test-only: the source coordinates dfr_reproject itself uses (same device
 * functions, same tile tables), DEVICE double [n][out_ny][out_nx] each.
 * src_ny/src_nx are needed because the fast path's tiling depends on them. */
int dfr_src_coords(int32_t n, int32_t src_ny, int32_t src_nx,
                   const dfr_wcs *src_wcs, const dfr_wcs *tgt_wcs,
                   int32_t out_ny, int32_t out_nx, int32_t order,
                   double *x, double *y, void *stream, int32_t path);

/* ---- helpers ----------------------------------------------------------- */

/* CD_ij = CDELT_i * PC_ij (FITS Paper I). HOST only. */
int dfr_wcs_set_pc_cdelt(dfr_wcs *w, const double pc[4], const double cdelt[2]);

/* Inverse SIP polynomials for a WCS that lacks them (PAPER.md:51 assumes SIP_INV_A /
 * SIP_INV_B exist). HOST only. Fits AP, BP of the given order
 * (1..9, full triangle 0 <= p+q <= order) by least squares so that
 *   u ~= U + AP(U, V),  v ~= V + BP(U, V)   with (U, V) = (u + A(u,v), v + B(u,v))
 * on a 64 x 64 uniform grid of pixel centres over [0, nx-1] x [0, ny-1] (Householder QR,
 * columns scaled to [-1, 1]). Overwrites w->ap, w->bp (entries outside the triangle are
 * zeroed) and sets w->ap_order = w->bp_order = order. *max_resid_px (optional) receives
 * the largest |u - (U + AP)|, |v - (V + BP)| over the grid: raise the order if it is too
 * large for the application. The forward side of *w must be valid. */
int dfr_wcs_fit_inverse_sip(dfr_wcs *w, int32_t order, int32_t nx, int32_t ny, double *max_resid_px);

/* Counters of the last dfr_reproject* call on this thread (HOST):
 * stats[0] = tiles on the fast path, [1] = tiles on the exact path,
 * [2] = tiles entirely outside the footprint, [3] = kernels launched.
 * The counters and the event that guards them exist once per (host thread, device), not per
 * stream: they describe the last call only if this thread's calls on that device were issued on
 * ONE stream. With calls in flight on several streams an earlier call may finish later and
 * overwrite them. The same holds for dfr_profile_last. Outputs are never affected. */
int dfr_last_stats(int64_t stats[4]);

/* Timing hooks used by bench.py: when enabled (per host thread), dfr_reproject*
 * records CUDA events on the caller's stream around its own kernels.
 * dfr_profile_last waits for the last call and returns ms[0] = setup kernels
 * (per-tile fit), ms[1] = main reprojection kernel. */
int dfr_profile_enable(int on);
int dfr_profile_last(float ms[2]);

/* What the library keeps between calls, per device: a private cudaMemPool for stream-ordered
 * scratch (the application's default pool is never touched), per host thread a few KB of pinned
 * staging memory, three events and 16 bytes of mapped counters, and — after a *_host call — the
 * pipeline's device buffers (3 x batch x (input + output frames)), reused by later calls.
 * dfr_release() synchronises the CURRENT device, frees the calling thread's state for it, every
 * idle pipeline on it, and trims the scratch pool. Safe to call at any time between calls. */
int dfr_release(void);

const char *dfr_strerror(int code);
const char *dfr_last_error(void);
int dfr_version(void);           /* 10000*major + 100*minor + patch */

#ifdef __cplusplus
}
#endif
#endif /* DFR_H */
