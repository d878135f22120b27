/*
 * microlens.h -- C ABI of the B200-native direct inverse ray-shooting library.
 *
 * What it computes (citations: /root/reference/PAPER.md line, section/equation):
 *   A regular grid of light rays covering an image-plane "shooting rectangle" is
 *   propagated backwards through a lens plane of N* unit-mass point lenses plus a
 *   smooth convergence sigma_c and an external shear gamma (eq.4):
 *
 *       y1 = (1 - gamma - sigma_c) x1 - sum_i (x1 - xi1)/|x - xi|^2
 *       y2 = (1 + gamma - sigma_c) x2 - sum_i (x2 - xi2)/|x - xi|^2
 *
 *   and each ray is counted into the source-plane pixel it reaches; the map of
 *   counts N_ij gives the magnification mu_ij = N_ij / N_rays (eq.3).
 *   This is the "GPU-D" direct code of PAPER.md:119-138 (section 2.3), redesigned: rays are
 *   generated in-kernel from their grid index, deflected by an all-pairs FP32 sum
 *   over shared-memory lens tiles, and binned by warp-aggregated atomics in the
 *   same kernel.  Lengths are in Einstein radii of one lens; masses are 1
 *   (PAPER.md:165).
 *
 * Conventions
 *   - Every function returns an int: ML_OK (0) or a negative ML_ERR_* code.  The
 *     library never throws, aborts or prints.  ml_strerror() names a code.
 *   - "host" / "device" below says where a pointer must live.  The caller owns
 *     every buffer it passes; the library copies what it needs before returning.
 *   - A context is not thread-safe; separate contexts are independent.
 *   - There is no CPU fallback: without a CUDA device ml_create fails with
 *     ML_ERR_CUDA.
 *
 * Geometry derived by ml_create (all fp64; DESIGN.md "Readings" R1-R8):
 *   kappa_star = stellar_fraction*sigma, kappa_c = sigma - kappa_star
 *   pixel = L/n_pix;  ray spacing delta = pixel/sqrt(n_rays)
 *   a1 = 1.2 (L/2)/|1-sigma-gamma|, a2 = 1.2 (L/2)/|1-sigma+gamma|      (eq.11)
 *   n1 = ceil(2 a1/delta - 1e-9), n2 likewise; ray (i,j), 0<=i<n1, 0<=j<n2, sits at
 *   x = ((i-(n1-1)/2) delta, (j-(n2-1)/2) delta)
 *   R* = 1.3 sqrt(a1^2+a2^2);  N*_expected = floor(kappa_star R*^2 + 0.5) (eq.5)
 *   pixel (i',j') of y: i' = floor((y1+L/2)/pixel), j' = floor((y2+L/2)/pixel);
 *   counted iff 0 <= i',j' < n_pix.  Map layout: map[j'*n_pix + i'] (uint32).
 */
#ifndef MICROLENS_H
#define MICROLENS_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ml_ctx ml_ctx; /* opaque */

enum {
    ML_OK = 0,
    ML_ERR_INVALID_ARG = -1, /* bad argument (see each call)                        */
    ML_ERR_CUDA = -2,        /* a CUDA runtime call failed / no device              */
    ML_ERR_OOM = -3,         /* host or device allocation failed                    */
    ML_ERR_STATE = -4,       /* call sequence error (e.g. shoot before set_lenses)  */
    ML_ERR_LIMIT = -5        /* the input needs more than the fixed built-in scratch of a call that never
                                allocates (ml_delta_m_histogram_static)                */
};

/* Arithmetic of the deflection sum (eq.8 leaves the summation order open;
 * DESIGN.md "Summation order and precision" fixes it for each mode). */
enum {
    ML_PREC_FP32_TILED = 0,       /* default: tile-local FP32 terms, FP32 partial sums over K
                                     lenses flushed into fp64 accumulators, fp64 epilogue    */
    ML_PREC_FP32_COMPENSATED = 1, /* as above, Newton-refined reciprocal and a flush every
                                     16 lenses (8 with random rays): ~3x smaller errors      */
    ML_PREC_FP64 = 2              /* everything in fp64 (reciprocal refined to an ulp)       */
};

/* Where the rays start.  REGULAR: the cell-centred regular grid of the configs
 * (the tree codes' way).  RANDOM: the paper's GPU-D shoots rays "from random positions in the shooting
 * grid"; here ray (i,j) starts at a uniformly random point of its own grid cell,
 *     x = ((i + u1 - n1/2) delta, (j + u2 - n2/2) delta),
 * (u1, u2) = two 53-bit uniforms from Philox-4x32-10 with counter (ray id lo, hi, 0, 0), ray id = j n1 + i,
 * and key = seed (reading R17): the same number of rays, the same mean density, regions and
 * sharding unchanged; the rays share no coordinate differences, so a kernel with per-ray offsets runs
 * (shoot_kernel_rpipe in the FP32 modes: 57-60 % of FP32 peak against 74-76 % on the regular grid). */
enum {
    ML_RAYS_REGULAR = 0,
    ML_RAYS_RANDOM = 1,
    ML_RAYS_UNIFORM = 2  /* the literal reading of PAPER.md:131, :167 (reading R20): the n1 n2 rays are independent
                            uniform points of the whole shooting rectangle,
                                x = ((u1 n1 - n1/2) delta, (u2 n2 - n2/2) delta),  (u1, u2) drawn as above from ray id = j n1 + i,
                            so the counts carry the Poisson noise the paper describes (ML_RAYS_RANDOM's one ray per cell is a
                            stratified sample with less).  (i, j) only numbers the rays: a region of ml_shoot_region /
                            ml_capture_region selects ray ids, not a patch of the image plane.  The library sorts the rays
                            into buckets of 128 x 63 grid cells on the device (8 bytes of scratch per ray, kept by the context until
                            ml_destroy or until another ray mode is selected, up to
                            45 % of the device memory; more rays are done in several passes) and shoots each bucket in
                            coordinates local to it; ml_info.tile_w / tile_h report the bucket.  The lens loop is not split
                            over CTAs in this mode. */
};

typedef struct {
    double kappa_star, kappa_c;      /* sigma_*, sigma_c                                    */
    double a1, a2;                   /* half-sides of the shooting rectangle (R_E)          */
    double ray_spacing;              /* delta                                               */
    double r_star;                   /* lens-disk radius R*                                 */
    double pixel_side;               /* L / n_pix                                           */
    double mu_theory;                /* 1/((1-sigma)^2-gamma^2), signed (eq.12) */
    int64_t n1, n2;                  /* rays along axis 1 / axis 2                          */
    int64_t n_star_expected;         /* N* of eq.5 for the disk above                       */
    int64_t n_lenses;                /* lenses currently set (-1 before ml_set_lenses)      */
    int32_t n_pix;                   /* pixels per side                                     */
    int32_t tile_w, tile_h;          /* ray tile of one CTA in the current precision mode   */
    int32_t precision;               /* ML_PREC_*                                           */
    int32_t device;                  /* CUDA device ordinal                                 */
    int32_t sm_count;                /* multiProcessorCount of that device                  */
    int32_t sm_clock_khz;            /* cudaDevAttrClockRate (max SM clock)                 */
    int32_t ray_mode;                /* ML_RAYS_*                                           */
    uint64_t ray_seed;               /* key of the ray generator (ML_RAYS_RANDOM / _UNIFORM) */
} ml_info;

typedef struct {
    uint64_t rays_shot;    /* rays processed by the last shoot (sum over accumulated regions) */
    uint64_t rays_in_map;  /* rays counted into the map                                       */
    uint64_t rays_dropped; /* rays whose y was not finite: not binned.  A ray exactly ON a lens is dropped in
                              ML_PREC_FP64; in the FP32 modes it does not see that one lens (R12)     */
    uint64_t interactions; /* rays_shot * n_lenses (eq.6 without N_FLOP)       */
    uint64_t kernel_launches; /* launches of the shoot kernel since the map was last zeroed   */
    double kernel_ms;      /* device time of those launches, CUDA events on the ctx stream    */
    double total_ms;       /* host wall time of the last ml_shoot / ml_shoot_region call      */
    uint64_t capture_ctas; /* CTAs of the last launch that split its lens loop (tiles x lens ranges:
                              ml_probe / ml_capture_region / a small ml_shoot_region at N* >= 8192); else 0 */
} ml_stats;

/* Create a context for one map.  Arguments are the paper's statement of the problem
 * (PAPER.md:152-158, :25): total convergence sigma, stellar fraction sigma_* / sigma
 * (= 1 - s of PAPER.md:158), shear gamma, pixels per side n_pix, mean rays per pixel
 * n_rays, source-plane side L (Einstein radii); `device` is the CUDA ordinal.
 * Allocates the n_pix^2 uint32 device map.  *out is owned by the library until
 * ml_destroy.  ML_ERR_INVALID_ARG if out is NULL, any value is not finite, sigma < 0,
 * stellar_fraction outside [0,1], n_pix <= 0 or > 32768, n_rays <= 0, L <= 0,
 * |1-sigma-gamma| or |1-sigma+gamma| < 1e-6 (critical line: unbounded rectangle,
 * PAPER.md:285) or n1*n2 >= 2^62. */
int ml_create(double sigma, double stellar_fraction, double gamma, int32_t n_pix,
              double n_rays, double L, int32_t device, ml_ctx **out);

/* Frees everything.  NULL is a no-op. */
void ml_destroy(ml_ctx *ctx);

/* Derived geometry and device facts (host struct filled). */
int ml_get_info(const ml_ctx *ctx, ml_info *out);

/* Lens positions (PAPER.md:130 step 1, :138): xy = n interleaved (x, y) HOST fp64
 * pairs in Einstein radii, unit masses.  Copied before the call returns (into a pinned
 * staging buffer of the context, and from there to the device on the context's stream,
 * ordered before the next shoot; the call does not wait for the device and, once its
 * buffers have grown to the largest field seen, allocates nothing); the caller keeps xy.
 * n >= 0 and need not equal n_star_expected (n = 0: no stars).  A non-finite
 * coordinate gives ML_ERR_INVALID_ARG and leaves the previous lenses in place. */
int ml_set_lenses(ml_ctx *ctx, const double *xy, int64_t n);

/* Same with the lens masses m_i of eq.4: mass = n HOST fp64 values > 0 in units of the
 * mass whose Einstein radius is the unit of length, or NULL for unit masses (= ml_set_lenses; the
 * paper sets all masses equal).  The deflection of lens i is m_i (x - xi_i)/|x - xi_i|^2;
 * the kernels multiply 1/r^2 by m_i (one extra FP32 multiply per ray pair and lens).  For a mean mass
 * <M> the lens count of eq.5 is n_star_expected / <M>.  ML_ERR_INVALID_ARG for a non-finite or
 * non-positive mass; the previous lenses stay in place on ML_ERR_INVALID_ARG and ML_ERR_OOM (after
 * ML_ERR_CUDA no lenses are set). */
int ml_set_lens_masses(ml_ctx *ctx, const double *xy, const double *mass, int64_t n);

/* Select ML_RAYS_* (see the enum); seed keys the generator of ML_RAYS_RANDOM / ML_RAYS_UNIFORM and is ignored otherwise.
 * Takes effect at the next shoot / capture / probe.  ML_ERR_INVALID_ARG for any other mode. */
int ml_set_ray_mode(ml_ctx *ctx, int mode, uint64_t seed);

/* Select ML_PREC_*; ML_ERR_INVALID_ARG for any other value. */
int ml_set_precision(ml_ctx *ctx, int mode);

/* Zero the map and the statistics, shoot the whole n1 x n2 grid (PAPER.md:128-136 steps
 * 2-7 as one fused kernel per <= 2^31-1 tiles), synchronise.  ML_ERR_STATE before
 * ml_set_lenses. */
int ml_shoot(ml_ctx *ctx);

/* Same for the ray-index rectangle [i0,i1) x [j0,j1) only.  accumulate = 0 zeroes the
 * map and statistics first; != 0 adds to them.  Tiles are aligned to the global
 * grid, so a ray's arithmetic does not depend on the region it is shot in: any
 * partition of the grid into regions gives bit-identical counts to ml_shoot.
 * ML_ERR_INVALID_ARG unless 0 <= i0 <= i1 <= n1 and 0 <= j0 <= j1 <= n2. */
int ml_shoot_region(ml_ctx *ctx, int64_t i0, int64_t i1, int64_t j0, int64_t j1, int accumulate);

/* Copy the n_pix^2 counts to a HOST buffer of out_len >= n_pix^2 elements
 * (else ML_ERR_INVALID_ARG).  out[j'*n_pix + i'], i' <-> y1 (fast), j' <-> y2. */
int ml_get_map(const ml_ctx *ctx, uint32_t *out, size_t out_len);

/* Borrowed DEVICE pointer to the map (valid until ml_destroy / ml_use_device_map). */
int ml_get_map_device(const ml_ctx *ctx, void **dptr);

/* Use caller-owned DEVICE memory (>= n_pix^2 uint32, e.g. a torch tensor) as the map
 * from now on; NULL returns to the library's own buffer.  The caller keeps ownership.
 * ML_ERR_INVALID_ARG if dptr is not 4-byte-aligned device (or managed) memory of the context's
 * device; the size cannot be checked and is the caller's responsibility. */
int ml_use_device_map(ml_ctx *ctx, void *dptr);

/* Launch on this CUDA stream (a cudaStream_t as void*, e.g. torch's current stream;
 * NULL = the legacy default stream) instead of the context's own. */
int ml_attach_stream(ml_ctx *ctx, void *cuda_stream);

/* Counters and timings of the last shoot. */
int ml_get_stats(const ml_ctx *ctx, ml_stats *out);

/* Source-plane position (y1, y2) of EVERY ray of [i0,i1) x [j0,j1), computed by the
 * shoot kernel itself (same tile membership, summation order and epilogue; the
 * capture instantiation stores y instead of binning).  y_out = HOST buffer of
 * 2*(i1-i0)*(j1-j0) doubles, y_out[2*((j-j0)*(i1-i0) + (i-i0)) + {0,1}]; a dropped
 * ray gives NaN.  Does not touch the map.  ML_ERR_INVALID_ARG for a bad region,
 * ML_ERR_OOM if (i1-i0)*(j1-j0) > 2^28 rays. */
int ml_capture_region(ml_ctx *ctx, int64_t i0, int64_t i1, int64_t j0, int64_t j1, double *y_out);

/* Same for n listed rays (HOST int64 arrays ray_i, ray_j): y_out[2k], y_out[2k+1].
 * Cost: one whole tile per distinct tile touched. */
int ml_probe(ml_ctx *ctx, int64_t n, const int64_t *ray_i, const int64_t *ray_j, double *y_out);

/* ---------------------------------------------------------------------------------------
 * Map comparison (section 3.1): the paper's two accuracy measures between
 * magnification maps -- the root-mean-square difference in magnitudes and a two-sample
 * Kolmogorov-Smirnov test on the distributions of
 *       Delta m_ij = -2.5 log10(mu_ij),   mu_ij = N_ij / N_rays        (eq. 10 :171, eq. 3 :47)
 * computed on the device from two count maps (fp64 arithmetic, one fused pass over both
 * maps plus small scans, readings M1-M4).
 * --------------------------------------------------------------------------------------- */
enum {
    ML_MEM_HOST = 0,  /* the map pointers are HOST memory (copied to the device inside the call) */
    ML_MEM_DEVICE = 1 /* the map pointers are DEVICE memory on `device` (e.g. ml_get_map_device)  */
};

typedef struct {
    uint64_t n_pixels;             /* n                                                          */
    uint64_t n_valid;              /* pixels with a count > 0 in BOTH maps (enter the RMS, M1)   */
    uint64_t n_empty_a, n_empty_b; /* pixels with count 0                                        */
    uint64_t sum_a, sum_b;         /* total counts                                               */
    uint32_t max_a, max_b;         /* largest count                                              */
    double mean_mu_a, mean_mu_b;   /* sum / (n * n_rays)  (eq. 3; compare with eq. 12)           */
    double rms_delta_m;            /* sqrt(mean over the n_valid pixels of (dm_a - dm_b)^2), mag */
    double ks_d;                   /* sup_x |F_a(x) - F_b(x)| over the Delta m of ALL pixels (an
                                      empty pixel is a sample at +inf, M2)                       */
    double ks_prob;                /* Q_KS((sqrt(Ne)+0.12+0.11/sqrt(Ne)) ks_d), Ne = n/2 (M3):
                                      probability of a distance >= ks_d under the null hypothesis */
    double kernel_ms;              /* device time of the whole call (one memset and seven kernels,
                                      no host round trip between them), CUDA events              */
    double pass_kernel_ms;         /* device time of the fused pass over the maps alone          */
} ml_map_compare_result;

/* Compare two count maps of n pixels each (same layout; n >= 1).  a, b: uint32 counts in HOST or
 * DEVICE memory according to `where`; n_rays_a, n_rays_b > 0 are the maps' N_rays.  `cuda_stream`
 * (cudaStream_t as void*, NULL = default stream) is used for all work; the call synchronises it.
 * out = HOST struct.  K-S ties between the two maps are decided exactly when n_rays_a, n_rays_b
 * have <= 26 significant bits.  ML_ERR_INVALID_ARG for NULL pointers, n < 1, n > 2^31-1,
 * non-positive or non-finite n_rays, or a bad `where`; ML_ERR_OOM if a count >= 2^27 makes the
 * count histogram too large; ML_ERR_CUDA without a device.  Scratch memory (histograms, scans, events,
 * a pinned result) is kept per device between calls; concurrent calls are serialised inside the library. */
int ml_map_compare(const uint32_t *a, double n_rays_a, const uint32_t *b, double n_rays_b, int64_t n,
                   int where, int32_t device, void *cuda_stream, ml_map_compare_result *out);

/* Histogram of Delta m of one map (the "probability distribution for change in magnitude" of
 * PAPER.md:169): hist_out[k] (HOST, n_bins uint64) = number of pixels with count > 0 and
 * lo + k w <= Delta m < lo + (k+1) w, w = (hi-lo)/n_bins (half-open bins, M4); pixels outside
 * [lo, hi) and empty pixels are not counted.  ML_ERR_INVALID_ARG unless lo < hi, 1 <= n_bins <= 2^20. */
int ml_delta_m_histogram(const uint32_t *counts, double n_rays, int64_t n, double lo, double hi,
                         int32_t n_bins, int where, int32_t device, void *cuda_stream, uint64_t *hist_out);

/* ml_delta_m_histogram for callers that must not allocate device memory.
 *
 * Who that is: a program that has handed (nearly) all of the GPU's memory to its own pool before it calls in here -- a
 * torch process whose caching allocator already holds the HBM, an inference server that reserved its arena at start-up --
 * so that a late cudaMalloc inside this library fails although the program itself still has room; and a program that
 * renders maps in a loop next to other GPU work and cannot accept that cudaMalloc / cudaFree stall every stream of the
 * device while they run.  ml_delta_m_histogram keeps a growing per-device cache (count histogram, partial sums, a
 * staging copy of the output) that it cudaMalloc's on first use and when a map is brighter than anything seen before.
 * This variant computes the same histogram with the same kernels but takes its scratch from a fixed array that is part
 * of the library image (a file-scope __device__ array in csrc/mapstats.cu); it calls no cudaMalloc, cudaFree,
 * cudaMallocHost, cudaEventCreate or any other allocating routine, on any call.
 *
 *   counts    DEVICE, n uint32 counts (e.g. the pointer of ml_get_map_device, or a torch tensor)       -- input, read only
 *   hist_out  DEVICE, n_bins uint64, 8-byte aligned, owned by the caller -- output; the call overwrites all n_bins
 *             entries (whatever was there before is discarded) with the histogram ml_delta_m_histogram defines
 *   n_rays, n, lo, hi, n_bins, device, cuda_stream: as for ml_delta_m_histogram.  There is no `where`: host pointers are
 *             not accepted, because staging them would need a device buffer.
 *
 * The limit.  The built-in scratch is ML_STATIC_SCRATCH_BYTES (1 MiB + 16 KiB): a count histogram of
 * ML_STATIC_MAX_COUNT = 2^18 bins, 256 per-CTA partial sums and one totals record.  Every GPU on which this process
 * uses the library holds that array from the moment the library's code is loaded on it until the process exits,
 * whether or not this function is ever called.  Therefore every count must be < ML_STATIC_MAX_COUNT (262144; the
 * BASELINE configs peak below 1e5).  A brighter pixel is detected on the device and the call returns ML_ERR_LIMIT
 * ("more than the built-in scratch holds"); hist_out is then unspecified.  Use ml_delta_m_histogram for such maps.
 * ML_ERR_INVALID_ARG for NULL / misaligned pointers and for the argument errors of ml_delta_m_histogram;
 * ML_ERR_CUDA if a runtime call fails.
 *
 * Set-up.  The first call on each device looks up the device address of the built-in array (cudaGetSymbolAddress with
 * that device current) and raises the pass kernel's shared-memory limit; later calls on that device reuse both.
 * Make that first call early, outside any stream capture: it is the only one that talks to the driver about more than
 * launches and memsets.
 *
 * Sharing.  All calls on a device use the one array, and it keeps what the previous call left in it; each call clears
 * the part that has to start at zero on `cuda_stream` before its kernels run.  Two calls whose GPU work overlaps would
 * corrupt each other's histograms.  Inside one process that cannot happen -- a call holds the library's lock until it
 * has synchronised `cuda_stream` -- but nothing orders this call against GPU work the caller has queued on OTHER
 * streams: do not let such work write `counts` or touch `hist_out` while the call runs. */
#define ML_STATIC_MAX_COUNT (1u << 18)
#define ML_STATIC_SCRATCH_BYTES ((1u << 20) + (1u << 14))
int ml_delta_m_histogram_static(const uint32_t *counts, double n_rays, int64_t n, double lo, double hi,
                                int32_t n_bins, int32_t device, void *cuda_stream, uint64_t *hist_out);

/* Static description of a return code. */
const char *ml_strerror(int code);

/* Library version string, e.g. "microlens-b200 0.1 (sm_100a)". */
const char *ml_version(void);

#ifdef __cplusplus
}
#endif
#endif /* MICROLENS_H */
