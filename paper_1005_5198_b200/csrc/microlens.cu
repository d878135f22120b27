// microlens.cu -- host side of the C ABI declared in include/microlens.h.
//
// Holds the problem geometry (PAPER.md:56-60 eq.5, :275-285 eq.11, :287-292 eq.12 with the
// concrete rules of BASELINE.json:configs[0]; readings R1-R8), the device
// buffers and the launch logic.  All arithmetic on rays happens in shoot_kernel.cuh.
// There is no CPU path: every entry point that computes needs a CUDA device.
#include "../../include/microlens.h"
#include "shoot_kernel.cuh"

#include <algorithm>
#include <atomic>
#include <chrono>
#include <cmath>
#include <cstring>
#include <new>
#include <vector>

using namespace mlb200;

struct ml_ctx {
    // problem statement
    double sigma, stellar_fraction, gamma, n_rays, L;
    int32_t n_pix;
    // derived
    double kappa_star, kappa_c, pixel, delta, a1, a2, r_star, mu_th;
    int64_t n1, n2, n_star_expected;
    // device state
    int device;
    int sm_count, sm_clock_khz;
    cudaStream_t own_stream, stream;
    cudaEvent_t ev0, ev1;
    unsigned int *map_own, *map;
    double2 *lens;
    double *mass;     // device masses m_i (eq.4), nullptr = unit masses
    int64_t n_lenses; // -1: never set
    // ml_set_lenses without a device allocation or a synchronisation per call: device buffers and a pinned staging copy
    // that only grow, and an event that says when the staging copy may be overwritten
    size_t lens_cap, mass_cap;      // elements the device buffers `lens` / `mass_buf` hold
    double *mass_buf;               // device masses buffer (kept when a later call sets unit masses); `mass` = it or nullptr
    unsigned char *h_stage;         // pinned: [n double2 | n double]
    size_t stage_bytes;
    cudaEvent_t ev_stage;           // recorded after the copies out of h_stage
    // device scratch of probes / captures / split-lens shoots (tile lists, captured positions, partial sums): kept between
    // calls while small, so that a probe loop does not pay two device-synchronising allocator calls per probe
    void *scratch[3];
    size_t scratch_bytes[3];
    unsigned long long *counters; // device [3]: running totals, never reset (a shoot reports the difference)
    unsigned long long *h_counters; // pinned host copy of the same
    unsigned long long seen[3];     // device totals after the last shoot
    unsigned long long base[3];     // device totals when the current (non-accumulating) run began
    int precision;
    int ray_mode;            // ML_RAYS_*
    unsigned long long ray_seed;
    // ML_RAYS_UNIFORM scratch, grown on demand and kept: bucketed ray lists, fill counts (+ 1 word: their maximum)
    unsigned long long *uni_list;
    size_t uni_list_entries;
    unsigned int *uni_fill;
    size_t uni_fill_entries;
    unsigned int *h_uni_max; // pinned
    ml_stats stats;
};

namespace {

struct DeviceGuard {
    int prev;
    bool ok;
    explicit DeviceGuard(int dev) : prev(0), ok(false)
    {
        if (cudaGetDevice(&prev) != cudaSuccess) return;
        ok = (prev == dev) || (cudaSetDevice(dev) == cudaSuccess);
    }
    ~DeviceGuard()
    {
        if (ok) cudaSetDevice(prev);
    }
};

// Device scratch for one call (see ml_ctx::scratch).  Slots up to kKeepScratchBytes stay with the context and only grow;
// a larger request is allocated for this call alone and freed when the lease ends (a context does not sit on gigabytes
// because of one large capture).  Every user synchronises the stream before its lease ends, so a kept slot is idle
// between calls.
constexpr size_t kKeepScratchBytes = 64ull << 20;
struct ScratchLease {
    void *ptr = nullptr;
    bool own = false; // allocated for this call only
    ScratchLease() = default;
    ScratchLease(const ScratchLease &) = delete;
    ScratchLease &operator=(const ScratchLease &) = delete;
    ~ScratchLease()
    {
        if (own && ptr) cudaFree(ptr);
    }
    // false: out of memory (nothing leased)
    bool take(ml_ctx *c, int slot, size_t bytes)
    {
        if (bytes == 0) bytes = 1;
        if (bytes > kKeepScratchBytes) {
            own = cudaMalloc(&ptr, bytes) == cudaSuccess;
            if (!own) { cudaGetLastError(); ptr = nullptr; }
            return own;
        }
        if (bytes > c->scratch_bytes[slot]) {
            if (c->scratch[slot]) cudaFree(c->scratch[slot]);
            c->scratch[slot] = nullptr;
            c->scratch_bytes[slot] = 0;
            if (cudaMalloc(&c->scratch[slot], bytes) != cudaSuccess) { cudaGetLastError(); c->scratch[slot] = nullptr; return false; }
            c->scratch_bytes[slot] = bytes;
        }
        ptr = c->scratch[slot];
        return true;
    }
    template <typename T> T *as() const { return static_cast<T *>(ptr); }
};
enum { kSlotList = 0, kSlotBuf = 1, kSlotPart = 2 };

// Tile shape and kernel instantiations per precision mode.
struct Mode {
    int tw, th;
};
#ifndef ML_KFF
#define ML_KFF 64
#endif
constexpr int RXF = 4, RYF = 4, KFF = ML_KFF;  // FP32_TILED (shoot_kernel_pipe) and FP32_COMPENSATED
constexpr int WARPS_T = 4, SHARED_T = 4, MINB_T = 3; // FP32_TILED: 128-thread CTAs, 3 per SM, all rows share
// source-order knobs of shoot_kernel_pipe (same arithmetic, different ptxas schedule), picked by a sweep of all 256
// values on the B200: 44 = rows reversed in stage 1, pair B's 1/r^2 after pair A's accumulations, sy before sx
// (C2 slab 72.4 -> 73.7 % of FP32 peak, C4 slab 73.3 -> 74.9 %, N* = 135: 66.2 -> 67.2 %)
// The instantiations with masses and with the Newton step have other optima (same sweep: masses 4 -> 65.4 / 66.3 %,
// against 63.6 / 64.3 % with 44; Newton 2 -> 56.3 / 56.6 %).
#ifndef ML_PIPE_TUNE
#define ML_PIPE_TUNE 44
#endif
constexpr int tune_of(bool mass, bool newton) { return newton ? 2 : (mass ? 4 : ML_PIPE_TUNE); }
constexpr int KFCP = 16;                   // FP32_COMPENSATED, regular grid: the pipe kernel with a Newton step
constexpr int RXD = 4, RYD = 2, KFD = 64;  // FP64

constexpr int RXR = 4, RYR = kRandRY;      // FP32 modes with random rays (shoot_kernel_rpipe): every ray carries its own offsets
static_assert(kRandWarps == kWarps, "mode_of: the random-ray kernels use 256-thread CTAs");

Mode mode_of(int precision, int ray_mode)
{
    if (ray_mode == ML_RAYS_UNIFORM) return {kUniBW, kUniBH}; // the patch of the image plane one CTA's rays come from
    if (precision == ML_PREC_FP64) return {32 * RXD, kWarps * RYD};
    if (ray_mode == ML_RAYS_RANDOM) return {32 * RXR, kWarps * RYR};
    return {32 * RXF, WARPS_T * RYF};
}

Mode mode_of(const ml_ctx *c) { return mode_of(c->precision, c->ray_mode); }

template <bool CAPTURE, bool MASS> cudaError_t launch_m(int precision, dim3 g, const ShootParams &p, cudaStream_t s)
{
    switch (precision) {
    case ML_PREC_FP64:
        shoot_kernel<double, RXD, RYD, KFD, false, CAPTURE, MASS><<<g, kThreads, 0, s>>>(p);
        break;
    case ML_PREC_FP32_COMPENSATED:
        shoot_kernel_pipe<SHARED_T, KFCP, WARPS_T, MINB_T, true, CAPTURE, MASS, true, tune_of(MASS, true)><<<g, WARPS_T * 32, 0, s>>>(p);
        break;
    default:
        shoot_kernel_pipe<SHARED_T, KFF, WARPS_T, MINB_T, true, CAPTURE, MASS, false, tune_of(MASS, false)><<<g, WARPS_T * 32, 0, s>>>(p);
        break;
    }
    return cudaGetLastError();
}

// shoot_kernel_rpipe: own reciprocals on the last row of every lens (OWN = 2) and source-order knobs 10, from a sweep of
// OWN x TUNE on the B200 (C2 slab: 53.7 % of FP32 peak with everything shared, 56.8 % with these; C4 slab 55.5 -> 59.0 %)
#ifndef ML_RPIPE_OWN
#define ML_RPIPE_OWN 2
#endif
#ifndef ML_RPIPE_TUNE
#define ML_RPIPE_TUNE 10
#endif
// More than 48 KB of dynamic shared memory needs cudaFuncAttributeMaxDynamicSharedMemorySize, and that attribute belongs to
// the (function, device) pair: a process that shoots from contexts on several GPUs has to opt in on each of them.  `done`
// (one per kernel instantiation) has bit d set once device d is done; the launch runs with the context's device current.
template <typename Kernel> cudaError_t opt_in_shared_memory(Kernel kernel, size_t smem, std::atomic<unsigned long long> &done)
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    const bool tracked = dev >= 0 && dev < 64;
    if (tracked && ((done.load(std::memory_order_acquire) >> dev) & 1ull)) return cudaSuccess;
    e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem); // idempotent: a race repeats it harmlessly
    if (e == cudaSuccess && tracked) done.fetch_or(1ull << dev, std::memory_order_release);
    return e;
}

// random ray positions (reading R17): the packed random-ray kernel in the FP32 modes, the generic
// kernel with per-ray offsets in fp64
template <int KF, bool CAPTURE, bool MASS, bool NEWTON> cudaError_t launch_rpipe(dim3 g, const ShootParams &p, cudaStream_t s)
{
    constexpr size_t smem = rpipe_smem_bytes(MASS);
    static std::atomic<unsigned long long> opted_in{0ull}; // per device, see opt_in_shared_memory
    const cudaError_t e = opt_in_shared_memory(shoot_kernel_rpipe<KF, 2, CAPTURE, MASS, NEWTON, ML_RPIPE_OWN, ML_RPIPE_TUNE>, smem, opted_in);
    if (e != cudaSuccess) return e;
    shoot_kernel_rpipe<KF, 2, CAPTURE, MASS, NEWTON, ML_RPIPE_OWN, ML_RPIPE_TUNE><<<g, kRandWarps * 32, smem, s>>>(p);
    return cudaGetLastError();
}

template <bool CAPTURE, bool MASS> cudaError_t launch_r(int precision, dim3 g, const ShootParams &p, cudaStream_t s)
{
    switch (precision) {
    case ML_PREC_FP64:
        shoot_kernel<double, RXD, RYD, KFD, false, CAPTURE, MASS, true><<<g, kThreads, 0, s>>>(p);
        return cudaGetLastError();
    case ML_PREC_FP32_COMPENSATED:
        return launch_rpipe<KFCP, CAPTURE, MASS, true>(g, p, s);
    default:
        return launch_rpipe<KFF, CAPTURE, MASS, false>(g, p, s);
    }
}

// unit masses (every map of the paper) run the instantiations without the mass multiply
template <bool CAPTURE> cudaError_t launch(int precision, int ray_mode, dim3 g, const ShootParams &p, cudaStream_t s)
{
    if (g.x == 0 || g.y == 0) return cudaSuccess;
    if (ray_mode == ML_RAYS_RANDOM)
        return p.mass ? launch_r<CAPTURE, true>(precision, g, p, s) : launch_r<CAPTURE, false>(precision, g, p, s);
    return p.mass ? launch_m<CAPTURE, true>(precision, g, p, s) : launch_m<CAPTURE, false>(precision, g, p, s);
}

// uniformly random rays over the whole rectangle (reading R20): bucketed ray lists, one CTA per
// kUniSlots entries; shoot_kernel_upipe in the FP32 modes, the generic kernel in fp64
// source-order knobs of shoot_kernel_upipe (same arithmetic, another ptxas schedule), from a sweep of all 32 values on the
// B200: 29 = accumulations as sx, sx, sy, sy; both lenses' differences before the first r^2; ray pair B's reciprocals
// first; both 1/r^2 pairs of a row before the first accumulation (C2 step 1397 -> 1382 ms, C4 55.8 -> 56.6 % of FP32 peak)
#ifndef ML_UPIPE_TUNE
#define ML_UPIPE_TUNE 29
#endif
template <int KF, bool CAPTURE, bool MASS, bool NEWTON> cudaError_t launch_upipe(dim3 g, const ShootParams &p, cudaStream_t s)
{
    constexpr size_t smem = upipe_smem_bytes(MASS);
    static std::atomic<unsigned long long> opted_in{0ull}; // per device, see opt_in_shared_memory
    const cudaError_t e = opt_in_shared_memory(shoot_kernel_upipe<KF, 4, CAPTURE, MASS, NEWTON, ML_UPIPE_TUNE>, smem, opted_in);
    if (e != cudaSuccess) return e;
    shoot_kernel_upipe<KF, 4, CAPTURE, MASS, NEWTON, ML_UPIPE_TUNE><<<g, kUniWarps * 32, smem, s>>>(p);
    return cudaGetLastError();
}

// list entries one CTA takes: 128 threads x 8 rays (shoot_kernel_upipe), 256 x 8 (the generic kernel in fp64)
unsigned int uniform_slots(int precision) { return precision == ML_PREC_FP64 ? kThreads * RXD * RYD : kUniWarps * 32 * 4 * kRandRY; }

// g.y = the largest bucket fill; turned into list slices of the kernel's size here
template <bool CAPTURE, bool MASS> cudaError_t launch_u(int precision, dim3 g, const ShootParams &p, cudaStream_t s)
{
    g.y = (g.y + uniform_slots(precision) - 1) / uniform_slots(precision);
    switch (precision) {
    case ML_PREC_FP64:
        shoot_kernel<double, RXD, RYD, KFD, false, CAPTURE, MASS, true, true><<<g, kThreads, 0, s>>>(p);
        return cudaGetLastError();
    case ML_PREC_FP32_COMPENSATED:
        return launch_upipe<KFCP, CAPTURE, MASS, true>(g, p, s);
    default:
        return launch_upipe<KFF, CAPTURE, MASS, false>(g, p, s);
    }
}

__global__ void max_fill_kernel(const unsigned int *fill, long long n, unsigned int *out)
{
    unsigned int m = 0;
    for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (long long)gridDim.x * blockDim.x) m = max(m, fill[k]);
    m = __reduce_max_sync(0xffffffffu, m);
    if ((threadIdx.x & 31) == 0 && m) atomicMax(out, m);
}

ShootParams base_params(const ml_ctx *c)
{
    ShootParams p;
    std::memset(&p, 0, sizeof(p));
    p.lens = c->lens;
    p.mass = c->mass;
    p.n_lens = (int)c->n_lenses;
    p.n_pix = c->n_pix;
    p.delta = c->delta;
    p.half1 = (double)(c->n1 - 1) / 2.0;
    p.half2 = (double)(c->n2 - 1) / 2.0;
    p.c1 = 1.0 - c->gamma - c->kappa_c;
    p.c2 = 1.0 + c->gamma - c->kappa_c;
    p.halfL = c->L / 2.0;
    p.inv_pixel = (double)c->n_pix / c->L;
    p.k1 = p.c1 * p.inv_pixel;
    p.k2 = p.c2 * p.inv_pixel;
    p.hoff = p.halfL * p.inv_pixel;
    p.map = c->map;
    p.counters = c->counters;
    p.n1 = c->n1;
    p.ray_seed = c->ray_seed;
    p.n1d = (double)c->n1;
    p.n2d = (double)c->n2;
    return p;
}

#ifndef ML_UNIFORM_LIST_BYTES
#define ML_UNIFORM_LIST_BYTES 0
#endif
constexpr long long kUniformListBytes = ML_UNIFORM_LIST_BYTES; // 0: sized from the device memory (below)
#ifndef ML_UNIFORM_FAIL_ALLOCS
#define ML_UNIFORM_FAIL_ALLOCS 0
#endif
// (test builds: the first ML_UNIFORM_FAIL_ALLOCS list allocations of the process report failure, to drive the retry below)
inline bool uniform_alloc_fails_in_this_test_build()
{
    static int left = ML_UNIFORM_FAIL_ALLOCS;
    if (left <= 0) return false;
    --left;
    return true;
}

// ML_RAYS_UNIFORM: shoot (or capture) the rays behind handles 0 .. n_handles - 1 (p.list_w / p.probe_ids say which).
// The image plane is cut into buckets of kUniBW x kUniBH grid cells; as many bucket rows as the list memory holds are
// done per pass: zero the fill counts, scatter the handles (every pass draws every ray again and keeps those of its
// rows), read back the largest fill (it sizes the grid; a fill above the capacity repeats the pass with more room),
// shoot.  Events ev0 / ev1 bracket everything.  Does not synchronise after the last launch.
int uniform_run(ml_ctx *c, ShootParams p, long long n_handles, bool capture, uint64_t *launches)
{
    const long long nbx = (c->n1 + kUniBW - 1) / kUniBW, nby = (c->n2 + kUniBH - 1) / kUniBH;
    const double mean = (double)n_handles * (double)kUniBW * (double)kUniBH / ((double)c->n1 * (double)c->n2);
    unsigned int cap = (unsigned int)std::min(4.0e9, std::ceil(mean + 6.0 * std::sqrt(mean) + 32.0));
    if (cudaEventRecord(c->ev0, c->stream) != cudaSuccess) return ML_ERR_CUDA;
    long long row0 = 0;
    while (row0 < nby) {
        cap = (cap + 3u) & ~3u;
        // list memory: at most 45 % of the device (82 GB of a B200's 180: C2's 8.4e9 rays in one pass), and never more
        // than what is already held plus what is free less 8 GiB
        size_t free_b = 0, total_b = 0;
        if (cudaMemGetInfo(&free_b, &total_b) != cudaSuccess) return ML_ERR_CUDA;
        double budget = std::min(0.45 * (double)total_b, (double)c->uni_list_entries * 8.0 + (double)free_b - 8.0 * 1073741824.0);
        if (kUniformListBytes > 0) budget = (double)kUniformListBytes; // (test builds: many passes on a small problem)
        long long rows = (long long)(budget / ((double)nbx * cap * 8.0));
        rows = std::max<long long>(1, std::min(rows, nby - row0));
        if ((double)rows * (double)nbx > 2.0e9) rows = std::max<long long>(1, (long long)(2.0e9 / (double)nbx));
        size_t n_b = (size_t)rows * (size_t)nbx, need = n_b * cap;
        if (need > c->uni_list_entries) {
            if (c->uni_list) cudaFree(c->uni_list);
            c->uni_list = nullptr;
            c->uni_list_entries = 0;
            // cudaMemGetInfo is a snapshot: another context or a caching allocator on the same device may have taken the
            // memory since.  A stripe of half as many bucket rows needs half the list: retry down to one row.
            for (;;) {
                if (!uniform_alloc_fails_in_this_test_build() && cudaMalloc(&c->uni_list, need * sizeof(unsigned long long)) == cudaSuccess) break;
                cudaGetLastError();
                c->uni_list = nullptr;
                if (rows <= 1) return ML_ERR_OOM;
                rows = (rows + 1) / 2;
                n_b = (size_t)rows * (size_t)nbx;
                need = n_b * cap;
            }
            c->uni_list_entries = need;
        }
        if (n_b + 1 > c->uni_fill_entries) {
            if (c->uni_fill) cudaFree(c->uni_fill);
            c->uni_fill = nullptr;
            c->uni_fill_entries = 0;
            if (cudaMalloc(&c->uni_fill, (n_b + 1) * sizeof(unsigned int)) != cudaSuccess) { cudaGetLastError(); return ML_ERR_OOM; }
            c->uni_fill_entries = n_b + 1;
        }
        p.ray_list = c->uni_list;
        p.bucket_fill = c->uni_fill;
        p.bucket_cap = cap;
        p.bucket_nx = nbx;
        p.bucket_row0 = row0;
        ScatterParams q;
        q.sp = p;
        q.n_handles = n_handles;
        q.bucket_row1 = row0 + rows;
        q.fill = c->uni_fill;
        q.list = c->uni_list;
        const int sblocks = (int)std::min<long long>((n_handles + kScatterRun - 1) / kScatterRun, (long long)c->sm_count * 32);
        const int mblocks = (int)std::min<long long>(((long long)n_b + 255) / 256, (long long)c->sm_count * 8);
        if (cudaMemsetAsync(c->uni_fill, 0, (n_b + 1) * sizeof(unsigned int), c->stream) != cudaSuccess) return ML_ERR_CUDA;
        uniform_scatter_kernel<<<sblocks, 256, 0, c->stream>>>(q);
        max_fill_kernel<<<mblocks, 256, 0, c->stream>>>(c->uni_fill, (long long)n_b, c->uni_fill + n_b);
        if (cudaGetLastError() != cudaSuccess ||
            cudaMemcpyAsync(c->h_uni_max, c->uni_fill + n_b, sizeof(unsigned int), cudaMemcpyDeviceToHost, c->stream) != cudaSuccess ||
            cudaStreamSynchronize(c->stream) != cudaSuccess)
            return ML_ERR_CUDA;
        *launches += 2;
        const unsigned int mx = *c->h_uni_max;
        if (mx > cap) { // (6 sigma above the mean: about once in 1e9 buckets)
            if (mx >= 0xfffffff0u) return ML_ERR_OOM;
            cap = mx;
            continue;
        }
        if (mx > 0) {
            const dim3 grid((unsigned int)n_b, mx, 1); // (y: launch_u turns the largest fill into list slices)
            cudaError_t e;
            if (capture) e = p.mass ? launch_u<true, true>(c->precision, grid, p, c->stream) : launch_u<true, false>(c->precision, grid, p, c->stream);
            else e = p.mass ? launch_u<false, true>(c->precision, grid, p, c->stream) : launch_u<false, false>(c->precision, grid, p, c->stream);
            if (e != cudaSuccess) return ML_ERR_CUDA;
            *launches += 1;
        }
        row0 += rows;
    }
    if (cudaEventRecord(c->ev1, c->stream) != cudaSuccess) return ML_ERR_CUDA;
    return ML_OK;
}

// Second half of a split launch (see lens_range in shoot_kernel.cuh): add the partial sums of the lens ranges, then
// write the positions (CAPTURE) or bin the rays.
template <bool CAPTURE>
cudaError_t launch_combine(int precision, int ray_mode, unsigned int n_tiles, const ShootParams &p, int n_splits, cudaStream_t s)
{
    const dim3 g(n_tiles, 1, 1);
    if (precision == ML_PREC_FP64) {
        if (ray_mode == ML_RAYS_RANDOM) combine_kernel<RXD, RYD, kWarps, true, CAPTURE><<<g, kThreads, 0, s>>>(p, n_splits);
        else combine_kernel<RXD, RYD, kWarps, false, CAPTURE><<<g, kThreads, 0, s>>>(p, n_splits);
    } else if (ray_mode == ML_RAYS_RANDOM) {
        combine_kernel<RXR, RYR, kRandWarps, true, CAPTURE><<<g, kRandWarps * 32, 0, s>>>(p, n_splits);
    } else {
        combine_kernel<RXF, RYF, WARPS_T, false, CAPTURE><<<g, WARPS_T * 32, 0, s>>>(p, n_splits);
    }
    return cudaGetLastError();
}

// Lens ranges for a launch of nb tiles: none while the tiles alone give every SM work or the lens list is
// short; otherwise enough ranges (multiples of the 512-lens chunk, at least 2048 lenses each) for about two CTAs
// per SM, within `max_splits` (memory of the partial sums).
int plan_lens_split(const ml_ctx *c, long long nb, long long max_splits, int *split_len)
{
    *split_len = 0;
    const long long want_ctas = 2ll * c->sm_count;
    if (c->n_lenses < 8192 || nb >= want_ctas || max_splits < 2) return 1;
    long long splits = std::min<long long>({(want_ctas + nb - 1) / nb, c->n_lenses / 2048, max_splits});
    if (splits < 2) return 1;
    long long len = (c->n_lenses + splits - 1) / splits;
    len = (len + kChunk - 1) / kChunk * kChunk;
    splits = (c->n_lenses + len - 1) / len;
    if (splits < 2) return 1;
    *split_len = (int)len;
    return (int)splits;
}

// ml_shoot_region over a handful of tiles and very many lenses: the capture instantiation (which bins nothing) runs
// once per (tile, lens range) and leaves fp64 partial sums; combine_kernel<.., CAPTURE = false> adds them in range
// order and bins the rays with the region masks.  Synchronises (the scratch is idle again when it returns).
int shoot_split(ml_ctx *c, ShootParams p, const Mode &m, long long ti0, long long tj0, long long tiles_x, long long tiles_y,
                int n_splits, int split_len, float *ms)
{
    const long long n_tiles = tiles_x * tiles_y;
    std::vector<long long> tiles;
    try {
        tiles.reserve((size_t)(2 * n_tiles));
        for (long long ty = 0; ty < tiles_y; ++ty)
            for (long long tx = 0; tx < tiles_x; ++tx) {
                tiles.push_back(ti0 + tx);
                tiles.push_back(tj0 + ty);
            }
    } catch (const std::bad_alloc &) {
        return ML_ERR_OOM;
    }
    ScratchLease list, part;
    int rc = ML_OK;
    if (!list.take(c, kSlotList, tiles.size() * sizeof(long long)) ||
        !part.take(c, kSlotPart, (size_t)n_splits * n_tiles * m.tw * m.th * sizeof(double2)))
        rc = ML_ERR_OOM;
    if (rc == ML_OK) {
        long long *d_list = list.as<long long>();
        p.tile_list = d_list;
        p.split_len = split_len;
        p.partial = part.as<double2>();
        if (cudaMemcpyAsync(d_list, tiles.data(), tiles.size() * sizeof(long long), cudaMemcpyHostToDevice, c->stream) != cudaSuccess ||
            cudaEventRecord(c->ev0, c->stream) != cudaSuccess ||
            launch<true>(c->precision, c->ray_mode, dim3((unsigned int)n_tiles, (unsigned int)n_splits, 1), p, c->stream) != cudaSuccess ||
            launch_combine<false>(c->precision, c->ray_mode, (unsigned int)n_tiles, p, n_splits, c->stream) != cudaSuccess ||
            cudaEventRecord(c->ev1, c->stream) != cudaSuccess || cudaStreamSynchronize(c->stream) != cudaSuccess ||
            cudaEventElapsedTime(ms, c->ev0, c->ev1) != cudaSuccess) {
            rc = ML_ERR_CUDA;
            cudaStreamSynchronize(c->stream); // the leases end below: nothing may still be running in them
        }
    }
    if (rc == ML_OK) c->stats.capture_ctas = (uint64_t)n_tiles * (uint64_t)n_splits;
    return rc;
}

// One shoot launch is a 2-D grid of tiles (x = tile column, y = tile row).  A grid holds at most 2^31 - 1 CTAs along x
// and 65535 along y; larger regions are cut into several launches that continue the same tile raster (tile_i0 / tile_j0
// of each launch).  The limits are macros so that a test build (-DML_MAX_GRID_X=7 -DML_MAX_GRID_Y=50) can exercise the
// split on a small problem.
#ifndef ML_MAX_GRID_X
#define ML_MAX_GRID_X 0x7fffffffLL
#endif
#ifndef ML_MAX_GRID_Y
#define ML_MAX_GRID_Y 65535LL
#endif
constexpr long long kMaxGridX = ML_MAX_GRID_X, kMaxGridY = ML_MAX_GRID_Y;
static_assert(kMaxGridX >= 1 && kMaxGridX <= 0x7fffffffLL && kMaxGridY >= 1 && kMaxGridY <= 65535LL, "grid limits");

int shoot_region_run(ml_ctx *c, int64_t i0, int64_t i1, int64_t j0, int64_t j1, int accumulate);

// The device counters are running totals; `seen` (their value after the last shoot) becomes the next run's `base`.  A run
// that fails after some of its kernels were enqueued has already moved the totals, so on every error exit they are read
// again (best effort): otherwise the next run's rays_shot / rays_in_map / interactions would include the failed run's rays.
int shoot_region_impl(ml_ctx *c, int64_t i0, int64_t i1, int64_t j0, int64_t j1, int accumulate)
{
    if (!c) return ML_ERR_INVALID_ARG;
    if (c->n_lenses < 0) return ML_ERR_STATE;
    if (i0 < 0 || j0 < 0 || i1 > c->n1 || j1 > c->n2 || i0 > i1 || j0 > j1) return ML_ERR_INVALID_ARG;
    DeviceGuard g(c->device);
    if (!g.ok) return ML_ERR_CUDA;
    const int rc = shoot_region_run(c, i0, i1, j0, j1, accumulate);
    if (rc != ML_OK) {
        cudaGetLastError();
        if (cudaMemcpyAsync(c->h_counters, c->counters, 3 * sizeof(unsigned long long), cudaMemcpyDeviceToHost, c->stream) == cudaSuccess &&
            cudaStreamSynchronize(c->stream) == cudaSuccess)
            std::memcpy(c->seen, c->h_counters, sizeof(c->seen));
        else
            cudaGetLastError();
    }
    return rc;
}

int shoot_region_run(ml_ctx *c, int64_t i0, int64_t i1, int64_t j0, int64_t j1, int accumulate)
{
    const auto t0 = std::chrono::steady_clock::now();
    if (!accumulate) {
        // one memset: the counters are running totals and are never zeroed (the run's statistics are differences)
        if (cudaMemsetAsync(c->map, 0, (size_t)c->n_pix * c->n_pix * sizeof(unsigned int), c->stream) != cudaSuccess)
            return ML_ERR_CUDA;
        std::memset(&c->stats, 0, sizeof(c->stats));
        std::memcpy(c->base, c->seen, sizeof(c->base));
    }
    float ms = 0.f;
    uint64_t launches = 0;
    if (i1 > i0 && j1 > j0) {
        const Mode m = mode_of(c);
        ShootParams p = base_params(c);
        p.i0 = i0; p.i1 = i1; p.j0 = j0; p.j1 = j1;
        if (c->ray_mode == ML_RAYS_UNIFORM) { // the region selects ray ids; where the rays are is the generator's business
            p.list_w = i1 - i0;
            const int rc = uniform_run(c, p, (i1 - i0) * (j1 - j0), false, &launches);
            if (rc != ML_OK) return rc;
        } else {
        const long long ti0 = i0 / m.tw, tj0 = j0 / m.th;
        const long long tiles_x = (i1 - 1) / m.tw - ti0 + 1, tiles_y = (j1 - 1) / m.th - tj0 + 1;
        int split_len = 0;
        const int n_splits = (double)tiles_x * (double)tiles_y < 4096.0
                                 ? plan_lens_split(c, tiles_x * tiles_y, (1024ll << 20) / (tiles_x * tiles_y * m.tw * m.th * (long long)sizeof(double2)), &split_len)
                                 : 1;
        if (n_splits > 1) { // few rays, very many lenses: split the lens loop over CTAs, then combine and bin
            const int rc = shoot_split(c, p, m, ti0, tj0, tiles_x, tiles_y, n_splits, split_len, &ms);
            if (rc != ML_OK) return rc;
            launches = 2;
        } else {
        if (cudaEventRecord(c->ev0, c->stream) != cudaSuccess) return ML_ERR_CUDA;
        for (long long by = 0; by < tiles_y; by += kMaxGridY)
            for (long long bx = 0; bx < tiles_x; bx += kMaxGridX) {
                p.tile_i0 = ti0 + bx;
                p.tile_j0 = tj0 + by;
                const dim3 grid((unsigned int)std::min(kMaxGridX, tiles_x - bx), (unsigned int)std::min(kMaxGridY, tiles_y - by), 1);
                if (launch<false>(c->precision, c->ray_mode, grid, p, c->stream) != cudaSuccess) return ML_ERR_CUDA;
                ++launches;
            }
        if (cudaEventRecord(c->ev1, c->stream) != cudaSuccess) return ML_ERR_CUDA;
        }
        } // not ML_RAYS_UNIFORM
    }
    if (cudaMemcpyAsync(c->h_counters, c->counters, 3 * sizeof(unsigned long long), cudaMemcpyDeviceToHost, c->stream) != cudaSuccess ||
        cudaStreamSynchronize(c->stream) != cudaSuccess)
        return ML_ERR_CUDA;
    if (launches && ms == 0.f && cudaEventElapsedTime(&ms, c->ev0, c->ev1) != cudaSuccess) return ML_ERR_CUDA;
    std::memcpy(c->seen, c->h_counters, sizeof(c->seen));
    c->stats.rays_shot = c->seen[0] - c->base[0];
    c->stats.rays_in_map = c->seen[1] - c->base[1];
    c->stats.rays_dropped = c->seen[2] - c->base[2];
    c->stats.interactions = c->stats.rays_shot * (uint64_t)c->n_lenses;
    c->stats.kernel_launches += launches;
    c->stats.kernel_ms += ms;
    c->stats.total_ms = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t0).count();
    return ML_OK;
}

// Run the capture instantiation on an explicit list of global tiles and hand every
// batch of results to `sink(first_tile_in_list, n_tiles_in_batch, host_buffer)`.
template <typename Sink>
int capture_tiles(ml_ctx *c, const std::vector<long long> &tiles /* pairs */, Sink sink)
{
    const Mode m = mode_of(c);
    const size_t per_tile = (size_t)m.tw * m.th;
    const long long n_tiles = (long long)(tiles.size() / 2);
    if (n_tiles == 0) return ML_OK;
    const long long batch = std::max<long long>(1, std::min<long long>(n_tiles, (256ll << 20) / (long long)(per_tile * sizeof(double2))));
    int split_len = 0;
    const int n_splits = plan_lens_split(c, batch, (1024ll << 20) / (long long)(batch * per_tile * sizeof(double2)), &split_len);
    ScratchLease list, buf, part;
    std::vector<double2> h_buf;
    try {
        h_buf.resize((size_t)batch * per_tile);
    } catch (const std::bad_alloc &) {
        return ML_ERR_OOM;
    }
    int rc = ML_OK;
    if (!list.take(c, kSlotList, tiles.size() * sizeof(long long)) || !buf.take(c, kSlotBuf, (size_t)batch * per_tile * sizeof(double2)) ||
        (n_splits > 1 && !part.take(c, kSlotPart, (size_t)n_splits * batch * per_tile * sizeof(double2))))
        return ML_ERR_OOM;
    long long *d_list = list.as<long long>();
    double2 *d_buf = buf.as<double2>(), *d_part = part.as<double2>();
    if (rc == ML_OK && cudaMemcpyAsync(d_list, tiles.data(), tiles.size() * sizeof(long long), cudaMemcpyHostToDevice, c->stream) != cudaSuccess)
        rc = ML_ERR_CUDA;
    for (long long first = 0; rc == ML_OK && first < n_tiles; first += batch) {
        const long long nb = std::min(batch, n_tiles - first);
        ShootParams p = base_params(c);
        p.capture = d_buf;
        p.tile_list = d_list + 2 * first;
        cudaError_t e;
        if (n_splits > 1) {
            p.split_len = split_len;
            p.partial = d_part;
            e = launch<true>(c->precision, c->ray_mode, dim3((unsigned int)nb, (unsigned int)n_splits, 1), p, c->stream);
            if (e == cudaSuccess) e = launch_combine<true>(c->precision, c->ray_mode, (unsigned int)nb, p, n_splits, c->stream);
        } else {
            e = launch<true>(c->precision, c->ray_mode, dim3((unsigned int)nb, 1, 1), p, c->stream);
        }
        if (e != cudaSuccess ||
            cudaMemcpyAsync(h_buf.data(), d_buf, (size_t)nb * per_tile * sizeof(double2), cudaMemcpyDeviceToHost, c->stream) != cudaSuccess ||
            cudaStreamSynchronize(c->stream) != cudaSuccess) {
            rc = ML_ERR_CUDA;
            break;
        }
        c->stats.capture_ctas = n_splits > 1 ? (uint64_t)nb * (uint64_t)n_splits : 0;
        sink(first, nb, h_buf.data());
    }
    if (rc != ML_OK) cudaStreamSynchronize(c->stream); // the leases end here: nothing may still be running in them
    return rc;
}

// ML_RAYS_UNIFORM: positions of the rays behind handles 0 .. n - 1 (region-relative indices, or entries of `ids`).
int capture_uniform(ml_ctx *c, ShootParams p, long long n, const std::vector<long long> *ids, double *y_out)
{
    ScratchLease buf, idl;
    if (!buf.take(c, kSlotBuf, (size_t)n * sizeof(double2)) || (ids && !idl.take(c, kSlotList, (size_t)n * sizeof(long long)))) return ML_ERR_OOM;
    double2 *d_buf = buf.as<double2>();
    long long *d_ids = ids ? idl.as<long long>() : nullptr;
    int rc = ML_OK;
    if (rc == ML_OK && ids &&
        cudaMemcpyAsync(d_ids, ids->data(), (size_t)n * sizeof(long long), cudaMemcpyHostToDevice, c->stream) != cudaSuccess)
        rc = ML_ERR_CUDA;
    if (rc == ML_OK) {
        p.capture = d_buf;
        p.probe_ids = d_ids;
        uint64_t launches = 0;
        rc = uniform_run(c, p, n, true, &launches);
    }
    if (rc == ML_OK && (cudaMemcpyAsync(y_out, d_buf, (size_t)n * sizeof(double2), cudaMemcpyDeviceToHost, c->stream) != cudaSuccess ||
                        cudaStreamSynchronize(c->stream) != cudaSuccess))
        rc = ML_ERR_CUDA;
    if (rc != ML_OK) cudaStreamSynchronize(c->stream); // the leases end here: nothing may still be running in them
    return rc;
}

} // namespace

extern "C" {

int ml_create(double sigma, double stellar_fraction, double gamma, int32_t n_pix, double n_rays, double L,
              int32_t device, ml_ctx **out)
{
    if (!out) return ML_ERR_INVALID_ARG;
    *out = nullptr;
    if (!std::isfinite(sigma) || !std::isfinite(stellar_fraction) || !std::isfinite(gamma) || !std::isfinite(n_rays) ||
        !std::isfinite(L))
        return ML_ERR_INVALID_ARG;
    if (sigma < 0.0 || stellar_fraction < 0.0 || stellar_fraction > 1.0 || n_pix <= 0 || n_pix > 32768 ||
        n_rays <= 0.0 || L <= 0.0)
        return ML_ERR_INVALID_ARG;
    const double minus = 1.0 - sigma - gamma, plus = 1.0 - sigma + gamma;
    if (std::fabs(minus) < 1e-6 || std::fabs(plus) < 1e-6) return ML_ERR_INVALID_ARG;

    ml_ctx *c = new (std::nothrow) ml_ctx;
    if (!c) return ML_ERR_OOM;
    std::memset(c, 0, sizeof(*c));
    c->sigma = sigma; c->stellar_fraction = stellar_fraction; c->gamma = gamma;
    c->n_rays = n_rays; c->L = L; c->n_pix = n_pix;
    c->kappa_star = stellar_fraction * sigma;
    c->kappa_c = sigma - c->kappa_star;
    c->pixel = L / (double)n_pix;
    c->delta = c->pixel / std::sqrt(n_rays);
    c->a1 = 1.2 * (L / 2.0) / std::fabs(minus);
    c->a2 = 1.2 * (L / 2.0) / std::fabs(plus);
    const double f1 = std::ceil(2.0 * c->a1 / c->delta - 1e-9), f2 = std::ceil(2.0 * c->a2 / c->delta - 1e-9);
    if (!(f1 >= 1.0) || !(f2 >= 1.0) || f1 * f2 >= 4.611686018427388e18 || f1 >= 9.0e15 || f2 >= 9.0e15) {
        delete c;
        return ML_ERR_INVALID_ARG;
    }
    c->n1 = (int64_t)f1;
    c->n2 = (int64_t)f2;
    c->r_star = 1.3 * std::sqrt(c->a1 * c->a1 + c->a2 * c->a2);
    c->n_star_expected = (int64_t)std::floor(c->kappa_star * c->r_star * c->r_star + 0.5);
    c->mu_th = 1.0 / ((1.0 - sigma) * (1.0 - sigma) - gamma * gamma);
    c->n_lenses = -1;
    c->precision = ML_PREC_FP32_TILED;
    c->ray_mode = ML_RAYS_REGULAR;
    c->device = device;

    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) {
        cudaGetLastError();
        delete c;
        return ML_ERR_CUDA;
    }
    DeviceGuard g(device);
    int rc = g.ok ? ML_OK : ML_ERR_CUDA;
    if (rc == ML_OK &&
        (cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, device) != cudaSuccess ||
         cudaDeviceGetAttribute(&c->sm_clock_khz, cudaDevAttrClockRate, device) != cudaSuccess ||
         cudaStreamCreateWithFlags(&c->own_stream, cudaStreamNonBlocking) != cudaSuccess ||
         cudaEventCreate(&c->ev0) != cudaSuccess || cudaEventCreate(&c->ev1) != cudaSuccess))
        rc = ML_ERR_CUDA;
    if (rc == ML_OK) {
        c->stream = c->own_stream;
        if (cudaMalloc(&c->map_own, (size_t)n_pix * n_pix * sizeof(unsigned int)) != cudaSuccess ||
            cudaMalloc(&c->counters, 3 * sizeof(unsigned long long)) != cudaSuccess ||
            cudaMallocHost(&c->h_counters, 3 * sizeof(unsigned long long)) != cudaSuccess ||
            cudaMallocHost(&c->h_uni_max, sizeof(unsigned int)) != cudaSuccess) {
            cudaGetLastError();
            rc = ML_ERR_OOM;
        }
    }
    if (rc == ML_OK) {
        c->map = c->map_own;
        if (cudaMemsetAsync(c->map, 0, (size_t)n_pix * n_pix * sizeof(unsigned int), c->stream) != cudaSuccess ||
            cudaMemsetAsync(c->counters, 0, 3 * sizeof(unsigned long long), c->stream) != cudaSuccess ||
            cudaStreamSynchronize(c->stream) != cudaSuccess)
            rc = ML_ERR_CUDA;
    }
    if (rc != ML_OK) {
        ml_destroy(c);
        return rc;
    }
    *out = c;
    return ML_OK;
}

void ml_destroy(ml_ctx *c)
{
    if (!c) return;
    {
        DeviceGuard g(c->device);
        if (g.ok) {
            if (c->own_stream) cudaStreamSynchronize(c->own_stream);
            if (c->map_own) cudaFree(c->map_own);
            if (c->lens) cudaFree(c->lens);
            if (c->mass_buf) cudaFree(c->mass_buf);
            for (void *q : c->scratch)
                if (q) cudaFree(q);
            if (c->h_stage) cudaFreeHost(c->h_stage);
            if (c->ev_stage) cudaEventDestroy(c->ev_stage);
            if (c->counters) cudaFree(c->counters);
            if (c->h_counters) cudaFreeHost(c->h_counters);
            if (c->h_uni_max) cudaFreeHost(c->h_uni_max);
            if (c->uni_list) cudaFree(c->uni_list);
            if (c->uni_fill) cudaFree(c->uni_fill);
            if (c->ev0) cudaEventDestroy(c->ev0);
            if (c->ev1) cudaEventDestroy(c->ev1);
            if (c->own_stream) cudaStreamDestroy(c->own_stream);
        }
    }
    delete c;
}

int ml_get_info(const ml_ctx *c, ml_info *o)
{
    if (!c || !o) return ML_ERR_INVALID_ARG;
    std::memset(o, 0, sizeof(*o));
    o->kappa_star = c->kappa_star; o->kappa_c = c->kappa_c;
    o->a1 = c->a1; o->a2 = c->a2;
    o->ray_spacing = c->delta; o->r_star = c->r_star; o->pixel_side = c->pixel; o->mu_theory = c->mu_th;
    o->n1 = c->n1; o->n2 = c->n2; o->n_star_expected = c->n_star_expected; o->n_lenses = c->n_lenses;
    o->n_pix = c->n_pix;
    const Mode m = mode_of(c);
    o->tile_w = m.tw; o->tile_h = m.th;
    o->precision = c->precision; o->device = c->device;
    o->sm_count = c->sm_count; o->sm_clock_khz = c->sm_clock_khz;
    o->ray_mode = c->ray_mode; o->ray_seed = c->ray_seed;
    return ML_OK;
}

int ml_set_lens_masses(ml_ctx *c, const double *xy, const double *mass, int64_t n)
{
    if (!c || n < 0 || n > 0x7ffffe00LL || (n > 0 && !xy)) return ML_ERR_INVALID_ARG; // base + 512 must fit an int in the kernels
    for (int64_t k = 0; k < 2 * n; ++k)
        if (!std::isfinite(xy[k])) return ML_ERR_INVALID_ARG;
    if (mass)
        for (int64_t k = 0; k < n; ++k)
            if (!std::isfinite(mass[k]) || !(mass[k] > 0.0)) return ML_ERR_INVALID_ARG;
    DeviceGuard g(c->device);
    if (!g.ok) return ML_ERR_CUDA;
    // The caller's arrays are copied into the pinned staging buffer before returning (the caller keeps xy / mass, pinned or
    // not), and from there to the device on the context's stream: the next shoot is ordered after the copy, nothing waits
    // here.  Every buffer only grows, so a map-per-lens-field loop allocates nothing after its first pass.  The stream is
    // idle whenever this runs (every shoot / capture ends with a synchronisation), so the lens array is not in use.
    const size_t cnt = (size_t)std::max<int64_t>(n, 1);
    const size_t need_stage = cnt * (sizeof(double2) + sizeof(double));
    if (c->ev_stage && cudaEventSynchronize(c->ev_stage) != cudaSuccess) { cudaGetLastError(); return ML_ERR_CUDA; } // previous copy out of h_stage
    if (need_stage > c->stage_bytes) {
        unsigned char *h = nullptr;
        if (cudaMallocHost(&h, need_stage) != cudaSuccess) { cudaGetLastError(); return ML_ERR_OOM; }
        if (c->h_stage) cudaFreeHost(c->h_stage);
        c->h_stage = h;
        c->stage_bytes = need_stage;
    }
    if (!c->ev_stage && cudaEventCreateWithFlags(&c->ev_stage, cudaEventDisableTiming) != cudaSuccess) { cudaGetLastError(); return ML_ERR_CUDA; }
    // grow the device buffers: both allocations first, so that on failure the previous lenses are still in place
    double2 *d = nullptr;
    double *dm = nullptr;
    if ((cnt > c->lens_cap && cudaMalloc(&d, cnt * sizeof(double2)) != cudaSuccess) ||
        (mass && cnt > c->mass_cap && cudaMalloc(&dm, cnt * sizeof(double)) != cudaSuccess)) {
        cudaGetLastError();
        if (d) cudaFree(d);
        return ML_ERR_OOM;
    }
    if (d) {
        if (c->lens) cudaFree(c->lens); // (synchronises the device: only when a larger field arrives)
        c->lens = d;
        c->lens_cap = cnt;
    }
    if (dm) {
        if (c->mass_buf) cudaFree(c->mass_buf);
        c->mass_buf = dm;
        c->mass_cap = cnt;
    }
    double2 *h_xy = reinterpret_cast<double2 *>(c->h_stage);
    double *h_m = reinterpret_cast<double *>(c->h_stage + cnt * sizeof(double2));
    if (n > 0) {
        std::memcpy(h_xy, xy, (size_t)n * sizeof(double2));
        if (mass) std::memcpy(h_m, mass, (size_t)n * sizeof(double));
        if (cudaMemcpyAsync(c->lens, h_xy, (size_t)n * sizeof(double2), cudaMemcpyHostToDevice, c->stream) != cudaSuccess ||
            (mass && cudaMemcpyAsync(c->mass_buf, h_m, (size_t)n * sizeof(double), cudaMemcpyHostToDevice, c->stream) != cudaSuccess) ||
            cudaEventRecord(c->ev_stage, c->stream) != cudaSuccess) {
            cudaGetLastError();
            c->n_lenses = -1; // the device array may hold a mixture now: ml_shoot refuses until lenses are set again
            return ML_ERR_CUDA;
        }
    }
    c->mass = mass ? c->mass_buf : nullptr;
    c->n_lenses = n;
    return ML_OK;
}

int ml_set_lenses(ml_ctx *c, const double *xy, int64_t n) { return ml_set_lens_masses(c, xy, nullptr, n); }

int ml_set_precision(ml_ctx *c, int mode)
{
    if (!c || (mode != ML_PREC_FP32_TILED && mode != ML_PREC_FP32_COMPENSATED && mode != ML_PREC_FP64))
        return ML_ERR_INVALID_ARG;
    c->precision = mode;
    return ML_OK;
}

int ml_set_ray_mode(ml_ctx *c, int mode, uint64_t seed)
{
    if (!c || (mode != ML_RAYS_REGULAR && mode != ML_RAYS_RANDOM && mode != ML_RAYS_UNIFORM)) return ML_ERR_INVALID_ARG;
    if (mode != ML_RAYS_UNIFORM && c->uni_list) { // leaving the uniform mode: give its bucket lists (8.5 B per ray) back
        DeviceGuard g(c->device);
        if (g.ok) {
            cudaStreamSynchronize(c->stream);
            cudaFree(c->uni_list);
            if (c->uni_fill) cudaFree(c->uni_fill);
            c->uni_list = nullptr; c->uni_fill = nullptr;
            c->uni_list_entries = 0; c->uni_fill_entries = 0;
        }
    }
    c->ray_mode = mode;
    c->ray_seed = mode == ML_RAYS_REGULAR ? 0 : seed;
    return ML_OK;
}

int ml_shoot(ml_ctx *c)
{
    if (!c) return ML_ERR_INVALID_ARG;
    return shoot_region_impl(c, 0, c->n1, 0, c->n2, 0);
}

int ml_shoot_region(ml_ctx *c, int64_t i0, int64_t i1, int64_t j0, int64_t j1, int accumulate)
{
    return shoot_region_impl(c, i0, i1, j0, j1, accumulate);
}

int ml_get_map(const ml_ctx *c, uint32_t *out, size_t out_len)
{
    if (!c || !out || out_len < (size_t)c->n_pix * c->n_pix) return ML_ERR_INVALID_ARG;
    DeviceGuard g(c->device);
    if (!g.ok) return ML_ERR_CUDA;
    if (cudaMemcpyAsync(out, c->map, (size_t)c->n_pix * c->n_pix * sizeof(uint32_t), cudaMemcpyDeviceToHost, c->stream) != cudaSuccess ||
        cudaStreamSynchronize(c->stream) != cudaSuccess)
        return ML_ERR_CUDA;
    return ML_OK;
}

int ml_get_map_device(const ml_ctx *c, void **dptr)
{
    if (!c || !dptr) return ML_ERR_INVALID_ARG;
    *dptr = c->map;
    return ML_OK;
}

int ml_use_device_map(ml_ctx *c, void *dptr)
{
    if (!c) return ML_ERR_INVALID_ARG;
    if (dptr) { // must be device (or managed) memory of this context's device, 4-byte aligned; the size is the caller's word
        cudaPointerAttributes a;
        if (cudaPointerGetAttributes(&a, dptr) != cudaSuccess) {
            cudaGetLastError();
            return ML_ERR_INVALID_ARG;
        }
        if ((a.type != cudaMemoryTypeDevice && a.type != cudaMemoryTypeManaged) || a.device != c->device ||
            (reinterpret_cast<uintptr_t>(dptr) & 3) != 0)
            return ML_ERR_INVALID_ARG;
    }
    c->map = dptr ? (unsigned int *)dptr : c->map_own;
    return ML_OK;
}

int ml_attach_stream(ml_ctx *c, void *cuda_stream)
{
    if (!c) return ML_ERR_INVALID_ARG;
    if (c->ev_stage && (cudaStream_t)cuda_stream != c->stream) {
        // lenses set on the previous stream may still be on their way to the device: the new stream waits for that copy
        DeviceGuard g(c->device);
        if (!g.ok || cudaStreamWaitEvent((cudaStream_t)cuda_stream, c->ev_stage, 0) != cudaSuccess) { cudaGetLastError(); return ML_ERR_CUDA; }
    }
    c->stream = (cudaStream_t)cuda_stream;
    return ML_OK;
}

int ml_get_stats(const ml_ctx *c, ml_stats *o)
{
    if (!c || !o) return ML_ERR_INVALID_ARG;
    *o = c->stats;
    return ML_OK;
}

int ml_capture_region(ml_ctx *c, int64_t i0, int64_t i1, int64_t j0, int64_t j1, double *y_out)
{
    if (!c) return ML_ERR_INVALID_ARG;
    if (c->n_lenses < 0) return ML_ERR_STATE;
    if (i0 < 0 || j0 < 0 || i1 > c->n1 || j1 > c->n2 || i0 > i1 || j0 > j1) return ML_ERR_INVALID_ARG;
    if (i1 == i0 || j1 == j0) return ML_OK;
    if (!y_out) return ML_ERR_INVALID_ARG;
    if ((double)(i1 - i0) * (double)(j1 - j0) > 268435456.0) return ML_ERR_OOM;
    DeviceGuard g(c->device);
    if (!g.ok) return ML_ERR_CUDA;
    if (c->ray_mode == ML_RAYS_UNIFORM) {
        ShootParams p = base_params(c);
        p.i0 = i0; p.i1 = i1; p.j0 = j0; p.j1 = j1;
        p.list_w = i1 - i0;
        return capture_uniform(c, p, (i1 - i0) * (j1 - j0), nullptr, y_out);
    }
    const Mode m = mode_of(c);
    std::vector<long long> tiles;
    try {
        for (long long tj = j0 / m.th; tj <= (j1 - 1) / m.th; ++tj)
            for (long long ti = i0 / m.tw; ti <= (i1 - 1) / m.tw; ++ti) {
                tiles.push_back(ti);
                tiles.push_back(tj);
            }
    } catch (const std::bad_alloc &) {
        return ML_ERR_OOM;
    }
    const int64_t w = i1 - i0;
    return capture_tiles(c, tiles, [&](long long first, long long nb, const double2 *buf) {
        for (long long q = 0; q < nb; ++q) {
            const long long ti = tiles[2 * (first + q)], tj = tiles[2 * (first + q) + 1];
            const double2 *tb = buf + (size_t)q * m.tw * m.th;
            for (int ly = 0; ly < m.th; ++ly) {
                const int64_t j = tj * m.th + ly;
                if (j < j0 || j >= j1) continue;
                for (int lx = 0; lx < m.tw; ++lx) {
                    const int64_t i = ti * m.tw + lx;
                    if (i < i0 || i >= i1) continue;
                    const double2 v = tb[(size_t)ly * m.tw + lx];
                    double *o = y_out + 2 * ((j - j0) * w + (i - i0));
                    o[0] = v.x;
                    o[1] = v.y;
                }
            }
        }
    });
}

int ml_probe(ml_ctx *c, int64_t n, const int64_t *ray_i, const int64_t *ray_j, double *y_out)
{
    if (!c || n < 0) return ML_ERR_INVALID_ARG;
    if (c->n_lenses < 0) return ML_ERR_STATE;
    if (n == 0) return ML_OK;
    if (!ray_i || !ray_j || !y_out) return ML_ERR_INVALID_ARG;
    for (int64_t k = 0; k < n; ++k)
        if (ray_i[k] < 0 || ray_i[k] >= c->n1 || ray_j[k] < 0 || ray_j[k] >= c->n2) return ML_ERR_INVALID_ARG;
    DeviceGuard g(c->device);
    if (!g.ok) return ML_ERR_CUDA;
    if (c->ray_mode == ML_RAYS_UNIFORM) {
        std::vector<long long> ids;
        try {
            ids.resize((size_t)n);
        } catch (const std::bad_alloc &) {
            return ML_ERR_OOM;
        }
        for (int64_t k = 0; k < n; ++k) ids[(size_t)k] = ray_j[k] * c->n1 + ray_i[k];
        return capture_uniform(c, base_params(c), n, &ids, y_out);
    }
    const Mode m = mode_of(c);
    // rays sorted by the tile that owns them; one capture tile per distinct tile
    std::vector<int64_t> order;
    std::vector<long long> tiles;
    std::vector<int64_t> first_ray_of_tile; // index into `order`
    try {
        order.resize((size_t)n);
        for (int64_t k = 0; k < n; ++k) order[(size_t)k] = k;
        auto key = [&](int64_t k) { return std::make_pair(ray_j[k] / m.th, ray_i[k] / m.tw); };
        std::sort(order.begin(), order.end(), [&](int64_t a, int64_t b) { return key(a) < key(b); });
        for (int64_t q = 0; q < n; ++q) {
            const int64_t k = order[(size_t)q];
            const long long ti = ray_i[k] / m.tw, tj = ray_j[k] / m.th;
            if (tiles.empty() || tiles[tiles.size() - 2] != ti || tiles[tiles.size() - 1] != tj) {
                tiles.push_back(ti);
                tiles.push_back(tj);
                first_ray_of_tile.push_back(q);
            }
        }
        first_ray_of_tile.push_back(n);
    } catch (const std::bad_alloc &) {
        return ML_ERR_OOM;
    }
    return capture_tiles(c, tiles, [&](long long first, long long nb, const double2 *buf) {
        for (long long q = 0; q < nb; ++q) {
            const long long ti = tiles[2 * (first + q)], tj = tiles[2 * (first + q) + 1];
            const double2 *tb = buf + (size_t)q * m.tw * m.th;
            for (int64_t s = first_ray_of_tile[(size_t)(first + q)]; s < first_ray_of_tile[(size_t)(first + q) + 1]; ++s) {
                const int64_t k = order[(size_t)s];
                const double2 v = tb[(size_t)(ray_j[k] - tj * m.th) * m.tw + (size_t)(ray_i[k] - ti * m.tw)];
                y_out[2 * k] = v.x;
                y_out[2 * k + 1] = v.y;
            }
        }
    });
}

const char *ml_strerror(int code)
{
    switch (code) {
    case ML_OK: return "ok";
    case ML_ERR_INVALID_ARG: return "invalid argument";
    case ML_ERR_CUDA: return "CUDA runtime error or no CUDA device";
    case ML_ERR_OOM: return "out of memory";
    case ML_ERR_STATE: return "call sequence error (lenses not set)";
    case ML_ERR_LIMIT: return "the input needs more than the built-in scratch of a no-allocation entry point holds";
    default: return "unknown error code";
    }
}

const char *ml_version(void) { return "microlens-b200 0.1 (sm_100a)"; }

} // extern "C"
