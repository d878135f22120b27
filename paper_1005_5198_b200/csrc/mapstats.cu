// mapstats.cu -- map comparison on the device (include/microlens.h, "Map comparison").
//
// The paper's two accuracy measures between magnification maps (section 3.1):
// RMS difference in magnitudes and a two-sample Kolmogorov-Smirnov test on the distributions of
// Delta m = -2.5 log10(mu) (eq. 10), mu = N/N_rays (eq. 3).
//
// Counts are integers, so the K-S distance needs no sort: one fused pass over both maps gathers
// the RMS sums, the map statistics and the two count histograms (per-CTA shared-memory bins, flushed once);
// prefix sums of the histograms are the two empirical distributions, and
//   D = max over sample points x of |F_a(x) - F_b(x)|
// is evaluated at the sample points of both maps (x = c/n_rays_a and x = c/n_rays_b, compared in
// mu, which orders the samples exactly as Delta m does, reversed).  All sums that feed a
// floating-point result are reduced in a fixed order: results are bit-reproducible.
//
// Host side: nothing is allocated, created or synchronised per call beyond the one read-back of the result; the
// scratch (histograms, scans, events, a pinned result) lives in a per-device cache that grows when needed.
#include "../../include/microlens.h"

#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

#include <mutex>

namespace mlstats {

constexpr int kThreads = 256;
constexpr unsigned int kCap0 = 1u << 18;  // bins of the count histograms a scratch starts with (it grows on overflow)
constexpr unsigned int kCapMax = 1u << 27;
constexpr int kScanItems = 16;            // elements per thread in the scan kernels
constexpr int kScanTile = kThreads * kScanItems;

struct Partial {
    double ssq;                       // sum of (dm_a - dm_b)^2 over valid pixels
    unsigned long long n_valid, n_empty_a, n_empty_b, sum_a, sum_b;
    unsigned int max_a, max_b;
};

// Device-resident state of one call, filled by reduce_partials_kernel and read by the kernels after it.
struct Totals {
    Partial t;
    unsigned int cap_eff;  // max count + 1, clipped to the histogram size: the bins that matter
    unsigned int overflow; // a count did not fit the histogram: the host repeats the call with more bins
};

constexpr int kPassThreads = 1024;        // one CTA per SM
constexpr unsigned int kShBins = 16384;   // per map: counts below this are histogrammed in shared memory
constexpr unsigned int kLut = 8192;       // log10(c) for c < kLut is tabulated (global, copied to shared memory per CTA)

__global__ void lut_kernel(double *lut)
{
    const unsigned int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k < kLut) lut[k] = log10((double)k); // [0] = -inf, never read
}

__device__ __forceinline__ void hist_add(unsigned int *sh, unsigned int *hist, unsigned int cap, unsigned int c)
{
    if (c < kShBins) atomicAdd(&sh[c], 1u);
    else if (c < cap) atomicAdd(&hist[c], 1u); // bright pixels: RED into the global histogram (L2)
}

// One pass over the maps: RMS sums, statistics, count histograms (privatised per CTA in shared memory for
// counts < kShBins, flushed once at the end).  TWO = false: one map (ml_delta_m_histogram).
// log10 of a count < kLut comes from a table (`lut`, built once per device by lut_kernel) that every CTA copies into
// its shared memory: a pixel costs two table reads instead of two fp64 logarithms.
template <bool TWO>
__global__ void __launch_bounds__(kPassThreads, 1) pass_kernel(const unsigned int *__restrict__ a, const unsigned int *__restrict__ b,
                                                               long long n, double n_rays_a, double n_rays_b, unsigned int *hist_a,
                                                               unsigned int *hist_b, unsigned int cap, Partial *partials,
                                                               const double *__restrict__ lut)
{
    extern __shared__ __align__(8) unsigned char sh_raw[]; // [kLut] doubles, then [kShBins] bins for a and for b
    double *sh_log = reinterpret_cast<double *>(sh_raw);
    unsigned int *sh_hist = reinterpret_cast<unsigned int *>(sh_raw + kLut * sizeof(double));
    unsigned int *sh_a = sh_hist, *sh_b = sh_hist + kShBins;
    for (unsigned int k = threadIdx.x; k < (TWO ? 2 : 1) * kShBins; k += kPassThreads) sh_hist[k] = 0u;
    if (TWO)
        for (unsigned int k = threadIdx.x; k < kLut; k += kPassThreads) sh_log[k] = lut[k]; // [0] = -inf, never read
    const double log_rays = (n_rays_a == n_rays_b) ? 0.0 : log10(n_rays_a / n_rays_b);
    __syncthreads();

    Partial p;
    p.ssq = 0.0;
    p.n_valid = p.n_empty_a = p.n_empty_b = p.sum_a = p.sum_b = 0ull;
    p.max_a = p.max_b = 0u;
    const bool vec = ((reinterpret_cast<uintptr_t>(a) & 15) == 0) && (!TWO || (reinterpret_cast<uintptr_t>(b) & 15) == 0);
    const long long stride = (long long)gridDim.x * kPassThreads * 4;
    unsigned int n_valid = 0, n_empty_a = 0, n_empty_b = 0; // per thread: < 2^31 / (gridDim.x * 1024) pixels each

    auto load4 = [&](long long i, unsigned int (&ca)[4], unsigned int (&cb)[4]) {
#pragma unroll
        for (int q = 0; q < 4; ++q) { ca[q] = 0u; cb[q] = 0u; }
        if (i >= n) return;
        if (vec && i + 3 < n) {
            const uint4 va = __ldcs(reinterpret_cast<const uint4 *>(a + i)); // streamed: every pixel is read once
            ca[0] = va.x; ca[1] = va.y; ca[2] = va.z; ca[3] = va.w;
            if (TWO) {
                const uint4 vb = __ldcs(reinterpret_cast<const uint4 *>(b + i));
                cb[0] = vb.x; cb[1] = vb.y; cb[2] = vb.z; cb[3] = vb.w;
            }
        } else {
#pragma unroll
            for (int q = 0; q < 4; ++q)
                if (i + q < n) {
                    ca[q] = a[i + q];
                    if (TWO) cb[q] = b[i + q];
                }
        }
    };
    auto process4 = [&](long long i, const unsigned int (&ca)[4], const unsigned int (&cb)[4]) {
        if (i >= n) return;
        const unsigned int big = ca[0] | ca[1] | ca[2] | ca[3] | cb[0] | cb[1] | cb[2] | cb[3];
        if (i + 3 < n && big < kLut) {
            // common case: four pixels, every count inside the log table and the shared-memory bins: no range checks
            unsigned int s_a = 0, s_b = 0;
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                atomicAdd(&sh_a[ca[q]], 1u);
                if (TWO) atomicAdd(&sh_b[cb[q]], 1u);
                {
                    s_a += ca[q];
                    p.max_a = max(p.max_a, ca[q]);
                    n_empty_a += (ca[q] == 0);
                    if (TWO) {
                        s_b += cb[q];
                        p.max_b = max(p.max_b, cb[q]);
                        n_empty_b += (cb[q] == 0);
                        const bool valid = (ca[q] != 0) & (cb[q] != 0);
                        // dm_a - dm_b = -2.5 (log10 N_a - log10 N_b - log10(n_rays_a / n_rays_b))   (eq. 10)
                        const double d = -2.5 * ((sh_log[ca[q]] - sh_log[cb[q]]) - log_rays);
                        p.ssq += valid ? d * d : 0.0;
                        n_valid += valid;
                    }
                }
            }
            p.sum_a += s_a;
            p.sum_b += s_b;
            return;
        }
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            if (i + q >= n) break;
            hist_add(sh_a, hist_a, cap, ca[q]);
            if (TWO) hist_add(sh_b, hist_b, cap, cb[q]);
            {
                p.sum_a += ca[q];
                p.max_a = max(p.max_a, ca[q]);
                n_empty_a += (ca[q] == 0);
                if (TWO) {
                    p.sum_b += cb[q];
                    p.max_b = max(p.max_b, cb[q]);
                    n_empty_b += (cb[q] == 0);
                    if (ca[q] > 0 && cb[q] > 0) {
                        const double la = ca[q] < kLut ? sh_log[ca[q]] : log10((double)ca[q]);
                        const double lb = cb[q] < kLut ? sh_log[cb[q]] : log10((double)cb[q]);
                        const double d = -2.5 * ((la - lb) - log_rays);
                        p.ssq += d * d;
                        n_valid += 1;
                    }
                }
            }
        }
    };
    // two quads in flight per thread: the loads of the second are issued before the first is processed
    for (long long i = ((long long)blockIdx.x * kPassThreads + threadIdx.x) * 4; i < n; i += 2 * stride) {
        unsigned int ca0[4], cb0[4], ca1[4], cb1[4];
        load4(i, ca0, cb0);
        load4(i + stride, ca1, cb1);
        process4(i, ca0, cb0);
        process4(i + stride, ca1, cb1);
    }
    p.n_valid = n_valid; p.n_empty_a = n_empty_a; p.n_empty_b = n_empty_b;
    __syncthreads();
    for (unsigned int k = threadIdx.x; k < kShBins; k += kPassThreads) {
        const unsigned int va = sh_a[k];
        if (va) atomicAdd(&hist_a[k], va);
        if (TWO) {
            const unsigned int vb = sh_b[k];
            if (vb) atomicAdd(&hist_b[k], vb);
        }
    }
    {
        // block reduction in a fixed order: lanes by shuffle tree, then warps in index order
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            p.ssq += __shfl_down_sync(0xffffffffu, p.ssq, o);
            p.n_valid += __shfl_down_sync(0xffffffffu, p.n_valid, o);
            p.n_empty_a += __shfl_down_sync(0xffffffffu, p.n_empty_a, o);
            p.n_empty_b += __shfl_down_sync(0xffffffffu, p.n_empty_b, o);
            p.sum_a += __shfl_down_sync(0xffffffffu, p.sum_a, o);
            p.sum_b += __shfl_down_sync(0xffffffffu, p.sum_b, o);
            p.max_a = max(p.max_a, __shfl_down_sync(0xffffffffu, p.max_a, o));
            p.max_b = max(p.max_b, __shfl_down_sync(0xffffffffu, p.max_b, o));
        }
        __shared__ Partial wp[kPassThreads / 32];
        if ((threadIdx.x & 31) == 0) wp[threadIdx.x >> 5] = p;
        __syncthreads();
        if (threadIdx.x == 0) {
            Partial t = wp[0];
            for (int w = 1; w < kPassThreads / 32; ++w) {
                t.ssq += wp[w].ssq;
                t.n_valid += wp[w].n_valid; t.n_empty_a += wp[w].n_empty_a; t.n_empty_b += wp[w].n_empty_b;
                t.sum_a += wp[w].sum_a; t.sum_b += wp[w].sum_b;
                t.max_a = max(t.max_a, wp[w].max_a); t.max_b = max(t.max_b, wp[w].max_b);
            }
            partials[blockIdx.x] = t;
        }
    }
}

__device__ __forceinline__ void add_partial(Partial &t, const Partial &q)
{
    t.ssq += q.ssq;
    t.n_valid += q.n_valid; t.n_empty_a += q.n_empty_a; t.n_empty_b += q.n_empty_b;
    t.sum_a += q.sum_a; t.sum_b += q.sum_b;
    t.max_a = max(t.max_a, q.max_a); t.max_b = max(t.max_b, q.max_b);
}

// Sum the per-block partials in a fixed order: one warp, lane l takes blocks l, l+32, ..., then a shuffle tree.
// Also fixes how many histogram bins the rest of the call has to look at.
__global__ void reduce_partials_kernel(const Partial *partials, int n_blocks, unsigned int cap, Totals *out)
{
    const int lane = threadIdx.x;
    Partial t;
    t.ssq = 0.0;
    t.n_valid = t.n_empty_a = t.n_empty_b = t.sum_a = t.sum_b = 0ull;
    t.max_a = t.max_b = 0u;
    for (int k = lane; k < n_blocks; k += 32) add_partial(t, partials[k]);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        Partial q;
        q.ssq = __shfl_down_sync(0xffffffffu, t.ssq, o);
        q.n_valid = __shfl_down_sync(0xffffffffu, t.n_valid, o);
        q.n_empty_a = __shfl_down_sync(0xffffffffu, t.n_empty_a, o);
        q.n_empty_b = __shfl_down_sync(0xffffffffu, t.n_empty_b, o);
        q.sum_a = __shfl_down_sync(0xffffffffu, t.sum_a, o);
        q.sum_b = __shfl_down_sync(0xffffffffu, t.sum_b, o);
        q.max_a = __shfl_down_sync(0xffffffffu, t.max_a, o);
        q.max_b = __shfl_down_sync(0xffffffffu, t.max_b, o);
        add_partial(t, q);
    }
    if (lane == 0) {
        const unsigned int mx = max(t.max_a, t.max_b);
        out->t = t;
        out->overflow = mx >= cap ? 1u : 0u;
        out->cap_eff = mx >= cap ? cap : mx + 1u;
    }
}

// ---- inclusive prefix sums of the count histograms (three small kernels, tiles of kScanTile bins; blockIdx.y = map;
//      the grids are sized for the whole histogram and blocks beyond cap_eff leave at once)
__global__ void __launch_bounds__(kThreads) scan_tile_sums_kernel(const unsigned int *hist, unsigned int cap, const Totals *tot,
                                                                  unsigned int *tile_sums, int n_tiles)
{
    const unsigned int cap_eff = tot->cap_eff;
    const unsigned int base = blockIdx.x * kScanTile;
    if (base >= cap_eff) return;
    hist += (size_t)blockIdx.y * cap;
    unsigned int s = 0;
    for (int q = 0; q < kScanItems; ++q) {
        const unsigned int k = base + q * kThreads + threadIdx.x;
        if (k < cap_eff) s += hist[k];
    }
    __shared__ unsigned int ws[kThreads / 32];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_down_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0) ws[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned int t = 0;
        for (int w = 0; w < kThreads / 32; ++w) t += ws[w];
        tile_sums[blockIdx.y * n_tiles + blockIdx.x] = t;
    }
}

__global__ void scan_tile_offsets_kernel(unsigned int *tile_sums, int n_tiles, const Totals *tot)
{
    if (threadIdx.x != 0) return;
    const int used = (int)((tot->cap_eff + kScanTile - 1) / kScanTile);
    unsigned int *ts = tile_sums + blockIdx.x * n_tiles; // blockIdx.x = map
    unsigned int run = 0;
    for (int k = 0; k < used; ++k) {
        const unsigned int v = ts[k];
        ts[k] = run; // exclusive
        run += v;
    }
}

__global__ void __launch_bounds__(kThreads) scan_apply_kernel(const unsigned int *hist, unsigned int cap, const Totals *tot,
                                                              const unsigned int *tile_offsets, int n_tiles, unsigned int *cum)
{
    const unsigned int cap_eff = tot->cap_eff;
    if (blockIdx.x * kScanTile >= cap_eff) return;
    hist += (size_t)blockIdx.y * cap;
    cum += (size_t)blockIdx.y * cap;
    // thread t owns the kScanItems consecutive bins starting at base + t*kScanItems
    const unsigned int base = blockIdx.x * kScanTile + threadIdx.x * kScanItems;
    unsigned int v[kScanItems];
    unsigned int s = 0;
#pragma unroll
    for (int q = 0; q < kScanItems; ++q) {
        v[q] = (base + q < cap_eff) ? hist[base + q] : 0u;
        s += v[q];
    }
    // exclusive scan of the per-thread sums over the block
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    unsigned int incl = s;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const unsigned int u = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += u;
    }
    __shared__ unsigned int ws[kThreads / 32];
    if (lane == 31) ws[warp] = incl;
    __syncthreads();
    unsigned int off = tile_offsets[blockIdx.y * n_tiles + blockIdx.x];
    for (int w = 0; w < warp; ++w) off += ws[w];
    unsigned int run = off + incl - s;
#pragma unroll
    for (int q = 0; q < kScanItems; ++q) {
        run += v[q];
        if (base + q < cap_eff) cum[base + q] = run;
    }
}

// floor(c * num / den) clipped to `last`; exact when num, den have <= 26 significant bits.
__device__ __forceinline__ unsigned int floor_ratio(unsigned int c, double num, double den, unsigned int last)
{
    const double t = (double)c * num;
    double q = floor(t / den);
    if ((q + 1.0) * den <= t) q += 1.0;
    else if (q * den > t) q -= 1.0;
    if (q >= (double)last) return last;
    return q < 0.0 ? 0u : (unsigned int)q;
}

// D = max_x |F_a(x) - F_b(x)| at the sample points of both maps (x in mu = count / n_rays).
__global__ void __launch_bounds__(kThreads) ks_kernel(const unsigned int *cum, unsigned int cap, const Totals *tot, double n,
                                                      double n_rays_a, double n_rays_b, unsigned long long *d_bits)
{
    const unsigned int cap_eff = tot->cap_eff;
    const unsigned int *cum_a = cum, *cum_b = cum + cap;
    double d = 0.0;
    const unsigned int last = cap_eff - 1;
    for (unsigned int c = blockIdx.x * kThreads + threadIdx.x; c < cap_eff; c += gridDim.x * kThreads) {
        // x = c / n_rays_a : F_a = cum_a[c], F_b = #{N_b <= c n_rays_b / n_rays_a}
        const double fa1 = (double)cum_a[c] / n, fb1 = (double)cum_b[floor_ratio(c, n_rays_b, n_rays_a, last)] / n;
        // x = c / n_rays_b
        const double fb2 = (double)cum_b[c] / n, fa2 = (double)cum_a[floor_ratio(c, n_rays_a, n_rays_b, last)] / n;
        d = fmax(d, fmax(fabs(fa1 - fb1), fabs(fa2 - fb2)));
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) d = fmax(d, __shfl_down_sync(0xffffffffu, d, o));
    if ((threadIdx.x & 31) == 0 && d > 0.0) atomicMax(d_bits, (unsigned long long)__double_as_longlong(d)); // d >= 0: bit order = value order
}

// Delta m histogram from the count histogram: one evaluation of eq. 10 per distinct count.
__global__ void __launch_bounds__(kThreads) delta_m_hist_kernel(const unsigned int *hist, const Totals *tot, double n_rays, double lo, double hi,
                                                                int n_bins, unsigned long long *out)
{
    const unsigned int cap_eff = tot->cap_eff;
    const double w = (hi - lo) / (double)n_bins;
    for (unsigned int c = 1 + blockIdx.x * kThreads + threadIdx.x; c < cap_eff; c += gridDim.x * kThreads) {
        const unsigned int h = hist[c];
        if (!h) continue;
        const double x = -2.5 * log10((double)c / n_rays);
        if (!(x >= lo)) continue;
        const double k = floor((x - lo) / w);
        if (k >= 0.0 && k < (double)n_bins) atomicAdd(&out[(int)k], (unsigned long long)h);
    }
}

// Q_KS(lambda) = 2 sum_{j>=1} (-1)^(j-1) exp(-2 j^2 lambda^2), lambda = (sqrt(Ne) + 0.12 + 0.11/sqrt(Ne)) D.
__global__ void finalize_kernel(const Totals *tot, const unsigned long long *d_bits, double n, double n_rays_a, double n_rays_b,
                                ml_map_compare_result *out)
{
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    const Partial t = tot->t;
    ml_map_compare_result r;
    r.n_pixels = (uint64_t)n;
    r.n_valid = t.n_valid; r.n_empty_a = t.n_empty_a; r.n_empty_b = t.n_empty_b;
    r.sum_a = t.sum_a; r.sum_b = t.sum_b; r.max_a = t.max_a; r.max_b = t.max_b;
    r.mean_mu_a = ((double)t.sum_a / n) / n_rays_a;
    r.mean_mu_b = ((double)t.sum_b / n) / n_rays_b;
    r.rms_delta_m = t.n_valid ? sqrt(t.ssq / (double)t.n_valid) : 0.0;
    const double d = __longlong_as_double((long long)*d_bits);
    r.ks_d = d;
    const double ne = n * n / (n + n);
    const double lam = (sqrt(ne) + 0.12 + 0.11 / sqrt(ne)) * d;
    // two series for the same function: the theta-function form converges fast where the alternating one does not
    double q;
    if (lam < 0.04) {
        q = 1.0;
    } else if (lam < 1.18) {
        const double y = exp(-1.2337005501361697 / (lam * lam)); // exp(-pi^2 / (8 lambda^2))
        const double y2 = y * y, y4 = y2 * y2, y8 = y4 * y4;
        // sum_{j=1..4} y^((2j-1)^2) = y + y^9 + y^25 + y^49
        q = 1.0 - (2.5066282746310002 / lam) * (y + y8 * y + y8 * y8 * y8 * y + y8 * y8 * y8 * y8 * y8 * y8 * y);
    } else {
        const double x = exp(-2.0 * lam * lam);
        const double x2 = x * x, x4 = x2 * x2, x8 = x4 * x4;
        // sum_{j=1..4} (-1)^(j-1) x^(j^2) = x - x^4 + x^9 - x^16
        q = 2.0 * (x - x4 + x8 * x - x8 * x8);
    }
    q = fmin(1.0, fmax(0.0, q));
    r.ks_prob = q;
    r.kernel_ms = 0.0;
    r.pass_kernel_ms = 0.0;
    *out = r;
}

} // namespace mlstats

// ---------------------------------------------------------------------------------------- host side
namespace {

using namespace mlstats;

constexpr int kMaxDevices = 64;
constexpr size_t kPassSmem = kLut * sizeof(double) + 2 * kShBins * sizeof(unsigned int);

// Everything a call needs on one device, created on first use and kept: no allocation, event creation or
// synchronisation per call besides the read-back of the result.  Calls are serialised by `lock` (a call ends with a
// stream synchronisation, so the scratch is idle whenever the lock is free).
struct Scratch {
    bool ready = false;
    int sm_count = 0;
    unsigned int cap = 0;          // bins per histogram
    unsigned char *zeroed = nullptr; // [2*cap hist | d_bits]: one memset per call
    unsigned int *hist = nullptr;  // = zeroed: [2][cap]
    unsigned long long *d_bits = nullptr;
    unsigned long long *dm_out = nullptr; // [2^20] bins of ml_delta_m_histogram (allocated by its first call)
    unsigned int *cum = nullptr;   // [2][cap]
    unsigned int *tile_sums = nullptr; // [2][n_tiles]
    Partial *partials = nullptr;   // [sm_count]
    Totals *totals = nullptr;
    double *lut = nullptr;         // [kLut] log10 table, built once
    ml_map_compare_result *d_res = nullptr;
    struct Pinned { ml_map_compare_result res; Totals tot; } *pinned = nullptr;
    unsigned int *map_a = nullptr, *map_b = nullptr; // device copies of host maps
    size_t map_cap = 0;
    cudaEvent_t ev0 = nullptr, ev1 = nullptr, evp0 = nullptr, evp1 = nullptr; // whole call; the fused pass alone
    void free_hist()
    {
        if (zeroed) cudaFree(zeroed);
        if (cum) cudaFree(cum);
        if (tile_sums) cudaFree(tile_sums);
        zeroed = nullptr; cum = nullptr; tile_sums = nullptr; hist = nullptr; d_bits = nullptr;
        cap = 0;
    }
    size_t zeroed_bytes(bool two) const { return two ? 2 * (size_t)cap * 4 + 8 : (size_t)cap * 4; }
    int n_tiles() const { return (int)((cap + kScanTile - 1) / kScanTile); }
    bool set_cap(unsigned int want)
    {
        if (want <= cap) return true;
        free_hist();
        cap = want;
        if (cudaMalloc(&zeroed, zeroed_bytes(true)) != cudaSuccess || cudaMalloc(&cum, 2 * (size_t)cap * 4) != cudaSuccess ||
            cudaMalloc(&tile_sums, 2 * (size_t)n_tiles() * 4) != cudaSuccess) {
            cudaGetLastError();
            free_hist();
            return false;
        }
        hist = reinterpret_cast<unsigned int *>(zeroed);
        d_bits = reinterpret_cast<unsigned long long *>(zeroed + 2 * (size_t)cap * 4);
        return true;
    }
    bool set_maps(size_t n, bool two)
    {
        if (n <= map_cap && (!two || map_b)) return true;
        if (map_a) cudaFree(map_a);
        if (map_b) cudaFree(map_b);
        map_a = map_b = nullptr;
        map_cap = 0;
        if (cudaMalloc(&map_a, n * 4) != cudaSuccess || cudaMalloc(&map_b, n * 4) != cudaSuccess) {
            cudaGetLastError();
            if (map_a) cudaFree(map_a);
            map_a = map_b = nullptr;
            return false;
        }
        map_cap = n;
        return true;
    }
    int init(int device)
    {
        if (ready) return ML_OK;
        if (cudaDeviceGetAttribute(&sm_count, cudaDevAttrMultiProcessorCount, device) != cudaSuccess) return ML_ERR_CUDA;
        if (cudaFuncSetAttribute(pass_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kPassSmem) != cudaSuccess ||
            cudaFuncSetAttribute(pass_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kPassSmem) != cudaSuccess)
            return ML_ERR_CUDA;
        if (cudaMalloc(&partials, (size_t)sm_count * sizeof(Partial)) != cudaSuccess || cudaMalloc(&totals, sizeof(Totals)) != cudaSuccess ||
            cudaMalloc(&lut, kLut * sizeof(double)) != cudaSuccess ||
            cudaMalloc(&d_res, sizeof(ml_map_compare_result)) != cudaSuccess || cudaMallocHost(&pinned, sizeof(Pinned)) != cudaSuccess) {
            cudaGetLastError();
            return ML_ERR_OOM;
        }
        if (cudaEventCreate(&ev0) != cudaSuccess || cudaEventCreate(&ev1) != cudaSuccess || cudaEventCreate(&evp0) != cudaSuccess ||
            cudaEventCreate(&evp1) != cudaSuccess)
            return ML_ERR_CUDA;
        if (!set_cap(kCap0)) return ML_ERR_OOM;
        lut_kernel<<<kLut / 256, 256>>>(lut); // legacy stream; the synchronisation below orders it before every later call
        if (cudaGetLastError() != cudaSuccess || cudaDeviceSynchronize() != cudaSuccess) return ML_ERR_CUDA;
        ready = true;
        return ML_OK;
    }
};

Scratch g_scratch[kMaxDevices];
std::mutex g_lock;

struct DeviceScope { // device selection for the duration of a call
    int prev = 0;
    bool ok = false;
    explicit DeviceScope(int dev)
    {
        int ndev = 0;
        if (cudaGetDeviceCount(&ndev) != cudaSuccess || dev < 0 || dev >= ndev || dev >= kMaxDevices) { cudaGetLastError(); return; }
        if (cudaGetDevice(&prev) != cudaSuccess) return;
        ok = (prev == dev) || (cudaSetDevice(dev) == cudaSuccess);
    }
    ~DeviceScope()
    {
        if (ok) cudaSetDevice(prev);
    }
};

int grid_for(long long n, int sm_count)
{
    const long long want = (n + (long long)kPassThreads * 4 - 1) / ((long long)kPassThreads * 4);
    return (int)(want < 1 ? 1 : (want < sm_count ? want : sm_count)); // one CTA of 1024 threads per SM
}

// Front half of both entry points: device copies of host maps, one memset, the fused pass, the reduced statistics.
// Leaves Totals on the device (nothing is read back here).
int run_pass(Scratch &sc, cudaStream_t s, const uint32_t *a, const uint32_t *b, int64_t n, double na, double nb, int where,
             const unsigned int **da, const unsigned int **db)
{
    const bool two = b != nullptr;
    *da = a; *db = b;
    if (where == ML_MEM_HOST) {
        if (!sc.set_maps((size_t)n, two)) return ML_ERR_OOM;
        if (cudaMemcpyAsync(sc.map_a, a, (size_t)n * 4, cudaMemcpyHostToDevice, s) != cudaSuccess ||
            (two && cudaMemcpyAsync(sc.map_b, b, (size_t)n * 4, cudaMemcpyHostToDevice, s) != cudaSuccess))
            return ML_ERR_CUDA;
        *da = sc.map_a; *db = two ? sc.map_b : nullptr;
    }
    const int grid = grid_for(n, sc.sm_count);
    if (cudaEventRecord(sc.ev0, s) != cudaSuccess || cudaMemsetAsync(sc.zeroed, 0, sc.zeroed_bytes(two), s) != cudaSuccess ||
        cudaEventRecord(sc.evp0, s) != cudaSuccess)
        return ML_ERR_CUDA;
    if (two) pass_kernel<true><<<grid, kPassThreads, kPassSmem, s>>>(*da, *db, n, na, nb, sc.hist, sc.hist + sc.cap, sc.cap, sc.partials, sc.lut);
    else pass_kernel<false><<<grid, kPassThreads, kPassSmem, s>>>(*da, nullptr, n, na, nb, sc.hist, nullptr, sc.cap, sc.partials, sc.lut);
    if (cudaGetLastError() != cudaSuccess || cudaEventRecord(sc.evp1, s) != cudaSuccess) return ML_ERR_CUDA;
    reduce_partials_kernel<<<1, 32, 0, s>>>(sc.partials, grid, sc.cap, sc.totals);
    return cudaGetLastError() == cudaSuccess ? ML_OK : ML_ERR_CUDA;
}

// After an overflow (a count >= the histogram size) the call is repeated once with enough bins.
bool grow_after_overflow(Scratch &sc, const Totals &t, int *rc)
{
    if (!t.overflow) return false;
    const unsigned int mx = t.t.max_a > t.t.max_b ? t.t.max_a : t.t.max_b;
    if (mx >= kCapMax) { *rc = ML_ERR_OOM; return false; }
    unsigned int want = sc.cap;
    while (want <= mx) want *= 2;
    if (!sc.set_cap(want)) { *rc = ML_ERR_OOM; return false; }
    return true;
}

bool bad_rays(double v) { return !(v > 0.0) || !isfinite(v); }

} // namespace

extern "C" {

int ml_map_compare(const uint32_t *a, double n_rays_a, const uint32_t *b, double n_rays_b, int64_t n, int where, int32_t device,
                   void *cuda_stream, ml_map_compare_result *out)
{
    if (!a || !b || !out || n < 1 || n > 0x7fffffffLL || bad_rays(n_rays_a) || bad_rays(n_rays_b) ||
        (where != ML_MEM_HOST && where != ML_MEM_DEVICE))
        return ML_ERR_INVALID_ARG;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    DeviceScope g(device);
    if (!g.ok) return ML_ERR_CUDA;
    std::lock_guard<std::mutex> hold(g_lock);
    Scratch &sc = g_scratch[device];
    int rc = sc.init(device);
    if (rc != ML_OK) return rc;
    for (int attempt = 0; attempt < 2; ++attempt) {
        const unsigned int *da, *db;
        rc = run_pass(sc, s, a, b, n, n_rays_a, n_rays_b, where, &da, &db);
        if (rc != ML_OK) return rc;
        const int n_tiles = sc.n_tiles();
        scan_tile_sums_kernel<<<dim3(n_tiles, 2), kThreads, 0, s>>>(sc.hist, sc.cap, sc.totals, sc.tile_sums, n_tiles);
        scan_tile_offsets_kernel<<<2, 32, 0, s>>>(sc.tile_sums, n_tiles, sc.totals);
        scan_apply_kernel<<<dim3(n_tiles, 2), kThreads, 0, s>>>(sc.hist, sc.cap, sc.totals, sc.tile_sums, n_tiles, sc.cum);
        const int want = (int)((sc.cap + kThreads - 1) / kThreads);
        ks_kernel<<<want < sc.sm_count * 8 ? want : sc.sm_count * 8, kThreads, 0, s>>>(sc.cum, sc.cap, sc.totals, (double)n, n_rays_a, n_rays_b, sc.d_bits);
        finalize_kernel<<<1, 32, 0, s>>>(sc.totals, sc.d_bits, (double)n, n_rays_a, n_rays_b, sc.d_res);
        if (cudaGetLastError() != cudaSuccess || cudaEventRecord(sc.ev1, s) != cudaSuccess) return ML_ERR_CUDA;
        if (cudaMemcpyAsync(&sc.pinned->res, sc.d_res, sizeof(ml_map_compare_result), cudaMemcpyDeviceToHost, s) != cudaSuccess ||
            cudaMemcpyAsync(&sc.pinned->tot, sc.totals, sizeof(Totals), cudaMemcpyDeviceToHost, s) != cudaSuccess ||
            cudaStreamSynchronize(s) != cudaSuccess)
            return ML_ERR_CUDA;
        if (grow_after_overflow(sc, sc.pinned->tot, &rc)) continue;
        if (rc != ML_OK) return rc;
        break;
    }
    float ms = 0.f, pass_ms = 0.f;
    if (cudaEventElapsedTime(&ms, sc.ev0, sc.ev1) != cudaSuccess || cudaEventElapsedTime(&pass_ms, sc.evp0, sc.evp1) != cudaSuccess)
        return ML_ERR_CUDA;
    *out = sc.pinned->res;
    out->kernel_ms = ms;
    out->pass_kernel_ms = pass_ms;
    return ML_OK;
}

int ml_delta_m_histogram(const uint32_t *counts, double n_rays, int64_t n, double lo, double hi, int32_t n_bins, int where,
                         int32_t device, void *cuda_stream, uint64_t *hist_out)
{
    if (!counts || !hist_out || n < 1 || n > 0x7fffffffLL || bad_rays(n_rays) || !(lo < hi) || !isfinite(lo) || !isfinite(hi) ||
        n_bins < 1 || n_bins > (1 << 20) || (where != ML_MEM_HOST && where != ML_MEM_DEVICE))
        return ML_ERR_INVALID_ARG;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    DeviceScope g(device);
    if (!g.ok) return ML_ERR_CUDA;
    std::lock_guard<std::mutex> hold(g_lock);
    Scratch &sc = g_scratch[device];
    int rc = sc.init(device);
    if (rc != ML_OK) return rc;
    if (!sc.dm_out && cudaMalloc(&sc.dm_out, (size_t)(1 << 20) * 8) != cudaSuccess) {
        cudaGetLastError();
        sc.dm_out = nullptr;
        return ML_ERR_OOM;
    }
    for (int attempt = 0; attempt < 2; ++attempt) {
        const unsigned int *da, *db;
        rc = run_pass(sc, s, counts, nullptr, n, n_rays, n_rays, where, &da, &db);
        if (rc != ML_OK) return rc;
        if (cudaMemsetAsync(sc.dm_out, 0, (size_t)n_bins * 8, s) != cudaSuccess) return ML_ERR_CUDA;
        const int want = (int)((sc.cap + kThreads - 1) / kThreads);
        delta_m_hist_kernel<<<want < sc.sm_count * 8 ? want : sc.sm_count * 8, kThreads, 0, s>>>(sc.hist, sc.totals, n_rays, lo, hi, n_bins, sc.dm_out);
        if (cudaGetLastError() != cudaSuccess) return ML_ERR_CUDA;
        if (cudaMemcpyAsync(hist_out, sc.dm_out, (size_t)n_bins * 8, cudaMemcpyDeviceToHost, s) != cudaSuccess ||
            cudaMemcpyAsync(&sc.pinned->tot, sc.totals, sizeof(Totals), cudaMemcpyDeviceToHost, s) != cudaSuccess ||
            cudaStreamSynchronize(s) != cudaSuccess)
            return ML_ERR_CUDA;
        if (grow_after_overflow(sc, sc.pinned->tot, &rc)) continue;
        if (rc != ML_OK) return rc;
        break;
    }
    return ML_OK;
}

} // extern "C"

// ---------------------------------------------------------------------------------------- no-allocation variant
// ml_delta_m_histogram_static (include/microlens.h): the same pass / reduce / Delta-m kernels as ml_delta_m_histogram,
// but their scratch is this fixed array inside the library image instead of the cudaMalloc'ed per-device cache above.
// For callers whose process cannot (its own pool owns the memory) or must not (cudaMalloc / cudaFree stall the whole
// device) allocate.  Each device that loads this module holds ML_STATIC_SCRATCH_BYTES for it until the process exits.
namespace {

constexpr unsigned int kStaticBins = ML_STATIC_MAX_COUNT; // bins of the count histogram: counts must stay below this
constexpr int kStaticMaxBlocks = 256;                     // per-CTA partial sums (the pass runs one CTA per SM, at most this many)

struct StaticLayout {
    unsigned int hist[kStaticBins];       // must be zero when the pass starts: cleared on the stream by every call
    Partial partials[kStaticMaxBlocks];   // [0, grid) fully rewritten by the pass
    Totals totals;                        // fully rewritten by reduce_partials_kernel
};
static_assert(sizeof(StaticLayout) <= ML_STATIC_SCRATCH_BYTES, "the documented size of the built-in scratch is too small");

// NOTE for host code: `g_static_scratch` names the host-side shadow of the symbol, not device memory.  Passing it to a
// kernel would fault (or quietly use host memory on systems where the GPU can reach it).  Host code below only ever
// uses the address cudaGetSymbolAddress returns for the current device.
static __device__ __align__(256) unsigned char g_static_scratch[ML_STATIC_SCRATCH_BYTES];

struct StaticDevice {
    bool ready = false;
    int sm_count = 0;
    StaticLayout *scratch = nullptr; // device address of g_static_scratch on this device
};
StaticDevice g_static[kMaxDevices];

// Once per device, with that device current (the caller holds a DeviceScope and g_lock).  Allocates nothing.
int static_setup(StaticDevice &sd, int device)
{
    if (sd.ready) return ML_OK;
    void *ptr = nullptr;
    if (cudaGetSymbolAddress(&ptr, g_static_scratch) != cudaSuccess || !ptr) { cudaGetLastError(); return ML_ERR_CUDA; }
    if (cudaDeviceGetAttribute(&sd.sm_count, cudaDevAttrMultiProcessorCount, device) != cudaSuccess) { cudaGetLastError(); return ML_ERR_CUDA; }
    // per-device attribute; the allocating path sets the same value in Scratch::init, so the order of first use does not matter
    if (cudaFuncSetAttribute(pass_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kPassSmem) != cudaSuccess) {
        cudaGetLastError();
        return ML_ERR_CUDA;
    }
    sd.scratch = static_cast<StaticLayout *>(ptr);
    sd.ready = true;
    return ML_OK;
}

} // namespace

extern "C" int ml_delta_m_histogram_static(const uint32_t *counts, double n_rays, int64_t n, double lo, double hi, int32_t n_bins,
                                           int32_t device, void *cuda_stream, uint64_t *hist_out)
{
    if (!counts || !hist_out || (reinterpret_cast<uintptr_t>(counts) & 3) || (reinterpret_cast<uintptr_t>(hist_out) & 7) || n < 1 ||
        n > 0x7fffffffLL || bad_rays(n_rays) || !(lo < hi) || !isfinite(lo) || !isfinite(hi) || n_bins < 1 || n_bins > (1 << 20))
        return ML_ERR_INVALID_ARG;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    DeviceScope g(device);
    if (!g.ok) return ML_ERR_CUDA;
    std::lock_guard<std::mutex> hold(g_lock); // one call at a time per process: every call works in the same array
    StaticDevice &sd = g_static[device];
    int rc = static_setup(sd, device);
    if (rc != ML_OK) return rc;
    StaticLayout *sc = sd.scratch;
    int grid = grid_for(n, sd.sm_count);
    if (grid > kStaticMaxBlocks) grid = kStaticMaxBlocks; // a device with more SMs than partial-sum slots: grid-stride loop covers the rest
    // the array still holds the previous call's histogram: clear it (stream-ordered), and the caller's output bins
    if (cudaMemsetAsync(sc->hist, 0, sizeof(sc->hist), s) != cudaSuccess ||
        cudaMemsetAsync(hist_out, 0, (size_t)n_bins * sizeof(uint64_t), s) != cudaSuccess) {
        cudaGetLastError();
        return ML_ERR_CUDA;
    }
    pass_kernel<false><<<grid, kPassThreads, kPassSmem, s>>>(counts, nullptr, n, n_rays, n_rays, sc->hist, nullptr, kStaticBins, sc->partials,
                                                             nullptr);
    reduce_partials_kernel<<<1, 32, 0, s>>>(sc->partials, grid, kStaticBins, &sc->totals);
    const int want = (int)(kStaticBins / kThreads);
    delta_m_hist_kernel<<<want < sd.sm_count * 8 ? want : sd.sm_count * 8, kThreads, 0, s>>>(
        sc->hist, &sc->totals, n_rays, lo, hi, n_bins, reinterpret_cast<unsigned long long *>(hist_out));
    if (cudaGetLastError() != cudaSuccess) return ML_ERR_CUDA;
    // 4 bytes back into a stack variable (pageable: the runtime stages the copy itself, nothing is allocated here)
    unsigned int overflow = 0;
    if (cudaMemcpyAsync(&overflow, &sc->totals.overflow, sizeof(overflow), cudaMemcpyDeviceToHost, s) != cudaSuccess ||
        cudaStreamSynchronize(s) != cudaSuccess) {
        cudaGetLastError();
        return ML_ERR_CUDA;
    }
    return overflow ? ML_ERR_LIMIT : ML_OK; // a count >= ML_STATIC_MAX_COUNT was not histogrammed
}
