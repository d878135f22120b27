// shoot_kernel.cuh -- the fused ray-generation + deflection + binning kernel (sm_100a).
//
// One CTA shoots one tile of TW x TH rays of the regular image-plane grid through all
// N* lenses (eq.4, unit masses PAPER.md:165) and bins them into the
// source-plane count map (eq.3).  Steps a1-a6 of SURVEY.md section 8(a):
//
//   a1 lens staging   lens positions (fp64, L2-resident) are re-centred on the tile centre
//                     with an fp64 subtract, rounded to the working type and staged into
//                     shared memory in chunks of CHUNK lenses, double-buffered: global loads
//                     for chunk n+1 are issued before the arithmetic on chunk n.
//   a2 ray generation ray (i,j) -> x from the tile / thread index; nothing is stored.
//   a3 deflection     each thread owns an RX x RY block of rays; per lens the RX column
//                     differences / squares and RY row differences / squares are shared, so
//                     one interaction is FADD (r^2) + MUFU.RCP + 2 FFMA, plus
//                     2(RX+RY)/(RX*RY) amortised FADD/FMUL.
//   a4 macro terms    y = (1 -/+ gamma - kappa_c) x - S in fp64.
//   a5 binning        pixel index in fp64; per register slot the 32 lanes of a warp hold 32
//                     rays of one row, RX apart: runs of equal pixel along the lanes are
//                     found with shfl_up + ballot and the run head issues ONE
//                     atomicAdd(run length) (red.global.add.u32 resolved in L2).
//   a6 scheduling     one tile per CTA, tiles aligned to the GLOBAL grid and rasterised
//                     row-major so that concurrently resident CTAs touch a narrow band of
//                     the map; rays outside the requested region are masked.
//
// Summation order and precision:
//   lenses in index order; FP32 partial sums over groups of KF consecutive lenses (groups
//   aligned to multiples of KF in lens index) are added, in order, to one fp64
//   accumulator per ray and component.  With Real = double the partials are fp64 too
//   and the reciprocal is an IEEE division.
//   Every FP32 operation is written with an explicit-rounding intrinsic so that the
//   compiler can neither contract nor reassociate: the arithmetic of a ray does not
//   depend on the template instantiation (shoot vs capture) it runs in.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <type_traits>

namespace mlb200 {

struct ShootParams {
    const double2 *lens;      // [n_lens] fp64 (x, y), device
    const double *mass;       // [n_lens] fp64 lens masses m_i of eq.4 (MASS instantiations only)
    int n_lens;
    int n_pix;
    long long i0, i1, j0, j1; // region of ray indices to count (others are masked)
    long long tile_i0, tile_j0; // global tile index of block (0, 0) of this launch: tile = (tile_i0 + blockIdx.x,
                              // tile_j0 + blockIdx.y); regions larger than one grid are split into several launches
    double delta;             // ray spacing
    double half1, half2;      // (n1-1)/2, (n2-1)/2
    double c1, c2;            // 1 - gamma - kappa_c, 1 + gamma - kappa_c
    double halfL, inv_pixel;  // L/2, n_pix/L
    double k1, k2, hoff;      // c1 * inv_pixel, c2 * inv_pixel, halfL * inv_pixel: pixel coordinate u = k x + hoff - S inv_pixel
    unsigned int *map;        // [n_pix*n_pix] counts, device
    unsigned long long *counters; // [0] shot [1] in map [2] dropped
    double2 *capture;         // CAPTURE: [n_tiles_in_list * TW*TH] source-plane positions
    const long long *tile_list; // CAPTURE: pairs (tile_i, tile_j), global tile indices
    int split_len;            // CAPTURE, > 0: CTA (t, blockIdx.y) sums lenses [blockIdx.y*split_len, +split_len) only
    double2 *partial;         // CAPTURE with split_len > 0: [gridDim.y][gridDim.x][TW*TH] partial sums (Sx, Sy)
    long long n1;             // rays per row of the whole grid (ray id = j*n1 + i, RANDOM instantiations)
    unsigned long long ray_seed; // key of the ray generator (RANDOM instantiations)
    // ---- ML_RAYS_UNIFORM (shoot_kernel_upipe): rays sorted into buckets of kUniBW x kUniBH grid cells
    const unsigned long long *ray_list; // [buckets of this launch][bucket_cap] ray handles (see uniform_ray_id)
    const unsigned int *bucket_fill;    // [buckets of this launch] rays scattered into each bucket (may exceed bucket_cap)
    unsigned int bucket_cap;
    long long bucket_nx, bucket_row0;   // buckets per row of the bucket grid; bucket row of block x = 0
    double n1d, n2d;                    // n1, n2 as doubles
    long long list_w;                   // handle -> ray: width of the region the handles index (0 with probe_ids)
    const long long *probe_ids;         // handle -> ray id by table (ml_probe); nullptr: handle = (j - j0) list_w + (i - i0)
};

constexpr int kThreads = 256;
constexpr int kWarps = kThreads / 32;
#ifndef ML_CHUNK
#define ML_CHUNK 512
#endif
constexpr int kChunk = ML_CHUNK; // lenses per shared-memory stage

template <typename Real> struct Vec2;
template <> struct Vec2<float> { using type = float2; };
template <> struct Vec2<double> { using type = double2; };

// A lens this far away contributes exactly zero: d^2 overflows to +inf, 1/inf = +0,
// d * 0 = 0 (d itself stays finite).  Used to pad the last chunk to a multiple of 8.
template <typename Real, bool NEWTON> __device__ __forceinline__ Real pad_coordinate();
template <> __device__ __forceinline__ float pad_coordinate<float, false>() { return 1e30f; }
// with the Newton step inf * 0 would give NaN: stay finite (term ~ 5e-19, below every rounding)
template <> __device__ __forceinline__ float pad_coordinate<float, true>() { return 1e18f; }
// fp64: r^2 = 2e200 stays finite (the Newton-refined reciprocal below would turn inf * 0 into NaN); term ~ 5e-101
template <> __device__ __forceinline__ double pad_coordinate<double, false>() { return 1e100; }
template <> __device__ __forceinline__ double pad_coordinate<double, true>() { return 1e100; }

__device__ __forceinline__ float rcp_approx(float a)
{
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(a)); // one MUFU.RCP
    return r;
}

template <bool NEWTON> __device__ __forceinline__ float recip(float a)
{
    float r = rcp_approx(a);
    if (NEWTON) { // one Newton-Raphson step removes the approximation's error to < 1 ulp
        float e = __fmaf_rn(-a, r, 1.0f);
        r = __fmaf_rn(r, e, r);
    }
    return r;
}
// fp64 reciprocal: MUFU.RCP64H seed (rcp.approx.ftz.f64, ~20 bits) + two Newton-Raphson steps (4 DFMA): within an
// ulp of 1/a for the normal, finite r^2 that occur, without the IEEE division's slow-path fix-up (about half its
// instructions).  a = 0 (ray on a lens) gives inf -> NaN -> the ray is dropped (reading R12).
template <bool NEWTON> __device__ __forceinline__ double recip(double a)
{
    double x;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(x) : "d"(a));
    double e = __fma_rn(-a, x, 1.0);
    x = __fma_rn(x, e, x);
    e = __fma_rn(-a, x, 1.0);
    return __fma_rn(x, e, x);
}

__device__ __forceinline__ float sub_rn(float a, float b) { return __fsub_rn(a, b); }
__device__ __forceinline__ double sub_rn(double a, double b) { return __dsub_rn(a, b); }
__device__ __forceinline__ float add_rn(float a, float b) { return __fadd_rn(a, b); }
__device__ __forceinline__ double add_rn(double a, double b) { return __dadd_rn(a, b); }
__device__ __forceinline__ float mul_rn(float a, float b) { return __fmul_rn(a, b); }
__device__ __forceinline__ double mul_rn(double a, double b) { return __dmul_rn(a, b); }
__device__ __forceinline__ float fma_rn(float a, float b, float c) { return __fmaf_rn(a, b, c); }
__device__ __forceinline__ double fma_rn(double a, double b, double c) { return __fma_rn(a, b, c); }

// Philox-4x32-10 (Salmon et al., SC'11), counter = (ray id lo, hi, 0, 0), key = seed: two 53-bit uniforms in
// [0,1) per ray.  GPU-D shoots rays from random positions; reading R17 draws one ray
// uniformly inside each grid cell, so ray (i,j) stays in the tile that owns cell (i,j).
__device__ __forceinline__ void ray_words(unsigned long long ray_id, unsigned long long seed, unsigned int &c0, unsigned int &c1,
                                          unsigned int &c2, unsigned int &c3)
{
    c0 = (unsigned int)ray_id; c1 = (unsigned int)(ray_id >> 32); c2 = 0u; c3 = 0u;
    unsigned int k0 = (unsigned int)seed, k1 = (unsigned int)(seed >> 32);
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const unsigned int h0 = __umulhi(0xD2511F53u, c0), l0 = 0xD2511F53u * c0;
        const unsigned int h1 = __umulhi(0xCD9E8D57u, c2), l1 = 0xCD9E8D57u * c2;
        c0 = h1 ^ c1 ^ k0; c1 = l1; c2 = h0 ^ c3 ^ k1; c3 = l0;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
}

__device__ __forceinline__ void ray_uniforms(unsigned long long ray_id, unsigned long long seed, double &u1, double &u2)
{
    unsigned int c0, c1, c2, c3;
    ray_words(ray_id, seed, c0, c1, c2, c3);
    u1 = ((double)(c0 >> 5) * 67108864.0 + (double)(c1 >> 6)) * (1.0 / 9007199254740992.0);
    u2 = ((double)(c2 >> 5) * 67108864.0 + (double)(c3 >> 6)) * (1.0 / 9007199254740992.0);
}

// ML_RAYS_UNIFORM (see shoot_kernel_upipe below): bucket size and the ray a list entry stands for
// bucket: grid cells along axis 1 / axis 2.  Small, because the FP32 error of a close passage grows with the distance of ray
// and lens from the local origin (R15); 128 x 63 = 8064 cells, because a full shoot puts one ray per cell on
// average and CTAs take 1024 (fp64: 2048) list entries: 8064 + 1.4 sigma = 8192, so 92 % of the buckets need exactly 8 CTAs
// (at 128 x 64 half of them would need a ninth for a handful of rays).
constexpr int kUniBW = 128, kUniBH = 63;
constexpr int kUniWarps = 4;             // shoot_kernel_upipe: 128 threads x 8 rays = 1024 list entries per CTA, 4 CTAs per SM

__host__ __device__ __forceinline__ unsigned long long uniform_ray_id(const ShootParams &p, unsigned long long handle)
{
    if (p.probe_ids) return (unsigned long long)p.probe_ids[handle];
    const long long jj = (long long)handle / p.list_w, ii = (long long)handle - jj * p.list_w;
    return (unsigned long long)((p.j0 + jj) * p.n1 + (p.i0 + ii));
}

// a4 + a5 (+ statistics) for one thread's RX x RY rays: macro terms and pixel index in
// fp64, run-length aggregated binning.  Shared by every instantiation of the kernels below.
//
// Binning works on the pixel coordinate directly: u = (y + L/2) n_pix/L with y = c x - S (eq.4) is evaluated as
//     u = fma(-S, n_pix/L, fma(x, c n_pix/L, (L/2) n_pix/L))
// (two fp64 FMAs per component, the inner one shared by a column / row of the regular grid), floored with one
// F2I.F64.FLOOR; the ray is in the map iff both floors are < n_pix as unsigned integers and u is finite (exponent
// field of u not all ones: F2I maps NaN to 0, so the test cannot be skipped).  CAPTURE writes y itself.
// RANDOM instantiations either pass the (u1, u2) they drew in the prologue (UV_SMEM: shared memory, [ray][thread]) or
// have them drawn again here (same counter, same key: the same numbers).
// UNIFORM (ML_RAYS_UNIFORM, reading R20): slot (r, c) of thread t is entry (r RX + c) THREADS + t of the CTA's slice of a
// bucket's ray list (`handles`, `n_valid` entries); the ray's position is x = ((u1 n1 - n1/2) delta, (u2 n2 - n2/2) delta)
// with the uniforms of its ray id, kept in `uv`.  CAPTURE writes y to capture[handle].
template <int RX, int RY, bool CAPTURE, int WARPS = kWarps, bool RANDOM = false, bool UV_SMEM = false, bool UNIFORM = false>
__device__ __forceinline__ void finish_tile(const ShootParams &p, long long ti, long long tj, long long t, int lane,
                                            int warp, const double (&Sx)[RY][RX], const double (&Sy)[RY][RX],
                                            unsigned int *cta_count, const double2 *uv = nullptr, int n_valid = 0,
                                            const unsigned long long *handles = nullptr)
{
    constexpr int TW = 32 * RX;
    constexpr int TH = WARPS * RY;
    constexpr int THREADS = WARPS * 32;
    unsigned int n_shot = 0, n_in = 0, n_drop = 0; // per thread; reduced over the warp once, after the loop
    const unsigned int full = 0xffffffffu;
    auto draw = [&](int r, int c) {
        double2 w = make_double2(0.0, 0.0);
        if (RANDOM) {
            if (UV_SMEM) {
                w = uv[(r * RX + c) * THREADS + threadIdx.x];
            } else {
                const unsigned long long i = (unsigned long long)(ti * TW + lane * RX + c), j = (unsigned long long)(tj * TH + warp * RY + r);
                ray_uniforms(j * (unsigned long long)p.n1 + i, p.ray_seed, w.x, w.y);
            }
        }
        return w;
    };
    // ray indices as exact doubles: (double)(ti*TW) + small integer = (double)i, no 64-bit conversions per ray
    const double ib = (double)(ti * TW) + (double)(lane * RX), jb = (double)(tj * TH) + (double)(warp * RY);
    if (CAPTURE) {
#pragma unroll
        for (int r = 0; r < RY; ++r)
#pragma unroll
            for (int c = 0; c < RX; ++c) {
                double x1, x2;
                if (UNIFORM) {
                    const int slot = (r * RX + c) * THREADS + (int)threadIdx.x;
                    if (slot >= n_valid) continue;
                    double2 w;
                    if (UV_SMEM) w = uv[slot];
                    else ray_uniforms(uniform_ray_id(p, handles[slot]), p.ray_seed, w.x, w.y);
                    x1 = __dmul_rn(__dsub_rn(__dmul_rn(w.x, p.n1d), 0.5 * p.n1d), p.delta);
                    x2 = __dmul_rn(__dsub_rn(__dmul_rn(w.y, p.n2d), 0.5 * p.n2d), p.delta);
                    const double y1 = p.c1 * x1 - Sx[r][c], y2 = p.c2 * x2 - Sy[r][c];
                    const bool finite = (fabs(y1) <= 1.7976931348623157e308) && (fabs(y2) <= 1.7976931348623157e308);
                    const double qnan = __longlong_as_double(0x7ff8000000000000LL);
                    p.capture[handles[slot]] = make_double2(finite ? y1 : qnan, finite ? y2 : qnan);
                    continue;
                }
                if (RANDOM) { // the ray's own position in its cell (the draw of the prologue)
                    const double2 w = draw(r, c);
                    x1 = ((ib + (double)c) + w.x - (p.half1 + 0.5)) * p.delta;
                    x2 = ((jb + (double)r) + w.y - (p.half2 + 0.5)) * p.delta;
                } else {
                    x1 = ((ib + (double)c) - p.half1) * p.delta;
                    x2 = ((jb + (double)r) - p.half2) * p.delta;
                }
                const double y1 = p.c1 * x1 - Sx[r][c];
                const double y2 = p.c2 * x2 - Sy[r][c];
                const bool finite = (fabs(y1) <= 1.7976931348623157e308) && (fabs(y2) <= 1.7976931348623157e308);
                const double qnan = __longlong_as_double(0x7ff8000000000000LL);
                double2 o;
                o.x = finite ? y1 : qnan;
                o.y = finite ? y2 : qnan;
                p.capture[(size_t)t * (TW * TH) + (size_t)(warp * RY + r) * TW + lane * RX + c] = o;
            }
        return;
    }
    // ---- a4 + a5: macro terms folded into the pixel coordinate, binning
    // "inside the requested region" bits per column / row, and the x-part of the pixel coordinate per column
    unsigned int colmask = 0u, rowmask = 0u;
    double U1[RX];
#pragma unroll
    for (int c = 0; c < RX; ++c) {
        const long long i = ti * TW + lane * RX + c;
        colmask |= ((i >= p.i0) && (i < p.i1)) ? (1u << c) : 0u;
        if (!RANDOM) U1[c] = __fma_rn(((ib + (double)c) - p.half1) * p.delta, p.k1, p.hoff);
    }
#pragma unroll
    for (int r = 0; r < RY; ++r) {
        const long long j = tj * TH + warp * RY + r;
        rowmask |= ((j >= p.j0) && (j < p.j1)) ? (1u << r) : 0u;
    }
    if (UNIFORM) { colmask = 0xffffffffu; rowmask = 0xffffffffu; } // every listed ray belongs to the region: slots decide
    const unsigned int n_pix_u = (unsigned int)p.n_pix;
    const double nip = -p.inv_pixel;
#pragma unroll
    for (int r = 0; r < RY; ++r) {
        double U2 = 0.0;
        if (!RANDOM) U2 = __fma_rn(((jb + (double)r) - p.half2) * p.delta, p.k2, p.hoff);
#pragma unroll
        for (int c = 0; c < RX; ++c) {
            double b1, b2;
            bool in_list = true;
            if (UNIFORM) {
                const int slot = (r * RX + c) * THREADS + (int)threadIdx.x;
                in_list = slot < n_valid;
                double2 w = make_double2(0.5, 0.5);
                if (UV_SMEM) w = uv[slot];
                else if (in_list) ray_uniforms(uniform_ray_id(p, handles[slot]), p.ray_seed, w.x, w.y);
                b1 = __fma_rn(__dmul_rn(__dsub_rn(__dmul_rn(w.x, p.n1d), 0.5 * p.n1d), p.delta), p.k1, p.hoff);
                b2 = __fma_rn(__dmul_rn(__dsub_rn(__dmul_rn(w.y, p.n2d), 0.5 * p.n2d), p.delta), p.k2, p.hoff);
            } else if (RANDOM) {
                const double2 w = draw(r, c);
                b1 = __fma_rn(((ib + (double)c) + w.x - (p.half1 + 0.5)) * p.delta, p.k1, p.hoff);
                b2 = __fma_rn(((jb + (double)r) + w.y - (p.half2 + 0.5)) * p.delta, p.k2, p.hoff);
            } else {
                b1 = U1[c];
                b2 = U2;
            }
            const double u1 = __fma_rn(Sx[r][c], nip, b1);
            const double u2 = __fma_rn(Sy[r][c], nip, b2);
            // finite <=> exponent field not all ones, in both components
            const bool finite = ((~__double2hiint(u1) & 0x7ff00000) != 0) && ((~__double2hiint(u2) & 0x7ff00000) != 0);
            const bool valid = UNIFORM ? in_list : (((colmask >> c) & (rowmask >> r) & 1u) != 0u);
            // floor to int (saturating): 0 <= u < n_pix  <=>  (unsigned)floor(u) < n_pix for every finite u
            const int pi = __double2int_rd(u1), pj = __double2int_rd(u2);
            const bool inside = ((unsigned int)pi < n_pix_u) && ((unsigned int)pj < n_pix_u);
            const int pix = (valid && finite && inside) ? pj * p.n_pix + pi : -1;
            // run-length aggregation along the lanes of the warp
            const int prev = __shfl_up_sync(full, pix, 1);
            const bool head = (lane == 0) || (pix != prev);
            const unsigned int heads = __ballot_sync(full, head);
            if (head && pix >= 0) {
                const unsigned int above = heads & ~((2u << lane) - 1u);
                const int next = above ? (__ffs(above) - 1) : 32;
                atomicAdd(&p.map[pix], (unsigned int)(next - lane));
            }
            n_in += (pix >= 0);
            n_shot += valid;
            n_drop += (valid && !finite);
        }
    }
    n_shot = __reduce_add_sync(full, n_shot); // REDUX.SUM: one instruction per counter instead of a vote per ray
    n_in = __reduce_add_sync(full, n_in);
    n_drop = __reduce_add_sync(full, n_drop);
    if (lane == 0) {
        atomicAdd(&cta_count[0], n_shot);
        atomicAdd(&cta_count[1], n_in);
        if (n_drop) atomicAdd(&cta_count[2], n_drop);
    }
    __syncthreads();
    if (threadIdx.x < 3 && cta_count[threadIdx.x])
        atomicAdd(&p.counters[threadIdx.x], (unsigned long long)cta_count[threadIdx.x]);
}

// a6: which tile this CTA shoots.  Shoot launches use a 2-D grid (x = tile column, y = tile row: the hardware
// rasterises x first, so concurrently resident CTAs touch a narrow band of the map) and need no division; capture
// launches take their tiles from an explicit list.
template <bool CAPTURE>
__device__ __forceinline__ void which_tile(const ShootParams &p, long long &t, long long &ti, long long &tj)
{
    if (CAPTURE) {
        t = (long long)blockIdx.x;
        ti = p.tile_list[2 * t];
        tj = p.tile_list[2 * t + 1];
    } else {
        t = 0;
        ti = p.tile_i0 + blockIdx.x;
        tj = p.tile_j0 + blockIdx.y;
    }
}

// Lens range of this CTA.  Shoot launches walk every lens.  Capture launches of a few tiles over many lenses
// (ml_probe / ml_capture_region at N* >= 1e5) split the lens loop over
// blockIdx.y: ranges are multiples of the 512-lens chunk, so chunk and flush-group boundaries fall where they do in
// the unsplit loop; each CTA writes its fp64 partial sums and combine_kernel adds them in range order.
template <bool CAPTURE> __device__ __forceinline__ void lens_range(const ShootParams &p, int &lb, int &le)
{
    lb = 0;
    le = p.n_lens;
    if (CAPTURE && p.split_len > 0) {
        const long long b = (long long)blockIdx.y * p.split_len;
        lb = (int)b;
        le = (int)min(b + (long long)p.split_len, (long long)p.n_lens);
    }
}

template <int RX, int RY, int WARPS>
__device__ __forceinline__ void store_partials(const ShootParams &p, long long t, int lane, int warp, const double (&Sx)[RY][RX],
                                               const double (&Sy)[RY][RX])
{
    constexpr int TW = 32 * RX, TH = WARPS * RY;
    double2 *dst = p.partial + ((size_t)blockIdx.y * gridDim.x + (size_t)t) * (TW * TH);
#pragma unroll
    for (int r = 0; r < RY; ++r)
#pragma unroll
        for (int c = 0; c < RX; ++c) dst[(size_t)(warp * RY + r) * TW + lane * RX + c] = make_double2(Sx[r][c], Sy[r][c]);
}

// Second half of a split launch: one CTA per tile, the thread-to-ray mapping of the shoot kernels; the partial sums
// of the lens ranges are added in range order (fp64), then the usual epilogue runs: CAPTURE writes the positions,
// otherwise the rays are binned (a small region shot through very many lenses, ml_shoot_region).
template <int RX, int RY, int WARPS, bool RANDOM, bool CAPTURE>
__global__ void __launch_bounds__(WARPS * 32) combine_kernel(const ShootParams p, int n_splits)
{
    constexpr int TW = 32 * RX, TH = WARPS * RY;
    __shared__ unsigned int cta_count[3];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    long long t, ti, tj;
    which_tile<true>(p, t, ti, tj);
    if (threadIdx.x < 3) cta_count[threadIdx.x] = 0;
    __syncthreads();
    double Sx[RY][RX], Sy[RY][RX];
#pragma unroll
    for (int r = 0; r < RY; ++r)
#pragma unroll
        for (int c = 0; c < RX; ++c) { Sx[r][c] = 0.0; Sy[r][c] = 0.0; }
    for (int s = 0; s < n_splits; ++s) {
        const double2 *src = p.partial + ((size_t)s * gridDim.x + (size_t)t) * (TW * TH);
#pragma unroll
        for (int r = 0; r < RY; ++r)
#pragma unroll
            for (int c = 0; c < RX; ++c) {
                const double2 v = src[(size_t)(warp * RY + r) * TW + lane * RX + c];
                Sx[r][c] += v.x;
                Sy[r][c] += v.y;
            }
    }
    finish_tile<RX, RY, CAPTURE, WARPS, RANDOM, false>(p, ti, tj, t, lane, warp, Sx, Sy, cta_count);
}

template <typename Real, int RX, int RY, int KF, bool NEWTON, bool CAPTURE, bool MASS = false, bool RANDOM = false, bool UNIFORM = false>
__global__ void __launch_bounds__(kThreads, 2) shoot_kernel(const ShootParams p)
{
    static_assert(!UNIFORM || RANDOM, "UNIFORM: per-ray offsets");
    constexpr int SLOTS = kThreads * RX * RY; // UNIFORM: list entries per CTA
    using Real2 = typename Vec2<Real>::type;
    constexpr int TW = 32 * RX;
    constexpr int TH = kWarps * RY;
    static_assert(kChunk % KF == 0 && KF % 8 == 0, "flush groups must tile a chunk");
    static_assert(kChunk % kThreads == 0, "staging assumes whole lenses per thread");
    constexpr int PER_THREAD = kChunk / kThreads;

    __shared__ __align__(16) Real2 lens_s[2][kChunk];
    __shared__ Real mass_s[2][MASS ? kChunk : 1]; // m_i of eq.4, unit masses otherwise
    __shared__ unsigned int cta_count[3];

    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;

    // ---- a6: which tile (UNIFORM: which slice of which bucket's ray list, as in shoot_kernel_upipe)
    long long t = 0, ti = 0, tj = 0;
    int lb, le; // this CTA's lens range: [0, n_lens) except in split capture launches
    int n_valid = 0;
    const unsigned long long *handles = nullptr;
    double cx, cy, ccx = 0.0, ccy = 0.0;
    if (UNIFORM) {
        const long long b = (long long)blockIdx.x;
        const unsigned int filled = min(p.bucket_fill[b], p.bucket_cap);
        const long long first = (long long)blockIdx.y * SLOTS;
        if (first >= (long long)filled) return; // (whole CTA: before any barrier)
        n_valid = (int)min((long long)SLOTS, (long long)filled - first);
        handles = p.ray_list + (size_t)b * p.bucket_cap + first;
        lens_range<false>(p, lb, le);
        ccx = (double)((b % p.bucket_nx) * kUniBW) + 0.5 * kUniBW;
        ccy = (double)((p.bucket_row0 + b / p.bucket_nx) * kUniBH) + 0.5 * kUniBH;
        cx = (ccx - 0.5 * p.n1d) * p.delta;
        cy = (ccy - 0.5 * p.n2d) * p.delta;
    } else {
        which_tile<CAPTURE>(p, t, ti, tj);
        lens_range<CAPTURE>(p, lb, le);
        // ---- a2: tile centre (fp64) and this thread's ray offsets from it
        cx = ((double)(ti * TW) + 0.5 * (TW - 1) - p.half1) * p.delta;
        cy = ((double)(tj * TH) + 0.5 * (TH - 1) - p.half2) * p.delta;
    }
    if (threadIdx.x < 3) cta_count[threadIdx.x] = 0;
    Real ox[RX], oy[RY];
#pragma unroll
    for (int c = 0; c < RX; ++c) ox[c] = (Real)(((double)(lane * RX + c) - 0.5 * (TW - 1)) * p.delta);
#pragma unroll
    for (int r = 0; r < RY; ++r) oy[r] = (Real)(((double)(warp * RY + r) - 0.5 * (TH - 1)) * p.delta);
    // RANDOM: every ray has its own offset from the tile centre (no shared column / row differences)
    Real oxr[RANDOM ? RY : 1][RANDOM ? RX : 1], oyr[RANDOM ? RY : 1][RANDOM ? RX : 1];
    if (RANDOM) {
#pragma unroll
        for (int r = 0; r < RY; ++r)
#pragma unroll
            for (int c = 0; c < RX; ++c) {
                double u1, u2;
                if (UNIFORM) { // an empty slot shoots a ray from the bucket centre and throws it away
                    const int slot = (r * RX + c) * kThreads + (int)threadIdx.x;
                    Real fx = (Real)0, fy = (Real)0;
                    if (slot < n_valid) {
                        ray_uniforms(uniform_ray_id(p, handles[slot]), p.ray_seed, u1, u2);
                        fx = (Real)((__dmul_rn(u1, p.n1d) - ccx) * p.delta);
                        fy = (Real)((__dmul_rn(u2, p.n2d) - ccy) * p.delta);
                    }
                    oxr[RANDOM ? r : 0][RANDOM ? c : 0] = fx;
                    oyr[RANDOM ? r : 0][RANDOM ? c : 0] = fy;
                    continue;
                }
                const unsigned long long i = (unsigned long long)(ti * TW + lane * RX + c), j = (unsigned long long)(tj * TH + warp * RY + r);
                ray_uniforms(j * (unsigned long long)p.n1 + i, p.ray_seed, u1, u2);
                oxr[RANDOM ? r : 0][RANDOM ? c : 0] = (Real)(((double)(lane * RX + c) + u1 - 0.5 * TW) * p.delta);
                oyr[RANDOM ? r : 0][RANDOM ? c : 0] = (Real)(((double)(warp * RY + r) + u2 - 0.5 * TH) * p.delta);
            }
    }

    double Sx[RY][RX], Sy[RY][RX]; // fp64 accumulators of the deflection sum
    Real sx[RY][RX], sy[RY][RX];   // partial sums of the current flush group
#pragma unroll
    for (int r = 0; r < RY; ++r)
#pragma unroll
        for (int c = 0; c < RX; ++c) {
            Sx[r][c] = 0.0; Sy[r][c] = 0.0;
            sx[r][c] = (Real)0; sy[r][c] = (Real)0;
        }

    // ---- a1: stage chunk 0
    const Real pad = pad_coordinate<Real, NEWTON>();
    double2 pre[PER_THREAD];
    double pre_m[MASS ? PER_THREAD : 1];
    auto fetch = [&](int base) {
#pragma unroll
        for (int q = 0; q < PER_THREAD; ++q) {
            const int k = base + q * kThreads + threadIdx.x;
            if (k < le) {
                pre[q] = __ldg(&p.lens[k]);
                if (MASS) pre_m[q] = __ldg(&p.mass[k]);
            }
        }
    };
    auto stage = [&](int base, int buf) {
#pragma unroll
        for (int q = 0; q < PER_THREAD; ++q) {
            const int k = base + q * kThreads + threadIdx.x;
            Real2 v;
            Real m = (Real)0;
            if (k < le) {
                v.x = (Real)(pre[q].x - cx);
                v.y = (Real)(pre[q].y - cy);
                if (MASS) m = (Real)pre_m[q];
            } else {
                v.x = pad; v.y = pad;
            }
            lens_s[buf][q * kThreads + threadIdx.x] = v;
            if (MASS) mass_s[buf][q * kThreads + threadIdx.x] = m;
        }
    };
    fetch(lb);
    stage(lb, 0);
    __syncthreads();

    // ---- a3: all-pairs deflection sum
    int buf = 0;
    for (int base = lb; base < le; base += kChunk) {
        const bool more = base + kChunk < le;
        if (more) fetch(base + kChunk);
        const int cnt = min(kChunk, le - base);
        const int cntp = (cnt + 7) & ~7; // padded with zero-contribution lenses
        const Real2 *ls = lens_s[buf];
        const Real *ms = mass_s[buf];
        for (int k0 = 0; k0 < cntp; k0 += KF) {
            const int kend = min(k0 + KF, cntp);
#pragma unroll 1
            for (int k = k0; k < kend; k += 2) {
#pragma unroll
                for (int u = 0; u < 2; ++u) {
                    const Real2 l = ls[k + u];
                    const Real m = MASS ? ms[k + u] : (Real)1;
                    if constexpr (RANDOM) { // 2 sub, mul, fma, rcp, 2 fma per interaction: the paper's 10 flop, nothing shared
#pragma unroll
                        for (int r = 0; r < RY; ++r)
#pragma unroll
                            for (int c = 0; c < RX; ++c) {
                                const Real ex = sub_rn(oxr[RANDOM ? r : 0][RANDOM ? c : 0], l.x);
                                const Real ey = sub_rn(oyr[RANDOM ? r : 0][RANDOM ? c : 0], l.y);
                                Real inv = recip<NEWTON>(fma_rn(ey, ey, mul_rn(ex, ex)));
                                if (MASS) inv = mul_rn(inv, m);
                                sx[r][c] = fma_rn(ex, inv, sx[r][c]);
                                sy[r][c] = fma_rn(ey, inv, sy[r][c]);
                            }
                    } else {
                    Real dx[RX], dx2[RX], dy[RY], dy2[RY];
#pragma unroll
                    for (int c = 0; c < RX; ++c) { dx[c] = sub_rn(ox[c], l.x); dx2[c] = mul_rn(dx[c], dx[c]); }
#pragma unroll
                    for (int r = 0; r < RY; ++r) { dy[r] = sub_rn(oy[r], l.y); dy2[r] = mul_rn(dy[r], dy[r]); }
#pragma unroll
                    for (int r = 0; r < RY; ++r)
#pragma unroll
                        for (int c = 0; c < RX; ++c) {
                            Real inv = recip<NEWTON>(add_rn(dx2[c], dy2[r]));
                            if (MASS) inv = mul_rn(inv, m); // m_i / r^2
                            sx[r][c] = fma_rn(dx[c], inv, sx[r][c]);
                            sy[r][c] = fma_rn(dy[r], inv, sy[r][c]);
                        }
                    } // regular grid
                }
            }
            // flush the group's partial sums into the fp64 accumulators
#pragma unroll
            for (int r = 0; r < RY; ++r)
#pragma unroll
                for (int c = 0; c < RX; ++c) {
                    Sx[r][c] += (double)sx[r][c]; sx[r][c] = (Real)0;
                    Sy[r][c] += (double)sy[r][c]; sy[r][c] = (Real)0;
                }
        }
        if (more) stage(base + kChunk, buf ^ 1);
        __syncthreads();
        buf ^= 1;
    }

    if (UNIFORM) {
        finish_tile<RX, RY, CAPTURE, kWarps, true, false, true>(p, 0, 0, 0, lane, warp, Sx, Sy, cta_count, nullptr, n_valid, handles);
        return;
    }
    if (CAPTURE && p.partial) { store_partials<RX, RY, kWarps>(p, t, lane, warp, Sx, Sy); return; }
    finish_tile<RX, RY, CAPTURE, kWarps, RANDOM>(p, ti, tj, t, lane, warp, Sx, Sy, cta_count);
}

// ---------------------------------------------------------------------------------------
// The default FP32 kernel (ML_PREC_FP32_TILED): packed f32x2 arithmetic, shared reciprocals,
// software-pipelined over lenses.
//
// The generic kernel above issues one MUFU.RCP per interaction, and the special-function unit
// (16 results per clock per SM) caps it at 62.5 % of the FP32 peak in the paper's 10-flop
// accounting.  Here a thread still owns 4 x 4 rays, but
//   * every FP32 instruction on the rays is a packed FADD2 / FMUL2 / FFMA2 on two rays that are
//     adjacent along axis 1 (columns 0,1 = "A", columns 2,3 = "B"): half the issue slots, so the
//     MUFU instructions issue beside a busy FMA pipe;
//   * on SHARED of the 4 rows one reciprocal serves two interactions:
//         R = 1/(r2A * r2B),   1/r2A = R * r2B,   1/r2B = R * r2A      (3 FMUL2, 2 MUFU per 4)
//     instead of 4 MUFU.  SHARED = 4: 40 packed + 4 scalar FP32 instructions and 8 MUFU per lens
//     per thread (16 interactions) = 5.25 FMA-pipe lane-cycles and 0.5 MUFU per interaction;
//   * the lens tile is staged as float4 (-x, -x, -y, -y): one LDS.128 broadcast per lens feeds
//     the packed subtractions without any register shuffling;
//   * stage 1 (differences, r^2, products, MUFU) of lens k+1 is issued before stage 2
//     (1/r^2 = R * r2, the four accumulating FFMA2 per row) of lens k, so that no instruction
//     waits on a reciprocal it has just issued (PipeRegs carries a lens between the stages).
// r^2 = dy*dy + (dx*dx + 2^-80): the 2^-80 keeps a ray that coincides with a lens in its
// FP32 tile-local coordinates from producing 0 * inf = NaN in its partner's term (the lens
// is then simply not seen by that one ray, R12); it is below half an ulp of r^2 for
// every ray that ends closer than 1e8 R_E to the map.
// Summation order: as above (lens index order, groups of KF, fp64 accumulators).  A padding
// lens sits at 1e15: r^2 = 2e30 stays finite, the shared product overflows to +inf, 1/inf = +0,
// so its terms are exactly 0 on shared rows and 5e-16 on the others.
template <int RY> struct PipeRegs {
    float2 dxA, dxB;
    float m; // lens mass (MASS instantiations)
    float dy[RY];
    float2 r2A[RY], r2B[RY]; // shared rows: r^2; other rows: 1/r^2
    float2 R[RY];
};

// TUNE: source-order knobs that change nothing in the arithmetic of a ray (same operations, same operands, same
// rounding) but steer ptxas towards different instruction schedules of the loop; the value the library uses was
// picked by measurement on the B200.  bit 0: pipeline two lenses ahead instead of
// one; bits 1-2: order of the four accumulations of a row; bit 3: 1/r^2 of pair B after the accumulations of pair A;
// bit 4: rows in reverse order in stage 2; bit 5: rows in reverse order in stage 1; bit 6: stage 1 forms r^2 of
// all rows before the first reciprocal; bit 7: stage 2 forms every 1/r^2 before the first accumulation.
// bit 8 does change the arithmetic (shoot and capture instantiations alike): on the last row of every odd lens the two
// ray pairs take their own reciprocals (4 MUFU.RCP) instead of the shared one (2 MUFU.RCP + 3 FMUL2).
template <int SHARED, int KF, int WARPS, int MINB, bool SCALAR_DY, bool CAPTURE, bool MASS = false, bool NEWTON = false, int TUNE = 0>
__global__ void __launch_bounds__(WARPS * 32, MINB) shoot_kernel_pipe(const ShootParams p)
{
    constexpr int RX = 4, RY = 4;
    constexpr int THREADS = WARPS * 32;
    constexpr int TW = 32 * RX;
    constexpr int TH = WARPS * RY;
    static_assert(kChunk % KF == 0 && KF % 2 == 0, "flush groups must tile a chunk");
    constexpr int PER_THREAD = kChunk / THREADS;

    __shared__ __align__(16) float4 lens_s[2][kChunk + 2];
    __shared__ float mass_s[2][MASS ? kChunk + 2 : 1]; // m_i of eq.4; one extra FMUL2 per row and lens
    __shared__ unsigned int cta_count[3];

    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;

    long long t, ti, tj;
    which_tile<CAPTURE>(p, t, ti, tj);
    int lb, le; // this CTA's lens range: [0, n_lens) except in split capture launches
    lens_range<CAPTURE>(p, lb, le);
    if (threadIdx.x < 3) cta_count[threadIdx.x] = 0;
    // NEWTON: the padding lens must keep r2A * r2B finite (inf * 0 in the refinement would be NaN): 1e9 -> product 4e36,
    // its terms are 5e-10 R_E (at most two padding lenses per launch are ever evaluated: below every tolerance)
    const float padc = NEWTON ? -1e9f : -1e15f;
    if (threadIdx.x < 4) lens_s[threadIdx.x >> 1][kChunk + (threadIdx.x & 1)] = make_float4(padc, padc, padc, padc);
    if (MASS && threadIdx.x < 4) mass_s[threadIdx.x >> 1][(MASS ? kChunk : 0) + (MASS ? (threadIdx.x & 1) : 0)] = 0.f;

    const double cx = ((double)(ti * TW) + 0.5 * (TW - 1) - p.half1) * p.delta;
    const double cy = ((double)(tj * TH) + 0.5 * (TH - 1) - p.half2) * p.delta;
    float2 oxA, oxB;
    float oy[RY];
    oxA.x = (float)(((double)(lane * RX + 0) - 0.5 * (TW - 1)) * p.delta);
    oxA.y = (float)(((double)(lane * RX + 1) - 0.5 * (TW - 1)) * p.delta);
    oxB.x = (float)(((double)(lane * RX + 2) - 0.5 * (TW - 1)) * p.delta);
    oxB.y = (float)(((double)(lane * RX + 3) - 0.5 * (TW - 1)) * p.delta);
#pragma unroll
    for (int r = 0; r < RY; ++r) oy[r] = (float)(((double)(warp * RY + r) - 0.5 * (TH - 1)) * p.delta);

    double Sx[RY][RX], Sy[RY][RX];
    float2 sxA[RY], sxB[RY], syA[RY], syB[RY];
#pragma unroll
    for (int r = 0; r < RY; ++r) {
#pragma unroll
        for (int c = 0; c < RX; ++c) { Sx[r][c] = 0.0; Sy[r][c] = 0.0; }
        sxA[r] = make_float2(0.f, 0.f); sxB[r] = sxA[r]; syA[r] = sxA[r]; syB[r] = sxA[r];
    }

    double2 pre[PER_THREAD];
    double pre_m[MASS ? PER_THREAD : 1];
    auto fetch = [&](int base) {
#pragma unroll
        for (int q = 0; q < PER_THREAD; ++q) {
            const int k = base + q * THREADS + threadIdx.x;
            if (k < le) {
                pre[q] = __ldg(&p.lens[k]);
                if (MASS) pre_m[q] = __ldg(&p.mass[k]);
            }
        }
    };
    auto stage = [&](int base, int buf) {
#pragma unroll
        for (int q = 0; q < PER_THREAD; ++q) {
            const int k = base + q * THREADS + threadIdx.x;
            float nx = padc, ny = padc, m = 0.f;
            if (k < le) {
                nx = -(float)(pre[q].x - cx);
                ny = -(float)(pre[q].y - cy);
                if (MASS) m = (float)pre_m[q];
            }
            lens_s[buf][q * THREADS + threadIdx.x] = make_float4(nx, nx, ny, ny);
            if (MASS) mass_s[buf][q * THREADS + threadIdx.x] = m;
        }
    };
    fetch(lb);
    stage(lb, 0);
    __syncthreads();

    const float2 eps2 = make_float2(0x1p-80f, 0x1p-80f);
    static_assert(!(NEWTON && ((TUNE & 256) || SHARED < RY)), "the Newton step is written for shared reciprocals only");
    // rows whose two ray pairs share one reciprocal: all SHARED first rows, except (TUNE bit 8) the last row of odd lenses
    auto shares = [](int r, bool odd) { return r < SHARED && !((TUNE & 256) && odd && r == RY - 1); };
    auto stage1 = [&](auto odd, const float4 l, const float m, PipeRegs<RY> &s) {
        const float2 nlx = make_float2(l.x, l.y), nly = make_float2(l.z, l.w);
        s.m = m;
        s.dxA = __fadd2_rn(oxA, nlx);
        s.dxB = __fadd2_rn(oxB, nlx);
        const float2 qA = __ffma2_rn(s.dxA, s.dxA, eps2), qB = __ffma2_rn(s.dxB, s.dxB, eps2);
        auto row_r2 = [&](int r) {
            float2 dy;
            if (SCALAR_DY) {
                s.dy[r] = __fadd_rn(oy[r], l.z);
                dy = make_float2(s.dy[r], s.dy[r]);
            } else {
                dy = __fadd2_rn(make_float2(oy[r], oy[r]), nly);
                s.dy[r] = dy.x;
            }
            s.r2A[r] = __ffma2_rn(dy, dy, qA);
            s.r2B[r] = __ffma2_rn(dy, dy, qB);
        };
        auto row_rcp = [&](int r) {
            if (shares(r, decltype(odd)::value)) {
                const float2 P = __fmul2_rn(s.r2A[r], s.r2B[r]);
                s.R[r].x = rcp_approx(P.x);
                s.R[r].y = rcp_approx(P.y);
            } else {
                s.r2A[r].x = rcp_approx(s.r2A[r].x); s.r2A[r].y = rcp_approx(s.r2A[r].y);
                s.r2B[r].x = rcp_approx(s.r2B[r].x); s.r2B[r].y = rcp_approx(s.r2B[r].y);
            }
        };
        if (TUNE & 64) { // all r^2 first, then the products and reciprocals
#pragma unroll
            for (int rr = 0; rr < RY; ++rr) row_r2((TUNE & 32) ? RY - 1 - rr : rr);
#pragma unroll
            for (int rr = 0; rr < RY; ++rr) row_rcp((TUNE & 32) ? RY - 1 - rr : rr);
        } else {
#pragma unroll
            for (int rr = 0; rr < RY; ++rr) {
                const int r = (TUNE & 32) ? RY - 1 - rr : rr;
                row_r2(r);
                row_rcp(r);
            }
        }
    };
    auto stage2 = [&](auto odd, const PipeRegs<RY> &s) {
        float2 iAs[RY], iBs[RY];
        auto inv_r2 = [&](int r, float2 &iA, float2 &iB, float2 &R, bool both) {
            R = s.R[r];
            if (shares(r, decltype(odd)::value)) {
                if (NEWTON) { // one Newton-Raphson step on the shared reciprocal: R <- R + R (1 - P R), P = r2A r2B
                    const float2 P = __fmul2_rn(s.r2A[r], s.r2B[r]);
                    const float2 e = __ffma2_rn(make_float2(-P.x, -P.y), R, make_float2(1.f, 1.f));
                    R = __ffma2_rn(R, e, R);
                }
                if (MASS) R = __fmul2_rn(R, make_float2(s.m, s.m)); // m_i / (r2A r2B)
                iA = __fmul2_rn(R, s.r2B[r]);
                if (both) iB = __fmul2_rn(R, s.r2A[r]);
            } else {
                iA = MASS ? __fmul2_rn(s.r2A[r], make_float2(s.m, s.m)) : s.r2A[r];
                iB = MASS ? __fmul2_rn(s.r2B[r], make_float2(s.m, s.m)) : s.r2B[r];
            }
        };
        if (TUNE & 128) {
#pragma unroll
            for (int rr = 0; rr < RY; ++rr) {
                const int r = (TUNE & 16) ? RY - 1 - rr : rr;
                float2 R;
                inv_r2(r, iAs[r], iBs[r], R, true);
            }
        }
#pragma unroll
        for (int rr = 0; rr < RY; ++rr) {
            const int r = (TUNE & 16) ? RY - 1 - rr : rr;
            float2 iA, iB, R;
            const bool late_b = (TUNE & 8) && !(TUNE & 128) && shares(r, decltype(odd)::value);
            if (TUNE & 128) { iA = iAs[r]; iB = iBs[r]; }
            else inv_r2(r, iA, iB, R, !late_b);
            const float2 dy = make_float2(s.dy[r], s.dy[r]);
            constexpr int ORD = (TUNE >> 1) & 3;
            if (late_b) { // pair A first, then 1/r^2 of pair B and its accumulations
                if (ORD & 1) { syA[r] = __ffma2_rn(dy, iA, syA[r]); sxA[r] = __ffma2_rn(s.dxA, iA, sxA[r]); }
                else { sxA[r] = __ffma2_rn(s.dxA, iA, sxA[r]); syA[r] = __ffma2_rn(dy, iA, syA[r]); }
                iB = __fmul2_rn(R, s.r2A[r]);
                if (ORD & 2) { syB[r] = __ffma2_rn(dy, iB, syB[r]); sxB[r] = __ffma2_rn(s.dxB, iB, sxB[r]); }
                else { sxB[r] = __ffma2_rn(s.dxB, iB, sxB[r]); syB[r] = __ffma2_rn(dy, iB, syB[r]); }
            } else if (ORD == 0) {
                sxA[r] = __ffma2_rn(s.dxA, iA, sxA[r]);
                sxB[r] = __ffma2_rn(s.dxB, iB, sxB[r]);
                syA[r] = __ffma2_rn(dy, iA, syA[r]);
                syB[r] = __ffma2_rn(dy, iB, syB[r]);
            } else if (ORD == 1) {
                sxA[r] = __ffma2_rn(s.dxA, iA, sxA[r]);
                syA[r] = __ffma2_rn(dy, iA, syA[r]);
                sxB[r] = __ffma2_rn(s.dxB, iB, sxB[r]);
                syB[r] = __ffma2_rn(dy, iB, syB[r]);
            } else if (ORD == 2) {
                syA[r] = __ffma2_rn(dy, iA, syA[r]);
                syB[r] = __ffma2_rn(dy, iB, syB[r]);
                sxA[r] = __ffma2_rn(s.dxA, iA, sxA[r]);
                sxB[r] = __ffma2_rn(s.dxB, iB, sxB[r]);
            } else {
                syA[r] = __ffma2_rn(dy, iA, syA[r]);
                sxA[r] = __ffma2_rn(s.dxA, iA, sxA[r]);
                syB[r] = __ffma2_rn(dy, iB, syB[r]);
                sxB[r] = __ffma2_rn(s.dxB, iB, sxB[r]);
            }
        }
    };

    int buf = 0;
    for (int base = lb; base < le; base += kChunk) {
        const bool more = base + kChunk < le;
        if (more) fetch(base + kChunk);
        const int cnt = min(kChunk, le - base);
        const int cntp = (cnt + 1) & ~1;
        const float4 *ls = lens_s[buf];
        const float *ms = mass_s[buf];
        auto mass_of = [&](int k) { return MASS ? ms[k] : 1.f; };
        PipeRegs<RY> a, b; // a: even lenses of the chunk, b: odd lenses
        const std::integral_constant<bool, false> even;
        const std::integral_constant<bool, true> odd;
        stage1(even, ls[0], mass_of(0), a);
        if (TUNE & 1) stage1(odd, ls[1], mass_of(1), b);
        for (int k0 = 0; k0 < cntp; k0 += KF) {
            const int kend = min(k0 + KF, cntp);
#pragma unroll 1
            for (int k = k0; k < kend; k += 2) {
                if (TUNE & 1) { // lenses k, k+1 are staged; stage k+2, k+3 (<= cntp + 1: a padding lens) behind their use
                    stage2(even, a);
                    stage1(even, ls[k + 2], mass_of(k + 2), a);
                    stage2(odd, b);
                    stage1(odd, ls[k + 3], mass_of(k + 3), b);
                } else {
                    stage1(odd, ls[k + 1], mass_of(k + 1), b);
                    stage2(even, a);
                    stage1(even, ls[k + 2], mass_of(k + 2), a);
                    stage2(odd, b);
                }
            }
#pragma unroll
            for (int r = 0; r < RY; ++r) {
                Sx[r][0] += (double)sxA[r].x; Sx[r][1] += (double)sxA[r].y;
                Sx[r][2] += (double)sxB[r].x; Sx[r][3] += (double)sxB[r].y;
                Sy[r][0] += (double)syA[r].x; Sy[r][1] += (double)syA[r].y;
                Sy[r][2] += (double)syB[r].x; Sy[r][3] += (double)syB[r].y;
                sxA[r] = make_float2(0.f, 0.f); sxB[r] = sxA[r]; syA[r] = sxA[r]; syB[r] = sxA[r];
            }
        }
        if (more) stage(base + kChunk, buf ^ 1);
        __syncthreads();
        buf ^= 1;
    }
    if (CAPTURE && p.partial) { store_partials<RX, RY, WARPS>(p, t, lane, warp, Sx, Sy); return; }
    finish_tile<RX, RY, CAPTURE, WARPS>(p, ti, tj, t, lane, warp, Sx, Sy, cta_count);
}


// ---------------------------------------------------------------------------------------
// Random ray positions (ML_RAYS_RANDOM: GPU-D's own ray generation; R17), FP32 modes.
//
// Every ray starts at its own point of its grid cell, so no column / row difference is shared between the rays
// of a thread and the regular-grid kernel above does not apply.  The rest of its design does: a thread owns
// 4 x 2 rays as packed pairs along axis 1 (columns 0,1 = "A", 2,3 = "B"), every FP32 instruction on the rays is a
// packed FADD2 / FMUL2 / FFMA2, one reciprocal serves two interactions (R = 1/(r2A r2B), 1/r2A = R r2B,
// 1/r2B = R r2A) and the loop is software-pipelined over lenses.  Per lens and row: 4 FADD2 (dx, dy of A and B),
// 4 FFMA2 (r^2 = dy dy + (dx dx + 2^-80)), 3 FMUL2, 2 MUFU.RCP, 4 FFMA2 = 15 packed instructions for 4 interactions
// (7.5 FMA-pipe lane-cycles per interaction against 5.25 on the regular grid: the price of per-ray offsets).
// The two 53-bit uniforms of a ray are drawn once (Philox-4x32-10, counter = ray id) and kept in shared memory for
// the epilogue, which needs them again for the fp64 position.  Summation order and padding as in shoot_kernel_pipe.
template <int RY> struct RPipeRegs {
    float m;
    float2 dxA[RY], dxB[RY], dyA[RY], dyB[RY];
    float2 r2A[RY], r2B[RY]; // r^2
    float2 R[RY], Rb[RY];    // shared rows: R = 1/(r2A r2B); own-reciprocal rows: R = 1/r2A, Rb = 1/r2B
};

constexpr int kRandWarps = 8, kRandRY = 2;
constexpr size_t rpipe_smem_bytes(bool mass)
{
    return 2 * (kChunk + 2) * sizeof(float4) + (size_t)4 * kRandRY * kRandWarps * 32 * sizeof(double2) +
           (mass ? 2 * (kChunk + 2) * sizeof(float) : 0);
}

// OWN = 1: on the last row of every odd lens the two ray pairs take their own reciprocals (4 MUFU, no FMUL2) instead
// of the shared one (2 MUFU + 3 FMUL2): the XU pipe has room for more reciprocals (48 % busy with everything shared) and
// the FMA pipe, which bounds the loop, loses 3 of its 60 packed instructions per lens pair.
// OWN = 2: the same on the last row of every lens.  TUNE: source-order knobs as in shoot_kernel_pipe (bits 0-1: order
// of the four accumulations of a row; bit 2 / bit 3: rows in reverse order in stage 2 / stage 1).
template <int KF, int MINB, bool CAPTURE, bool MASS = false, bool NEWTON = false, int OWN = 1, int TUNE = 0>
__global__ void __launch_bounds__(kRandWarps * 32, MINB) shoot_kernel_rpipe(const ShootParams p)
{
    constexpr int RX = 4, RY = kRandRY, WARPS = kRandWarps;
    constexpr int THREADS = WARPS * 32;
    constexpr int TW = 32 * RX;
    constexpr int TH = WARPS * RY;
    static_assert(kChunk % KF == 0 && KF % 2 == 0, "flush groups must tile a chunk");
    constexpr int PER_THREAD = kChunk / THREADS;

    extern __shared__ __align__(16) unsigned char rp_smem[];
    float4 *lens_s = reinterpret_cast<float4 *>(rp_smem);                                      // [2][kChunk + 2]
    double2 *uv_s = reinterpret_cast<double2 *>(rp_smem + 2 * (kChunk + 2) * sizeof(float4)); // [RX*RY][THREADS]
    float *mass_s = reinterpret_cast<float *>(rp_smem + 2 * (kChunk + 2) * sizeof(float4) +
                                              (size_t)RX * RY * THREADS * sizeof(double2));   // [2][kChunk + 2]
    __shared__ unsigned int cta_count[3];

    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    long long t, ti, tj;
    which_tile<CAPTURE>(p, t, ti, tj);
    int lb, le; // this CTA's lens range: [0, n_lens) except in split capture launches
    lens_range<CAPTURE>(p, lb, le);
    if (threadIdx.x < 3) cta_count[threadIdx.x] = 0;
    const float padc = NEWTON ? -1e9f : -1e15f; // see shoot_kernel_pipe
    if (threadIdx.x < 4) lens_s[(threadIdx.x >> 1) * (kChunk + 2) + kChunk + (threadIdx.x & 1)] = make_float4(padc, padc, padc, padc);
    if (MASS && threadIdx.x < 4) mass_s[(threadIdx.x >> 1) * (kChunk + 2) + kChunk + (threadIdx.x & 1)] = 0.f;

    // ---- a2: tile centre (fp64) and every ray's own offset from it
    const double cx = ((double)(ti * TW) + 0.5 * (TW - 1) - p.half1) * p.delta;
    const double cy = ((double)(tj * TH) + 0.5 * (TH - 1) - p.half2) * p.delta;
    float2 oxA[RY], oxB[RY], oyA[RY], oyB[RY];
#pragma unroll
    for (int r = 0; r < RY; ++r) {
        float ox[RX], oy[RX];
#pragma unroll
        for (int c = 0; c < RX; ++c) {
            const unsigned long long i = (unsigned long long)(ti * TW + lane * RX + c), j = (unsigned long long)(tj * TH + warp * RY + r);
            double2 w;
            ray_uniforms(j * (unsigned long long)p.n1 + i, p.ray_seed, w.x, w.y);
            uv_s[(r * RX + c) * THREADS + threadIdx.x] = w;
            ox[c] = (float)(((double)(lane * RX + c) + w.x - 0.5 * TW) * p.delta);
            oy[c] = (float)(((double)(warp * RY + r) + w.y - 0.5 * TH) * p.delta);
        }
        oxA[r] = make_float2(ox[0], ox[1]); oxB[r] = make_float2(ox[2], ox[3]);
        oyA[r] = make_float2(oy[0], oy[1]); oyB[r] = make_float2(oy[2], oy[3]);
    }

    double Sx[RY][RX], Sy[RY][RX];
    float2 sxA[RY], sxB[RY], syA[RY], syB[RY];
#pragma unroll
    for (int r = 0; r < RY; ++r) {
#pragma unroll
        for (int c = 0; c < RX; ++c) { Sx[r][c] = 0.0; Sy[r][c] = 0.0; }
        sxA[r] = make_float2(0.f, 0.f); sxB[r] = sxA[r]; syA[r] = sxA[r]; syB[r] = sxA[r];
    }

    // ---- a1: lens staging (as in shoot_kernel_pipe)
    double2 pre[PER_THREAD];
    double pre_m[MASS ? PER_THREAD : 1];
    auto fetch = [&](int base) {
#pragma unroll
        for (int q = 0; q < PER_THREAD; ++q) {
            const int k = base + q * THREADS + threadIdx.x;
            if (k < le) {
                pre[q] = __ldg(&p.lens[k]);
                if (MASS) pre_m[q] = __ldg(&p.mass[k]);
            }
        }
    };
    auto stage = [&](int base, int buf) {
#pragma unroll
        for (int q = 0; q < PER_THREAD; ++q) {
            const int k = base + q * THREADS + threadIdx.x;
            float nx = padc, ny = padc, m = 0.f;
            if (k < le) {
                nx = -(float)(pre[q].x - cx);
                ny = -(float)(pre[q].y - cy);
                if (MASS) m = (float)pre_m[q];
            }
            lens_s[buf * (kChunk + 2) + q * THREADS + threadIdx.x] = make_float4(nx, nx, ny, ny);
            if (MASS) mass_s[buf * (kChunk + 2) + q * THREADS + threadIdx.x] = m;
        }
    };
    fetch(lb);
    stage(lb, 0);
    __syncthreads();

    // ---- a3: all-pairs deflection sum
    const float2 eps2 = make_float2(0x1p-80f, 0x1p-80f);
    auto stage1 = [&](auto odd, const float4 l, const float m, RPipeRegs<RY> &s) {
        const float2 nlx = make_float2(l.x, l.y), nly = make_float2(l.z, l.w);
        s.m = m;
#pragma unroll
        for (int rr = 0; rr < RY; ++rr) {
            const int r = (TUNE & 8) ? RY - 1 - rr : rr;
            s.dxA[r] = __fadd2_rn(oxA[r], nlx);
            s.dxB[r] = __fadd2_rn(oxB[r], nlx);
            s.dyA[r] = __fadd2_rn(oyA[r], nly);
            s.dyB[r] = __fadd2_rn(oyB[r], nly);
            s.r2A[r] = __ffma2_rn(s.dyA[r], s.dyA[r], __ffma2_rn(s.dxA[r], s.dxA[r], eps2));
            s.r2B[r] = __ffma2_rn(s.dyB[r], s.dyB[r], __ffma2_rn(s.dxB[r], s.dxB[r], eps2));
            if (r == RY - 1 && (OWN == 2 || (OWN == 1 && decltype(odd)::value))) {
                s.R[r].x = rcp_approx(s.r2A[r].x); s.R[r].y = rcp_approx(s.r2A[r].y);
                s.Rb[r].x = rcp_approx(s.r2B[r].x); s.Rb[r].y = rcp_approx(s.r2B[r].y);
            } else {
                const float2 P = __fmul2_rn(s.r2A[r], s.r2B[r]);
                s.R[r].x = rcp_approx(P.x);
                s.R[r].y = rcp_approx(P.y);
            }
        }
    };
    auto newton = [](float2 a, float2 R) { // one Newton-Raphson step: R <- R + R (1 - a R)
        const float2 e = __ffma2_rn(make_float2(-a.x, -a.y), R, make_float2(1.f, 1.f));
        return __ffma2_rn(R, e, R);
    };
    auto stage2 = [&](auto odd, const RPipeRegs<RY> &s) {
#pragma unroll
        for (int rr = 0; rr < RY; ++rr) {
            const int r = (TUNE & 4) ? RY - 1 - rr : rr;
            float2 iA, iB;
            if (r == RY - 1 && (OWN == 2 || (OWN == 1 && decltype(odd)::value))) {
                iA = s.R[r];
                iB = s.Rb[r];
                if (NEWTON) { iA = newton(s.r2A[r], iA); iB = newton(s.r2B[r], iB); }
                if (MASS) { iA = __fmul2_rn(iA, make_float2(s.m, s.m)); iB = __fmul2_rn(iB, make_float2(s.m, s.m)); }
            } else {
                float2 R = s.R[r];
                if (NEWTON) R = newton(__fmul2_rn(s.r2A[r], s.r2B[r]), R); // on the shared reciprocal, P = r2A r2B
                if (MASS) R = __fmul2_rn(R, make_float2(s.m, s.m)); // m_i / (r2A r2B)
                iA = __fmul2_rn(R, s.r2B[r]);
                iB = __fmul2_rn(R, s.r2A[r]);
            }
            constexpr int ORD = TUNE & 3;
            if (ORD == 0) {
                sxA[r] = __ffma2_rn(s.dxA[r], iA, sxA[r]);
                syA[r] = __ffma2_rn(s.dyA[r], iA, syA[r]);
                sxB[r] = __ffma2_rn(s.dxB[r], iB, sxB[r]);
                syB[r] = __ffma2_rn(s.dyB[r], iB, syB[r]);
            } else if (ORD == 1) {
                sxA[r] = __ffma2_rn(s.dxA[r], iA, sxA[r]);
                sxB[r] = __ffma2_rn(s.dxB[r], iB, sxB[r]);
                syA[r] = __ffma2_rn(s.dyA[r], iA, syA[r]);
                syB[r] = __ffma2_rn(s.dyB[r], iB, syB[r]);
            } else if (ORD == 2) {
                syA[r] = __ffma2_rn(s.dyA[r], iA, syA[r]);
                syB[r] = __ffma2_rn(s.dyB[r], iB, syB[r]);
                sxA[r] = __ffma2_rn(s.dxA[r], iA, sxA[r]);
                sxB[r] = __ffma2_rn(s.dxB[r], iB, sxB[r]);
            } else {
                syA[r] = __ffma2_rn(s.dyA[r], iA, syA[r]);
                sxA[r] = __ffma2_rn(s.dxA[r], iA, sxA[r]);
                syB[r] = __ffma2_rn(s.dyB[r], iB, syB[r]);
                sxB[r] = __ffma2_rn(s.dxB[r], iB, sxB[r]);
            }
        }
    };

    int buf = 0;
    for (int base = lb; base < le; base += kChunk) {
        const bool more = base + kChunk < le;
        if (more) fetch(base + kChunk);
        const int cnt = min(kChunk, le - base);
        const int cntp = (cnt + 1) & ~1;
        const float4 *ls = lens_s + buf * (kChunk + 2);
        const float *ms = mass_s + buf * (kChunk + 2);
        auto mass_of = [&](int k) { return MASS ? ms[k] : 1.f; };
        RPipeRegs<RY> a, b;
        const std::integral_constant<bool, false> even;
        const std::integral_constant<bool, true> odd;
        stage1(even, ls[0], mass_of(0), a);
        for (int k0 = 0; k0 < cntp; k0 += KF) {
            const int kend = min(k0 + KF, cntp);
#pragma unroll 1
            for (int k = k0; k < kend; k += 2) {
                stage1(odd, ls[k + 1], mass_of(k + 1), b);
                stage2(even, a);
                stage1(even, ls[k + 2], mass_of(k + 2), a);
                stage2(odd, b);
            }
#pragma unroll
            for (int r = 0; r < RY; ++r) {
                Sx[r][0] += (double)sxA[r].x; Sx[r][1] += (double)sxA[r].y;
                Sx[r][2] += (double)sxB[r].x; Sx[r][3] += (double)sxB[r].y;
                Sy[r][0] += (double)syA[r].x; Sy[r][1] += (double)syA[r].y;
                Sy[r][2] += (double)syB[r].x; Sy[r][3] += (double)syB[r].y;
                sxA[r] = make_float2(0.f, 0.f); sxB[r] = sxA[r]; syA[r] = sxA[r]; syB[r] = sxA[r];
            }
        }
        if (more) stage(base + kChunk, buf ^ 1);
        __syncthreads();
        buf ^= 1;
    }
    if (CAPTURE && p.partial) { store_partials<RX, RY, WARPS>(p, t, lane, warp, Sx, Sy); return; }
    finish_tile<RX, RY, CAPTURE, WARPS, true, true>(p, ti, tj, t, lane, warp, Sx, Sy, cta_count, uv_s);
}

// ---------------------------------------------------------------------------------------
// Uniformly random ray positions over the whole shooting rectangle (ML_RAYS_UNIFORM: the literal GPU-D ray
// generation, "a batch of 2^17 random ray positions" PAPER.md:131, "shot from random positions in the shooting grid ...
// This will introduce Poisson noise" PAPER.md:167; reading R20).
//
// Ray id = j n1 + i only numbers the rays: its position is ((u1 n1 - n1/2) delta, (u2 n2 - n2/2) delta) with the two
// uniforms of Philox-4x32-10(counter = id, key = seed).  FP32 terms need coordinates local to a small patch of the image
// plane, so the rays are first sorted by position: uniform_scatter_kernel draws every ray of the requested id range and
// appends its handle to the list of the bucket (kUniBW x kUniBH grid cells) it falls in; shoot_kernel_upipe then shoots
// one CTA per 1024 list entries with the bucket centre as the local origin.  The list order depends on the order of the
// atomics, the results do not: the arithmetic of a ray involves no other ray.  That is why the shared reciprocal pairs two
// LENSES of one ray here, R = 1/(r2_k r2_k+1), 1/r2_k = R r2_k+1, 1/r2_k+1 = R r2_k (k even), not two rays of one lens as
// in the kernels above; every second lens pair takes its own reciprocals instead (4 MUFU, no FMUL2: the XU pipe has room,
// the FMA pipe is the bound), for every ray alike.  A thread owns 8 list entries as two "rows" of two packed pairs;
// per row and lens pair: 8 FADD2, 8 FFMA2 (r^2), 3 FMUL2 + 2 x 2 MUFU (or 8 MUFU), 8 FFMA2: the instruction mix of
// shoot_kernel_rpipe.  Lenses are added in index order, FP32 partial sums over KF lenses, fp64 accumulators, as everywhere.
struct ScatterParams {
    ShootParams sp;        // i0, j0, n1, n1d, n2d, ray_seed, list_w, probe_ids, bucket_nx, bucket_row0, bucket_cap
    long long n_handles;   // rays to scatter: handles 0 .. n_handles - 1
    long long bucket_row1; // bucket rows [bucket_row0, bucket_row1) are kept by this pass
    unsigned int *fill;    // [rows x bucket_nx], zeroed by the caller
    unsigned long long *list;
};

// Each block takes runs of kScatterRun consecutive handles; a thread steps through its run 256 handles at a time and
// carries (row, column) of the region along, so the handle -> ray id division happens once per run.  The bucket is
// taken from the integer part of u n (u as the 64-bit fraction c0:c1 / 2^64): within 1e-10 of a grid cell of the
// double-precision position the shoot kernel uses -- a ray that close to a bucket edge may sit in either bucket.
constexpr int kScatterRun = 256 * 16;
__global__ void __launch_bounds__(256) uniform_scatter_kernel(const ScatterParams q)
{
    const unsigned long long n1 = (unsigned long long)q.sp.n1, n2 = (unsigned long long)q.sp.n2d;
    // list tails are written 8 bytes at a time: ask the L2 to keep them until their sectors are full
    unsigned long long keep;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(keep));
    for (long long run = (long long)blockIdx.x * kScatterRun; run < q.n_handles; run += (long long)gridDim.x * kScatterRun) {
        long long h = run + threadIdx.x;
        const long long end = min(run + (long long)kScatterRun, q.n_handles);
        long long jj = 0, ii = 0;
        if (!q.sp.probe_ids && h < end) { jj = h / q.sp.list_w; ii = h - jj * q.sp.list_w; }
        for (; h < end; h += 256) {
            const unsigned long long id = q.sp.probe_ids ? (unsigned long long)q.sp.probe_ids[h]
                                                         : (unsigned long long)((q.sp.j0 + jj) * q.sp.n1 + (q.sp.i0 + ii));
            unsigned int c0, c1, c2, c3;
            ray_words(id, q.sp.ray_seed, c0, c1, c2, c3);
            const long long bx = (long long)(__umul64hi(((unsigned long long)c0 << 32) | c1, n1) / kUniBW);
            const long long by = (long long)(__umul64hi(((unsigned long long)c2 << 32) | c3, n2) / kUniBH);
            if (by >= q.sp.bucket_row0 && by < q.bucket_row1) {
                const long long b = (by - q.sp.bucket_row0) * q.sp.bucket_nx + bx;
                const unsigned int slot = atomicAdd(&q.fill[b], 1u);
                if (slot < q.sp.bucket_cap)
                    asm volatile("st.global.L2::cache_hint.u64 [%0], %1, %2;" ::"l"(q.list + (size_t)b * q.sp.bucket_cap + slot),
                                 "l"((unsigned long long)h), "l"(keep)
                                 : "memory");
            }
            ii += 256;
            while (ii >= q.sp.list_w && !q.sp.probe_ids) { ii -= q.sp.list_w; ++jj; }
        }
    }
}

template <int RY> struct UPipeRegs {   // one row of a thread (two packed ray pairs A, B) x one lens pair (lenses 0, 1)
    float m[2];
    float2 dx[2][2], dy[2][2]; // [lens][ray pair]
    float2 r2[2][2];           // r^2; own-reciprocal pairs: 1/r^2
    float2 R[2];               // shared pairs: 1/(r2[0] r2[1]) per ray pair
};

// TUNE: source-order knobs as in the kernels above (same operations, operands and rounding; another ptxas schedule).
// bit 0: the accumulations of a ray pair as sx, sx, sy, sy instead of sx, sy, sx, sy; bit 1: ray pair B before A in
// stage 2; bit 2: stage 1 forms the differences of both lenses before the first r^2; bit 3: ray pair B before A in stage 1's
// reciprocals; bit 4: in stage 2 both 1/r^2 pairs of a row before the first accumulation.
template <int KF, int MINB, bool CAPTURE, bool MASS = false, bool NEWTON = false, int TUNE = 0>
__global__ void __launch_bounds__(kUniWarps * 32, MINB) shoot_kernel_upipe(const ShootParams p)
{
    constexpr int RX = 4, RY = kRandRY, WARPS = kUniWarps;
    constexpr int THREADS = WARPS * 32;
    constexpr int SLOTS = THREADS * RX * RY; // list entries per CTA
    static_assert(kChunk % KF == 0 && KF % 4 == 0, "flush groups must tile a chunk in double lens pairs");
    static_assert(RY == 2, "two rows per thread");
    constexpr int PER_THREAD = kChunk / THREADS;

    extern __shared__ __align__(16) unsigned char rp_smem[];
    float4 *lens_s = reinterpret_cast<float4 *>(rp_smem);                                      // [2][kChunk + 4]
    double2 *uv_s = reinterpret_cast<double2 *>(rp_smem + 2 * (kChunk + 4) * sizeof(float4)); // [RX*RY][THREADS]
    float *mass_s = reinterpret_cast<float *>(rp_smem + 2 * (kChunk + 4) * sizeof(float4) +
                                              (size_t)RX * RY * THREADS * sizeof(double2));   // [2][kChunk + 4]
    __shared__ unsigned int cta_count[3];

    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    // ---- which slice of which bucket list
    const long long b = (long long)blockIdx.x;
    const unsigned int filled = min(p.bucket_fill[b], p.bucket_cap);
    const long long first = (long long)blockIdx.y * SLOTS;
    if (first >= (long long)filled) return; // (whole CTA: before any barrier)
    const int n_valid = (int)min((long long)SLOTS, (long long)filled - first);
    const unsigned long long *handles = p.ray_list + (size_t)b * p.bucket_cap + first;
    int lb, le;
    lens_range<false>(p, lb, le);
    if (threadIdx.x < 3) cta_count[threadIdx.x] = 0;
    const float padc = -1e9f; // a padding lens must keep the shared product finite (see shoot_kernel_pipe, NEWTON)
    if (threadIdx.x < 8) lens_s[(threadIdx.x >> 2) * (kChunk + 4) + kChunk + (threadIdx.x & 3)] = make_float4(padc, padc, padc, padc);
    if (MASS && threadIdx.x < 8) mass_s[(threadIdx.x >> 2) * (kChunk + 4) + kChunk + (threadIdx.x & 3)] = 0.f;

    // ---- a2: bucket centre (grid cells, fp64) and every listed ray's offset from it
    const long long bxi = b % p.bucket_nx, byi = p.bucket_row0 + b / p.bucket_nx;
    const double ccx = (double)(bxi * kUniBW) + 0.5 * kUniBW, ccy = (double)(byi * kUniBH) + 0.5 * kUniBH;
    const double cx = (ccx - 0.5 * p.n1d) * p.delta, cy = (ccy - 0.5 * p.n2d) * p.delta;
    float2 oxA[RY], oxB[RY], oyA[RY], oyB[RY];
#pragma unroll
    for (int r = 0; r < RY; ++r) {
        float ox[RX], oy[RX];
#pragma unroll
        for (int c = 0; c < RX; ++c) {
            const int slot = (r * RX + c) * THREADS + (int)threadIdx.x;
            double2 w = make_double2(0.5, 0.5);
            ox[c] = 0.f; oy[c] = 0.f; // an empty slot shoots a ray from the bucket centre and throws it away
            if (slot < n_valid) {
                ray_uniforms(uniform_ray_id(p, handles[slot]), p.ray_seed, w.x, w.y);
                ox[c] = (float)((__dmul_rn(w.x, p.n1d) - ccx) * p.delta);
                oy[c] = (float)((__dmul_rn(w.y, p.n2d) - ccy) * p.delta);
            }
            uv_s[slot] = w;
        }
        oxA[r] = make_float2(ox[0], ox[1]); oxB[r] = make_float2(ox[2], ox[3]);
        oyA[r] = make_float2(oy[0], oy[1]); oyB[r] = make_float2(oy[2], oy[3]);
    }

    double Sx[RY][RX], Sy[RY][RX];
    float2 sxA[RY], sxB[RY], syA[RY], syB[RY];
#pragma unroll
    for (int r = 0; r < RY; ++r) {
#pragma unroll
        for (int c = 0; c < RX; ++c) { Sx[r][c] = 0.0; Sy[r][c] = 0.0; }
        sxA[r] = make_float2(0.f, 0.f); sxB[r] = sxA[r]; syA[r] = sxA[r]; syB[r] = sxA[r];
    }

    // ---- a1: lens staging (as in shoot_kernel_pipe)
    double2 pre[PER_THREAD];
    double pre_m[MASS ? PER_THREAD : 1];
    auto fetch = [&](int base) {
#pragma unroll
        for (int q = 0; q < PER_THREAD; ++q) {
            const int k = base + q * THREADS + threadIdx.x;
            if (k < le) {
                pre[q] = __ldg(&p.lens[k]);
                if (MASS) pre_m[q] = __ldg(&p.mass[k]);
            }
        }
    };
    auto stage = [&](int base, int buf) {
#pragma unroll
        for (int q = 0; q < PER_THREAD; ++q) {
            const int k = base + q * THREADS + threadIdx.x;
            float nx = padc, ny = padc, m = 0.f;
            if (k < le) {
                nx = -(float)(pre[q].x - cx);
                ny = -(float)(pre[q].y - cy);
                if (MASS) m = (float)pre_m[q];
            }
            lens_s[buf * (kChunk + 4) + q * THREADS + threadIdx.x] = make_float4(nx, nx, ny, ny);
            if (MASS) mass_s[buf * (kChunk + 4) + q * THREADS + threadIdx.x] = m;
        }
    };
    fetch(lb);
    stage(lb, 0);
    __syncthreads();

    // ---- a3: all-pairs deflection sum, two lenses at a time
    const float2 eps2 = make_float2(0x1p-80f, 0x1p-80f);
    auto newton = [](float2 a, float2 R) { // one Newton-Raphson step: R <- R + R (1 - a R)
        const float2 e = __ffma2_rn(make_float2(-a.x, -a.y), R, make_float2(1.f, 1.f));
        return __ffma2_rn(R, e, R);
    };
    // stage 1 of (row r, lens pair l0 l1): differences, r^2, reciprocals (own: of each r^2; shared: of the products)
    auto stage1 = [&](auto own, int r, const float4 l0, const float4 l1, const float m0, const float m1, UPipeRegs<RY> &s) {
        s.m[0] = m0; s.m[1] = m1;
        auto diffs = [&](int L) {
            const float4 l = L ? l1 : l0;
            const float2 nlx = make_float2(l.x, l.y), nly = make_float2(l.z, l.w);
            s.dx[L][0] = __fadd2_rn(oxA[r], nlx); s.dx[L][1] = __fadd2_rn(oxB[r], nlx);
            s.dy[L][0] = __fadd2_rn(oyA[r], nly); s.dy[L][1] = __fadd2_rn(oyB[r], nly);
        };
        auto squares = [&](int L) {
#pragma unroll
            for (int X = 0; X < 2; ++X) s.r2[L][X] = __ffma2_rn(s.dy[L][X], s.dy[L][X], __ffma2_rn(s.dx[L][X], s.dx[L][X], eps2));
        };
        if (TUNE & 4) { diffs(0); diffs(1); squares(0); squares(1); }
        else { diffs(0); squares(0); diffs(1); squares(1); }
#pragma unroll
        for (int XX = 0; XX < 2; ++XX) {
            const int X = (TUNE & 8) ? 1 - XX : XX;
            if (decltype(own)::value) {
#pragma unroll
                for (int L = 0; L < 2; ++L) {
                    float2 i;
                    i.x = rcp_approx(s.r2[L][X].x); i.y = rcp_approx(s.r2[L][X].y);
                    if (NEWTON) i = newton(s.r2[L][X], i);
                    s.r2[L][X] = i;
                }
            } else {
                const float2 P = __fmul2_rn(s.r2[0][X], s.r2[1][X]);
                s.R[X].x = rcp_approx(P.x); s.R[X].y = rcp_approx(P.y);
            }
        }
    };
    // stage 2: 1/r^2 of both lenses and the accumulations, lens 0 before lens 1 (index order)
    auto stage2 = [&](auto own, int r, const UPipeRegs<RY> &s) {
        float2 i0s[2], i1s[2];
        auto inv = [&](int X, float2 &i0, float2 &i1) {
            if (decltype(own)::value) {
                i0 = s.r2[0][X]; i1 = s.r2[1][X];
            } else {
                float2 R = s.R[X];
                if (NEWTON) R = newton(__fmul2_rn(s.r2[0][X], s.r2[1][X]), R);
                i0 = __fmul2_rn(R, s.r2[1][X]);
                i1 = __fmul2_rn(R, s.r2[0][X]);
            }
            if (MASS) { i0 = __fmul2_rn(i0, make_float2(s.m[0], s.m[0])); i1 = __fmul2_rn(i1, make_float2(s.m[1], s.m[1])); }
        };
        if (TUNE & 16) { inv(0, i0s[0], i1s[0]); inv(1, i0s[1], i1s[1]); }
#pragma unroll
        for (int XX = 0; XX < 2; ++XX) {
            const int X = (TUNE & 2) ? 1 - XX : XX;
            float2 i0, i1;
            if (TUNE & 16) { i0 = i0s[X]; i1 = i1s[X]; }
            else inv(X, i0, i1);
            float2 &sx = X ? sxB[r] : sxA[r], &sy = X ? syB[r] : syA[r];
            if (TUNE & 1) {
                sx = __ffma2_rn(s.dx[0][X], i0, sx);
                sx = __ffma2_rn(s.dx[1][X], i1, sx);
                sy = __ffma2_rn(s.dy[0][X], i0, sy);
                sy = __ffma2_rn(s.dy[1][X], i1, sy);
            } else {
                sx = __ffma2_rn(s.dx[0][X], i0, sx);
                sy = __ffma2_rn(s.dy[0][X], i0, sy);
                sx = __ffma2_rn(s.dx[1][X], i1, sx);
                sy = __ffma2_rn(s.dy[1][X], i1, sy);
            }
        }
    };

    int buf = 0;
    for (int base = lb; base < le; base += kChunk) {
        const bool more = base + kChunk < le;
        if (more) fetch(base + kChunk);
        const int cnt = min(kChunk, le - base);
        const int cntp = (cnt + 3) & ~3; // whole double pairs: up to three padding lenses at the very end
        const float4 *ls = lens_s + buf * (kChunk + 4);
        const float *ms = mass_s + buf * (kChunk + 4);
        auto mass_of = [&](int k) { return MASS ? ms[k] : 1.f; };
        UPipeRegs<RY> a, c;
        const std::integral_constant<bool, false> shared;
        const std::integral_constant<bool, true> own;
        stage1(shared, 0, ls[0], ls[1], mass_of(0), mass_of(1), a);
        for (int k0 = 0; k0 < cntp; k0 += KF) {
            const int kend = min(k0 + KF, cntp);
#pragma unroll 1
            for (int k = k0; k < kend; k += 4) { // lens pairs (k, k+1): shared reciprocals; (k+2, k+3): own
                stage1(shared, 1, ls[k], ls[k + 1], mass_of(k), mass_of(k + 1), c);
                stage2(shared, 0, a);
                stage1(own, 0, ls[k + 2], ls[k + 3], mass_of(k + 2), mass_of(k + 3), a);
                stage2(shared, 1, c);
                stage1(own, 1, ls[k + 2], ls[k + 3], mass_of(k + 2), mass_of(k + 3), c);
                stage2(own, 0, a);
                stage1(shared, 0, ls[k + 4], ls[k + 5], mass_of(k + 4), mass_of(k + 5), a); // (<= cntp + 1 <= kChunk + 3)
                stage2(own, 1, c);
            }
#pragma unroll
            for (int r = 0; r < RY; ++r) {
                Sx[r][0] += (double)sxA[r].x; Sx[r][1] += (double)sxA[r].y;
                Sx[r][2] += (double)sxB[r].x; Sx[r][3] += (double)sxB[r].y;
                Sy[r][0] += (double)syA[r].x; Sy[r][1] += (double)syA[r].y;
                Sy[r][2] += (double)syB[r].x; Sy[r][3] += (double)syB[r].y;
                sxA[r] = make_float2(0.f, 0.f); sxB[r] = sxA[r]; syA[r] = sxA[r]; syB[r] = sxA[r];
            }
        }
        if (more) stage(base + kChunk, buf ^ 1);
        __syncthreads();
        buf ^= 1;
    }
    finish_tile<RX, RY, CAPTURE, WARPS, true, true, true>(p, 0, 0, 0, lane, warp, Sx, Sy, cta_count, uv_s, n_valid, handles);
}

constexpr size_t upipe_smem_bytes(bool mass)
{
    return 2 * (kChunk + 4) * sizeof(float4) + (size_t)4 * kRandRY * kUniWarps * 32 * sizeof(double2) +
           (mass ? 2 * (kChunk + 4) * sizeof(float) : 0);
}

} // namespace mlb200
