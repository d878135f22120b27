/*
 * microlens_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU restatement of direct inverse ray-shooting, written from
 * the paper (Bate, Fluke, Barsdell, Garsden & Lewis 2010, /root/reference/PAPER.md)
 * so that the CUDA library can be checked against something that is not itself.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference legs may build, load or call this file.  It shares no code, header,
 * constant or helper with paper_1005_5198_b200/ and is never imported by it.
 *
 * The direct method is the definition ("includes contributions from all lenses
 * without approximations"), so each function below is that
 * definition written out, in the paper's order, with no blocking, fusion or
 * reordering.  OpenMP only splits the independent rays over threads.
 *
 * What each function follows:
 *   ora_derive          PAPER.md:56-60 eq.(5), :275-285 eq.(11), :287-292 eq.(12),
 *                       and the concrete rules of BASELINE.json:configs[0]
 *                       (readings R1-R4, R7 in DESIGN.md).
 *   ora_ray_x           BASELINE.json:configs[0] "regular grid over the rectangle";
 *                       PAPER.md:167 (regular grid).  Readings R7, R8.  ray_mode 1: GPU-D's random
 *                       ray positions, one per grid cell (reading R17), drawn
 *                       with Philox-4x32-10 keyed by the seed, counter = ray id.  ray_mode 2: the
 *                       same draw spread over the WHOLE shooting rectangle -- every ray an independent
 *                       uniform point of it, the literal reading of PAPER.md:131, :167 ("random
 *                       positions in the shooting grid ... will introduce Poisson noise"; reading R20).
 *   ora_lens_equation   PAPER.md:49-54 eq.(4) with m_i = 1; the *_m variants take
 *                       the masses m_i of eq.(4).
 *   ora_pixel           PAPER.md:45-47 (rays "mapped to a grid of pixels in the
 *                       source plane"); readings R10, R11.
 *   ora_shoot_region    PAPER.md:45-47 eq.(3): N_ij = number of rays reaching
 *                       pixel (i,j).
 *
 * Pins (tests/test_oracle_pins.py, all -m "not gpu"): paper N* lists
 * (PAPER.md:156-157), Fig. 1 N*=558, eq.(12) uniform map without
 * stars, point-lens A(u), 2-D Gauss theorem on a ring of lenses, ray
 * conservation, mirror / transpose symmetries, an independent numpy brute force
 * on C1, Phi bookkeeping of eq.(6)/(9); for the *_m variants: unit masses reproduce the
 * unit-mass path bit for bit, two coincident unit lenses = one lens of mass 2, the Einstein
 * radius of a mass-m lens is sqrt(m), Gauss theorem for a ring of unequal masses, numpy
 * brute force; for the random-ray modes (tests/test_oracle_random_rays.py, tests/test_oracle_uniform_rays.py): the
 * published Philox known-answer vectors, a second Python restatement of the draws and positions, cell containment
 * (mode 1) / rectangle coverage and uniformity (mode 2), index of dispersion < 0.5 (mode 1) and 1 (mode 2) on a no-star
 * map with eq.(12) in the mean, point-lens A(u), region partition by ray id, brute-force maps.
 * No function here is "parity unpinned".
 *
 * Build: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC (see oracle/oracle.py).
 * -ffp-contract=off keeps every multiply and add separately rounded, so the
 * results do not depend on whether the host CPU has FMA.
 */
#include <math.h>
#include <stdint.h>
#include <stddef.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    double sigma;            /* total convergence sigma = sigma_c + sigma_*   */
    double stellar_fraction; /* sigma_* / sigma = 1 - s, s = sigma_c/sigma */
    double gamma;            /* external shear */
    int32_t n_pix;           /* pixels per side of the square map                          */
    double n_rays;           /* mean rays per pixel without lensing */
    double L;                /* source-plane side length, Einstein radii */
    int32_t ray_mode;        /* 0: regular grid (configs); 1: random position inside
                                each grid cell (the GPU-D way; reading R17);
                                2: random position in the whole shooting rectangle (reading R20)   */
    uint64_t ray_seed;       /* key of the counter-based generator for ray_modes 1 and 2           */
} ora_problem;

typedef struct {
    double kappa_star; /* sigma_*                                                     */
    double kappa_c;    /* sigma_c                                                     */
    double pixel;      /* pixel side = L / n_pix                                      */
    double delta;      /* ray spacing = pixel / sqrt(N_rays)                          */
    double a1, a2;     /* half-sides of the shooting rectangle                        */
    double r_star;     /* lens-disk radius                                            */
    double mu_th;      /* 1/((1-sigma)^2-gamma^2), signed          */
    int64_t n1, n2;    /* rays along axis 1 / axis 2                                  */
    int64_t n_star;    /* N_* of eq.(5)                                               */
} ora_geometry;

enum { ORA_OK = 0, ORA_BAD = -1 };

/* eq.(5): N_* = sigma_* A / (pi <M>), A = pi R^2, <M> = 1  =>  sigma_* R^2,
 * rounded to the nearest integer (reading R4: floor(x + 0.5)). */
int64_t ora_n_star(double kappa_star, double r_disk)
{
    return (int64_t)floor(kappa_star * r_disk * r_disk + 0.5);
}

int ora_derive(const ora_problem *p, ora_geometry *g)
{
    if (!p || !g) return ORA_BAD;
    if (!(p->sigma >= 0.0) || !(p->stellar_fraction >= 0.0) || !(p->stellar_fraction <= 1.0) ||
        p->n_pix <= 0 || !(p->n_rays > 0.0) || !(p->L > 0.0) || !isfinite(p->gamma) ||
        !isfinite(p->sigma) || !isfinite(p->n_rays) || !isfinite(p->L) || (p->ray_mode < 0 || p->ray_mode > 2))
        return ORA_BAD;
    double minus = 1.0 - p->sigma - p->gamma; /* axis-1 smooth stretch (eq.4, eq.11) */
    double plus = 1.0 - p->sigma + p->gamma;  /* axis-2 smooth stretch               */
    if (fabs(minus) < 1e-6 || fabs(plus) < 1e-6) return ORA_BAD;

    g->kappa_star = p->stellar_fraction * p->sigma;
    g->kappa_c = p->sigma - g->kappa_star;
    g->pixel = p->L / (double)p->n_pix;
    g->delta = g->pixel / sqrt(p->n_rays);
    /* eq.(11) PAPER.md:283 L_pm = L_map/(1 - sigma pm gamma); configs[0] takes the
     * absolute value and a 1.2 margin, half-sides. */
    g->a1 = 1.2 * (p->L / 2.0) / fabs(minus);
    g->a2 = 1.2 * (p->L / 2.0) / fabs(plus);
    /* reading R7: keep delta exact, round the ray count up; the 1e-9 keeps
     * exactly-integer ratios from being bumped by rounding fuzz. */
    g->n1 = (int64_t)ceil(2.0 * g->a1 / g->delta - 1e-9);
    g->n2 = (int64_t)ceil(2.0 * g->a2 / g->delta - 1e-9);
    /* configs[0]: R* = 1.3 sqrt(a1^2 + a2^2)  (wider than the long axis) */
    g->r_star = 1.3 * sqrt(g->a1 * g->a1 + g->a2 * g->a2);
    g->n_star = ora_n_star(g->kappa_star, g->r_star);
    /* eq.(12) */
    g->mu_th = 1.0 / ((1.0 - p->sigma) * (1.0 - p->sigma) - p->gamma * p->gamma);
    return ORA_OK;
}

/* Philox-4x32-10 (Salmon, Moraes, Dror & Shaw, SC'11): counter-based generator, 10 rounds of
 *   (c0,c1,c2,c3) <- (hi(M1 c2) ^ c1 ^ k0, lo(M1 c2), hi(M0 c0) ^ c3 ^ k1, lo(M0 c0)),  k <- k + (W0, W1).
 * Pinned by the published known-answer vectors (tests/golden/philox4x32_10_kat.txt). */
void ora_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3], k0 = key[0], k1 = key[1];
    for (int r = 0; r < 10; ++r) {
        uint64_t p0 = (uint64_t)0xD2511F53u * c0, p1 = (uint64_t)0xCD9E8D57u * c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0, n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1, n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* Two uniform deviates in [0,1) for ray id = j*n1 + i: counter (id_lo, id_hi, 0, 0), key (seed_lo, seed_hi);
 * 53 bits each: u = ((r_a >> 5) 2^26 + (r_b >> 6)) 2^-53. */
void ora_ray_uniforms(uint64_t ray_id, uint64_t seed, double u[2])
{
    uint32_t ctr[4] = {(uint32_t)ray_id, (uint32_t)(ray_id >> 32), 0u, 0u};
    uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)}, r[4];
    ora_philox4x32_10(ctr, key, r);
    u[0] = ((double)(r[0] >> 5) * 67108864.0 + (double)(r[1] >> 6)) * (1.0 / 9007199254740992.0);
    u[1] = ((double)(r[2] >> 5) * 67108864.0 + (double)(r[3] >> 6)) * (1.0 / 9007199254740992.0);
}

/* Image-plane position of ray (i, j).  ray_mode 0: cell-centred regular grid, symmetric about the
 * origin (reading R7).  ray_mode 1: a uniformly random point of the same grid cell
 * [(i - n1/2) delta, (i + 1 - n1/2) delta) x [...]: the paper's GPU-D shoots rays "from random positions in
 * the shooting grid"; reading R17 keeps one ray per cell so that ray (i, j) stays
 * where the tile-local arithmetic and the region / sharding logic expect it (the regular grid is u = 1/2).
 * ray_mode 2 (reading R20): the n1 n2 rays are independent uniform points of the whole rectangle
 * [-n1 delta/2, n1 delta/2) x [-n2 delta/2, n2 delta/2) -- what "a batch of 2^17 random ray positions"
 * "in the shooting grid" says literally; (i, j) only numbers the rays
 * (id = j n1 + i is the counter), it says nothing about where the ray is.  Counts in any fixed area are then
 * binomial ~ Poisson, the noise PAPER.md:167 describes. */
static void ora_ray_x(const ora_problem *p, const ora_geometry *g, int64_t i, int64_t j, double x[2])
{
    if (p->ray_mode == 2) {
        double u[2];
        ora_ray_uniforms((uint64_t)j * (uint64_t)g->n1 + (uint64_t)i, p->ray_seed, u);
        x[0] = (u[0] * (double)g->n1 - (double)g->n1 / 2.0) * g->delta;
        x[1] = (u[1] * (double)g->n2 - (double)g->n2 / 2.0) * g->delta;
        return;
    }
    if (p->ray_mode == 1) {
        double u[2];
        ora_ray_uniforms((uint64_t)j * (uint64_t)g->n1 + (uint64_t)i, p->ray_seed, u);
        x[0] = ((double)i + u[0] - (double)g->n1 / 2.0) * g->delta;
        x[1] = ((double)j + u[1] - (double)g->n2 / 2.0) * g->delta;
        return;
    }
    x[0] = ((double)i - (double)(g->n1 - 1) / 2.0) * g->delta;
    x[1] = ((double)j - (double)(g->n2 - 1) / 2.0) * g->delta;
}

/* Image-plane positions of the listed rays (x_out = 2*n doubles): exposes ray generation to the pins. */
int ora_ray_positions(const ora_problem *p, int64_t n, const int64_t *ray_i, const int64_t *ray_j, double *x_out)
{
    ora_geometry g;
    if (ora_derive(p, &g) != ORA_OK || n < 0) return ORA_BAD;
    for (int64_t k = 0; k < n; ++k) ora_ray_x(p, &g, ray_i[k], ray_j[k], x_out + 2 * k);
    return ORA_OK;
}

/* eq.(4), PAPER.md:51:
 *   y = diag(1-gamma, 1+gamma) x - sigma_c x - sum_i m_i (x - x_i)/|x - x_i|^2
 * mass = NULL means m_i = 1 (every map of the paper).  Lenses in index order,
 * plain fp64 accumulation.  Returns 1 if the ray sits exactly on a lens (|x - x_i|^2 == 0) or y
 * is not finite (reading R12: such a ray is "dropped"), else 0. */
int ora_lens_equation_m(double gamma, double kappa_c, const double *lens_xy, const double *mass,
                        int64_t n_lens, const double x[2], double y[2])
{
    double s1 = 0.0, s2 = 0.0;
    int bad = 0;
    for (int64_t k = 0; k < n_lens; ++k) {
        double d1 = x[0] - lens_xy[2 * k];
        double d2 = x[1] - lens_xy[2 * k + 1];
        double r2 = d1 * d1 + d2 * d2;
        if (r2 == 0.0) bad = 1;
        if (mass) {
            s1 += mass[k] * d1 / r2;
            s2 += mass[k] * d2 / r2;
        } else {
            s1 += d1 / r2;
            s2 += d2 / r2;
        }
    }
    y[0] = (1.0 - gamma) * x[0] - kappa_c * x[0] - s1;
    y[1] = (1.0 + gamma) * x[1] - kappa_c * x[1] - s2;
    if (!isfinite(y[0]) || !isfinite(y[1])) bad = 1;
    return bad;
}

int ora_lens_equation(double gamma, double kappa_c, const double *lens_xy, int64_t n_lens,
                      const double x[2], double y[2])
{
    return ora_lens_equation_m(gamma, kappa_c, lens_xy, NULL, n_lens, x, y);
}

/* Source-plane pixel of y: half-open pixels, map covers [-L/2, L/2)^2, axis 1 is
 * the fast index (readings R10, R11).  Returns 0 and sets *pi,*pj if inside. */
static int ora_pixel(const ora_problem *p, const ora_geometry *g, const double y[2],
                     int64_t *pi, int64_t *pj)
{
    double u1 = floor((y[0] + p->L / 2.0) / g->pixel);
    double u2 = floor((y[1] + p->L / 2.0) / g->pixel);
    if (!(u1 >= 0.0) || !(u1 < (double)p->n_pix) || !(u2 >= 0.0) || !(u2 < (double)p->n_pix))
        return 1;
    *pi = (int64_t)u1;
    *pj = (int64_t)u2;
    return 0;
}

/* Shoot rays [i0,i1) x [j0,j1) and ADD them to map (n_pix*n_pix uint32, row-major,
 * map[j'*n_pix + i'], i' <-> y1).  stats[0..3] += shot, in-map, out-of-map, dropped. */
int ora_shoot_region_m(const ora_problem *p, const double *lens_xy, const double *mass, int64_t n_lens,
                       int64_t i0, int64_t i1, int64_t j0, int64_t j1,
                       uint32_t *map, uint64_t stats[4])
{
    ora_geometry g;
    if (ora_derive(p, &g) != ORA_OK || n_lens < 0 || (n_lens > 0 && !lens_xy) || !map || !stats)
        return ORA_BAD;
    if (i0 < 0 || j0 < 0 || i1 > g.n1 || j1 > g.n2 || i0 > i1 || j0 > j1) return ORA_BAD;
    uint64_t shot = 0, inmap = 0, outmap = 0, dropped = 0;
#pragma omp parallel for schedule(dynamic, 1) reduction(+ : shot, inmap, outmap, dropped)
    for (int64_t j = j0; j < j1; ++j) {
        for (int64_t i = i0; i < i1; ++i) {
            double x[2], y[2];
            int64_t pi, pj;
            ora_ray_x(p, &g, i, j, x);
            ++shot;
            if (ora_lens_equation_m(p->gamma, g.kappa_c, lens_xy, mass, n_lens, x, y)) {
                ++dropped;
            } else if (ora_pixel(p, &g, y, &pi, &pj)) {
                ++outmap;
            } else {
                ++inmap;
#pragma omp atomic
                map[pj * (int64_t)p->n_pix + pi] += 1u;
            }
        }
    }
    stats[0] += shot;
    stats[1] += inmap;
    stats[2] += outmap;
    stats[3] += dropped;
    return ORA_OK;
}

int ora_shoot_region(const ora_problem *p, const double *lens_xy, int64_t n_lens,
                     int64_t i0, int64_t i1, int64_t j0, int64_t j1,
                     uint32_t *map, uint64_t stats[4])
{
    return ora_shoot_region_m(p, lens_xy, NULL, n_lens, i0, i1, j0, j1, map, stats);
}

/* Source-plane positions of every ray of [i0,i1) x [j0,j1), row-major in (j, i):
 * y_out[2*((j-j0)*(i1-i0) + (i-i0)) + {0,1}].  Dropped rays get NaN. */
int ora_capture_region_m(const ora_problem *p, const double *lens_xy, const double *mass, int64_t n_lens,
                         int64_t i0, int64_t i1, int64_t j0, int64_t j1, double *y_out)
{
    ora_geometry g;
    if (ora_derive(p, &g) != ORA_OK || n_lens < 0 || (n_lens > 0 && !lens_xy) || !y_out)
        return ORA_BAD;
    if (i0 < 0 || j0 < 0 || i1 > g.n1 || j1 > g.n2 || i0 > i1 || j0 > j1) return ORA_BAD;
    int64_t w = i1 - i0;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t j = j0; j < j1; ++j) {
        for (int64_t i = i0; i < i1; ++i) {
            double x[2], y[2];
            ora_ray_x(p, &g, i, j, x);
            if (ora_lens_equation_m(p->gamma, g.kappa_c, lens_xy, mass, n_lens, x, y)) {
                y[0] = NAN;
                y[1] = NAN;
            }
            y_out[2 * ((j - j0) * w + (i - i0))] = y[0];
            y_out[2 * ((j - j0) * w + (i - i0)) + 1] = y[1];
        }
    }
    return ORA_OK;
}

int ora_capture_region(const ora_problem *p, const double *lens_xy, int64_t n_lens,
                       int64_t i0, int64_t i1, int64_t j0, int64_t j1, double *y_out)
{
    return ora_capture_region_m(p, lens_xy, NULL, n_lens, i0, i1, j0, j1, y_out);
}

/* Source-plane positions of the listed rays.  y_out = 2*n doubles. */
int ora_probe(const ora_problem *p, const double *lens_xy, int64_t n_lens,
              int64_t n, const int64_t *ray_i, const int64_t *ray_j, double *y_out)
{
    ora_geometry g;
    if (ora_derive(p, &g) != ORA_OK || n_lens < 0 || (n_lens > 0 && !lens_xy) || n < 0) return ORA_BAD;
    for (int64_t k = 0; k < n; ++k)
        if (ray_i[k] < 0 || ray_i[k] >= g.n1 || ray_j[k] < 0 || ray_j[k] >= g.n2) return ORA_BAD;
#pragma omp parallel for schedule(static)
    for (int64_t k = 0; k < n; ++k) {
        double x[2], y[2];
        ora_ray_x(p, &g, ray_i[k], ray_j[k], x);
        if (ora_lens_equation(p->gamma, g.kappa_c, lens_xy, n_lens, x, y)) {
            y[0] = NAN;
            y[1] = NAN;
        }
        y_out[2 * k] = y[0];
        y_out[2 * k + 1] = y[1];
    }
    return ORA_OK;
}

/* eq.(4) at arbitrary image-plane points (not only grid rays): x_in, y_out = 2*n doubles. */
int ora_deflect_points_m(double gamma, double kappa_c, const double *lens_xy, const double *mass, int64_t n_lens,
                         int64_t n, const double *x_in, double *y_out)
{
    if (n < 0 || n_lens < 0) return ORA_BAD;
    for (int64_t k = 0; k < n; ++k)
        ora_lens_equation_m(gamma, kappa_c, lens_xy, mass, n_lens, x_in + 2 * k, y_out + 2 * k);
    return ORA_OK;
}

int ora_deflect_points(double gamma, double kappa_c, const double *lens_xy, int64_t n_lens,
                       int64_t n, const double *x_in, double *y_out)
{
    return ora_deflect_points_m(gamma, kappa_c, lens_xy, NULL, n_lens, n, x_in, y_out);
}

/* eq.(5), with a mean lens mass: N_* = sigma_* A / (pi <M>) = sigma_* R^2 / <M>. */
int64_t ora_n_star_m(double kappa_star, double r_disk, double mean_mass)
{
    return (int64_t)floor(kappa_star * r_disk * r_disk / mean_mass + 0.5);
}

/* Pixel index (j'*n_pix + i') of source-plane positions, -1 outside / NaN. */
int ora_pixels_of(const ora_problem *p, int64_t n, const double *y, int64_t *pix_out)
{
    ora_geometry g;
    if (ora_derive(p, &g) != ORA_OK || n < 0) return ORA_BAD;
    for (int64_t k = 0; k < n; ++k) {
        int64_t pi, pj;
        if (!isfinite(y[2 * k]) || !isfinite(y[2 * k + 1]) || ora_pixel(p, &g, y + 2 * k, &pi, &pj))
            pix_out[k] = -1;
        else
            pix_out[k] = pj * (int64_t)p->n_pix + pi;
    }
    return ORA_OK;
}

int ora_num_threads(void)
{
    int n = 1;
#ifdef _OPENMP
#pragma omp parallel
    {
#pragma omp master
        n = omp_get_num_threads();
    }
#endif
    return n;
}
