/* Seeded synthetic light-field generator (input generation only -- none of HMLFC's arithmetic).
 *
 * Ray-casts a small 3-D scene with the light-slab cameras of DESIGN.md "Input recipe"
 * (SURVEY.md 8(d) D2): camera (iu,iv) at (uv_origin + (iu,iv)*uv_step, 0); pixel (is,it) of the
 * common image plane at (st_origin + (is,it)*st_step, z_st).  Objects: fronto-parallel textured
 * rectangles ("planes") and Lambertian textured spheres; nearest hit wins.  Texture = 4-octave
 * value noise over a hashed lattice, evaluated at continuous hit coordinates, so fractional
 * per-view disparities are meaningful.  Optional additive Gaussian noise per sample.
 *
 * Everything is a pure function of (scene arrays, seed): a counter-based 64-bit mix, no state.
 * Built with -ffp-contract=off so that the same binary gives the same bytes on every host.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    int32_t U, V, Ws, Ht;
    double uv_origin[2], uv_step[2], st_origin[2], st_step[2], z_st;
    int32_t n_planes, n_spheres;
    double noise_sigma;
    uint64_t seed;
    double light[3];      /* unit vector towards the light */
    double base_cell_px;  /* lattice cell of octave 0, in st-plane pixels */
} wl_scene;

/* plane k: z, x0, x1, y0, y1 (world rectangle at depth z; the background plane uses +-1e30), base rgb, tex id */
typedef struct { double z, x0, x1, y0, y1; double base[3]; uint64_t tex; } wl_plane;
typedef struct { double c[3], r; double base[3]; uint64_t tex; } wl_sphere;

static uint64_t mix64(uint64_t x)
{
    x += 0x9E3779B97F4A7C15ull;
    x = (x ^ (x >> 30)) * 0xBF58476D1CE4E5B9ull;
    x = (x ^ (x >> 27)) * 0x94D049BB133111EBull;
    return x ^ (x >> 31);
}
static uint64_t hash4(uint64_t a, uint64_t b, uint64_t c, uint64_t d)
{
    return mix64(mix64(mix64(mix64(a) ^ b) ^ c) ^ d);
}
static double u01(uint64_t h) { return (double)(h >> 11) * (1.0 / 9007199254740992.0); }

static double smooth(double t) { return t * t * (3.0 - 2.0 * t); }

/* 4 octaves, persistence 0.5, normalised to [0,1].  Lattice value at (ix, iy) = u01(hash4(tex, oct * 4 + ch, ix, iy)); the hash
 * chain mix64(mix64(mix64(mix64(tex) ^ k) ^ ix) ^ iy) is shared between the four corners as far as it goes. */
static double value_noise(uint64_t tex, int ch, double x, double y, double cell)
{
    double sum = 0.0, amp = 1.0, norm = 0.0;
    const uint64_t ht = mix64(tex);
    for (int o = 0; o < 4; ++o) {
        double fx = x / cell, fy = y / cell;
        double x0 = floor(fx), y0 = floor(fy);
        double tx = smooth(fx - x0), ty = smooth(fy - y0);
        int64_t ix = (int64_t)x0, iy = (int64_t)y0;
        const uint64_t hk = mix64(ht ^ (uint64_t)(o * 4 + ch));
        const uint64_t hx0 = mix64(hk ^ (uint64_t)ix), hx1 = mix64(hk ^ (uint64_t)(ix + 1));
        double a = u01(mix64(hx0 ^ (uint64_t)iy)), b = u01(mix64(hx1 ^ (uint64_t)iy));
        double c = u01(mix64(hx0 ^ (uint64_t)(iy + 1))), d = u01(mix64(hx1 ^ (uint64_t)(iy + 1)));
        double v = (a * (1.0 - tx) + b * tx) * (1.0 - ty) + (c * (1.0 - tx) + d * tx) * ty;
        sum += amp * v;
        norm += amp;
        amp *= 0.5;
        cell *= 0.5;
    }
    return sum / norm;
}

static double gauss(uint64_t seed, uint64_t idx)
{
    double a = u01(hash4(seed, 0x6e6f697365ull, idx, 0));
    double b = u01(hash4(seed, 0x6e6f697365ull, idx, 1));
    if (a < 1e-300) a = 1e-300;
    return sqrt(-2.0 * log(a)) * cos(6.283185307179586 * b);
}

int wl_generate_lf(const wl_scene *sc, const wl_plane *planes, const wl_sphere *spheres, uint8_t *lf, int nthreads)
{
    if (!sc || !lf || sc->n_planes < 1) return -1;
#ifdef _OPENMP
    if (nthreads <= 0) nthreads = omp_get_max_threads();
#else
    (void)nthreads;
#endif
    const int U = sc->U, V = sc->V, Ws = sc->Ws, Ht = sc->Ht;
    const double zst = sc->z_st;
    /* central camera: texture coordinates are st-plane pixel coordinates as seen from it */
    const double ccx = sc->uv_origin[0] + 0.5 * (U - 1) * sc->uv_step[0];
    const double ccy = sc->uv_origin[1] + 0.5 * (V - 1) * sc->uv_step[1];
#pragma omp parallel for schedule(dynamic, 1) num_threads(nthreads)
    for (int64_t row = 0; row < (int64_t)U * V * Ht; ++row) {
        int it = (int)(row % Ht);
        int vi = (int)(row / Ht);
        int iu = vi % U, iv = vi / U;
        double cx = sc->uv_origin[0] + iu * sc->uv_step[0];
        double cy = sc->uv_origin[1] + iv * sc->uv_step[1];
        double ty = sc->st_origin[1] + it * sc->st_step[1];
        for (int is = 0; is < Ws; ++is) {
            double tx = sc->st_origin[0] + is * sc->st_step[0];
            /* ray: P(z) = (cx,cy,0) + (z / zst) * (tx - cx, ty - cy, zst) */
            double dx = (tx - cx) / zst, dy = (ty - cy) / zst;
            /* nearest hit first (the last object that lowers best_z wins), then ONE texture evaluation for the winner */
            double best_z = 1e300;
            double col[3] = { 0.0, 0.0, 0.0 };
            int win_plane = -1, win_sphere = -1;
            for (int k = 0; k < sc->n_planes; ++k) {
                const wl_plane *pl = &planes[k];
                if (pl->z >= best_z) continue;
                double X = cx + dx * pl->z, Y = cy + dy * pl->z;
                if (X < pl->x0 || X > pl->x1 || Y < pl->y0 || Y > pl->y1) continue;
                best_z = pl->z;
                win_plane = k;
            }
            for (int k = 0; k < sc->n_spheres; ++k) {
                const wl_sphere *sp = &spheres[k];
                /* |o + z*d - c|^2 = r^2 with d = (dx,dy,1), o = (cx,cy,0), parameter z */
                double ox = cx - sp->c[0], oy = cy - sp->c[1], oz = -sp->c[2];
                double A = dx * dx + dy * dy + 1.0;
                double Bq = 2.0 * (ox * dx + oy * dy + oz);
                double Cq = ox * ox + oy * oy + oz * oz - sp->r * sp->r;
                double disc = Bq * Bq - 4.0 * A * Cq;
                if (disc < 0.0) continue;
                double z = (-Bq - sqrt(disc)) / (2.0 * A);
                if (z <= 0.0 || z >= best_z) continue;
                best_z = z;
                win_sphere = k;
            }
            if (win_sphere >= 0) {
                const wl_sphere *sp = &spheres[win_sphere];
                double z = best_z;
                double hx = cx + dx * z, hy = cy + dy * z, hz = z;
                double nx = (hx - sp->c[0]) / sp->r, ny = (hy - sp->c[1]) / sp->r, nz = (hz - sp->c[2]) / sp->r;
                double lam = nx * sc->light[0] + ny * sc->light[1] + nz * sc->light[2];
                if (lam < 0.0) lam = 0.0;
                double shade = 0.3 + 0.7 * lam;
                /* texture fixed to the sphere surface: pixel-scaled offsets from the centre */
                double px = (hx - sp->c[0]) * zst / sp->c[2] / sc->st_step[0];
                double py = (hy - sp->c[1]) * zst / sp->c[2] / sc->st_step[1];
                for (int c = 0; c < 3; ++c)
                    col[c] = shade * (0.5 * sp->base[c] + 0.5 * value_noise(sp->tex, c, px, py, sc->base_cell_px));
            } else if (win_plane >= 0) {
                const wl_plane *pl = &planes[win_plane];
                double X = cx + dx * pl->z, Y = cy + dy * pl->z;
                /* project the hit to the st plane through the central camera -> pixel units */
                double px = ((ccx + (X - ccx) * zst / pl->z) - sc->st_origin[0]) / sc->st_step[0];
                double py = ((ccy + (Y - ccy) * zst / pl->z) - sc->st_origin[1]) / sc->st_step[1];
                for (int c = 0; c < 3; ++c)
                    col[c] = 0.5 * pl->base[c] + 0.5 * value_noise(pl->tex, c, px, py, sc->base_cell_px);
            }
            uint8_t *o = lf + ((size_t)row * Ws + is) * 3;
            for (int c = 0; c < 3; ++c) {
                double v = 16.0 + 224.0 * col[c];
                if (sc->noise_sigma > 0.0) v += sc->noise_sigma * gauss(sc->seed, ((uint64_t)row * (uint64_t)Ws + (uint64_t)is) * 3u + (uint64_t)c);
                double r = floor(v + 0.5);
                o[c] = (uint8_t)(r < 0.0 ? 0.0 : (r > 255.0 ? 255.0 : r));
            }
        }
    }
    return 0;
}
