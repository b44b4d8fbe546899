/*
 * fdc_inputs/gen.c -- seeded synthetic INPUT generators (track database, phantoms).
 *
 * This module serves both the oracle and the CUDA path with identical input bytes.  It holds
 * none of the track-repeating method's arithmetic (no transport, no sampling of protons, no
 * deposit): it only manufactures the *inputs* the paper took from GEANT4 and a patient CT,
 * which are not available.  Recipes: BASELINE.json configs[0..4],
 * SURVEY.md §8(d) "Track generator recipe" / "Phantom generator", readings A14-A18; restated in
 * DESIGN.md §5.
 *
 * Machine independence: every value is a fixed sequence of IEEE-754 double operations
 * (+ - * / sqrt) -- the transcendental functions below are this file's own fixed-order series,
 * not libm -- and the file is compiled with -ffp-contract=off, so the same seed gives the same
 * bytes on any x86-64/aarch64 host.  That is what lets oracle digests computed off the GPU box
 * be compared with GPU results computed on it.
 *
 * Random numbers: this file's own Philox4x32-10 (Salmon et al., SC'11), keyed by the seed.
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#include <math.h>   /* sqrt, floor only (both exactly specified by IEEE-754 / C) */

/* ------------------------------------------------------------------ Philox4x32-10 */
static inline void gen_philox(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                              uint32_t k0, uint32_t k1, uint32_t out[4])
{
    for (int r = 0; r < 10; ++r) {
        uint64_t p0 = (uint64_t)0xD2511F53u * c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* ------------------------------------------------------------------ deterministic math */
static const double LN2_HI = 6.93147180369123816490e-01;
static const double LN2_LO = 1.90821492927058770002e-10;
static const double LN2    = 6.93147180559945286227e-01;
static const double PIO2_HI = 1.57079632673412561417e+00;
static const double PIO2_LO = 6.07710050650619224932e-11;
static const double TWO_PI  = 6.28318530717958623200e+00;

/* ln(x), x > 0 normal.  x = m 2^e, m in [sqrt(1/2), sqrt(2)); ln m = 2 atanh((m-1)/(m+1)). */
static double det_ln(double x)
{
    union { double d; uint64_t u; } v; v.d = x;
    int e = (int)((v.u >> 52) & 0x7ff) - 1022;
    v.u = (v.u & 0x000fffffffffffffULL) | 0x3fe0000000000000ULL;   /* m in [0.5, 1) */
    double m = v.d;
    if (m < 0.70710678118654757) { m = m * 2.0; e -= 1; }
    double z = (m - 1.0) / (m + 1.0), z2 = z * z;
    double s = 1.0 / 29.0;
    for (int n = 13; n >= 0; --n) s = s * z2 + 1.0 / (double)(2 * n + 1);
    return (double)e * LN2 + 2.0 * z * s;
}

/* exp(x) for |x| < 700. */
static double det_exp(double x)
{
    double kf = floor(x * 1.4426950408889634 + 0.5);
    double r = (x - kf * LN2_HI) - kf * LN2_LO;
    double s = 1.0;
    for (int n = 16; n >= 1; --n) s = 1.0 + (r / (double)n) * s;
    union { double d; uint64_t u; } v;
    v.u = (uint64_t)((int64_t)kf + 1023) << 52;
    return s * v.d;
}

static double det_pow(double x, double y) { return det_exp(y * det_ln(x)); }

/* sin and cos of x (|x| < 1e6). */
static void det_sincos(double x, double *sn, double *cs)
{
    double kf = floor(x * 0.63661977236758138 + 0.5);
    double r = (x - kf * PIO2_HI) - kf * PIO2_LO;
    double r2 = r * r;
    double s = 0.0, c = 0.0;
    /* sin r = r (1 - r2/6 (1 - r2/20 (...)));  cos r = 1 - r2/2 (1 - r2/12 (...)) */
    s = 1.0;
    for (int n = 9; n >= 1; --n) s = 1.0 - r2 / (double)((2 * n) * (2 * n + 1)) * s;
    s = r * s;
    c = 1.0;
    for (int n = 9; n >= 1; --n) c = 1.0 - r2 / (double)((2 * n - 1) * (2 * n)) * c;
    int q = (int)((int64_t)kf & 3);
    switch (q) {
        case 0: *sn = s;  *cs = c;  break;
        case 1: *sn = c;  *cs = -s; break;
        case 2: *sn = -s; *cs = -c; break;
        default: *sn = -c; *cs = s; break;
    }
}

static double det_tan(double x) { double s, c; det_sincos(x, &s, &c); return s / c; }

static inline double u01(uint32_t x) { return ((double)x + 0.5) * 2.3283064365386963e-10; }

/* Box-Muller: words (x0,x1) -> two unit Gaussians. */
static void gauss_pair(uint32_t x0, uint32_t x1, double *g0, double *g1)
{
    double rad = sqrt(-2.0 * det_ln(u01(x0)));
    double s, c; det_sincos(TWO_PI * u01(x1), &s, &c);
    *g0 = rad * c; *g1 = rad * s;
}

/* exported for the generator's own self-tests (tests/test_inputs.py) */
double fdcgen_ln(double x) { return det_ln(x); }
double fdcgen_exp(double x) { return det_exp(x); }
double fdcgen_sin(double x) { double s, c; det_sincos(x, &s, &c); return s; }
double fdcgen_cos(double x) { double s, c; det_sincos(x, &s, &c); return c; }
void fdcgen_philox(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{ gen_philox(ctr[0], ctr[1], ctr[2], ctr[3], key[0], key[1], out); }

/* ------------------------------------------------------------------ track database
 * configs[0]: 1 mm steps; mean energy loss from Bragg-Kleeman R = 0.022 E^1.77 mm; 1 % Gaussian
 * straggling per step (A14); Highland multiple scattering per step (A15); stop when the
 * post-step energy would be < 0.5 MeV, the last step taking everything left (A16).
 */
#define BK_ALPHA 0.022
#define BK_P     1.77
#define X0_MM    360.8
#define M_P      938.272

static double bk_range(double E) { return BK_ALPHA * det_pow(E, BK_P); }

/* upper bound on steps of a track of nominal energy E (for buffer sizing) */
static int64_t step_cap(double E) { return (int64_t)(bk_range(E) * 1.25) + 24; }

/* Generate one track into out arrays (capacity cap); returns number of steps. */
static int gen_track(uint64_t seed, uint64_t track_id, double E_nom, int cap,
                     float *dx, float *dy, float *dz, float *dE, float *Es)
{
    const uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
    double E = E_nom;
    double u[3] = {0, 0, 1}, a[3] = {1, 0, 0}, b[3] = {0, 1, 0};
    int n = 0;
    for (;;) {
        uint32_t w[4];
        gen_philox((uint32_t)track_id, (uint32_t)(track_id >> 32), (uint32_t)n, 0u, k0, k1, w);
        double gE, gx, gy, unused;
        gauss_pair(w[0], w[1], &gE, &gx);
        gauss_pair(w[2], w[3], &gy, &unused);

        double r = bk_range(E);
        double L = r < 1.0 ? r : 1.0;
        double Ep = (r <= L) ? 0.0 : det_pow((r - L) / BK_ALPHA, 1.0 / BK_P);
        double m = E - Ep;
        double de = m * (1.0 + 0.01 * gE);
        if (de < 1e-3 * m) de = 1e-3 * m;
        if (de > E) de = E;
        int last = (E - de < 0.5) || (n + 1 >= cap);
        if (last) de = E;
        float def = (float)de;

        dx[n] = (float)(L * u[0]); dy[n] = (float)(L * u[1]); dz[n] = (float)(L * u[2]);
        dE[n] = def; Es[n] = (float)E;
        ++n;
        if (last) break;

        /* Highland angle for the next step, at the start-of-step energy over length L */
        double pbc = (E * E + 2.0 * E * M_P) / (E + M_P);
        double xr = L / X0_MM;
        double corr = 1.0 + 0.038 * det_ln(xr);
        if (corr < 0.0) corr = 0.0;
        double th0 = 13.6 / pbc * sqrt(xr) * corr;
        double tx = det_tan(th0 * gx), ty = det_tan(th0 * gy);
        double v[3];
        for (int i = 0; i < 3; ++i) v[i] = u[i] + tx * a[i] + ty * b[i];
        double inv = 1.0 / sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
        for (int i = 0; i < 3; ++i) u[i] = v[i] * inv;
        /* re-orthogonalise: a <- normalise(a - (a.u)u); b <- u x a */
        double au = a[0] * u[0] + a[1] * u[1] + a[2] * u[2];
        for (int i = 0; i < 3; ++i) a[i] = a[i] - au * u[i];
        inv = 1.0 / sqrt(a[0] * a[0] + a[1] * a[1] + a[2] * a[2]);
        for (int i = 0; i < 3; ++i) a[i] *= inv;
        b[0] = u[1] * a[2] - u[2] * a[1];
        b[1] = u[2] * a[0] - u[0] * a[2];
        b[2] = u[0] * a[1] - u[1] * a[0];

        E -= (double)def;   /* state follows the stored float so sum(dE) == E_nom */
    }
    return n;
}

/* Upper bound on the total number of steps, for array allocation by the caller. */
int64_t fdcgen_tracks_capacity(double e_min, double e_bin, int n_bins, int tracks_per_bin,
                               const uint8_t *bin_mask /* n_bins, or NULL = all */)
{
    int64_t tot = 0;
    for (int b = 0; b < n_bins; ++b)
        if (!bin_mask || bin_mask[b]) tot += (int64_t)tracks_per_bin * step_cap(e_min + b * e_bin);
    return tot;
}

/*
 * Fill the SoA database.  Layout: bin-major, track-major, step-minor.  Bins whose mask byte is 0
 * are left empty (bin_first[b+1] == bin_first[b]); the global track id used as the Philox counter
 * is b*tracks_per_bin + n regardless of the mask, so a lazily built DB has the same tracks.
 * track_off must hold (number of generated tracks)+1 entries, bin_first n_bins+1.
 * Returns the total number of steps written.
 */
int64_t fdcgen_tracks(uint64_t seed, double e_min, double e_bin, int n_bins, int tracks_per_bin,
                      const uint8_t *bin_mask,
                      float *dx, float *dy, float *dz, float *dE, float *Es,
                      uint64_t *track_off, uint32_t *bin_first)
{
    int64_t pos = 0; uint32_t ntr = 0;
    enum { CHUNK = 2048 };
    int *cnt = (int *)malloc(sizeof(int) * CHUNK);
    bin_first[0] = 0; track_off[0] = 0;
    for (int b = 0; b < n_bins; ++b) {
        if (bin_mask && !bin_mask[b]) { bin_first[b + 1] = ntr; continue; }
        double E_nom = e_min + b * e_bin;
        int cap = (int)step_cap(E_nom);
        float *tmp = (float *)malloc(sizeof(float) * 5 * (size_t)cap * CHUNK);
        for (int t0 = 0; t0 < tracks_per_bin; t0 += CHUNK) {
            int nt = tracks_per_bin - t0 < CHUNK ? tracks_per_bin - t0 : CHUNK;
            #pragma omp parallel for schedule(dynamic, 16)
            for (int t = 0; t < nt; ++t) {
                float *base = tmp + (size_t)5 * cap * t;
                uint64_t tid = (uint64_t)b * (uint64_t)tracks_per_bin + (uint64_t)(t0 + t);
                cnt[t] = gen_track(seed, tid, E_nom, cap, base, base + cap, base + 2 * cap,
                                   base + 3 * cap, base + 4 * cap);
            }
            for (int t = 0; t < nt; ++t) {
                const float *base = tmp + (size_t)5 * cap * t;
                size_t nb = sizeof(float) * (size_t)cnt[t];
                memcpy(dx + pos, base, nb);
                memcpy(dy + pos, base + cap, nb);
                memcpy(dz + pos, base + 2 * cap, nb);
                memcpy(dE + pos, base + 3 * cap, nb);
                memcpy(Es + pos, base + 4 * cap, nb);
                pos += cnt[t];
                track_off[++ntr] = (uint64_t)pos;
            }
        }
        free(tmp);
        bin_first[b + 1] = ntr;
    }
    free(cnt);
    return pos;
}

/* ------------------------------------------------------------------ phantoms
 * kind 0: uniform `hu0` everywhere (config 1: 0 HU).
 * kind 1: z slabs, config 2 (A17): water [0,30) mm, -750 HU [30,60), +1000 HU [60,80), water.
 * kind 2: thorax (A18): extent 512 x 512 x 256 mm whatever the voxel size; body ellipse 0 HU,
 *         lungs -800 HU, spine +700 HU, outside -1000 HU; + N(0, noise_sigma) noise keyed by
 *         (seed, linear voxel index); rounded; clamped to [-1000, 3071].
 */
void fdcgen_phantom(int kind, uint64_t seed, int nx, int ny, int nz,
                    double sx, double sy, double sz, int hu0, double noise_sigma, int16_t *hu)
{
    const uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
    const double cx = 0.5 * nx * sx, cy = 0.5 * ny * sy;
    const double cz = 0.5 * nz * sz;
    #pragma omp parallel for schedule(static)
    for (int iz = 0; iz < nz; ++iz) {
        double z = (iz + 0.5) * sz;
        for (int iy = 0; iy < ny; ++iy) {
            double y = (iy + 0.5) * sy;
            for (int ix = 0; ix < nx; ++ix) {
                double x = (ix + 0.5) * sx;
                uint64_t lin = (uint64_t)ix + (uint64_t)nx * ((uint64_t)iy + (uint64_t)ny * iz);
                double base;
                if (kind == 0) base = hu0;
                else if (kind == 1) base = (z < 30.0) ? 0.0 : (z < 60.0) ? -750.0 : (z < 80.0) ? 1000.0 : 0.0;
                else {
                    double X = x - cx, Y = y - cy, Z = z - cz;
                    double body = (X / 150.0) * (X / 150.0) + (Y / 100.0) * (Y / 100.0);
                    double xl = (X - 70.0) / 55.0, xr = (X + 70.0) / 55.0;
                    double yl = Y / 75.0, zl = Z / 100.0;
                    double lungL = xl * xl + yl * yl + zl * zl, lungR = xr * xr + yl * yl + zl * zl;
                    double sp = X * X + (Y - 70.0) * (Y - 70.0);
                    if (sp <= 18.0 * 18.0) base = 700.0;
                    else if (lungL <= 1.0 || lungR <= 1.0) base = -800.0;
                    else if (body <= 1.0) base = 0.0;
                    else base = -1000.0;
                }
                if (noise_sigma > 0.0) {
                    uint32_t w[4]; double g, g2;
                    gen_philox((uint32_t)lin, (uint32_t)(lin >> 32), 0u, 0u, k0, k1, w);
                    gauss_pair(w[0], w[1], &g, &g2);
                    base = floor(base + noise_sigma * g + 0.5);
                    if (base < -1000.0) base = -1000.0;
                    if (base > 3071.0) base = 3071.0;
                }
                hu[lin] = (int16_t)base;
            }
        }
    }
}
