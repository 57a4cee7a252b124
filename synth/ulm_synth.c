/*
 * ulm_synth.c -- seeded synthetic RCA channel data (INPUT GENERATOR ONLY).
 *
 * Forward model of SURVEY.md 8(d) "Common echo model": point scatterer s at (x, y, z) with amplitude a
 * adds to event (row-tx or column-tx plane wave at angle th) and receive channel ch the pulse
 * a*p(t - tau), p(t) = exp(-t^2 / 2 sigma^2) cos(2 pi fc t), sigma = 2 / (2.355 fc); no directivity,
 * no spreading loss; white Gaussian noise from a counter-based generator; int16 quantisation.
 * Shapes follow the paper's acquisition (128+128 RCA, pitch 0.214 mm, plane waves,
 * 400 Hz, 300-volume buffers, 20-45 mm depth).
 *
 * This file holds none of the beamformer's arithmetic and is used by neither the oracle nor the CUDA
 * path; it only produces the inputs both consume.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#ifndef M_PI
#define M_PI 3.14159265358979323846
#endif

typedef struct {
    int32_t n_rows, n_cols;
    double pitch;
    int32_t n_row_tx, n_col_tx;
    const double *row_tx_angles, *col_tx_angles;
    double c, fs, fc;
    int32_t n_samples;
    double t_start;
    const double *t0;       /* per event, NULL = 0 */
    int32_t all_channels;   /* 1: n_rows+n_cols channels per event (rows first); 0: orthogonal only */
} ulm_synth_params;

static int n_channels(const ulm_synth_params *p)
{
    return p->all_channels ? p->n_rows + p->n_cols : (p->n_rows > p->n_cols ? p->n_rows : p->n_cols);
}

/* which aperture / element a stored channel of an event is: returns 0 and sets is_col, elem; -1 = unused */
static int channel_elem(const ulm_synth_params *p, int row_tx, int ch, int *is_col, int *elem)
{
    if (p->all_channels) {
        if (ch < p->n_rows) { *is_col = 0; *elem = ch; }
        else { *is_col = 1; *elem = ch - p->n_rows; }
        return 0;
    }
    *is_col = row_tx; /* orthogonal aperture: row-tx -> columns receive */
    *elem = ch;
    return ch < (row_tx ? p->n_cols : p->n_rows) ? 0 : -1;
}

/* noise-free line of one (event, channel): line[n] += a p(t_n - tau) for every scatterer */
static void render_line(const ulm_synth_params *p, const double *scat, int64_t n_scat, int e, int ch,
                        double *line)
{
    const int ns = p->n_samples;
    memset(line, 0, sizeof(double) * (size_t)ns);
    const int row_tx = e < p->n_row_tx;
    int is_col, elem;
    if (channel_elem(p, row_tx, ch, &is_col, &elem)) return;
    const double th = row_tx ? p->row_tx_angles[e] : p->col_tx_angles[e - p->n_row_tx];
    const double t0 = p->t0 ? p->t0[e] : 0.0;
    const double sigma = 2.0 / (2.355 * p->fc);
    const double half = 4.5 * sigma * p->fs; /* pulse support in samples (envelope < 4e-5 beyond) */
    const double pe = (elem - 0.5 * ((is_col ? p->n_cols : p->n_rows) - 1)) * p->pitch;
    for (int64_t s = 0; s < n_scat; ++s) {
        const double x = scat[4 * s], y = scat[4 * s + 1], z = scat[4 * s + 2], a = scat[4 * s + 3];
        /* plane wave steered along y for row-tx, along x for column-tx; line element of the
         * receiving aperture: a column (long in y) sees lateral offset in x, a row in y */
        const double tau_tx = t0 + (z * cos(th) + (row_tx ? y : x) * sin(th)) / p->c;
        const double off = (is_col ? x : y) - pe;
        const double tau = tau_tx + sqrt(off * off + z * z) / p->c;
        const double u = (tau - p->t_start) * p->fs;
        int n_lo = (int)ceil(u - half), n_hi = (int)floor(u + half);
        if (n_lo < 0) n_lo = 0;
        if (n_hi > ns - 1) n_hi = ns - 1;
        for (int n = n_lo; n <= n_hi; ++n) {
            const double dt = (n - u) / p->fs;
            line[n] += a * exp(-dt * dt / (2.0 * sigma * sigma)) * cos(2.0 * M_PI * p->fc * dt);
        }
    }
}

/* counter-based standard normal: splitmix64 of (seed, counter) -> Box-Muller */
static uint64_t mix64(uint64_t z)
{
    z += 0x9E3779B97F4A7C15ull;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}

static double normal_at(uint64_t seed, uint64_t counter)
{
    uint64_t a = mix64(seed * 0xD1342543DE82EF95ull + 2 * counter);
    uint64_t b = mix64(seed * 0xD1342543DE82EF95ull + 2 * counter + 1);
    double u1 = ((a >> 11) + 1.0) * (1.0 / 9007199254740993.0); /* (0, 1] */
    double u2 = (b >> 11) * (1.0 / 9007199254740992.0);
    return sqrt(-2.0 * log(u1)) * cos(2.0 * M_PI * u2);
}

int ulm_synth_channels(const ulm_synth_params *p) { return n_channels(p); }

/* max |value| and mean square of the noise-free data of one frame */
int ulm_synth_stats(const ulm_synth_params *p, const double *scat, int64_t n_scat, double *max_abs,
                    double *mean_sq)
{
    const int ne = p->n_row_tx + p->n_col_tx, nch = n_channels(p), ns = p->n_samples;
    double mx = 0.0, ss = 0.0;
#pragma omp parallel
    {
        double *line = (double *)malloc(sizeof(double) * (size_t)ns);
        double lmx = 0.0, lss = 0.0;
#pragma omp for schedule(dynamic, 4) collapse(2)
        for (int e = 0; e < ne; ++e)
            for (int ch = 0; ch < nch; ++ch) {
                render_line(p, scat, n_scat, e, ch, line);
                for (int n = 0; n < ns; ++n) {
                    double v = fabs(line[n]);
                    if (v > lmx) lmx = v;
                    lss += v * v;
                }
            }
#pragma omp critical
        {
            if (lmx > mx) mx = lmx;
            ss += lss;
        }
        free(line);
    }
    *max_abs = mx;
    *mean_sq = ss / ((double)ne * nch * ns);
    return 0;
}

/* out[event][channel][sample] = clip(round(scale * (line + noise_sigma * N(0,1)))) */
int ulm_synth_render(const ulm_synth_params *p, const double *scat, int64_t n_scat, double scale,
                     double noise_sigma, uint64_t seed, int64_t frame_index, int16_t *out)
{
    const int ne = p->n_row_tx + p->n_col_tx, nch = n_channels(p), ns = p->n_samples;
#pragma omp parallel
    {
        double *line = (double *)malloc(sizeof(double) * (size_t)ns);
#pragma omp for schedule(dynamic, 4) collapse(2)
        for (int e = 0; e < ne; ++e)
            for (int ch = 0; ch < nch; ++ch) {
                render_line(p, scat, n_scat, e, ch, line);
                const uint64_t base = (((uint64_t)frame_index * ne + e) * nch + ch) * (uint64_t)ns;
                int16_t *o = out + ((int64_t)e * nch + ch) * ns;
                for (int n = 0; n < ns; ++n) {
                    double v = line[n];
                    if (noise_sigma > 0.0) v += noise_sigma * normal_at(seed, base + n);
                    double q = nearbyint(scale * v);
                    if (q > 32767.0) q = 32767.0;
                    if (q < -32767.0) q = -32767.0;
                    o[n] = (int16_t)q;
                }
            }
        free(line);
    }
    return 0;
}
