/*
 * ulm_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE (see ulm_oracle.h).
 *
 * fp64, no tables, no tiling, no reordering beyond the definition in SURVEY.md 8(c) /
 * DESIGN.md "Definition".  Every function names the passage it follows.  The only parallelism is
 * an OpenMP "parallel for" over independent output pixels / points.
 */
#include "ulm_oracle.h"

#include <complex.h>
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#ifndef M_PI
#define M_PI 3.14159265358979323846
#endif

int ulm_oracle_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* centre coordinate of element e of an n-element aperture (SURVEY 8 "Notation"; pitch PAPER.md:113) */
static double elem_pos(int e, int n, double pitch) { return (e - 0.5 * (n - 1)) * pitch; }

static int n_events(const ulm_oracle_params *p) { return p->n_row_tx + p->n_col_tx; }

static int fir_half_len(const ulm_oracle_params *p)
{
    if (p->demod_taps > 0) return (p->demod_taps - 1) / 2;
    return 2 * (int)lround(p->fs / p->fc); /* L = 2*round(fs/fc): 17 taps at 20 MHz, 33 at 40 MHz */
}

static double sinc_pi(double x) { return x == 0.0 ? 1.0 : sin(M_PI * x) / (M_PI * x); }

/* h[m] ~ sinc(2 fc m / fs) * (0.54 + 0.46 cos(pi m / L)), sum h = 1 */
int ulm_oracle_fir(const ulm_oracle_params *p, double *h, int capacity)
{
    int L = fir_half_len(p);
    if (L < 0 || (p->demod_taps > 0 && p->demod_taps % 2 == 0)) return -1;
    if (capacity < 2 * L + 1) return -2;
    double s = 0.0;
    for (int m = -L; m <= L; ++m) {
        double win = L > 0 ? 0.54 + 0.46 * cos(M_PI * m / L) : 1.0;
        h[m + L] = sinc_pi(2.0 * p->fc * m / p->fs) * win;
        s += h[m + L];
    }
    for (int m = 0; m <= 2 * L; ++m) h[m] /= s;
    return L;
}

/* x[n] = rf[n] exp(-j 2 pi fc t_n); iq[n] = 2 sum_m h[m] x[n-m], x = 0 outside
 * the record.  IQ input: iq[n] = re + j im, no filtering. */
static int demod_channel(const ulm_oracle_params *p, const int16_t *in, double complex *iq,
                         const double *h, int L)
{
    const int ns = p->n_samples;
    if (p->input_kind == 1) {
        for (int n = 0; n < ns; ++n) iq[n] = (double)in[2 * n] + I * (double)in[2 * n + 1];
        return 0;
    }
    double complex *x = (double complex *)malloc(sizeof(double complex) * (size_t)ns);
    if (!x) return -1;
    for (int n = 0; n < ns; ++n) {
        double tn = p->t_start + n / p->fs;
        x[n] = (double)in[n] * cexp(-I * 2.0 * M_PI * p->fc * tn);
    }
    for (int n = 0; n < ns; ++n) {
        double complex s = 0.0;
        for (int m = -L; m <= L; ++m) {
            int q = n - m;
            if (q >= 0 && q < ns) s += h[m + L] * x[q];
        }
        iq[n] = 2.0 * s;
    }
    free(x);
    return 0;
}

int ulm_oracle_demod_channel(const ulm_oracle_params *p, const int16_t *in, double *out)
{
    double h[1025];
    int L = ulm_oracle_fir(p, h, 1025);
    if (L < 0) return -1;
    return demod_channel(p, in, (double complex *)out, h, L);
}

int64_t ulm_oracle_out_per_frame(const ulm_oracle_params *p)
{
    int64_t pxz = (int64_t)p->xz.n_lat * p->xz.n_ax, pyz = (int64_t)p->yz.n_lat * p->yz.n_ax;
    if (p->compound) return pxz + pyz;
    return p->n_row_tx * pxz + p->n_col_tx * pyz;
}

/* number of int16 values per channel record */
static int64_t rec_len(const ulm_oracle_params *p) { return (int64_t)p->n_samples * (p->input_kind == 1 ? 2 : 1); }

/* a row-tx event is received on the columns, a column-tx event on the rows; data may
 * carry all n_rows+n_cols channels (rows first) or only the orthogonal aperture. */
static int rx_channel(const ulm_oracle_params *p, int is_row_tx, int elem)
{
    int full = p->channels_per_event == p->n_rows + p->n_cols;
    if (is_row_tx) return full ? p->n_rows + elem : elem;
    return elem;
}

static int check(const ulm_oracle_params *p)
{
    if (!p || p->n_rows <= 0 || p->n_cols <= 0 || p->n_samples < 2) return -1;
    if (p->n_row_tx < 0 || p->n_col_tx < 0) return -1;
    if (p->channels_per_event != p->n_rows + p->n_cols &&
        !(p->n_rows == p->n_cols && p->channels_per_event == p->n_rows))
        return -1;
    return 0;
}

/* demodulate the receive aperture of every event of one frame: iq[(e*nrx_max + elem)*ns + n] */
static double complex *demod_frame(const ulm_oracle_params *p, const int16_t *frame, int *nrx_max_out)
{
    double h[1025];
    int L = ulm_oracle_fir(p, h, 1025);
    if (L < 0) return NULL;
    const int ne = n_events(p), ns = p->n_samples;
    const int nrx_max = p->n_rows > p->n_cols ? p->n_rows : p->n_cols;
    double complex *iq = (double complex *)calloc((size_t)ne * nrx_max * ns, sizeof(double complex));
    if (!iq) return NULL;
    int fail = 0;
#pragma omp parallel for schedule(static) collapse(2)
    for (int e = 0; e < ne; ++e)
        for (int elem = 0; elem < nrx_max; ++elem) {
            int is_row_tx = e < p->n_row_tx;
            int nrx = is_row_tx ? p->n_cols : p->n_rows;
            if (elem >= nrx) continue;
            const int16_t *rec =
                frame + ((int64_t)e * p->channels_per_event + rx_channel(p, is_row_tx, elem)) * rec_len(p);
            if (demod_channel(p, rec, iq + ((size_t)e * nrx_max + elem) * ns, h, L)) fail = 1;
        }
    if (fail) { free(iq); return NULL; }
    *nrx_max_out = nrx_max;
    return iq;
}

/* boxcar f-number mask, w_j = [f_number = 0 or |lat - lat_j| <= z / (2 f_number)],
 * evaluated in fp64 exactly as the definition writes it (the edge is inclusive). */
static int in_aperture(double f_number, double lat, double lat_elem, double z)
{
    if (f_number == 0.0) return 1;
    return fabs(lat - lat_elem) <= z / (2.0 * f_number);
}

/*
 * SURVEY 8(c) steps 1-2 for one image of one frame.
 *   tau = t0_k + (z cos(th_k) + ref sin(th_k))/c + sqrt((lat - lat_j)^2 + z^2)/c
 *   u = (tau - t_start) fs, n = floor(u), a = u - n; term = 0 unless 0 <= n and n+1 <= Ns-1
 *   v = (1-a) iq[n] + a iq[n+1]
 *   P(lat, z) = sum_k sum_j w_j(lat, z) v exp(+j 2 pi fc tau)          (no normalisation)
 * is_row_tx = 1: XZ image (lat = x, elements = columns, events 0..n_row_tx-1);
 * is_row_tx = 0: YZ image (lat = y, elements = rows, events n_row_tx..).
 * compound = 0: the k-sum is not taken and image k is written to out + k*n_lat*n_ax.
 */
static void project(const ulm_oracle_params *p, int is_row_tx, const double complex *iq, int nrx_max,
                    double complex *out)
{
    const ulm_oracle_grid *g = is_row_tx ? &p->xz : &p->yz;
    const int n_tx = is_row_tx ? p->n_row_tx : p->n_col_tx;
    const double *angles = is_row_tx ? p->row_tx_angles : p->col_tx_angles;
    const int e0 = is_row_tx ? 0 : p->n_row_tx;
    const int n_el = is_row_tx ? p->n_cols : p->n_rows;
    const double *win = p->elem_window ? p->elem_window + (is_row_tx ? 0 : p->n_cols) : NULL;
    const int ns = p->n_samples;
    const int64_t npix = (int64_t)g->n_lat * g->n_ax;

#pragma omp parallel for schedule(dynamic, 1)
    for (int il = 0; il < g->n_lat; ++il) {
        const double lat = g->lat0 + il * g->dlat;
        for (int iz = 0; iz < g->n_ax; ++iz) {
            const double z = g->z0 + iz * g->dz;
            double complex sum = 0.0;
            for (int k = 0; k < n_tx; ++k) {
                const double th = angles[k];
                const double t0 = p->t0 ? p->t0[e0 + k] : 0.0;
                double complex acc = 0.0;
                for (int j = 0; j < n_el; ++j) {
                    const double lat_j = elem_pos(j, n_el, p->pitch);
                    const double tau = t0 + (z * cos(th) + g->ref * sin(th)) / p->c +
                                       sqrt((lat - lat_j) * (lat - lat_j) + z * z) / p->c;
                    const double u = (tau - p->t_start) * p->fs;
                    const double nf = floor(u);
                    if (!(nf >= 0.0 && nf + 1.0 <= ns - 1)) continue;
                    const int n = (int)nf;
                    const double a = u - nf;
                    const double complex *s = iq + ((size_t)(e0 + k) * nrx_max + j) * ns;
                    const double complex v = (1.0 - a) * s[n] + a * s[n + 1];
                    double w = win ? win[j] : 1.0;
                    if (!in_aperture(p->f_number, lat, lat_j, z)) w = 0.0;
                    acc += w * v * cexp(I * 2.0 * M_PI * p->fc * tau);
                }
                if (p->compound) sum += acc;
                else out[(int64_t)k * npix + (int64_t)il * g->n_ax + iz] = acc;
            }
            if (p->compound) out[(int64_t)il * g->n_ax + iz] = sum;
        }
    }
}

int ulm_oracle_beamform(const ulm_oracle_params *p, const int16_t *channel, int32_t n_frames, double *out)
{
    if (check(p) || !channel || !out || n_frames < 0) return -1;
    const int64_t per_frame_in = (int64_t)n_events(p) * p->channels_per_event * rec_len(p);
    const int64_t per_frame_out = ulm_oracle_out_per_frame(p);
    const int64_t pxz = (int64_t)p->xz.n_lat * p->xz.n_ax;
    for (int f = 0; f < n_frames; ++f) {
        int nrx_max = 0;
        double complex *iq = demod_frame(p, channel + f * per_frame_in, &nrx_max);
        if (!iq) return -2;
        double complex *o = (double complex *)out + f * per_frame_out;
        project(p, 1, iq, nrx_max, o);
        project(p, 0, iq, nrx_max, o + (p->compound ? pxz : (int64_t)p->n_row_tx * pxz));
        free(iq);
    }
    return 0;
}

/*
 * SURVEY 8(c) step 4 (the "conventional 3D processing" of PAPER.md:45-47), written point-outer with
 * one loop over ALL events and its own delay expressions:
 *   RC event (tx rows, angle th, rx column j): tau = t0 + (z cos th + y sin th)/c + sqrt((x-x_j)^2+z^2)/c
 *   CR event (tx cols, angle th, rx row i):    tau = t0 + (z cos th + x sin th)/c + sqrt((y-y_i)^2+z^2)/c
 * V_RC and V_CR are returned separately (V = V_RC + V_CR, coherent sum).
 */
int ulm_oracle_das_points(const ulm_oracle_params *p, const int16_t *channel, const double *xyz,
                          int64_t n_pts, double *v_rc_out, double *v_cr_out)
{
    if (check(p) || !channel || !xyz || !v_rc_out || !v_cr_out || n_pts < 0) return -1;
    int nrx_max = 0;
    double complex *iq = demod_frame(p, channel, &nrx_max);
    if (!iq) return -2;
    double complex *v_rc = (double complex *)v_rc_out, *v_cr = (double complex *)v_cr_out;
    const int ns = p->n_samples, ne = n_events(p);
    const double two_pi_fc = 2.0 * M_PI * p->fc;

#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t q = 0; q < n_pts; ++q) {
        const double x = xyz[3 * q], y = xyz[3 * q + 1], z = xyz[3 * q + 2];
        double complex s_rc = 0.0, s_cr = 0.0;
        for (int e = 0; e < ne; ++e) {
            const int rc = e < p->n_row_tx;
            const double th = rc ? p->row_tx_angles[e] : p->col_tx_angles[e - p->n_row_tx];
            const double along_tx = rc ? y : x;   /* coordinate the plane wave is steered along */
            const double across = rc ? x : y;     /* coordinate resolved by the receive aperture */
            const int n_el = rc ? p->n_cols : p->n_rows;
            const double *win = p->elem_window ? p->elem_window + (rc ? 0 : p->n_cols) : NULL;
            const double tau_tx = (p->t0 ? p->t0[e] : 0.0) + (z * cos(th) + along_tx * sin(th)) / p->c;
            for (int el = 0; el < n_el; ++el) {
                const double pe = (el - (n_el - 1) / 2.0) * p->pitch;
                const double tau = tau_tx + hypot(across - pe, z) / p->c;
                const double u = (tau - p->t_start) * p->fs;
                const long n = (long)floor(u);
                if (n < 0 || n + 1 > ns - 1) continue;
                const double a = u - (double)n;
                const double complex *s = iq + ((size_t)e * nrx_max + el) * ns;
                double complex v = s[n] + a * (s[n + 1] - s[n]);
                double w = win ? win[el] : 1.0;
                if (!in_aperture(p->f_number, across, pe, z)) w = 0.0;
                v *= w * (cos(two_pi_fc * tau) + I * sin(two_pi_fc * tau));
                if (rc) s_rc += v; else s_cr += v;
            }
        }
        v_rc[q] = s_rc;
        v_cr[q] = s_cr;
    }
    free(iq);
    return 0;
}
