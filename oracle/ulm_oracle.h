/*
 * ulm_oracle.h -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, fp64 CPU statement of what the RCA Stage-1 projection beamformer of
 * arxiv 2511.21647 computes (Section II.A.1 "Beamforming"; grid sizes at
 * PAPER.md:117).  The paper gives no formula for this step, so the definition written out here
 * is the one fixed in SURVEY.md section 8(c) (readings A1-A13, restated in DESIGN.md).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * build, load or call this library.  It shares no code, header, table or constant with the CUDA
 * path under paper_2511_21647_b200/ and neither includes the other.
 *
 * Parity pins (tests/test_oracle_pins.py): P1 impulse closed form, P2 phase convention and the
 * f-number mask counted over whole grids against the fp64 inequality (near-edge and on-edge pairs),
 * P3 demodulation of a pure tone and the FIR taps against literal values and numpy's sinc / hamming,
 * P4 independently coded 3-D DAS == projection on the reference plane, P5 linearity,
 * P7 point-scatterer peak, P8 symmetries, P9 work count.
 * Every decision and every value in this file is fp64.  Parity unpinned: nothing in this file.
 */
#ifndef ULM_ORACLE_H
#define ULM_ORACLE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* One lateral x axial image grid (SURVEY.md 8(b) ulm_rca_grid): lateral coordinate of pixel il is
 * lat0 + il*dlat (x for the XZ image, y for the YZ image), depth of pixel iz is z0 + iz*dz;
 * ref is the coordinate of the reference slice along the transmit direction (y_ref for XZ,
 * x_ref for YZ; "central slices along the transmit directions", Fig. 1b). */
typedef struct {
    int32_t n_lat;
    double lat0, dlat;
    int32_t n_ax;
    double z0, dz;
    double ref;
} ulm_oracle_grid;

typedef struct {
    /* array: n_rows row elements (long in x, centred at y_i), n_cols column elements (long in y,
     * centred at x_j); centre coordinate of element e of n is (e - (n-1)/2)*pitch */
    int32_t n_rows, n_cols;
    double pitch;
    /* steering angles in radians: row-tx plane waves steer in the y-z plane, column-tx in x-z */
    int32_t n_row_tx, n_col_tx;
    const double *row_tx_angles;
    const double *col_tx_angles;
    double c, fs, fc;
    ulm_oracle_grid xz, yz;
    int32_t input_kind;         /* 0: RF int16 real; 1: IQ int16 interleaved (re, im)             */
    int32_t channels_per_event; /* n_rows + n_cols (rows first), or the orthogonal aperture only    */
    int32_t n_samples;
    double t_start;             /* time of sample 0                                                 */
    const double *t0;           /* per-event time offset [n_row_tx + n_col_tx], NULL = 0            */
    double f_number;            /* 0 = full aperture                                                */
    const double *elem_window;  /* static receive weight per receive element of each aperture:
                                   [n_cols] for XZ followed by [n_rows] for YZ; NULL = ones         */
    int32_t demod_taps;         /* odd; 0 = default 4*round(fs/fc)+1                                */
    int32_t compound;           /* 1: sum over angles; 0: emit per-event slices                     */
} ulm_oracle_params;

/* number of threads the OpenMP loops will use */
int ulm_oracle_threads(void);

/* SURVEY 8(c) step 0.  h[0..2L] <- normalised taps (h[m+L] for m=-L..L); returns L, or <0. */
int ulm_oracle_fir(const ulm_oracle_params *p, double *h, int capacity);

/* SURVEY 8(c) step 0 on one channel.  in: n_samples int16 (RF) or 2*n_samples (IQ);
 * out: n_samples interleaved (re, im) doubles. */
int ulm_oracle_demod_channel(const ulm_oracle_params *p, const int16_t *in, double *out);

/* number of complex output values per frame of ulm_oracle_beamform */
int64_t ulm_oracle_out_per_frame(const ulm_oracle_params *p);

/* SURVEY 8(c) steps 1-3.  channel: [frame][event][channel][sample] int16 (x2 for IQ input), events =
 * row-tx angles then column-tx angles.  out: interleaved complex doubles,
 * compound=1: [frame][XZ: n_lat*n_ax | YZ: n_lat*n_ax] (axial fastest);
 * compound=0: [frame][event][lat][ax] (row-tx events on the XZ grid, column-tx on the YZ grid). */
int ulm_oracle_beamform(const ulm_oracle_params *p, const int16_t *channel, int32_t n_frames,
                        double *out);

/* SURVEY 8(c) step 4, coded voxel-outer on an arbitrary list of points (independent of the
 * projection loops above; used for pin P4 and as the config-4 accuracy reference).
 * channel: ONE frame.  xyz: n_pts * 3 doubles.  v_rc, v_cr: n_pts interleaved complex each. */
int ulm_oracle_das_points(const ulm_oracle_params *p, const int16_t *channel, const double *xyz,
                          int64_t n_pts, double *v_rc, double *v_cr);

#ifdef __cplusplus
}
#endif
#endif
