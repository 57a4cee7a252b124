// ulm_rca_ring.cuh -- shared-memory ring DAS kernel (placeholder until the kernel lands: ring_plan()
// declines every shape, so the generic gather kernel runs).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

namespace ulm {

struct RingConfig {
    int frames = 0, tile_pixels = 0, window = 0, stages = 0, smem_bytes = 0;
};

struct RingTables {
    int n_tiles = 0;
};

struct RingApertureDesc {
    int n_tx, n_rx, n_lat, n_ax;
    double lat0, dlat, z0, dz, ref;
    const double *angles, *t0;
};

struct RingApertureArgs {
    int e0, n_tx, n_rx, n_lat, n_ax;
    const float *xs, *zs, *ejs, *xm, *zm, *ejm, *win;
    const int *n0;
    const float *f0m;
    long long out_base;
};

struct RingLaunch {
    const float4 *iq;
    int l_row, n_rx_max, n_events;
    float2 *out;
    long long out_frame_stride;
    int n_frames;
    double fcfs, fct;
    int n_lo;
    float two_f;
    RingApertureArgs ap[2];
};

inline bool ring_plan(const RingApertureDesc *, double, double, double, double, int, int, bool, RingConfig &,
                      RingTables &, RingTables &, const char **why) {
    if (why) *why = "not built yet";
    return false;
}

inline int ring_launch(const RingConfig &, const RingTables &, const RingTables &, const RingLaunch &, bool,
                       cudaStream_t) {
    return 0;
}

}  // namespace ulm
