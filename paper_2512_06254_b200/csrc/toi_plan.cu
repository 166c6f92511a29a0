// toi_plan.cu -- the C ABI of include/toi.h: plan (all memory, cuFFT plan, streams, events),
// the per-snapshot stage sequence a1..a7 and the streamed pipeline a8.
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <chrono>
#include <cmath>
#include <new>
#include <vector>

#include "toi_internal.cuh"

using namespace toi;

namespace {

thread_local char g_create_error[512] = "";

struct DevSlot {
    double *uvw = nullptr;
    float2 *vis = nullptr;
    float *weights = nullptr;
    uint8_t *flags = nullptr;
};

enum { EV_START = 0, EV_H2D, EV_FIT, EV_WEIGHT, EV_GRID, EV_FFT, EV_CROP, EV_COUNT };

}  // namespace

struct toi_plan {
    toi_config cfg;
    Geometry geo;
    double S1 = 0, S2 = 0;
    int n_sms = 148;
    int apply_jacobian = 1;
    size_t n_samples = 0, n_elems = 0;

    double *d_s = nullptr, *d_ipsi = nullptr, *d_V_inject = nullptr, *d_V_reproject = nullptr;
    SnapState *d_state = nullptr, *h_state = nullptr;    // d_state: the current snapshot's, one of
    SnapState *d_state_slots = nullptr;                  // two slots taken in turn: the plane fit of snapshot n + 1
    unsigned state_pos = 0;                              // never writes what consumers of snapshot n (re-projection) read
    DevSlot dev_in[2];
    toi_snapshot_buffers pin[2] = {{nullptr, nullptr, nullptr, nullptr}, {nullptr, nullptr, nullptr, nullptr}};
    // ONE gridding grid (with guard band) and ONE density map, both zero between snapshots: the
    // gridder / density pass mark the 128x8-cell tiles they write in a byte map and, once the first
    // FFT pass has read the grid OUT OF PLACE into d_work, only those tiles are zeroed again
    // (k_clear.cu).  The rest of the transform and the crop run on d_work.
    float2 *d_grid = nullptr, *d_grid_alloc = nullptr;   // d_grid = d_grid_alloc + grid_guard(G)
    float2 *d_work = nullptr;                            // FFT workspace, G x G
    float *d_dens = nullptr;
    uint8_t *d_tiles_grid = nullptr;
    size_t n_tiles = 0;
    bool s_monotone = true;      // channel scales monotone: the gridder can bound a strip's tiles by its ends
    float2 *d_grid_keep = nullptr;                       // cfg.debug_keep_grid
    float *d_dens_keep = nullptr;
    cudaEvent_t ev_done = nullptr;                       // end of the last imaging call, recorded only when the next
    cudaStream_t last_stream = nullptr;                  // call comes on ANOTHER stream than last_stream (an event
    bool have_last = false;                              // record between two kernels would break their launch overlap)
    cudaEvent_t ev_clear0 = nullptr, ev_clear1 = nullptr, ev_clear2 = nullptr;
    bool timed_density_clear = false;  // the last timed call cleared the density map between ev_clear1 and ev_clear2
    float *d_images = nullptr;
    int ring_depth = 5;
    long long ring_pos = 0;                              // image ring only
    bool inject = false, keep_grid = false;
    int snap_slot = 0;
    Inputs last_in = {nullptr, nullptr, nullptr, nullptr};

    cufftHandle fft = 0, fft_cols = 0, fft_rows = 0;
    bool fft_ok = false, fft_pruned = false;
    bool fft_custom = false;                             // k_fft.cu instead of cuFFT (+ k_correct_crop)
    float2 *d_tw = nullptr;                              // its twiddle table, G entries
    float2 *d_moment[2] = {nullptr, nullptr};            // 3-D mode: the cropped complex transform [N][N] of a pass, per lane
    cudaStream_t s_compute = nullptr, s_copy = nullptr, fft_stream = nullptr;
    cudaEvent_t ev[EV_COUNT] = {};
    cudaEvent_t ev_h2d_start[2] = {}, ev_h2d_done[2] = {}, ev_c_start[2] = {}, ev_c_done[2] = {}, ev_first = nullptr;

    // output side of the streamed run (toi_stream_set_output): re-projected image ring, difference
    // ping-pong, pinned depth-2 D2H ring on its own stream
    toi_stream_output out_cfg = {};
    float *d_products = nullptr, *d_diff[2] = {nullptr, nullptr}, *h_out[2] = {nullptr, nullptr};
    cudaStream_t s_d2h = nullptr;
    cudaEvent_t ev_out_ready[2] = {}, ev_d2h_start[2] = {}, ev_d2h_done[2] = {}, ev_tail = nullptr;

    // near-coplanar (3-D) mode (cfg.enable_3d): complex accumulator, r3 range on the device and in
    // pinned host memory, Bessel table; the passes run on d_grid / d_work like the 2-D path
    float2 *d_acc3 = nullptr, *d_slab3 = nullptr;        // total and per-slab sums of the 3-D mode, [N][N] each
    double *d_r3 = nullptr, *h_r3 = nullptr;
    float *d_jtab = nullptr;                             // Bessel table of the 3-D mode
    // second lane of the 3-D mode (hand-written transform only): odd passes grid, transform and combine
    // on their own grid / workspace / tile map on s_lane1, so that one pass's transform runs under the
    // next pass's gridding; the gridders and the combinations of the two lanes are chained by events
    float2 *d_grid1 = nullptr, *d_grid1_alloc = nullptr, *d_work1 = nullptr;
    uint8_t *d_tiles1 = nullptr;
    cudaStream_t s_lane1 = nullptr;
    cudaEvent_t ev_lane_grid[2] = {}, ev_lane_comb[2] = {}, ev_lane_setup = nullptr, ev_lane_cols0 = nullptr;
    double s_min = 0, s_max = 0;
    cudaEvent_t ev3_a = nullptr, ev3_b = nullptr;

    int deferred = TOI_OK;
    int last_launches = 0;
    char err[512] = "";
};

namespace {

int fail(toi_plan *p, int code, const char *fmt, const char *a = "", const char *b = "")
{
    char *dst = p ? p->err : g_create_error;
    snprintf(dst, 512, fmt, a, b);
    if (p && p->deferred == TOI_OK) p->deferred = code;
    return code;
}

#define CU_TRY(p, expr)                                                                 \
    do {                                                                                \
        cudaError_t e_ = (expr);                                                        \
        if (e_ != cudaSuccess) return fail((p), e_ == cudaErrorMemoryAllocation ? TOI_ERR_NOMEM : TOI_ERR_CUDA, \
                                           "%s: %s", #expr, cudaGetErrorString(e_));    \
    } while (0)

// ---- grid-correction table (G11) ------------------------------------------------
// psi(n) = int_{-W/2}^{W/2} phi(x) cos(2 pi x n / G) dx.  With x = (W/2) sin(theta) the square-root
// end-point behaviour of phi disappears:
//   psi(n) = W int_0^{pi/2} exp(beta_k (cos(theta) - 1)) cos(pi W n sin(theta) / G) cos(theta) dtheta,
// an analytic integrand that Gauss-Legendre integrates to rounding with a few dozen nodes.
void legendre_rule(int n, std::vector<double> &x, std::vector<double> &w)
{
    x.assign(n, 0.0);
    w.assign(n, 0.0);
    const double pi = 3.141592653589793238462643383279502884;
    for (int i = 0; i < n; ++i) {
        double z = cos(pi * (i + 0.75) / (n + 0.5)), dp = 1.0;
        for (int it = 0; it < 50; ++it) {
            double p0 = 1.0, p1 = z;                       // P_0, P_1
            for (int k = 2; k <= n; ++k) {
                const double pk = ((2 * k - 1) * z * p1 - (k - 1) * p0) / k;
                p0 = p1; p1 = pk;
            }
            dp = n * (z * p1 - p0) / (z * z - 1.0);        // P_n'(z)
            const double step = p1 / dp;
            z -= step;
            if (fabs(step) < 4e-16) break;
        }
        x[i] = z;
        w[i] = 2.0 / ((1.0 - z * z) * dp * dp);
    }
}

void correction_table(int N, int G, std::vector<double> &ipsi)
{
    const int nodes = 96;
    std::vector<double> x, w;
    legendre_rule(nodes, x, w);
    const double pi = 3.141592653589793238462643383279502884;
    const double beta = 2.30 * kW;
    std::vector<double> ct(nodes), st(nodes), wt(nodes);
    for (int k = 0; k < nodes; ++k) {
        const double th = 0.25 * pi * (x[k] + 1.0);        // [0, pi/2]
        ct[k] = cos(th); st[k] = sin(th);
        wt[k] = 0.25 * pi * w[k] * kW * exp(beta * (ct[k] - 1.0)) * ct[k];
    }
    ipsi.assign(N, 0.0);
    for (int i = 0; i < N; ++i) {
        const double f = pi * kW * (double)(i - N / 2) / (double)G;
        double acc = 0.0;
        for (int k = 0; k < nodes; ++k) acc += wt[k] * cos(f * st[k]);
        ipsi[i] = 1.0 / acc;
    }
}

int free_plan(toi_plan *p)
{
    if (!p) return TOI_OK;
    cudaSetDevice(p->cfg.device);
    if (p->s_compute) cudaStreamSynchronize(p->s_compute);
    if (p->s_copy) cudaStreamSynchronize(p->s_copy);
    if (p->fft_ok) cufftDestroy(p->fft);
    if (p->fft_pruned) { cufftDestroy(p->fft_cols); cufftDestroy(p->fft_rows); }
    cudaFree(p->d_s); cudaFree(p->d_ipsi); cudaFree(p->d_V_inject); cudaFree(p->d_V_reproject); cudaFree(p->d_state_slots);
    cudaFreeHost(p->h_state);
    for (int k = 0; k < 2; ++k) {
        cudaFree(p->dev_in[k].uvw); cudaFree(p->dev_in[k].vis);
        cudaFree(p->dev_in[k].weights); cudaFree(p->dev_in[k].flags);
        cudaFreeHost(p->pin[k].uvw_m); cudaFreeHost(p->pin[k].vis);
        cudaFreeHost(p->pin[k].weights); cudaFreeHost(p->pin[k].flags);
        if (p->ev_h2d_start[k]) cudaEventDestroy(p->ev_h2d_start[k]);
        if (p->ev_h2d_done[k]) cudaEventDestroy(p->ev_h2d_done[k]);
        if (p->ev_c_start[k]) cudaEventDestroy(p->ev_c_start[k]);
        if (p->ev_c_done[k]) cudaEventDestroy(p->ev_c_done[k]);
    }
    if (p->ev_first) cudaEventDestroy(p->ev_first);
    for (int k = 0; k < EV_COUNT; ++k)
        if (p->ev[k]) cudaEventDestroy(p->ev[k]);
    cudaFree(p->d_grid_alloc); cudaFree(p->d_work); cudaFree(p->d_dens); cudaFree(p->d_tw);
    cudaFree(p->d_moment[0]); cudaFree(p->d_moment[1]);
    cudaFree(p->d_tiles_grid);
    cudaFree(p->d_grid_keep); cudaFree(p->d_dens_keep);
    if (p->ev_done) cudaEventDestroy(p->ev_done);
    if (p->ev_clear0) cudaEventDestroy(p->ev_clear0);
    if (p->ev_clear1) cudaEventDestroy(p->ev_clear1);
    if (p->ev_clear2) cudaEventDestroy(p->ev_clear2);
    if (p->s_d2h) cudaStreamSynchronize(p->s_d2h);
    cudaFree(p->d_products);
    for (int k = 0; k < 2; ++k) {
        cudaFree(p->d_diff[k]);
        cudaFreeHost(p->h_out[k]);
        if (p->ev_out_ready[k]) cudaEventDestroy(p->ev_out_ready[k]);
        if (p->ev_d2h_start[k]) cudaEventDestroy(p->ev_d2h_start[k]);
        if (p->ev_d2h_done[k]) cudaEventDestroy(p->ev_d2h_done[k]);
    }
    if (p->ev_tail) cudaEventDestroy(p->ev_tail);
    if (p->s_d2h) cudaStreamDestroy(p->s_d2h);
    cudaFree(p->d_acc3); cudaFree(p->d_slab3); cudaFree(p->d_r3); cudaFree(p->d_jtab);
    if (p->s_lane1) cudaStreamSynchronize(p->s_lane1);
    cudaFree(p->d_grid1_alloc); cudaFree(p->d_work1); cudaFree(p->d_tiles1);
    for (int k = 0; k < 2; ++k) {
        if (p->ev_lane_grid[k]) cudaEventDestroy(p->ev_lane_grid[k]);
        if (p->ev_lane_comb[k]) cudaEventDestroy(p->ev_lane_comb[k]);
    }
    if (p->ev_lane_setup) cudaEventDestroy(p->ev_lane_setup);
    if (p->ev_lane_cols0) cudaEventDestroy(p->ev_lane_cols0);
    if (p->s_lane1) cudaStreamDestroy(p->s_lane1);
    cudaFreeHost(p->h_r3);
    if (p->ev3_a) cudaEventDestroy(p->ev3_a);
    if (p->ev3_b) cudaEventDestroy(p->ev3_b);
    cudaFree(p->d_images);
    if (p->s_compute) cudaStreamDestroy(p->s_compute);
    if (p->s_copy) cudaStreamDestroy(p->s_copy);
    cudaGetLastError();
    delete p;
    return TOI_OK;
}

int set_fft_stream(toi_plan *p, cudaStream_t stream)
{
    if (p->fft_stream == stream) return TOI_OK;
    if (p->fft_ok && cufftSetStream(p->fft, stream) != CUFFT_SUCCESS) return fail(p, TOI_ERR_CUFFT, "cufftSetStream failed");
    if (p->fft_pruned && (cufftSetStream(p->fft_cols, stream) != CUFFT_SUCCESS ||
                          cufftSetStream(p->fft_rows, stream) != CUFFT_SUCCESS))
        return fail(p, TOI_ERR_CUFFT, "cufftSetStream failed");
    p->fft_stream = stream;
    return TOI_OK;
}

// One grid, one workspace: a call on another stream than the previous call's waits for that call's last
// kernel; on the same stream the stream order already says so.  Also takes the next SnapState slot.
int follow_previous_call(toi_plan *p, cudaStream_t stream)
{
    if (p->have_last && p->last_stream != stream) {
        if (cudaEventRecord(p->ev_done, p->last_stream) == cudaSuccess) {
            CU_TRY(p, cudaStreamWaitEvent(stream, p->ev_done, 0));
        } else {                                 // the caller destroyed that stream: its work is done or draining
            cudaGetLastError();
            CU_TRY(p, cudaDeviceSynchronize());
        }
    }
    p->last_stream = stream;
    p->have_last = true;
    p->d_state = p->d_state_slots + (++p->state_pos & 1u);       // this snapshot's SnapState
    return TOI_OK;
}

// The gridder marks the tiles it writes only when the channel scales are monotone (it bounds a
// strip by its two end samples); otherwise, and for the strawman gridder, every tile is marked here.
uint8_t *gridder_tile_map(toi_plan *p, cudaStream_t stream, bool sliding, uint8_t *map)
{
    if (sliding && p->s_monotone) return map;
    cudaMemsetAsync(map, 1, p->n_tiles, stream);
    return nullptr;
}

// a6 + sparse clear (+ a7): the first transform pass reads the grid OUT OF PLACE into the workspace,
// after which the tiles the gridder touched are zeroed again for the next snapshot (or pass); the
// second pass runs on the workspace.  d_image != nullptr: correction + crop + normalisation into that
// image follow (fused into the second pass by the hand-written transform); nullptr (3-D mode): the
// complex transform is left in the workspace (cuFFT) or, cropped, in d_moment[lane] (hand-written
// transform).  `timed`: record the stage events of the 2-D path.
int transform_and_clear(toi_plan *p, cudaStream_t stream, float2 *d_grid, uint8_t *d_tiles, float2 *d_work,
                        bool clear_density, bool timed, float *d_image, int lane, cudaEvent_t before_cols, int *launches)
{
    const Geometry &g = p->geo;
    cufftComplex *A = (cufftComplex *)d_grid, *F = (cufftComplex *)d_work;
    if (p->fft_custom) {
        launch_fft_rows(g.N, g.G, d_grid, d_work, d_tiles, p->d_tw, p->n_sms, stream);
    } else if (p->fft_pruned) {
        // row transforms of all G rows (contiguous), then column transforms of only the N columns
        // the crop reads (columns n = -N/2..N/2-1 live at indices [0, N/2) and [G - N/2, G))
        if (cufftExecC2C(p->fft_rows, A, F, CUFFT_INVERSE) != CUFFT_SUCCESS) return fail(p, TOI_ERR_CUFFT, "cufftExecC2C failed");
    } else {
        if (cufftExecC2C(p->fft, A, F, CUFFT_INVERSE) != CUFFT_SUCCESS) return fail(p, TOI_ERR_CUFFT, "cufftExecC2C failed");
    }
    ++*launches;
    // The sparse clear: a launch of its own between the passes when the call is timed (ms_clear is then
    // what it costs by itself, and that is what the roofline accounting charges the gridding with);
    // otherwise, with the hand-written transform at G <= 4096, inside the column pass (its stores run
    // under that pass's shared-memory work: 0.006-0.014 ms per snapshot less at config 2; at G = 8192
    // and 16384 the column pass has one CTA of 8-16 warps per SM and the clear is faster by itself).
    const bool clear_in_cols = p->fft_custom && !timed && g.G <= 4096;
    float *dens_to_clear = clear_density ? p->d_dens : nullptr;
    if (!clear_in_cols && !timed) {
        launch_clear_tiles(d_grid, dens_to_clear, g.G, d_tiles, stream);
        ++*launches;
    } else if (!clear_in_cols) {
        // timed: the grid's clear (ms_clear, charged to the gridding) and the density map's
        // (ms_clear_density, charged to the weighting) as two launches, each between its own events
        CU_TRY(p, cudaEventRecord(p->ev_clear0, stream));
        launch_clear_tiles(d_grid, nullptr, g.G, d_tiles, stream, dens_to_clear == nullptr);
        ++*launches;
        CU_TRY(p, cudaEventRecord(p->ev_clear1, stream));
        p->timed_density_clear = dens_to_clear != nullptr;
        if (dens_to_clear) {
            launch_clear_tiles(nullptr, dens_to_clear, g.G, d_tiles, stream);
            ++*launches;
        }
        CU_TRY(p, cudaEventRecord(p->ev_clear2, stream));
    }
    if (before_cols) CU_TRY(p, cudaStreamWaitEvent(stream, before_cols, 0));     // what still reads this lane's moment
    if (p->fft_custom) {
        launch_fft_cols(g.N, g.G, d_work, p->d_tw, p->d_ipsi, p->d_state, p->apply_jacobian, d_image,
                        d_image ? nullptr : p->d_moment[lane], clear_in_cols ? d_grid : nullptr,
                        clear_in_cols ? dens_to_clear : nullptr, clear_in_cols ? d_tiles : nullptr, p->n_sms, stream);
        ++*launches;
        if (timed) CU_TRY(p, cudaEventRecord(p->ev[EV_FFT], stream));
        return TOI_OK;
    }
    if (p->fft_pruned) {
        cufftComplex *Fhi = F + (g.G - g.N / 2);
        if (cufftExecC2C(p->fft_cols, F, F, CUFFT_INVERSE) != CUFFT_SUCCESS ||
            cufftExecC2C(p->fft_cols, Fhi, Fhi, CUFFT_INVERSE) != CUFFT_SUCCESS)
            return fail(p, TOI_ERR_CUFFT, "cufftExecC2C failed");
        *launches += 2;
    }
    if (timed) CU_TRY(p, cudaEventRecord(p->ev[EV_FFT], stream));
    if (d_image) {
        launch_correct_crop(g, d_work, p->d_ipsi, p->d_state, p->apply_jacobian, d_image, stream);
        ++*launches;
    }
    return TOI_OK;
}

// Enqueue stages a1..a7 for the snapshot resident at `in` on `stream`; returns the image slot.
// `timed`: record the per-stage events toi_snapshot_info is read from (a timed event between two kernels
// costs 1-2 us of the stream's time; only calls that ask for the info pay for them).
int enqueue_imaging(toi_plan *p, const Inputs &in, cudaStream_t stream, float **d_image_out, bool timed)
{
    const Geometry &g = p->geo;
    const size_t GG = (size_t)g.G * g.G;
    int launches = 0;
    int rc = set_fft_stream(p, stream);
    if (rc) return rc;
    rc = follow_previous_call(p, stream);
    if (rc) return rc;
    const bool uniform = p->cfg.weighting == TOI_WEIGHT_UNIFORM;
    // a1-a2: plane fit (also resets the per-snapshot accumulators)
    launch_planefit(g, in.uvw, p->S1, p->S2, p->inject ? p->d_V_inject : nullptr, p->d_state, stream);
    ++launches;
    if (timed) CU_TRY(p, cudaEventRecord(p->ev[EV_FIT], stream));
    // a4: uniform-weighting density pass
    const float *dens = nullptr;
    if (uniform) {
        launch_density(g, in, p->d_state, p->d_dens, stream);
        dens = p->d_dens;
        ++launches;
    }
    if (timed) CU_TRY(p, cudaEventRecord(p->ev[EV_WEIGHT], stream));
    // a3 + a5: cell indices and gridding onto the zero grid
    const bool sliding = p->cfg.gridder != TOI_GRIDDER_ATOMIC;
    uint8_t *tiles = gridder_tile_map(p, stream, sliding, p->d_tiles_grid);
    if (sliding)
        launch_grid_pair8(g, in, p->d_state, dens, p->d_grid, tiles, p->n_sms, stream);
    else
        launch_grid_atomic(g, in, p->d_state, dens, p->d_grid, stream);
    launches += tiles ? 1 : 2;
    if (timed) CU_TRY(p, cudaEventRecord(p->ev[EV_GRID], stream));
    if (p->keep_grid) {
        CU_TRY(p, cudaMemcpyAsync(p->d_grid_keep, p->d_grid, GG * sizeof(float2), cudaMemcpyDeviceToDevice, stream));
        if (uniform) CU_TRY(p, cudaMemcpyAsync(p->d_dens_keep, p->d_dens, GG * sizeof(float), cudaMemcpyDeviceToDevice, stream));
    }
    // a6: inverse C2C FFT, grid -> workspace, with the sparse clear of the grid inside;
    // a7: correction + crop + normalisation into the image ring (fused into the transform's second
    // pass when the hand-written transform runs: ms_crop is then ~0 and ms_fft holds both)
    float *img = p->d_images + (size_t)(p->ring_pos % p->ring_depth) * g.N * g.N;
    ++p->ring_pos;
    rc = transform_and_clear(p, stream, p->d_grid, p->d_tiles_grid, p->d_work, uniform, timed, img, 0, nullptr, &launches);
    if (rc) return rc;
    if (timed) CU_TRY(p, cudaEventRecord(p->ev[EV_CROP], stream));
    CU_TRY(p, cudaGetLastError());
    p->last_in = in;
    p->last_launches = launches;
    if (d_image_out) *d_image_out = img;
    return TOI_OK;
}

int h2d_slot(toi_plan *p, int slot, const double *uvw, const void *vis, const float *weights,
             const uint8_t *flags, cudaStream_t stream, Inputs &in)
{
    DevSlot &d = p->dev_in[slot];
    const Geometry &g = p->geo;
    CU_TRY(p, cudaMemcpyAsync(d.uvw, uvw, (size_t)g.n_b * 3 * sizeof(double), cudaMemcpyHostToDevice, stream));
    CU_TRY(p, cudaMemcpyAsync(d.vis, vis, p->n_elems * sizeof(float2), cudaMemcpyHostToDevice, stream));
    if (weights) CU_TRY(p, cudaMemcpyAsync(d.weights, weights, p->n_elems * sizeof(float), cudaMemcpyHostToDevice, stream));
    if (flags) CU_TRY(p, cudaMemcpyAsync(d.flags, flags, p->n_elems, cudaMemcpyHostToDevice, stream));
    in.uvw = d.uvw; in.vis = d.vis;
    in.weights = weights ? d.weights : nullptr;
    in.flags = flags ? d.flags : nullptr;
    return TOI_OK;
}

size_t input_bytes(const toi_plan *p, bool w, bool f)
{
    return (size_t)p->geo.n_b * 24 + p->n_elems * (8 + (w ? 4 : 0) + (f ? 1 : 0));
}

int read_info(toi_plan *p, cudaStream_t stream, toi_snapshot_info *info, bool had_h2d)
{
    CU_TRY(p, cudaMemcpyAsync(p->h_state, p->d_state, sizeof(SnapState), cudaMemcpyDeviceToHost, stream));
    CU_TRY(p, cudaStreamSynchronize(stream));
    const SnapState &s = *p->h_state;
    memcpy(info->V, s.V, sizeof s.V);
    info->omega = s.omega;
    memcpy(info->sing, s.sing, sizeof s.sing);
    info->wsum = s.wsum;
    info->n_gridded = (int64_t)s.n_gridded;
    info->n_off_grid = (int64_t)s.n_off_grid;
    info->n_flagged = (int64_t)s.n_flagged;
    float ms = 0.0f;
    info->ms_h2d = 0.0f;
    if (had_h2d && cudaEventElapsedTime(&ms, p->ev[EV_START], p->ev[EV_H2D]) == cudaSuccess) info->ms_h2d = ms;
    cudaEventElapsedTime(&info->ms_planefit, p->ev[EV_H2D], p->ev[EV_FIT]);
    cudaEventElapsedTime(&info->ms_weight, p->ev[EV_FIT], p->ev[EV_WEIGHT]);
    cudaEventElapsedTime(&info->ms_grid, p->ev[EV_WEIGHT], p->ev[EV_GRID]);
    cudaEventElapsedTime(&info->ms_fft, p->ev[EV_GRID], p->ev[EV_FFT]);
    info->ms_clear = 0.0f;
    info->ms_clear_density = 0.0f;
    if (cudaEventElapsedTime(&ms, p->ev_clear0, p->ev_clear1) == cudaSuccess) info->ms_clear = ms;
    if (p->timed_density_clear && cudaEventElapsedTime(&ms, p->ev_clear1, p->ev_clear2) == cudaSuccess) info->ms_clear_density = ms;
    info->ms_fft -= info->ms_clear + info->ms_clear_density;
    cudaEventElapsedTime(&info->ms_crop, p->ev[EV_FFT], p->ev[EV_CROP]);
    cudaEventElapsedTime(&info->ms_total, p->ev[EV_START], p->ev[EV_CROP]);
    cudaGetLastError();
    if (s.status != TOI_OK)
        return fail(p, s.status, "degenerate geometry: the snapshot's baselines do not span a plane (or V33 < 1e-6)");
    return TOI_OK;
}

}  // namespace

extern "C" {

int toi_plan_create(const toi_config *cfg, toi_plan **out)
{
    if (out) *out = nullptr;
    if (!cfg || !out) return fail(nullptr, TOI_ERR_INVALID_ARG, "cfg and out must be non-NULL");
    const int N = cfg->image_size;
    const int G = cfg->grid_size > 0 ? cfg->grid_size : 2 * N;
    const int W = cfg->kernel_support > 0 ? cfg->kernel_support : kW;
    if (cfg->n_baselines < 1 || cfg->n_channels < 1) return fail(nullptr, TOI_ERR_INVALID_ARG, "n_baselines and n_channels must be >= 1");
    if (cfg->n_pols != 1 && cfg->n_pols != 2 && cfg->n_pols != 4) return fail(nullptr, TOI_ERR_INVALID_ARG, "n_pols must be 1, 2 or 4");
    if (cfg->pol_a < 0 || cfg->pol_a >= cfg->n_pols || cfg->pol_b < 0 || cfg->pol_b >= cfg->n_pols)
        return fail(nullptr, TOI_ERR_INVALID_ARG, "pol_a/pol_b out of range");
    if (!cfg->chan_freq_hz) return fail(nullptr, TOI_ERR_INVALID_ARG, "chan_freq_hz is NULL");
    if (N < 16 || (N & 1)) return fail(nullptr, TOI_ERR_INVALID_ARG, "image_size must be even and >= 16");
    // G <= 32768: the gridder packs a window's base cell into 2 x 16 bits
    if ((G & 1) || G < N || G > 32768) return fail(nullptr, TOI_ERR_INVALID_ARG, "grid_size must be even, >= image_size and <= 32768");
    if (!(cfg->cell_size_deg > 0.0) || !(cfg->cell_size_deg < 10.0)) return fail(nullptr, TOI_ERR_INVALID_ARG, "cell_size_deg must be in (0, 10)");
    if (W != kW) return fail(nullptr, TOI_ERR_UNSUPPORTED, "only kernel_support = 7 is built");
    if (cfg->weighting != TOI_WEIGHT_NATURAL && cfg->weighting != TOI_WEIGHT_UNIFORM) return fail(nullptr, TOI_ERR_INVALID_ARG, "unknown weighting");
    if (cfg->input_location != TOI_MEM_HOST && cfg->input_location != TOI_MEM_DEVICE) return fail(nullptr, TOI_ERR_INVALID_ARG, "unknown input_location");
    if (cfg->gridder != TOI_GRIDDER_SLIDING && cfg->gridder != TOI_GRIDDER_ATOMIC)
        return fail(nullptr, TOI_ERR_INVALID_ARG, "unknown gridder");
    if ((cfg->enable_3d != 0 && cfg->enable_3d != 1) || (cfg->debug_keep_grid != 0 && cfg->debug_keep_grid != 1))
        return fail(nullptr, TOI_ERR_INVALID_ARG, "enable_3d and debug_keep_grid must be 0 or 1");
    if (cfg->image_ring_depth < 0 || cfg->image_ring_depth > 64) return fail(nullptr, TOI_ERR_INVALID_ARG, "image_ring_depth must be in [0, 64]");
    if (cfg->apply_jacobian < 0 || cfg->apply_jacobian > 2) return fail(nullptr, TOI_ERR_INVALID_ARG, "apply_jacobian must be 0, 1 or 2");
    for (int k = 0; k < 5; ++k)
        if (cfg->reserved[k] != 0) return fail(nullptr, TOI_ERR_INVALID_ARG, "reserved fields must be 0");
    for (int c = 0; c < cfg->n_channels; ++c)
        if (!(cfg->chan_freq_hz[c] > 0.0) || !isfinite(cfg->chan_freq_hz[c]))
            return fail(nullptr, TOI_ERR_INVALID_ARG, "chan_freq_hz must be positive and finite");
    int n_dev = 0;
    if (cudaGetDeviceCount(&n_dev) != cudaSuccess || n_dev < 1) {
        cudaGetLastError();
        return fail(nullptr, TOI_ERR_CUDA, "no CUDA device: libtoi has no CPU fallback");
    }
    if (cfg->device < 0 || cfg->device >= n_dev) return fail(nullptr, TOI_ERR_INVALID_ARG, "device ordinal out of range");

    toi_plan *p = new (std::nothrow) toi_plan();
    if (!p) return fail(nullptr, TOI_ERR_NOMEM, "out of host memory");
    p->cfg = *cfg;
    p->cfg.chan_freq_hz = nullptr;
    p->cfg.grid_size = G;
    p->cfg.kernel_support = W;
    p->apply_jacobian = cfg->apply_jacobian == 2 ? 0 : 1;
    p->ring_depth = cfg->image_ring_depth > 0 ? cfg->image_ring_depth : 5;
    p->n_samples = (size_t)cfg->n_baselines * cfg->n_channels;
    p->n_elems = p->n_samples * cfg->n_pols;

#define CREATE_TRY(expr)                                                                             \
    do {                                                                                             \
        cudaError_t e_ = (expr);                                                                     \
        if (e_ != cudaSuccess) {                                                                     \
            int rc_ = fail(nullptr, e_ == cudaErrorMemoryAllocation ? TOI_ERR_NOMEM : TOI_ERR_CUDA, \
                           "%s: %s", #expr, cudaGetErrorString(e_));                                 \
            free_plan(p);                                                                            \
            return rc_;                                                                              \
        }                                                                                            \
    } while (0)

    CREATE_TRY(cudaSetDevice(cfg->device));
    cudaDeviceProp prop;
    CREATE_TRY(cudaGetDeviceProperties(&prop, cfg->device));
    p->n_sms = prop.multiProcessorCount;

    // plan-time scalars (fp64 on the host): s_c = nu_c / c0, kappa = G * beta_rad (normative forms)
    std::vector<double> s(cfg->n_channels);
    long double s1 = 0, s2 = 0;
    for (int c = 0; c < cfg->n_channels; ++c) {
        s[c] = cfg->chan_freq_hz[c] / 299792458.0;
        s1 += s[c];
        s2 += (long double)s[c] * s[c];
    }
    p->S1 = (double)s1;
    p->S2 = (double)s2;
    p->s_min = p->s_max = s[0];
    bool up = true, down = true;
    for (int c = 1; c < cfg->n_channels; ++c) {
        if (s[c] < p->s_min) p->s_min = s[c];
        if (s[c] > p->s_max) p->s_max = s[c];
        up = up && s[c] >= s[c - 1];
        down = down && s[c] <= s[c - 1];
    }
    p->s_monotone = up || down;
    Geometry &g = p->geo;
    g.n_b = cfg->n_baselines; g.n_c = cfg->n_channels; g.n_p = cfg->n_pols;
    g.pol_a = cfg->pol_a; g.pol_b = cfg->pol_b;
    g.N = N; g.G = G;
    g.kappa = (double)G * (cfg->cell_size_deg * (3.14159265358979323846 / 180.0));
    std::vector<double> ipsi;
    correction_table(N, G, ipsi);

    const size_t GG = (size_t)G * G;
    CREATE_TRY(cudaStreamCreateWithFlags(&p->s_compute, cudaStreamNonBlocking));
    CREATE_TRY(cudaStreamCreateWithFlags(&p->s_copy, cudaStreamNonBlocking));
    for (int k = 0; k < EV_COUNT; ++k) CREATE_TRY(cudaEventCreate(&p->ev[k]));
    for (int k = 0; k < 2; ++k) {
        CREATE_TRY(cudaEventCreate(&p->ev_h2d_start[k]));
        CREATE_TRY(cudaEventCreate(&p->ev_h2d_done[k]));
        CREATE_TRY(cudaEventCreate(&p->ev_c_start[k]));
        CREATE_TRY(cudaEventCreate(&p->ev_c_done[k]));
    }
    CREATE_TRY(cudaEventCreate(&p->ev_first));
    CREATE_TRY(cudaMalloc(&p->d_s, s.size() * sizeof(double)));
    CREATE_TRY(cudaMemcpy(p->d_s, s.data(), s.size() * sizeof(double), cudaMemcpyHostToDevice));
    g.s = p->d_s;
    CREATE_TRY(cudaMalloc(&p->d_ipsi, (size_t)N * sizeof(double)));
    CREATE_TRY(cudaMemcpy(p->d_ipsi, ipsi.data(), (size_t)N * sizeof(double), cudaMemcpyHostToDevice));
    CREATE_TRY(cudaMalloc(&p->d_V_inject, 9 * sizeof(double)));
    CREATE_TRY(cudaMalloc(&p->d_V_reproject, 9 * sizeof(double)));
    CREATE_TRY(cudaMalloc(&p->d_state_slots, 2 * sizeof(SnapState)));
    CREATE_TRY(cudaMemset(p->d_state_slots, 0, 2 * sizeof(SnapState)));
    p->d_state = p->d_state_slots;
    CREATE_TRY(cudaMallocHost(&p->h_state, sizeof(SnapState)));
    // the gridding grid with a guard band on both sides (the gridder's 8 x 8 window may overhang the
    // grid by one row or column of zero accumulators, whose flush must land in owned memory that
    // nothing reads), zero-filled ONCE here; the FFT workspace; the density map; the tile maps
    CREATE_TRY(cudaMalloc(&p->d_grid_alloc, (GG + 2 * grid_guard(G)) * sizeof(float2)));
    CREATE_TRY(cudaMemset(p->d_grid_alloc, 0, (GG + 2 * grid_guard(G)) * sizeof(float2)));
    p->d_grid = p->d_grid_alloc + grid_guard(G);
    CREATE_TRY(cudaMalloc(&p->d_work, GG * sizeof(float2)));
    p->n_tiles = (size_t)tiles_per_row(G) * tile_rows(G);
    CREATE_TRY(cudaMalloc(&p->d_tiles_grid, p->n_tiles));
    CREATE_TRY(cudaMemset(p->d_tiles_grid, 0, p->n_tiles));
    if (cfg->weighting == TOI_WEIGHT_UNIFORM) {
        CREATE_TRY(cudaMalloc(&p->d_dens, GG * sizeof(float)));
        CREATE_TRY(cudaMemset(p->d_dens, 0, GG * sizeof(float)));
    }
    CREATE_TRY(cudaEventCreateWithFlags(&p->ev_done, cudaEventDisableTiming));
    CREATE_TRY(cudaEventCreate(&p->ev_clear0));
    CREATE_TRY(cudaEventCreate(&p->ev_clear1));
    CREATE_TRY(cudaEventCreate(&p->ev_clear2));
    if (cfg->debug_keep_grid) {
        CREATE_TRY(cudaMalloc(&p->d_grid_keep, GG * sizeof(float2)));
        if (cfg->weighting == TOI_WEIGHT_UNIFORM) CREATE_TRY(cudaMalloc(&p->d_dens_keep, GG * sizeof(float)));
    }
    if (cfg->enable_3d) {
        CREATE_TRY(cudaMalloc(&p->d_acc3, (size_t)N * N * sizeof(float2)));
        CREATE_TRY(cudaMalloc(&p->d_slab3, (size_t)N * N * sizeof(float2)));
        CREATE_TRY(cudaMalloc(&p->d_r3, 2 * sizeof(double)));
        CREATE_TRY(cudaMalloc(&p->d_jtab, bessel_table_floats(64) * sizeof(float)));
        CREATE_TRY(cudaMallocHost(&p->h_r3, 2 * sizeof(double)));
        CREATE_TRY(cudaEventCreate(&p->ev3_a));
        CREATE_TRY(cudaEventCreate(&p->ev3_b));
        if (fft_custom_supported(N, G) && cfg->gridder == TOI_GRIDDER_SLIDING) {
            CREATE_TRY(cudaMalloc(&p->d_grid1_alloc, (GG + 2 * grid_guard(G)) * sizeof(float2)));
            CREATE_TRY(cudaMemset(p->d_grid1_alloc, 0, (GG + 2 * grid_guard(G)) * sizeof(float2)));
            p->d_grid1 = p->d_grid1_alloc + grid_guard(G);
            CREATE_TRY(cudaMalloc(&p->d_work1, GG * sizeof(float2)));
            CREATE_TRY(cudaMalloc(&p->d_moment[1], (size_t)N * N * sizeof(float2)));
            CREATE_TRY(cudaMalloc(&p->d_tiles1, p->n_tiles));
            CREATE_TRY(cudaMemset(p->d_tiles1, 0, p->n_tiles));
            CREATE_TRY(cudaStreamCreateWithFlags(&p->s_lane1, cudaStreamNonBlocking));
            for (int k = 0; k < 2; ++k) {
                CREATE_TRY(cudaEventCreateWithFlags(&p->ev_lane_grid[k], cudaEventDisableTiming));
                CREATE_TRY(cudaEventCreateWithFlags(&p->ev_lane_comb[k], cudaEventDisableTiming));
            }
            CREATE_TRY(cudaEventCreateWithFlags(&p->ev_lane_setup, cudaEventDisableTiming));
            CREATE_TRY(cudaEventCreateWithFlags(&p->ev_lane_cols0, cudaEventDisableTiming));
        }
    }
    CREATE_TRY(cudaMalloc(&p->d_images, (size_t)p->ring_depth * N * N * sizeof(float)));
    if (cfg->input_location == TOI_MEM_HOST) {
        for (int k = 0; k < 2; ++k) {                      // device input ring + pinned host ring, depth 2
            CREATE_TRY(cudaMalloc(&p->dev_in[k].uvw, (size_t)g.n_b * 3 * sizeof(double)));
            CREATE_TRY(cudaMalloc(&p->dev_in[k].vis, p->n_elems * sizeof(float2)));
            CREATE_TRY(cudaMalloc(&p->dev_in[k].weights, p->n_elems * sizeof(float)));
            CREATE_TRY(cudaMalloc(&p->dev_in[k].flags, p->n_elems));
            CREATE_TRY(cudaMallocHost(&p->pin[k].uvw_m, (size_t)g.n_b * 3 * sizeof(double)));
            CREATE_TRY(cudaMallocHost(&p->pin[k].vis, p->n_elems * sizeof(float2)));
            CREATE_TRY(cudaMallocHost(&p->pin[k].weights, p->n_elems * sizeof(float)));
            CREATE_TRY(cudaMallocHost(&p->pin[k].flags, p->n_elems));
        }
    }
    // Pruned transform (when the crop keeps at most 3/4 of the columns, e.g. the default G = 2N):
    // 1-D transforms of all G rows, then of only the N columns the crop reads -- cuFFT's strided
    // column pass is the expensive one (two kernels), so skipping G - N columns saves more than a
    // third of the FFT.  The skipped columns are left row-transformed only; nothing reads them.
    // Otherwise the plain 2-D plan.
    if (fft_custom_supported(N, G)) {
        // the hand-written pruned transform (k_fft.cu): no cuFFT plan at all
        std::vector<float2> tw((size_t)G);
        fft_twiddle_table(G, tw.data());
        CREATE_TRY(cudaMalloc(&p->d_tw, (size_t)G * sizeof(float2)));
        CREATE_TRY(cudaMemcpy(p->d_tw, tw.data(), (size_t)G * sizeof(float2), cudaMemcpyHostToDevice));
        if (cfg->enable_3d) CREATE_TRY(cudaMalloc(&p->d_moment[0], (size_t)N * N * sizeof(float2)));
        p->fft_custom = true;
    } else if (4 * N <= 3 * G) {
        int n[1] = {G};
        if (cufftPlanMany(&p->fft_cols, 1, n, n, G, 1, n, G, 1, CUFFT_C2C, N / 2) != CUFFT_SUCCESS ||
            cufftPlanMany(&p->fft_rows, 1, n, n, 1, G, n, 1, G, CUFFT_C2C, G) != CUFFT_SUCCESS) {
            fail(nullptr, TOI_ERR_CUFFT, "cufftPlanMany failed");
            free_plan(p);
            return TOI_ERR_CUFFT;
        }
        p->fft_pruned = true;
    } else {
        if (cufftPlan2d(&p->fft, G, G, CUFFT_C2C) != CUFFT_SUCCESS) {
            fail(nullptr, TOI_ERR_CUFFT, "cufftPlan2d failed");
            free_plan(p);
            return TOI_ERR_CUFFT;
        }
        p->fft_ok = true;
    }
    CREATE_TRY(cudaDeviceSynchronize());
#undef CREATE_TRY
    *out = p;
    return TOI_OK;
}

int toi_plan_destroy(toi_plan *plan) { return free_plan(plan); }

int toi_image_snapshot(toi_plan *p, const double *uvw_m, const void *vis, const float *weights,
                       const uint8_t *flags, void *cuda_stream, float **d_image_out, toi_snapshot_info *info)
{
    if (!p) return fail(nullptr, TOI_ERR_INVALID_ARG, "plan is NULL");
    if (!uvw_m || !vis || !d_image_out) return fail(p, TOI_ERR_INVALID_ARG, "uvw_m, vis and d_image_out must be non-NULL");
    CU_TRY(p, cudaSetDevice(p->cfg.device));
    cudaStream_t stream = cuda_stream ? (cudaStream_t)cuda_stream : p->s_compute;
    Inputs in;
    const bool timed = info != nullptr;
    if (timed) CU_TRY(p, cudaEventRecord(p->ev[EV_START], stream));
    const bool host = p->cfg.input_location == TOI_MEM_HOST;
    if (host) {
        p->snap_slot ^= 1;
        int rc = h2d_slot(p, p->snap_slot, uvw_m, vis, weights, flags, stream, in);
        if (rc) return rc;
    } else {
        in.uvw = uvw_m; in.vis = (const float2 *)vis; in.weights = weights; in.flags = flags;
    }
    if (timed) CU_TRY(p, cudaEventRecord(p->ev[EV_H2D], stream));
    int rc = enqueue_imaging(p, in, stream, d_image_out, timed);
    if (rc) return rc;
    if (info) return read_info(p, stream, info, host);
    return TOI_OK;
}

// ---- near-coplanar (3-D) mode: host-side parameter selection (Eqs. 25-27) ----
namespace {

// Eq. 17 at (t1, t2); NaN outside the sphere constraint
double t3_host(const double *V, double t1, double t2)
{
    const double a = t1 + V[2], b = t2 + V[5], rad = 1.0 - a * a - b * b;
    if (!(rad >= 0.0)) return NAN;
    return -V[8] + (V[8] < 0.0 ? -sqrt(rad) : sqrt(rad));
}

// Eq. 25 over the pixels of the N x N image: |t3| is extremal on the border of the image or at the
// pixels around the stationary point (t1, t2) = (-V13, -V23) of the square root
double t3_max_host(const double *V, int N, double beta)
{
    double best = 0.0;
    auto look = [&](int i, int j) {
        if (i < 0 || j < 0 || i >= N || j >= N) return;
        const double t3 = t3_host(V, -beta * (double)(i - N / 2), beta * (double)(j - N / 2));
        if (t3 == t3 && fabs(t3) > best) best = fabs(t3);
    };
    for (int k = 0; k < N; ++k) { look(k, 0); look(k, N - 1); look(0, k); look(N - 1, k); }
    const int ic = (int)floor(N / 2 + V[2] / beta), jc = (int)floor(N / 2 - V[5] / beta);
    for (int dj = -1; dj <= 2; ++dj)
        for (int di = -1; di <= 2; ++di) look(ic + di, jc + dj);
    // a border that leaves the sphere constraint: scan everything (small or all-sky images only)
    bool nan_border = false;
    for (int k = 0; k < N && !nan_border; ++k) {
        const double a = t3_host(V, -beta * (double)(k - N / 2), beta * (double)(0 - N / 2));
        const double b = t3_host(V, -beta * (double)(k - N / 2), beta * (double)(N - 1 - N / 2));
        const double c = t3_host(V, -beta * (double)(0 - N / 2), beta * (double)(k - N / 2));
        const double d = t3_host(V, -beta * (double)(N - 1 - N / 2), beta * (double)(k - N / 2));
        nan_border = !(a == a && b == b && c == c && d == d);
    }
    if (nan_border)
        for (int j = 0; j < N; ++j)
            for (int i = 0; i < N; ++i) look(i, j);
    return best;
}

// max over a 129 x 257 grid of [0, alpha_slab] x [-1, 1] of |exp(i a s) - sum_{k<K} c_k(a) T_k(s)| (G25)
double sampled_error_host(double alpha_slab, int K)
{
    const int na = 129, ns = 257;
    double worst = 0.0;
    std::vector<double> J(K), T(K);
    for (int ia = 0; ia < na; ++ia) {
        const double a = alpha_slab * ia / (na - 1);
        for (int k = 0; k < K; ++k) J[k] = std::cyl_bessel_j((double)k, a);
        for (int is = 0; is < ns; ++is) {
            const double sq = -1.0 + 2.0 * is / (ns - 1);
            T[0] = 1.0;
            if (K > 1) T[1] = sq;
            for (int k = 2; k < K; ++k) T[k] = 2.0 * sq * T[k - 1] - T[k - 2];
            double re = J[0], im = 0.0;                  // c_0 = J_0, c_k = 2 i^k J_k
            for (int k = 1; k < K; ++k) {
                const double v = 2.0 * J[k] * T[k];
                switch (k & 3) { case 0: re += v; break; case 1: im += v; break; case 2: re -= v; break; default: im -= v; break; }
            }
            const double er = cos(a * sq) - re, ei = sin(a * sq) - im;
            const double e = sqrt(er * er + ei * ei);
            if (e > worst) worst = e;
        }
    }
    return worst;
}

}  // namespace

int toi_image_snapshot_3d(toi_plan *p, const double *uvw_m, const void *vis, const float *weights, const uint8_t *flags,
                          void *cuda_stream, int32_t n_slab_in, int32_t K_in, float **d_image_out, toi_3d_info *info3,
                          toi_snapshot_info *info)
{
    if (!p) return fail(nullptr, TOI_ERR_INVALID_ARG, "plan is NULL");
    if (!uvw_m || !vis || !d_image_out) return fail(p, TOI_ERR_INVALID_ARG, "uvw_m, vis and d_image_out must be non-NULL");
    if (n_slab_in < 0 || n_slab_in > 1024 || K_in < 0 || K_in > 64) return fail(p, TOI_ERR_INVALID_ARG, "n_slab must be in [0, 1024], K in [0, 64]");
    if (!p->d_acc3) return fail(p, TOI_ERR_UNSUPPORTED, "the 3-D mode needs a plan created with enable_3d = 1");
    if (p->cfg.gridder == TOI_GRIDDER_ATOMIC) return fail(p, TOI_ERR_UNSUPPORTED, "the 3-D mode runs on the sliding gridders only");
    const Geometry &g = p->geo;
    CU_TRY(p, cudaSetDevice(p->cfg.device));
    cudaStream_t stream = cuda_stream ? (cudaStream_t)cuda_stream : p->s_compute;
    const size_t GG = (size_t)g.G * g.G, NN = (size_t)g.N * g.N;
    int rc = set_fft_stream(p, stream);
    if (rc) return rc;
    rc = follow_previous_call(p, stream);
    if (rc) return rc;
    CU_TRY(p, cudaEventRecord(p->ev3_a, stream));
    Inputs in;
    if (p->cfg.input_location == TOI_MEM_HOST) {
        p->snap_slot ^= 1;
        rc = h2d_slot(p, p->snap_slot, uvw_m, vis, weights, flags, stream, in);
        if (rc) return rc;
    } else {
        in.uvw = uvw_m; in.vis = (const float2 *)vis; in.weights = weights; in.flags = flags;
    }
    // plane fit, r3 range -> host (the one synchronisation of this mode)
    launch_planefit(g, in.uvw, p->S1, p->S2, p->inject ? p->d_V_inject : nullptr, p->d_state, stream);
    launch_r3_range(g.n_b, in.uvw, p->d_state, p->s_min, p->s_max, p->d_r3, stream);
    CU_TRY(p, cudaMemcpyAsync(p->h_state, p->d_state, sizeof(SnapState), cudaMemcpyDeviceToHost, stream));
    CU_TRY(p, cudaMemcpyAsync(p->h_r3, p->d_r3, 2 * sizeof(double), cudaMemcpyDeviceToHost, stream));
    CU_TRY(p, cudaStreamSynchronize(stream));
    float *img = p->d_images + (size_t)(p->ring_pos % p->ring_depth) * NN;
    ++p->ring_pos;
    *d_image_out = img;
    p->last_in = in;
    if (p->h_state->status != TOI_OK) {
        CU_TRY(p, cudaMemsetAsync(img, 0, NN * sizeof(float), stream));
        return fail(p, p->h_state->status, "degenerate geometry: the snapshot's baselines do not span a plane (or V33 < 1e-6)");
    }
    const double beta = p->cfg.cell_size_deg * (3.14159265358979323846 / 180.0);
    const double r3_min = p->h_r3[0], r3_max = p->h_r3[1];
    const double t3_max = t3_max_host(p->h_state->V, g.N, beta);
    const double phi_max = 2.0 * 3.14159265358979323846 * t3_max * (r3_max - r3_min) / 2.0;       // Eq. 26
    const int n_slab = n_slab_in > 0 ? n_slab_in : (int)fmax(1.0, ceil(phi_max / 10.0));          // Eq. 27
    if (n_slab > 1024) {
        CU_TRY(p, cudaMemsetAsync(img, 0, NN * sizeof(float), stream));
        return fail(p, TOI_ERR_UNSUPPORTED, "more than 1024 slabs: the snapshot is far from coplanar");
    }
    const double alpha_slab = phi_max / n_slab;
    int K = K_in;
    double err = -1.0;
    if (K == 0) {
        const int choices[4] = {8, 16, 24, 32};
        K = 32;
        for (int c = 0; c < 4; ++c) {
            const double e = sampled_error_host(alpha_slab, choices[c]);
            if (e < 1e-2) { K = choices[c]; err = e; break; }
        }
    }
    if (err < 0.0 && info3) err = sampled_error_host(alpha_slab, K);
    const double d = (r3_max - r3_min) / (2.0 * n_slab);                                           // G24
    const int slabs_run = d > 0.0 ? n_slab : 1;
    int launches = 2;
    // uniform weighting: the density map does not depend on the slab or the order
    const bool uniform = p->cfg.weighting == TOI_WEIGHT_UNIFORM;
    const float *dens = nullptr;
    if (uniform) {
        launch_density(g, in, p->d_state, p->d_dens, stream);
        dens = p->d_dens;
        ++launches;
    }
    // J_k(alpha) for every order, tabulated once over the range alpha takes in this image (Eq. 20)
    const double a_max = d > 0.0 ? 2.0 * 3.14159265358979323846 * d * t3_max * (1.0 + 1e-9) : 0.0;
    launch_bessel_table(K, a_max, p->d_jtab, stream);
    ++launches;
    // Two lanes (when the second set of buffers exists): even orders k on `stream`, odd ones on s_lane1,
    // each on its own grid / tile map / workspace / moment.  What the passes share is kept in order by
    // events: the task counter and the density map (gridder p + 1 waits for gridder p), the slab and total
    // sums (a combination waits for the one before), a lane's moment (its next column pass waits for the
    // combination that read it).  The two moments of a pair (k even, k + 1) are folded in by ONE
    // combination launch on the odd lane; a slab's unpaired last order (K odd), and every order when
    // there is one lane, by a launch of its own.
    const bool two_lanes = p->d_grid1 != nullptr;
    if (two_lanes) {
        CU_TRY(p, cudaEventRecord(p->ev_lane_setup, stream));
        CU_TRY(p, cudaStreamWaitEvent(p->s_lane1, p->ev_lane_setup, 0));
    }
    const int n_passes = slabs_run * K;
    bool have_comb[2] = {false, false};
    struct PdlOff {                              // no programmatic launches while two lanes share the SMs
        bool saved;
        explicit PdlOff(bool off) : saved(g_pdl_enabled) { if (off) g_pdl_enabled = false; }
        ~PdlOff() { g_pdl_enabled = saved; }
    } pdl_off(two_lanes);
    for (int pass = 0; pass < n_passes; ++pass) {
        const int sp = pass / K, k = pass % K;
        const int L = two_lanes ? (k & 1) : 0;
        cudaStream_t sL = L ? p->s_lane1 : stream;
        float2 *gridL = L ? p->d_grid1 : p->d_grid, *workL = L ? p->d_work1 : p->d_work;
        uint8_t *mapL = L ? p->d_tiles1 : p->d_tiles_grid;
        ChebArgs ca;
        ca.p = sp; ca.k = k; ca.n_slab = n_slab; ca.r3_min = r3_min; ca.d = d;
        ca.count = (k == 0 ? 1 : 0) | (pass == 0 ? 2 : 0);
        const bool last = pass == n_passes - 1;
        if (two_lanes && pass > 0) CU_TRY(p, cudaStreamWaitEvent(sL, p->ev_lane_grid[L ^ 1], 0));
        CU_TRY(p, cudaMemsetAsync(&p->d_state->task_counter, 0, sizeof(unsigned int), sL));
        uint8_t *tiles = gridder_tile_map(p, sL, true, mapL);
        launch_grid_pair8_cheb(g, in, p->d_state, dens, gridL, tiles, p->n_sms, ca, sL);
        launches += tiles ? 2 : 3;
        if (two_lanes) CU_TRY(p, cudaEventRecord(p->ev_lane_grid[L], sL));
        if (pass == 0 && p->keep_grid) {
            CU_TRY(p, cudaMemcpyAsync(p->d_grid_keep, gridL, GG * sizeof(float2), cudaMemcpyDeviceToDevice, sL));
            if (uniform) CU_TRY(p, cudaMemcpyAsync(p->d_dens_keep, p->d_dens, GG * sizeof(float), cudaMemcpyDeviceToDevice, sL));
        }
        // first transform pass out of place, sparse clear of the grid (and, after the last pass, of
        // the density map), second transform pass on the workspace
        rc = transform_and_clear(p, sL, gridL, mapL, workL, uniform && last, false, nullptr, L,
                                 two_lanes && have_comb[L ^ 1] ? p->ev_lane_comb[L ^ 1] : nullptr, &launches);
        if (rc) return rc;
        if (two_lanes && L == 0 && k != K - 1) {         // the odd lane's combination takes this moment along
            CU_TRY(p, cudaEventRecord(p->ev_lane_cols0, sL));
            continue;
        }
        const int nm = two_lanes && L == 1 ? 2 : 1, k0 = k - (nm - 1);
        const double r3_p = d > 0.0 ? r3_min + (2.0 * sp + 1.0) * d : r3_min;
        if (nm == 2) CU_TRY(p, cudaStreamWaitEvent(sL, p->ev_lane_cols0, 0));
        if (two_lanes && have_comb[L ^ 1]) CU_TRY(p, cudaStreamWaitEvent(sL, p->ev_lane_comb[L ^ 1], 0));
        const float2 *F0 = p->fft_custom ? p->d_moment[nm == 2 ? 0 : L] : workL;
        launch_cheb_combine(g, beta, p->d_state, k0, nm, r3_p, d, p->d_jtab, a_max, F0, p->d_moment[1], p->fft_custom ? 1 : 0,
                            p->d_ipsi, p->d_slab3, p->d_acc3, k0 == 0 ? 1 : 0, k0 + nm == K ? 1 : 0, sp == 0 ? 1 : 0, sL);
        ++launches;
        if (two_lanes) {
            CU_TRY(p, cudaEventRecord(p->ev_lane_comb[L], sL));
            have_comb[L] = true;
        }
    }
    // the last combination may sit on the other lane
    if (two_lanes && have_comb[1]) CU_TRY(p, cudaStreamWaitEvent(stream, p->ev_lane_comb[1], 0));
    launch_cheb_finish(g.N, beta, p->d_state, p->apply_jacobian, p->d_acc3, img, stream);
    ++launches;
    CU_TRY(p, cudaEventRecord(p->ev3_b, stream));
    CU_TRY(p, cudaGetLastError());
    p->last_launches = launches;
    if (info3 || info) {
        CU_TRY(p, cudaMemcpyAsync(p->h_state, p->d_state, sizeof(SnapState), cudaMemcpyDeviceToHost, stream));
        CU_TRY(p, cudaStreamSynchronize(stream));
    }
    if (info3) {
        memset(info3, 0, sizeof *info3);
        info3->n_slab = n_slab; info3->K = K; info3->n_passes = slabs_run * K;
        info3->phi_max = phi_max; info3->t3_max = t3_max; info3->r3_min = r3_min; info3->r3_max = r3_max;
        info3->alpha_slab = alpha_slab; info3->expansion_error = err;
        cudaEventElapsedTime(&info3->ms_total, p->ev3_a, p->ev3_b);
    }
    if (info) {
        memset(info, 0, sizeof *info);
        const SnapState &st = *p->h_state;
        memcpy(info->V, st.V, sizeof st.V);
        info->omega = st.omega;
        memcpy(info->sing, st.sing, sizeof st.sing);
        info->wsum = st.wsum;
        info->n_gridded = (int64_t)st.n_gridded;
        info->n_off_grid = (int64_t)st.n_off_grid;
        info->n_flagged = (int64_t)st.n_flagged;
        cudaEventElapsedTime(&info->ms_total, p->ev3_a, p->ev3_b);
    }
    return TOI_OK;
}

int toi_plan_sync(toi_plan *p)
{
    if (!p) return fail(nullptr, TOI_ERR_INVALID_ARG, "plan is NULL");
    CU_TRY(p, cudaSetDevice(p->cfg.device));
    CU_TRY(p, cudaDeviceSynchronize());
    CU_TRY(p, cudaMemcpy(p->h_state, p->d_state, sizeof(SnapState), cudaMemcpyDeviceToHost));
    int rc = p->deferred;
    p->deferred = TOI_OK;
    if (rc == TOI_OK && p->h_state->status != TOI_OK) {
        rc = p->h_state->status;
        snprintf(p->err, sizeof p->err, "degenerate geometry in the last snapshot");
    }
    return rc;
}

int toi_copy_image_to_host(toi_plan *p, const float *d_image, float *h_image)
{
    if (!p || !d_image || !h_image) return fail(p, TOI_ERR_INVALID_ARG, "NULL argument");
    CU_TRY(p, cudaSetDevice(p->cfg.device));
    CU_TRY(p, cudaDeviceSynchronize());
    CU_TRY(p, cudaMemcpy(h_image, d_image, (size_t)p->geo.N * p->geo.N * sizeof(float), cudaMemcpyDeviceToHost));
    return TOI_OK;
}

int toi_stream_set_output(toi_plan *p, const toi_stream_output *out)
{
    if (!p) return fail(nullptr, TOI_ERR_INVALID_ARG, "plan is NULL");
    toi_stream_output o;
    memset(&o, 0, sizeof o);
    if (out) o = *out;
    if (o.product != TOI_OUT_TILTED && o.product != TOI_OUT_REPROJECT_EXACT && o.product != TOI_OUT_REPROJECT_PAPER)
        return fail(p, TOI_ERR_INVALID_ARG, "unknown stream product");
    if ((o.difference != 0 && o.difference != 1) || (o.to_host != 0 && o.to_host != 1))
        return fail(p, TOI_ERR_INVALID_ARG, "difference and to_host must be 0 or 1");
    for (int k = 0; k < 5; ++k)
        if (o.reserved[k] != 0) return fail(p, TOI_ERR_INVALID_ARG, "reserved fields must be 0");
    if (o.to_host && !o.host_sink) return fail(p, TOI_ERR_INVALID_ARG, "to_host needs a host_sink callback");
    if (o.difference && p->ring_depth < 2) return fail(p, TOI_ERR_INVALID_ARG, "difference needs image_ring_depth >= 2");
    // the D2H of image n runs under the imaging of n + 1 and n + 2 (its pinned slot is reclaimed just
    // before n + 2 is enqueued... and the copy stream may lag): the ring slot it reads must not be
    // the one either of them writes
    if (o.to_host && p->ring_depth < 3) return fail(p, TOI_ERR_INVALID_ARG, "to_host needs image_ring_depth >= 3");
    CU_TRY(p, cudaSetDevice(p->cfg.device));
    CU_TRY(p, cudaDeviceSynchronize());
    const size_t img_bytes = (size_t)p->geo.N * p->geo.N * sizeof(float);
    if (!p->ev_tail) CU_TRY(p, cudaEventCreate(&p->ev_tail));
    if (o.product != TOI_OUT_TILTED && !p->d_products) CU_TRY(p, cudaMalloc(&p->d_products, (size_t)p->ring_depth * img_bytes));
    if (o.difference)
        for (int k = 0; k < 2; ++k)
            if (!p->d_diff[k]) CU_TRY(p, cudaMalloc(&p->d_diff[k], img_bytes));
    if (o.to_host) {
        if (!p->s_d2h) CU_TRY(p, cudaStreamCreateWithFlags(&p->s_d2h, cudaStreamNonBlocking));
        for (int k = 0; k < 2; ++k) {
            if (!p->h_out[k]) CU_TRY(p, cudaMallocHost(&p->h_out[k], img_bytes));
            if (!p->ev_out_ready[k]) CU_TRY(p, cudaEventCreateWithFlags(&p->ev_out_ready[k], cudaEventDisableTiming));
            if (!p->ev_d2h_start[k]) CU_TRY(p, cudaEventCreate(&p->ev_d2h_start[k]));
            if (!p->ev_d2h_done[k]) CU_TRY(p, cudaEventCreate(&p->ev_d2h_done[k]));
        }
    }
    p->out_cfg = o;
    return TOI_OK;
}

int toi_image_stream(toi_plan *p, int64_t n_snapshots, toi_fill_fn fill, void *fill_user, toi_sink_fn sink,
                     void *sink_user, int32_t want_info, toi_stream_stats *stats)
{
    if (!p) return fail(nullptr, TOI_ERR_INVALID_ARG, "plan is NULL");
    if (!fill || n_snapshots < 0) return fail(p, TOI_ERR_INVALID_ARG, "fill callback required, n_snapshots >= 0");
    if (p->cfg.input_location != TOI_MEM_HOST)
        return fail(p, TOI_ERR_UNSUPPORTED, "toi_image_stream needs a plan created with input_location = TOI_MEM_HOST");
    CU_TRY(p, cudaSetDevice(p->cfg.device));
    toi_stream_stats st;
    memset(&st, 0, sizeof st);
    const auto t0 = std::chrono::steady_clock::now();
    bool used[2] = {false, false};
    float ms = 0.0f;
    int rc = TOI_OK;
    auto harvest = [&](int slot) {     // timings of the snapshot that last used `slot` (already complete)
        if (cudaEventSynchronize(p->ev_c_done[slot]) != cudaSuccess) return;
        if (cudaEventElapsedTime(&ms, p->ev_h2d_start[slot], p->ev_h2d_done[slot]) == cudaSuccess) st.h2d_ms_sum += ms;
        if (cudaEventElapsedTime(&ms, p->ev_c_start[slot], p->ev_c_done[slot]) == cudaSuccess) st.compute_ms_sum += ms;
    };
    // ---- output side (toi_stream_set_output) ----
    const toi_stream_output oc = p->out_cfg;
    const size_t n_pix = (size_t)p->geo.N * p->geo.N;
    const double beta_rad = p->cfg.cell_size_deg * (3.14159265358979323846 / 180.0);
    const float *prev_prod = nullptr;
    int64_t out_idx[2] = {-1, -1}, n_out = 0;
    bool tail_used = false;
    auto finish_out = [&](int o, bool call) -> int {   // the D2H in pinned slot o has landed: hand it over
        if (out_idx[o] < 0) return TOI_OK;
        const int64_t idx = out_idx[o];
        out_idx[o] = -1;
        if (cudaEventSynchronize(p->ev_d2h_done[o]) != cudaSuccess) return fail(p, TOI_ERR_CUDA, "D2H of an output image failed");
        if (cudaEventElapsedTime(&ms, p->ev_d2h_start[o], p->ev_d2h_done[o]) == cudaSuccess) st.d2h_ms_sum += ms;
        if (call && oc.host_sink(oc.host_user, idx, p->h_out[o]) < 0) return fail(p, TOI_ERR_CALLBACK, "host sink callback failed");
        return TOI_OK;
    };
    int64_t n = 0;
    // inside the loop an error must not return before the streams are drained and the pending host
    // images handed over: record it and leave the loop
#define LOOP_TRY(expr)                                                                                \
    {                                                                                                 \
        cudaError_t e_ = (expr);                                                                      \
        if (e_ != cudaSuccess) {                                                                      \
            rc = fail(p, e_ == cudaErrorMemoryAllocation ? TOI_ERR_NOMEM : TOI_ERR_CUDA, "%s: %s", #expr, cudaGetErrorString(e_)); \
            break;                                                                                    \
        }                                                                                             \
    }
    for (; n < n_snapshots; ++n) {
        const int slot = (int)(n & 1);
        if (used[slot]) {
            // the pinned slot is free once its H2D finished; compute of n-2 is long done
            LOOP_TRY(cudaEventSynchronize(p->ev_h2d_done[slot]));
            harvest(slot);
        }
        toi_snapshot_buffers b = p->pin[slot];
        const int frc = fill(fill_user, n, &b);
        if (frc == 1) break;
        if (frc < 0) { rc = fail(p, TOI_ERR_CALLBACK, "fill callback failed"); break; }
        if (!b.uvw_m || !b.vis) { rc = fail(p, TOI_ERR_CALLBACK, "fill callback returned NULL uvw/vis"); break; }
        // device slot is free once the imaging that read it finished: GPU-side wait only
        if (used[slot]) LOOP_TRY(cudaStreamWaitEvent(p->s_copy, p->ev_c_done[slot], 0));
        if (n == 0) LOOP_TRY(cudaEventRecord(p->ev_first, p->s_copy));
        LOOP_TRY(cudaEventRecord(p->ev_h2d_start[slot], p->s_copy));
        Inputs in;
        rc = h2d_slot(p, slot, b.uvw_m, b.vis, b.weights, b.flags, p->s_copy, in);
        if (rc) break;
        LOOP_TRY(cudaEventRecord(p->ev_h2d_done[slot], p->s_copy));
        st.h2d_bytes += (double)input_bytes(p, b.weights != nullptr, b.flags != nullptr);
        LOOP_TRY(cudaStreamWaitEvent(p->s_compute, p->ev_h2d_done[slot], 0));
        LOOP_TRY(cudaEventRecord(p->ev_c_start[slot], p->s_compute));
        if (want_info) {
            LOOP_TRY(cudaEventRecord(p->ev[EV_START], p->s_compute));
            LOOP_TRY(cudaEventRecord(p->ev[EV_H2D], p->s_compute));
        }
        float *img = nullptr;
        rc = enqueue_imaging(p, in, p->s_compute, &img, want_info != 0);
        if (rc) break;
        LOOP_TRY(cudaEventRecord(p->ev_c_done[slot], p->s_compute));
        used[slot] = true;
        // interpolate stage: tilted plane -> (l, m) grid with this snapshot's V
        float *prod = img;
        if (oc.product != TOI_OUT_TILTED) {
            prod = p->d_products + (size_t)((p->ring_pos - 1) % p->ring_depth) * n_pix;
            launch_reproject(p->geo.N, beta_rad, p->d_state, nullptr,
                             oc.product == TOI_OUT_REPROJECT_PAPER ? TOI_REPROJECT_PAPER : TOI_REPROJECT_EXACT, img, prod,
                             p->s_compute);
        }
        const float *deliver = prod;
        bool to_host = oc.to_host != 0;
        const int o = (int)(n_out & 1);
        if (to_host && (!oc.difference || prev_prod)) {
            // pinned slot o (and the difference buffer it was copied from) is free once the D2H
            // two deliveries ago has landed; its image goes to the host sink now
            rc = finish_out(o, true);
            if (rc) break;
        }
        if (oc.difference) {
            if (prev_prod) {
                launch_difference(n_pix, prod, prev_prod, p->d_diff[n & 1], p->n_sms, p->s_compute);
                deliver = p->d_diff[n & 1];
            } else {
                to_host = false;                  // snapshot 0 has no predecessor
            }
            prev_prod = prod;
        }
        if (oc.product != TOI_OUT_TILTED || oc.difference) {
            LOOP_TRY(cudaGetLastError());
            LOOP_TRY(cudaEventRecord(p->ev_tail, p->s_compute));
            tail_used = true;
        }
        if (to_host) {
            // copy_cpu stage: third stream, pinned ring, events only
            LOOP_TRY(cudaEventRecord(p->ev_out_ready[o], p->s_compute));
            LOOP_TRY(cudaStreamWaitEvent(p->s_d2h, p->ev_out_ready[o], 0));
            LOOP_TRY(cudaEventRecord(p->ev_d2h_start[o], p->s_d2h));
            LOOP_TRY(cudaMemcpyAsync(p->h_out[o], deliver, n_pix * sizeof(float), cudaMemcpyDeviceToHost, p->s_d2h));
            LOOP_TRY(cudaEventRecord(p->ev_d2h_done[o], p->s_d2h));
            out_idx[o] = n;
            ++n_out;
            st.d2h_bytes += (double)(n_pix * sizeof(float));
        }
        toi_snapshot_info info;
        if (want_info) {
            rc = read_info(p, p->s_compute, &info, false);
            if (rc) break;
        }
        if (sink) {
            const int src = sink(sink_user, n, deliver, (void *)p->s_compute, want_info ? &info : nullptr);
            if (src < 0) { rc = fail(p, TOI_ERR_CALLBACK, "sink callback failed"); break; }
        }
    }
#undef LOOP_TRY
    cudaStreamSynchronize(p->s_copy);
    cudaStreamSynchronize(p->s_compute);
    if (p->s_d2h) cudaStreamSynchronize(p->s_d2h);
    {   // drain the host ring in index order
        const int first = (out_idx[0] >= 0 && (out_idx[1] < 0 || out_idx[0] < out_idx[1])) ? 0 : 1;
        float tail_ms = 0.0f;
        for (int k = 0; k < 2; ++k) {
            const int oo = k == 0 ? first : first ^ 1;
            if (out_idx[oo] < 0) continue;
            if (cudaEventElapsedTime(&ms, p->ev_first, p->ev_d2h_done[oo]) == cudaSuccess && ms > tail_ms) tail_ms = ms;
            const int frc = finish_out(oo, rc == TOI_OK);
            if (rc == TOI_OK) rc = frc;
        }
        if (tail_used && cudaEventElapsedTime(&ms, p->ev_first, p->ev_tail) == cudaSuccess && ms > tail_ms) tail_ms = ms;
        st.gpu_ms = tail_ms;
    }
    st.n_done = n;
    for (int slot = 0; slot < 2; ++slot)
        if (used[slot]) harvest(slot);
    if (n > 0) {
        const int last = (int)((n - 1) & 1);
        if (cudaEventElapsedTime(&ms, p->ev_first, p->ev_c_done[last]) == cudaSuccess && ms > st.gpu_ms) st.gpu_ms = ms;
    }
    cudaGetLastError();
    st.wall_s = std::chrono::duration<double>(std::chrono::steady_clock::now() - t0).count();
    if (stats) *stats = st;
    if (rc == TOI_OK) {
        cudaMemcpy(p->h_state, p->d_state, sizeof(SnapState), cudaMemcpyDeviceToHost);
        if (p->deferred != TOI_OK) { rc = p->deferred; p->deferred = TOI_OK; }
    }
    return rc;
}

int toi_reproject(toi_plan *p, const float *d_image, const double *V, int32_t mode, void *cuda_stream, float *d_out)
{
    if (!p) return fail(nullptr, TOI_ERR_INVALID_ARG, "plan is NULL");
    if (!d_image || !d_out || d_image == d_out) return fail(p, TOI_ERR_INVALID_ARG, "d_image and d_out must be non-NULL and distinct");
    if (mode != TOI_REPROJECT_EXACT && mode != TOI_REPROJECT_PAPER) return fail(p, TOI_ERR_INVALID_ARG, "unknown re-projection mode");
    CU_TRY(p, cudaSetDevice(p->cfg.device));
    cudaStream_t stream = cuda_stream ? (cudaStream_t)cuda_stream : p->s_compute;
    if (V) {
        for (int k = 0; k < 9; ++k)
            if (!isfinite(V[k])) return fail(p, TOI_ERR_INVALID_ARG, "V must be finite");
        if (!(fabs(V[8]) >= 1e-6)) return fail(p, TOI_ERR_DEGENERATE_GEOMETRY, "V33 < 1e-6: no tilted plane to re-project from");
        CU_TRY(p, cudaMemcpyAsync(p->d_V_reproject, V, 9 * sizeof(double), cudaMemcpyHostToDevice, stream));
    }
    const double beta_rad = p->cfg.cell_size_deg * (3.14159265358979323846 / 180.0);
    launch_reproject(p->geo.N, beta_rad, p->d_state, V ? p->d_V_reproject : nullptr, mode, d_image, d_out, stream);
    CU_TRY(p, cudaGetLastError());
    return TOI_OK;
}

int toi_difference(toi_plan *p, const float *d_a, const float *d_b, void *cuda_stream, float *d_out)
{
    if (!p) return fail(nullptr, TOI_ERR_INVALID_ARG, "plan is NULL");
    if (!d_a || !d_b || !d_out) return fail(p, TOI_ERR_INVALID_ARG, "NULL argument");
    CU_TRY(p, cudaSetDevice(p->cfg.device));
    cudaStream_t stream = cuda_stream ? (cudaStream_t)cuda_stream : p->s_compute;
    launch_difference((size_t)p->geo.N * p->geo.N, d_a, d_b, d_out, p->n_sms, stream);
    CU_TRY(p, cudaGetLastError());
    return TOI_OK;
}

const char *toi_last_error(const toi_plan *plan) { return plan ? plan->err : g_create_error; }

int toi_last_launch_count(const toi_plan *plan) { return plan ? plan->last_launches : 0; }

int toi_debug_set_transform(toi_plan *p, const double *V)
{
    if (!p) return fail(nullptr, TOI_ERR_INVALID_ARG, "plan is NULL");
    CU_TRY(p, cudaSetDevice(p->cfg.device));
    CU_TRY(p, cudaDeviceSynchronize());
    p->inject = V != nullptr;
    if (V) CU_TRY(p, cudaMemcpy(p->d_V_inject, V, 9 * sizeof(double), cudaMemcpyHostToDevice));
    return TOI_OK;
}

int toi_debug_cell_indices(toi_plan *p, int32_t *d_iu, int32_t *d_iv)
{
    if (!p || !d_iu || !d_iv) return fail(p, TOI_ERR_INVALID_ARG, "NULL argument");
    if (!p->last_in.uvw) return fail(p, TOI_ERR_INVALID_ARG, "no snapshot has been imaged yet");
    CU_TRY(p, cudaSetDevice(p->cfg.device));
    CU_TRY(p, cudaDeviceSynchronize());
    launch_cell_indices(p->geo, p->last_in.uvw, p->d_state, d_iu, d_iv, p->s_compute);
    CU_TRY(p, cudaGetLastError());
    CU_TRY(p, cudaStreamSynchronize(p->s_compute));
    return TOI_OK;
}

int toi_debug_keep_grid(toi_plan *p, int32_t on)
{
    if (!p) return fail(nullptr, TOI_ERR_INVALID_ARG, "plan is NULL");
    if (on && !p->d_grid_keep) return fail(p, TOI_ERR_UNSUPPORTED, "debug capture needs a plan created with debug_keep_grid = 1");
    p->keep_grid = on != 0;
    return TOI_OK;
}

int toi_debug_copy_grid(toi_plan *p, void *d_grid_c64)
{
    if (!p || !d_grid_c64) return fail(p, TOI_ERR_INVALID_ARG, "NULL argument");
    if (!p->keep_grid || !p->d_grid_keep) return fail(p, TOI_ERR_INVALID_ARG, "call toi_debug_keep_grid(plan, 1) before imaging");
    CU_TRY(p, cudaSetDevice(p->cfg.device));
    CU_TRY(p, cudaDeviceSynchronize());
    CU_TRY(p, cudaMemcpy(d_grid_c64, p->d_grid_keep, (size_t)p->geo.G * p->geo.G * sizeof(float2), cudaMemcpyDeviceToDevice));
    return TOI_OK;
}

int toi_debug_copy_density(toi_plan *p, float *d_density)
{
    if (!p || !d_density) return fail(p, TOI_ERR_INVALID_ARG, "NULL argument");
    if (!p->d_dens) return fail(p, TOI_ERR_INVALID_ARG, "plan was not created with uniform weighting");
    if (!p->keep_grid || !p->d_dens_keep) return fail(p, TOI_ERR_INVALID_ARG, "call toi_debug_keep_grid(plan, 1) before imaging");
    CU_TRY(p, cudaSetDevice(p->cfg.device));
    CU_TRY(p, cudaDeviceSynchronize());
    CU_TRY(p, cudaMemcpy(d_density, p->d_dens_keep, (size_t)p->geo.G * p->geo.G * sizeof(float), cudaMemcpyDeviceToDevice));
    return TOI_OK;
}

}  // extern "C"
