// toi_static.cu -- toi_cell_indices_static: steps a1-a3 (plane fit, rotation, centre-cell index of every
// sample, DESIGN.md section 3 steps 1-5) for callers that cannot allocate: code under
// CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.  No plan is needed and
// nothing is allocated, on the device or on the host: the scratch the kernels need -- the snapshot
// state the plane fit writes (SnapState: V, omega, singular values, status) and the channel scale
// table s_c = nu_c / c0 -- lives in ONE file-scope device array of fixed size, which every GPU that
// loads the library holds until the process exits (256 B + TOI_STATIC_MAX_CHANNELS x 8 B = 256.25 KB).
//
// Every call shares that array and finds the previous call's contents in it.  Nothing in it has to
// start at zero: the plane fit rewrites the whole SnapState and the call overwrites the n_channels
// table entries it reads.  Two calls that overlap on the GPU (different streams, or two host threads
// on one device) RACE on it; calls on one stream are ordered by the stream.
//
// The array's name is a host-side stand-in in host code, not a device address: its address is taken
// once per device with cudaGetSymbolAddress (that device current) and handed to the kernels.
#include <cstdio>
#include <mutex>

#include "toi_internal.cuh"

using namespace toi;

namespace {

constexpr int kMaxChannels = TOI_STATIC_MAX_CHANNELS;
constexpr size_t kStateBytes = 256;                      // SnapState, padded to the array's alignment
constexpr size_t kScratchBytes = kStateBytes + (size_t)kMaxChannels * sizeof(double);
static_assert(sizeof(SnapState) <= kStateBytes, "SnapState must fit its slot of the static scratch");

static __device__ __align__(256) unsigned char g_static_scratch[kScratchBytes];

constexpr int kMaxDevices = 64;
std::mutex g_mutex;                                      // address table and host staging table
unsigned char *g_scratch_addr[kMaxDevices] = {};         // device address of g_static_scratch, per device
double g_h_s[kMaxChannels];                              // host staging of the scale table (pageable, 256 KB)

int fail_static(char *err, int32_t err_len, int code, const char *what, const char *detail = "")
{
    if (err && err_len > 0) snprintf(err, (size_t)err_len, "toi_cell_indices_static: %s%s", what, detail);
    return code;
}

// The variant of k_cell_indices (k_planefit.cu) that takes the snapshot state and the scale table from
// the static scratch: same arithmetic (rotate_baseline, sample_cell: normative fp64 order).
__global__ void __launch_bounds__(256)
k_cell_indices_static(int n_b, int n_c, double kappa, const double *__restrict__ uvw,
                      const unsigned char *__restrict__ scratch, int32_t *__restrict__ iu_out,
                      int32_t *__restrict__ iv_out)
{
    const SnapState *st = reinterpret_cast<const SnapState *>(scratch);
    const double *s = reinterpret_cast<const double *>(scratch + kStateBytes);
    const long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= (long long)n_b * n_c) return;
    const int j = (int)(q / n_c), c = (int)(q % n_c);
    double rho1, rho2;
    int iu, iv;
    float xu, xv;
    rotate_baseline(st->V, uvw + 3 * j, rho1, rho2);
    sample_cell(rho1, rho2, s[c], kappa, iu, iv, xu, xv);
    iu_out[q] = iu;
    iv_out[q] = iv;
}

}  // namespace

#define STATIC_TRY(expr)                                                                           \
    do {                                                                                           \
        cudaError_t e_ = (expr);                                                                   \
        if (e_ != cudaSuccess) return fail_static(err, err_len, TOI_ERR_CUDA, #expr ": ", cudaGetErrorString(e_)); \
    } while (0)

extern "C" int toi_cell_indices_static(const double *d_uvw_m, int32_t n_baselines, const double *chan_freq_hz,
                                       int32_t n_channels, int32_t grid_size, double cell_size_deg, void *cuda_stream,
                                       int32_t *d_iu, int32_t *d_iv, double *d_fit_out, char *err, int32_t err_len)
{
    if (err && err_len > 0) err[0] = '\0';
    if (!d_uvw_m || !chan_freq_hz || !d_iu || !d_iv) return fail_static(err, err_len, TOI_ERR_INVALID_ARG, "d_uvw_m, chan_freq_hz, d_iu and d_iv must be non-NULL");
    if (n_baselines < 3) return fail_static(err, err_len, TOI_ERR_INVALID_ARG, "n_baselines must be >= 3");
    if (n_channels < 1) return fail_static(err, err_len, TOI_ERR_INVALID_ARG, "n_channels must be >= 1");
    if (n_channels > kMaxChannels) {
        char detail[96];
        snprintf(detail, sizeof detail, "%d > TOI_STATIC_MAX_CHANNELS = %d (the static scratch holds no more)", (int)n_channels, kMaxChannels);
        return fail_static(err, err_len, TOI_ERR_UNSUPPORTED, "n_channels ", detail);
    }
    if (grid_size < 2 || grid_size > 32768 || !(cell_size_deg > 0.0)) return fail_static(err, err_len, TOI_ERR_INVALID_ARG, "grid_size must be in [2, 32768] and cell_size_deg > 0");
    for (int c = 0; c < n_channels; ++c)
        if (!(chan_freq_hz[c] > 0.0)) return fail_static(err, err_len, TOI_ERR_INVALID_ARG, "channel frequencies must be positive");
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    int dev = -1;
    STATIC_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kMaxDevices) return fail_static(err, err_len, TOI_ERR_UNSUPPORTED, "device ordinal beyond the address table");

    std::lock_guard<std::mutex> lock(g_mutex);
    // set-up, once per device, with that device current: the device address of the static array
    if (!g_scratch_addr[dev]) {
        void *ptr = nullptr;
        STATIC_TRY(cudaGetSymbolAddress(&ptr, g_static_scratch));
        g_scratch_addr[dev] = static_cast<unsigned char *>(ptr);
    }
    unsigned char *scratch = g_scratch_addr[dev];

    // plan-time scalars exactly as toi_plan_create forms them (fp64 on the host)
    long double s1 = 0, s2 = 0;
    for (int c = 0; c < n_channels; ++c) {
        g_h_s[c] = chan_freq_hz[c] / 299792458.0;
        s1 += g_h_s[c];
        s2 += (long double)g_h_s[c] * g_h_s[c];
    }
    // pageable source: the call returns once the table is staged, so g_h_s is free again when the lock drops
    STATIC_TRY(cudaMemcpyAsync(scratch + kStateBytes, g_h_s, (size_t)n_channels * sizeof(double), cudaMemcpyHostToDevice, stream));

    Geometry g = {};
    g.n_b = n_baselines; g.n_c = n_channels; g.n_p = 1;
    g.G = grid_size; g.N = grid_size;
    g.kappa = (double)grid_size * (cell_size_deg * (3.14159265358979323846 / 180.0));
    g.s = reinterpret_cast<const double *>(scratch + kStateBytes);
    // a1-a2: the plane fit rewrites the whole SnapState slot (no programmatic launch: nothing to overlap with)
    const bool pdl_saved = g_pdl_enabled;
    g_pdl_enabled = false;
    launch_planefit(g, d_uvw_m, (double)s1, (double)s2, nullptr, reinterpret_cast<SnapState *>(scratch), stream);
    g_pdl_enabled = pdl_saved;
    STATIC_TRY(cudaGetLastError());
    // a3: cell indices
    const long long S = (long long)n_baselines * n_channels;
    k_cell_indices_static<<<(unsigned)((S + 255) / 256), 256, 0, stream>>>(n_baselines, n_channels, g.kappa, d_uvw_m, scratch, d_iu, d_iv);
    STATIC_TRY(cudaGetLastError());
    // V[9], omega, sing[3]: the first 13 doubles of SnapState
    if (d_fit_out) STATIC_TRY(cudaMemcpyAsync(d_fit_out, scratch, 13 * sizeof(double), cudaMemcpyDeviceToDevice, stream));
    return TOI_OK;
}
