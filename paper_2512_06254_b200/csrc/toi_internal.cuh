// toi_internal.cuh -- shared declarations of libtoi's translation units (CUDA path only).
// Nothing here is used by, or taken from, oracle/.
#pragma once
#include <cuda_runtime.h>
#include <cufft.h>
#include <stdint.h>
#include <stdlib.h>

#include "../../include/toi.h"

namespace toi {

constexpr int kW = 7;           // kernel support (G9)
constexpr int kH = 3;           // (W-1)/2
constexpr float kBetaK = 16.1f; // 2.30 * W
constexpr int kOffGrid = INT32_MIN;
// tiles of the sparse-clear maps (k_clear.cu): 128 cells wide (1 KB of complex64 per row: whole DRAM
// bursts) and 8 rows high
constexpr int kTileW = 128, kTileH = 8;
inline __host__ __device__ int tiles_per_row(int G) { return (G + kTileW - 1) / kTileW; }
inline __host__ __device__ int tile_rows(int G) { return (G + kTileH - 1) / kTileH; }

// Device-resident per-snapshot state: written by k_planefit, accumulated by the weighting and
// gridding kernels, read by k_correct_crop.  No host round trip between the stages.
struct SnapState {
    double V[9];
    double omega;
    double sing[3];
    double wsum;                       // sum f_q w_I,q over gridded samples
    unsigned long long n_gridded, n_off_grid, n_flagged;
    unsigned int task_counter;         // dynamic task queue of the sliding gridder
    int status;                        // TOI_OK or TOI_ERR_DEGENERATE_GEOMETRY
};

// Everything a kernel needs to know about the problem (passed by value).
struct Geometry {
    int n_b, n_c, n_p, pol_a, pol_b;
    int N, G;
    double kappa;                      // G * beta_rad, cells per wavelength
    const double *s;                   // device [n_c], s_c = nu_c / c0
};

struct Inputs {
    const double *uvw;                 // device [n_b][3]
    const float2 *vis;                 // device [n_b][n_c][n_p]
    const float *weights;              // device or nullptr
    const uint8_t *flags;              // device or nullptr
};

// ---- fp64 coordinates (DESIGN.md section 3 steps 4-5; expression order is normative) --------
// Every operation is individually rounded: __dmul_rn/__dadd_rn are never contracted to FMA.
__device__ __forceinline__ void rotate_baseline(const double *V, const double *uvw_j, double &rho1,
                                                double &rho2)
{
    const double u = uvw_j[0], v = uvw_j[1], w = uvw_j[2];
    rho1 = __dadd_rn(__dadd_rn(__dmul_rn(V[0], u), __dmul_rn(V[1], v)), __dmul_rn(V[2], w));
    rho2 = __dadd_rn(__dadd_rn(__dmul_rn(V[3], u), __dmul_rn(V[4], v)), __dmul_rn(V[5], w));
}

// third row: rho3 = V3 . uvw (metres), the residual coordinate kept by the near-coplanar mode
__device__ __forceinline__ double rotate_row3(const double *V, const double *uvw_j)
{
    return __dadd_rn(__dadd_rn(__dmul_rn(V[6], uvw_j[0]), __dmul_rn(V[7], uvw_j[1])), __dmul_rn(V[8], uvw_j[2]));
}

// One Chebyshev-moment pass of the near-coplanar mode (Eqs. 19-24): the gridder
// keeps only the samples of slab p and multiplies them by T_k(s_q).
struct ChebArgs {
    int p, k, n_slab;
    int count;              // bit 0: this pass accumulates Wsum and n_gridded (k == 0: once per slab);
                            // bit 1: it also counts the flagged and off-grid samples (p == 0, k == 0:
                            // once per snapshot -- every pass sees all of them)
    double r3_min;          // lower end of the r3 range
    double d;               // slab half-width Delta_r3 (0: all samples share one r3)
};

// floor(y) for |y| < 2^31 without the slow F2I/I2F conversion pipe: adding 2^52 + 2^51 with
// round-down leaves floor(y) in the low word of the sum (the ulp there is 1), and subtracting the
// constant again is exact.  Bit-identical to (int)floor(y).
constexpr double kFloorMagic = 6755399441055744.0;
__device__ __forceinline__ int floor_to_int(double y, double &fl)
{
    const double m = __dadd_rd(y, kFloorMagic);
    fl = __dsub_rn(m, kFloorMagic);
    return __double2loint(m);
}

// Normative order (DESIGN.md section 3 step 5): t = rho * s_c; g = -(t * kappa) resp. +(t * kappa);
// i = floor(g + 1/2).  xu, xv = g - i in [-1/2, 1/2] as fp32 (the sub-cell offsets).
__device__ __forceinline__ void sample_cell(double rho1, double rho2, double s_c, double kappa,
                                            int &iu, int &iv, float &xu, float &xv)
{
    const double gu = -__dmul_rn(__dmul_rn(rho1, s_c), kappa);   // the minus is Eq. 9's x = -beta(...)
    const double gv = __dmul_rn(__dmul_rn(rho2, s_c), kappa);
    double fu, fv;
    iu = floor_to_int(__dadd_rn(gu, 0.5), fu);
    iv = floor_to_int(__dadd_rn(gv, 0.5), fv);
    xu = (float)__dsub_rn(gu, fu);
    xv = (float)__dsub_rn(gv, fv);
    if (!(fabs(gu) < 1073741824.0 && fabs(gv) < 1073741824.0)) iu = iv = kOffGrid;   // also NaN
}

__device__ __forceinline__ bool cell_on_grid(int iu, int iv, int G)
{
    const int lo = -(G >> 1) + kH, hi = (G >> 1) - 1 - kH;
    return iu >= lo && iu <= hi && iv >= lo && iv <= hi;
}

// The grid (and the density map) are stored CENTRED: signed cell k in [-G/2, G/2) lives at array
// index k + G/2, so no address ever wraps while gridding.  cuFFT then sees the input shifted by
// G/2 on both axes, i.e. its output is (-1)^(n+m) times the transform of the unshifted grid
// (shift theorem); k_correct_crop applies that sign.  No fftshift pass exists anywhere.
__device__ __forceinline__ size_t centre_index(int iu, int iv, int G)
{
    return (size_t)(iv + (G >> 1)) * (size_t)G + (size_t)(iu + (G >> 1));
}

// ---- data handling (G12/G13): select, never multiply by zero --------
// positive and finite, i.e. bit pattern in [1, 0x7f7fffff]: one integer compare instead of two float ones
__device__ __forceinline__ bool weight_ok(float w) { return __float_as_uint(w) - 1u < 0x7f7fffffu; }

// Effective per-hand weights of sample q (element offset o = q * n_p) and the Stokes-I weight.
__device__ __forceinline__ void sample_weights(const Geometry &g, const Inputs &in, long long o, float &wa,
                                               float &wb)
{
    wa = in.weights ? __ldg(in.weights + o + g.pol_a) : 1.0f;
    if (!weight_ok(wa) || (in.flags && __ldg(in.flags + o + g.pol_a))) wa = 0.0f;
    wb = 0.0f;
    if (g.pol_b != g.pol_a) {
        wb = in.weights ? __ldg(in.weights + o + g.pol_b) : 1.0f;
        if (!weight_ok(wb) || (in.flags && __ldg(in.flags + o + g.pol_b))) wb = 0.0f;
    }
}

// z = w_a Vis_a + w_b Vis_b with a zero-weight hand skipped (its data may be NaN).
__device__ __forceinline__ float2 sample_stokes(const Geometry &g, const Inputs &in, long long o, float wa,
                                                float wb)
{
    float2 z = make_float2(0.0f, 0.0f);
    if (wa > 0.0f) {
        const float2 a = __ldg(in.vis + o + g.pol_a);
        z.x = wa * a.x; z.y = wa * a.y;
    }
    if (wb > 0.0f) {
        const float2 b = __ldg(in.vis + o + g.pol_b);
        z.x = fmaf(wb, b.x, z.x); z.y = fmaf(wb, b.y, z.y);
    }
    return z;
}

// ---- programmatic dependent launch (sm_90+) ------------------------------------------------------
// The kernels of a snapshot run back to back on one stream.  Launched with the programmatic-serialisation
// attribute, kernel n + 1's CTAs may become resident while kernel n drains (its CTAs have all passed
// pdl_trigger or exited) and sit in pdl_wait until kernel n has completed and its writes are visible:
// the launch latency between two kernels (~2 us) runs under the tail of the first.  Every kernel launched
// this way calls pdl_wait before it touches anything an earlier kernel wrote (or will still read).
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

// Off while the two lanes of the 3-D mode are being enqueued: there, early-resident CTAs of one lane's
// next kernel take SM room from the other lane's running kernel (measured: 19.3 -> 19.4-19.8 ms).
inline thread_local bool g_pdl_enabled = true;

template <class... P, class... A>
inline cudaError_t launch_pdl(void (*kernel)(P...), dim3 grid, dim3 block, size_t smem, cudaStream_t stream, A... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = stream;
    cudaLaunchAttribute attr;
    attr.id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr.val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = &attr;
    cfg.numAttrs = g_pdl_enabled ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kernel, P(args)...);
}

// ---- sparse clear (k_clear.cu; also run inside the transform's column pass) ------------------------
// One warp takes kClearTilesPerWarp consecutive map entries starting at t0 and clears the marked tiles
// one after the other (few tiles per warp: the marked tiles cluster around the uv origin, and a warp
// that finds all of its entries marked must not become the tail of the kernel).  A tile row of the
// grid is kTileW complex64 = 1 KB, written with 8-byte stores.
// The density map (uniform weighting) needs no map of its own: the density pass writes the centre
// cells of the samples -- inside the tiles the gridder marks for the same samples' windows -- and
// their mirror cells (-iu, -iv), i.e. array index (G - x, G - y) for (x, y).  For every marked tile
// the same rectangle of the density map and its point mirror are zeroed (4-byte stores: the mirrored
// rectangle starts on any column).
constexpr int kClearTilesPerWarp = 4;
__device__ __forceinline__ void clear_tiles_warp(float2 *__restrict__ grid, float *__restrict__ dens, int G,
                                                 uint8_t *__restrict__ map, int tpr, long long n_tiles, long long t0, int lane,
                                                 bool reset = true)
{
    if (t0 >= n_tiles) return;
    const long long mine = t0 + lane;
    const bool dirty = lane < kClearTilesPerWarp && mine < n_tiles && map[mine] != 0;
    if (dirty && reset) map[mine] = 0;     // reset == false: another clear launch follows on the same map
    unsigned todo = __ballot_sync(0xffffffffu, dirty);
    while (todo) {
        const int b = __ffs(todo) - 1;
        todo &= todo - 1;
        const long long t = t0 + b;
        const int x0 = (int)(t % tpr) * kTileW, y0 = (int)(t / tpr) * kTileH;
        const int rows = min(kTileH, G - y0);
        if (grid != nullptr) {
            float2 *row = grid + (size_t)y0 * G + x0;
            for (int r = 0; r < rows; ++r, row += G) {
#pragma unroll
                for (int k = 0; k < kTileW / 32; ++k)
                    if (x0 + k * 32 + lane < G) row[k * 32 + lane] = make_float2(0.0f, 0.0f);
            }
        }
        if (dens != nullptr) {
            for (int r = 0; r < rows; ++r) {
                float *own = dens + (size_t)(y0 + r) * G;
                const int ym = G - (y0 + r);                      // mirrored row; G itself is outside
                float *mir = dens + (size_t)(ym < G ? ym : 0) * G;
#pragma unroll
                for (int k = 0; k < kTileW / 32; ++k) {
                    const int x = x0 + k * 32 + lane, xm = G - x;
                    if (x < G) own[x] = 0.0f;
                    if (x < G && ym < G && xm < G) mir[xm] = 0.0f;
                }
            }
        }
    }
}

// ---- packed fp32 pairs (sm_100a FFMA2 / FMUL2: two fp32 lanes per instruction) ----------------
typedef unsigned long long u64;
__device__ __forceinline__ u64 pack2(float x, float y)
{
    u64 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(x), "f"(y));
    return r;
}
__device__ __forceinline__ float2 unpack2(u64 v)
{
    float2 r;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(r.x), "=f"(r.y) : "l"(v));
    return r;
}
__device__ __forceinline__ u64 fma2(u64 a, u64 b, u64 c)
{
    u64 d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
// acc += a * b with the accumulator tied to one register pair (keeps ptxas from renaming the
// accumulators across the branches of the sliding-window loop)
__device__ __forceinline__ void fma2_acc(u64 &acc, u64 a, u64 b)
{
    asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(acc) : "l"(a), "l"(b));
}
__device__ __forceinline__ u64 mul2(u64 a, u64 b)
{
    u64 d;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}

// Gridding kernel phi(x) = exp(beta_k (sqrt(1 - (2x/W)^2) - 1)) (G9) at the seven taps
// k = -3..3 of a sample whose sub-cell offsets are (xu, xv) = g - i in [-0.5, 0.5]: tap distance
// x = k - xoff.  phi is even, so phi(+-k - d) = E_k(d^2) +- d O_k(d^2) with one even and one odd
// polynomial per PAIR of taps (degrees 4 and 3 in s = d^2; coefficients in tap_poly.inc, written by
// gen_tap_poly.py from phi's definition; fit error <= 2.3e-8 absolute, below fp32 rounding of the
// centre taps).  Both axes are evaluated together as packed pairs (FFMA2 with broadcast immediate
// coefficients): 33 instructions for the 14 taps and nothing on the MUFU pipe, against 14 square
// roots + 14 exp2 before.
#include "tap_poly.inc"
__device__ __forceinline__ u64 bcast2(float c) { return pack2(c, c); }
__device__ __forceinline__ void kernel_taps2(float xu, float xv, float pu[kW], float pv[kW])
{
    const u64 X = pack2(xu, xv);
    const u64 NX = pack2(-xu, -xv);
    const u64 S = mul2(X, X);
#define TOI_EVEN(k)                                                                               \
    fma2(fma2(fma2(fma2(bcast2(TOI_TAP_E(k, 4)), S, bcast2(TOI_TAP_E(k, 3))), S, bcast2(TOI_TAP_E(k, 2))), S, \
              bcast2(TOI_TAP_E(k, 1))), S, bcast2(TOI_TAP_E(k, 0)))
#define TOI_ODD(k)                                                                                \
    fma2(fma2(fma2(bcast2(TOI_TAP_O(k, 3)), S, bcast2(TOI_TAP_O(k, 2))), S, bcast2(TOI_TAP_O(k, 1))), S, \
         bcast2(TOI_TAP_O(k, 0)))
#define TOI_PAIR(k)                                                                               \
    {                                                                                             \
        const u64 E = TOI_EVEN(k), O = TOI_ODD(k);                                                \
        const float2 hi = unpack2(fma2(X, O, E)), lo = unpack2(fma2(NX, O, E));                   \
        pu[kH + k] = hi.x; pv[kH + k] = hi.y;                                                     \
        pu[kH - k] = lo.x; pv[kH - k] = lo.y;                                                     \
    }
    {
        const float2 c = unpack2(TOI_EVEN(0));
        pu[kH] = c.x; pv[kH] = c.y;
    }
    TOI_PAIR(1)
    TOI_PAIR(2)
    TOI_PAIR(3)
#undef TOI_EVEN
#undef TOI_ODD
#undef TOI_PAIR
}

// Strip length of the sliding-window gridders: a task is `groups` strips of `strip` consecutive
// channels of one baseline.  Near `want` (tasks per resident warp), a multiple of `batch`, and such
// that the tasks of a row cover n_c with the least padding (a padded task still walks all its
// batches): n_c = 4096 with 4 groups and want = 96 gives 104 (10 tasks, 1.5 % padding) instead of
// 96 (11 tasks, 3 %); with 8 groups and want = 72 it gives 64 (8 tasks, none) instead of 72 (12 %).
inline int pick_strip(int n_c, int groups, int batch, long long want, int lo, int hi)
{
    if (want < lo) want = lo;
    if (want > hi) want = hi;
    const int share = ((n_c + groups - 1) / groups + batch - 1) / batch * batch;   // one task per row
    if (want >= share) return share;
    int best = (int)(want / batch * batch), best_pad = 1 << 30;
    for (int s = (int)(want * 3 / 4) / batch * batch; s <= want * 5 / 4; s += batch) {
        if (s < lo || s > hi || s > share) continue;
        const int t = (n_c + groups * s - 1) / (groups * s);
        const int pad = t * groups * s - n_c;
        if (pad < best_pad || (pad == best_pad && llabs(s - want) < llabs(best - want))) { best = s; best_pad = pad; }
    }
    return best;
}

// ---- host-side launchers, one per translation unit -------------------------------------------
void launch_planefit(const Geometry &g, const double *d_uvw, double S1, double S2, const double *d_V_inject,
                     SnapState *st, cudaStream_t stream);
// `tiles`: byte map of the kTileW x kTileH-cell tiles of the grid the gridder may write -- it sets the
// entries, launch_clear_tiles zeroes those tiles (and the density map under and opposite them) again
// and resets the entries.
void launch_density(const Geometry &g, const Inputs &in, SnapState *st, float *d_density, cudaStream_t stream);
void launch_grid_atomic(const Geometry &g, const Inputs &in, SnapState *st, const float *d_density,
                        float2 *d_grid, cudaStream_t stream);
// tiles == nullptr: the caller has marked every tile itself (channel scales not monotone)
void launch_grid_pair8(const Geometry &g, const Inputs &in, SnapState *st, const float *d_density,
                       float2 *d_grid, uint8_t *tiles, int n_sms, cudaStream_t stream);
// elements of guard band before and after the grid: k_grid_pair8's 8 x 8 window may overhang the
// grid by one row / column (of zeros); a multiple of 32 elements keeps the grid 256-byte aligned
inline size_t grid_guard(int G) { return ((size_t)G + 8 + 31) / 32 * 32; }
void launch_grid_pair8_cheb(const Geometry &g, const Inputs &in, SnapState *st, const float *d_density,
                            float2 *d_grid, uint8_t *tiles, int n_sms, const ChebArgs &cheb, cudaStream_t stream);
void launch_clear_tiles(float2 *d_grid, float *d_density, int G, uint8_t *d_map, cudaStream_t stream, bool reset_map = true);
// hand-written pruned transform (k_fft.cu): rows through the tile map, then columns with the crop fused
bool fft_custom_supported(int N, int G);
void fft_twiddle_table(int G, float2 *host_out);
void launch_fft_rows(int N, int G, const float2 *d_grid, float2 *d_work, const uint8_t *d_map, const float2 *d_tw,
                     int n_sms, cudaStream_t stream);
void launch_fft_cols(int N, int G, const float2 *d_work, const float2 *d_tw, const double *d_ipsi, const SnapState *st,
                     int apply_jacobian, float *d_image, float2 *d_moment, float2 *d_clear_grid, float *d_clear_density,
                     uint8_t *d_clear_map, int n_sms, cudaStream_t stream);
void launch_r3_range(int n_b, const double *d_uvw, const SnapState *st, double s_min, double s_max, double *d_out,
                     cudaStream_t stream);
size_t bessel_table_floats(int K);
void launch_bessel_table(int K, double a_max, float *d_tab, cudaStream_t stream);
void launch_cheb_combine(const Geometry &g, double beta_rad, const SnapState *st, int k0, int n_moments, double r3_p,
                         double d_r3, const float *d_tab, double a_max, const float2 *d_F0, const float2 *d_F1, int compact,
                         const double *d_ipsi, float2 *d_slab, float2 *d_acc, int first_k, int last_k, int first_slab,
                         cudaStream_t stream);
void launch_cheb_finish(int N, double beta_rad, const SnapState *st, int apply_jacobian, const float2 *d_acc,
                        float *d_image, cudaStream_t stream);
void launch_correct_crop(const Geometry &g, const float2 *d_F, const double *d_ipsi, const SnapState *st,
                         int apply_jacobian, float *d_image, cudaStream_t stream);
void launch_reproject(int N, double beta_rad, const SnapState *st, const double *d_V, int mode, const float *d_src,
                      float *d_dst, cudaStream_t stream);
void launch_difference(size_t n, const float *d_a, const float *d_b, float *d_out, int n_sms, cudaStream_t stream);
void launch_cell_indices(const Geometry &g, const double *d_uvw, const SnapState *st, int32_t *d_iu,
                         int32_t *d_iv, cudaStream_t stream);

}  // namespace toi
