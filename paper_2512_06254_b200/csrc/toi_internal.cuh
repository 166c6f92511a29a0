// toi_internal.cuh -- shared declarations of libtoi's translation units (CUDA path only).
// Nothing here is used by, or taken from, oracle/.
#pragma once
#include <cuda_runtime.h>
#include <cufft.h>
#include <stdint.h>

#include "../../include/toi.h"

namespace toi {

constexpr int kW = 7;           // kernel support (G9)
constexpr int kH = 3;           // (W-1)/2
constexpr float kBetaK = 16.1f; // 2.30 * W
constexpr int kOffGrid = INT32_MIN;

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

__device__ __forceinline__ void sample_cell(double rho1, double rho2, double s_c, double kappa,
                                            double &gu, double &gv, int &iu, int &iv)
{
    gu = -__dmul_rn(__dmul_rn(rho1, s_c), kappa);   // the minus is Eq. 9's x = -beta(...)
    gv = __dmul_rn(__dmul_rn(rho2, s_c), kappa);
    iu = (int)floor(__dadd_rn(gu, 0.5));
    iv = (int)floor(__dadd_rn(gv, 0.5));
}

__device__ __forceinline__ bool cell_on_grid(int iu, int iv, int G)
{
    const int lo = -(G >> 1) + kH, hi = (G >> 1) - 1 - kH;
    return iu >= lo && iu <= hi && iv >= lo && iv <= hi;
}

// signed cell k in [-G/2, G/2) -> array index (k + G) mod G  (no fftshift pass anywhere)
__device__ __forceinline__ int wrap_index(int k, int G) { return k < 0 ? k + G : k; }

// ---- data handling (G12/G13): select, never multiply by zero --------
__device__ __forceinline__ bool weight_ok(float w) { return w > 0.0f && w <= 3.402823466e+38f; }

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

// Gridding kernel phi(x) = exp(beta_k (sqrt(1 - (2x/W)^2) - 1)) (G9) at the seven taps
// du = -3..3 of a sample whose sub-cell offset is xoff = g - i in [-0.5, 0.5): tap distance du - xoff.
__device__ __forceinline__ void kernel_taps(float xoff, float p[kW])
{
    constexpr float k2w = 2.0f / kW;
    constexpr float kb2 = kBetaK * 1.4426950408889634f;   // beta_k * log2(e)
#pragma unroll
    for (int d = 0; d < kW; ++d) {
        const float t = fmaf(xoff, -k2w, (float)(d - kH) * k2w);
        float a = fmaf(-t, t, 1.0f);
        if (d == kW - 1) a = fmaxf(a, 0.0f);              // only du = +3 can reach |x| = W/2
        float r;
        asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(a));
        const float e = fmaf(r, kb2, -kb2);
        asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(p[d]) : "f"(e));
    }
}

// ---- host-side launchers, one per translation unit -------------------------------------------
void launch_planefit(const Geometry &g, const double *d_uvw, double S1, double S2, const double *d_V_inject,
                     SnapState *st, cudaStream_t stream);
void launch_density(const Geometry &g, const Inputs &in, SnapState *st, float *d_density, cudaStream_t stream);
void launch_grid_atomic(const Geometry &g, const Inputs &in, SnapState *st, const float *d_density,
                        float2 *d_grid, cudaStream_t stream);
void launch_grid_sliding(const Geometry &g, const Inputs &in, SnapState *st, const float *d_density,
                         float2 *d_grid, int n_sms, cudaStream_t stream);
void launch_correct_crop(const Geometry &g, const float2 *d_F, const double *d_ipsi, const SnapState *st,
                         int apply_jacobian, float *d_image, cudaStream_t stream);
void launch_cell_indices(const Geometry &g, const double *d_uvw, const SnapState *st, int32_t *d_iu,
                         int32_t *d_iv, cudaStream_t stream);

}  // namespace toi
