// k_cheb.cu -- helper kernels of the near-coplanar ("3-D") mode, PAPER.md:202-269 (section 3.4,
// Eqs. 17-27): the residual coordinate r3 is kept, its range is cut into slabs, and inside a slab
// the residual phase is expanded in Chebyshev polynomials (Jacobi-Anger, Eqs. 21-22), so that the
// image is a sum of N_slab * K two-dimensional reconstructions ("Chebyshev moments", Eq. 24), each
// made by the ordinary gridder (with the factor T_k(s_q) applied per sample) and cuFFT:
//   I(t1,t2) = Re{ sum_p exp(i 2 pi r3_p t3) sum_k c_k(2 pi Delta_r3 t3) M_pk(t1,t2) } / (omega Wsum)   (Eq. 23)
// Readings: DESIGN.md G24-G26 (equal-width slabs, K rule, valid region = inside the sphere constraint).
//
//   k_r3_range      r3 range of the snapshot (Eq. 26) -- r3 = rho3 * s_c is monotone in s_c, so the
//                   extremes sit at the band edges of the extreme baselines
//   k_crop_complex  correction + crop of one moment, complex (k_correct_crop keeps only Re)
//   k_cheb_combine  acc += exp(i 2 pi r3_p t3) c_k(alpha) M_pk per pixel, c_0 = J_0, c_k = 2 i^k J_k
//   k_cheb_finish   image = Re(acc) / (omega Wsum); NaN outside the sphere constraint of Eq. 17
#include <math_constants.h>

#include "toi_internal.cuh"

namespace toi {
namespace {

__global__ void __launch_bounds__(256)
k_r3_range(int n_b, const double *__restrict__ uvw, const SnapState *__restrict__ st, double s_min, double s_max,
           double *__restrict__ out /* [2]: r3_min, r3_max */)
{
    __shared__ double s_lo[256], s_hi[256];
    double lo = CUDART_INF, hi = -CUDART_INF;
    for (int j = threadIdx.x; j < n_b; j += blockDim.x) {
        const double rho3 = rotate_row3(st->V, uvw + 3 * j);
        const double a = __dmul_rn(rho3, s_min), b = __dmul_rn(rho3, s_max);   // the gridder's own expression
        lo = fmin(lo, fmin(a, b));
        hi = fmax(hi, fmax(a, b));
    }
    s_lo[threadIdx.x] = lo; s_hi[threadIdx.x] = hi;
    __syncthreads();
    for (int d = 128; d > 0; d >>= 1) {
        if (threadIdx.x < d) {
            s_lo[threadIdx.x] = fmin(s_lo[threadIdx.x], s_lo[threadIdx.x + d]);
            s_hi[threadIdx.x] = fmax(s_hi[threadIdx.x], s_hi[threadIdx.x + d]);
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) { out[0] = s_lo[0]; out[1] = s_hi[0]; }
}

__global__ void __launch_bounds__(256)
k_crop_complex(int N, int G, const float2 *__restrict__ F, const double *__restrict__ ipsi, float2 *__restrict__ M)
{
    const int i = blockIdx.x * 32 + (threadIdx.x & 31);
    const int j = blockIdx.y * 8 + (threadIdx.x >> 5);
    if (i >= N || j >= N) return;
    const int n = i - (N >> 1), m = j - (N >> 1);
    const float2 f = __ldg(F + (size_t)(m < 0 ? m + G : m) * G + (n < 0 ? n + G : n));
    double c = ipsi[i] * ipsi[j];
    if ((n + m) & 1) c = -c;                                 // (-1)^(n+m) of the centred grid
    M[(size_t)j * N + i] = make_float2((float)(f.x * c), (float)(f.y * c));
}

// t3 of Eq. 17 at pixel (i, j); NaN outside the sphere constraint
__device__ __forceinline__ double t3_pixel(const double *V, int N, double beta_rad, int i, int j)
{
    const double t1 = -beta_rad * (double)(i - (N >> 1)), t2 = beta_rad * (double)(j - (N >> 1));
    const double a = t1 + V[2], b = t2 + V[5];
    const double rad = 1.0 - a * a - b * b;
    if (!(rad >= 0.0)) return CUDART_NAN;
    return -V[8] + (V[8] < 0.0 ? -sqrt(rad) : sqrt(rad));
}

__global__ void __launch_bounds__(256)
k_cheb_combine(int N, double beta_rad, const SnapState *__restrict__ st, int k, double r3_p, double d_r3,
               const float2 *__restrict__ M, float2 *__restrict__ acc, int first)
{
    const int i = blockIdx.x * 32 + (threadIdx.x & 31);
    const int j = blockIdx.y * 8 + (threadIdx.x >> 5);
    if (i >= N || j >= N) return;
    const size_t o = (size_t)j * N + i;
    const double t3 = t3_pixel(st->V, N, beta_rad, i, j);
    float2 a = first ? make_float2(0.0f, 0.0f) : acc[o];
    if (t3 == t3) {
        const double two_pi = 6.283185307179586476925286766559;
        const double alpha = two_pi * d_r3 * t3;                         // Eq. 20
        double ck = jn(k, alpha);                                        // Eq. 22
        if (k > 0) ck *= 2.0;
        double sp, cp;
        sincos(two_pi * r3_p * t3, &sp, &cp);
        // w = exp(i 2 pi r3_p t3) * i^k * ck
        double wr, wi;
        switch (k & 3) {
        case 0: wr = cp; wi = sp; break;
        case 1: wr = -sp; wi = cp; break;
        case 2: wr = -cp; wi = -sp; break;
        default: wr = sp; wi = -cp; break;
        }
        wr *= ck; wi *= ck;
        const float2 m = M[o];
        a.x += (float)(wr * m.x - wi * m.y);
        a.y += (float)(wr * m.y + wi * m.x);
    }
    acc[o] = a;
}

__global__ void __launch_bounds__(256)
k_cheb_finish(int N, double beta_rad, const SnapState *__restrict__ st, int apply_jacobian,
              const float2 *__restrict__ acc, float *__restrict__ image)
{
    const int i = blockIdx.x * 32 + (threadIdx.x & 31);
    const int j = blockIdx.y * 8 + (threadIdx.x >> 5);
    if (i >= N || j >= N) return;
    const size_t o = (size_t)j * N + i;
    float out = 0.0f;
    const double wsum = st->wsum;
    if (st->status == TOI_OK && wsum > 0.0) {
        const double t3 = t3_pixel(st->V, N, beta_rad, i, j);
        out = (t3 == t3) ? (float)((double)acc[o].x / ((apply_jacobian ? st->omega : 1.0) * wsum)) : CUDART_NAN_F;
    }
    image[o] = out;
}

}  // namespace

void launch_r3_range(int n_b, const double *d_uvw, const SnapState *st, double s_min, double s_max, double *d_out,
                     cudaStream_t stream)
{
    k_r3_range<<<1, 256, 0, stream>>>(n_b, d_uvw, st, s_min, s_max, d_out);
}

void launch_crop_complex(const Geometry &g, const float2 *d_F, const double *d_ipsi, float2 *d_M, cudaStream_t stream)
{
    dim3 grid((g.N + 31) / 32, (g.N + 7) / 8);
    k_crop_complex<<<grid, 256, 0, stream>>>(g.N, g.G, d_F, d_ipsi, d_M);
}

void launch_cheb_combine(int N, double beta_rad, const SnapState *st, int k, double r3_p, double d_r3,
                         const float2 *d_M, float2 *d_acc, int first, cudaStream_t stream)
{
    dim3 grid((N + 31) / 32, (N + 7) / 8);
    k_cheb_combine<<<grid, 256, 0, stream>>>(N, beta_rad, st, k, r3_p, d_r3, d_M, d_acc, first);
}

void launch_cheb_finish(int N, double beta_rad, const SnapState *st, int apply_jacobian, const float2 *d_acc,
                        float *d_image, cudaStream_t stream)
{
    dim3 grid((N + 31) / 32, (N + 7) / 8);
    k_cheb_finish<<<grid, 256, 0, stream>>>(N, beta_rad, st, apply_jacobian, d_acc, d_image);
}

}  // namespace toi
