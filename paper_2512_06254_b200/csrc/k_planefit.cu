// k_planefit.cu -- step a1: basis estimate of PAPER.md:115-117 (section 3.1), fp64, on the device.
//
// The paper applies SVD/PCA to the centred baseline matrix Btilde = B - Bbar whose rows are all
// (baseline, channel) samples b_q = s_c * uvw_j in wavelengths.  Its right
// singular vectors are the eigenvectors of the 3x3 scatter matrix C = Btilde^T Btilde, and
// because every row is a baseline scaled by a channel factor, C factorises exactly:
//     sum_q b_q b_q^T = (sum_c s_c^2) * (sum_j uvw_j uvw_j^T),   Bbar = mean(s) * mean(uvw)
//     C = S2 * M2 - S * Bbar Bbar^T,    S = n_b * n_c, S1 = sum s_c, S2 = sum s_c^2
// so the fit costs O(n_b) on the device plus O(n_c) once at plan time instead of O(n_b n_c).
// The plane normal is the eigenvector of the smallest eigenvalue; the in-plane axes are the
// minimal rotation taking w onto that normal (reading G3); omega is Eq. 8
// (PAPER.md:148).  Also resets the per-snapshot accumulators of SnapState.
#include "toi_internal.cuh"

namespace toi {

namespace {

constexpr int kFitThreads = 256;

// Cyclic Jacobi on a symmetric 3x3 held as six numbers; returns eigenvalues in d[3] and the
// eigenvectors as the columns of Q (row-major 3x3).
__device__ void sym3_eigen(double a00, double a01, double a02, double a11, double a12, double a22,
                           double d[3], double Q[9])
{
    double A[3][3] = {{a00, a01, a02}, {a01, a11, a12}, {a02, a12, a22}};
    for (int i = 0; i < 9; ++i) Q[i] = (i % 4 == 0) ? 1.0 : 0.0;
    for (int sweep = 0; sweep < 60; ++sweep) {
        const double off = A[0][1] * A[0][1] + A[0][2] * A[0][2] + A[1][2] * A[1][2];
        const double diag = A[0][0] * A[0][0] + A[1][1] * A[1][1] + A[2][2] * A[2][2];
        if (off <= 1e-44 * diag || off == 0.0) break;
        const int P[3] = {0, 0, 1}, R[3] = {1, 2, 2};
        for (int e = 0; e < 3; ++e) {
            const int p = P[e], r = R[e];
            const double apr = A[p][r];
            if (apr == 0.0) continue;
            // rotation angle that annihilates A[p][r]
            const double tau = (A[r][r] - A[p][p]) / (2.0 * apr);
            const double t = copysign(1.0, tau) / (fabs(tau) + sqrt(1.0 + tau * tau));
            const double c = rsqrt(1.0 + t * t), s = t * c;
            const int q = 3 - p - r;   // the untouched index
            const double app = A[p][p], arr = A[r][r], aqp = A[q][p], aqr = A[q][r];
            A[p][p] = app - t * apr;
            A[r][r] = arr + t * apr;
            A[p][r] = A[r][p] = 0.0;
            A[q][p] = A[p][q] = c * aqp - s * aqr;
            A[q][r] = A[r][q] = s * aqp + c * aqr;
            for (int k = 0; k < 3; ++k) {
                const double qp = Q[3 * k + p], qr = Q[3 * k + r];
                Q[3 * k + p] = c * qp - s * qr;
                Q[3 * k + r] = s * qp + c * qr;
            }
        }
    }
    d[0] = A[0][0]; d[1] = A[1][1]; d[2] = A[2][2];
}

__global__ void __launch_bounds__(kFitThreads)
k_planefit(int n_b, int n_c, const double *__restrict__ uvw, double S1, double S2,
           const double *__restrict__ V_inject, SnapState *__restrict__ st)
{
    __shared__ double red[9][kFitThreads];
    const int tid = threadIdx.x;
    // uvw may have been produced on this stream by the caller's own kernel just before the call: wait for
    // whatever precedes (visibility of its writes is guaranteed only behind this wait) before reading it
    pdl_wait();
    pdl_trigger();
    double acc[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0};
    if (!V_inject) {
        for (int j = tid; j < n_b; j += kFitThreads) {
            const double u = uvw[3 * j], v = uvw[3 * j + 1], w = uvw[3 * j + 2];
            acc[0] += u; acc[1] += v; acc[2] += w;
            acc[3] += u * u; acc[4] += u * v; acc[5] += u * w;
            acc[6] += v * v; acc[7] += v * w; acc[8] += w * w;
        }
    }
    for (int k = 0; k < 9; ++k) red[k][tid] = acc[k];
    __syncthreads();
    for (int half = kFitThreads / 2; half > 0; half >>= 1) {   // fixed-shape tree: deterministic
        if (tid < half)
            for (int k = 0; k < 9; ++k) red[k][tid] += red[k][tid + half];
        __syncthreads();
    }
    if (tid != 0) return;

    st->wsum = 0.0;
    st->n_gridded = st->n_off_grid = st->n_flagged = 0ull;
    st->task_counter = 0u;
    st->status = TOI_OK;

    double V[9];
    if (V_inject) {
        for (int k = 0; k < 9; ++k) V[k] = V_inject[k];
        st->sing[0] = st->sing[1] = st->sing[2] = 0.0;
    } else {
        const double S = (double)n_b * (double)n_c;
        const double mu = red[0][0] / (double)n_b, mv = red[1][0] / (double)n_b, mw = red[2][0] / (double)n_b;
        const double ms = S1 / (double)n_c;
        const double bu = ms * mu, bv = ms * mv, bw = ms * mw;          // Bbar
        const double c00 = S2 * red[3][0] - S * bu * bu, c01 = S2 * red[4][0] - S * bu * bv,
                     c02 = S2 * red[5][0] - S * bu * bw, c11 = S2 * red[6][0] - S * bv * bv,
                     c12 = S2 * red[7][0] - S * bv * bw, c22 = S2 * red[8][0] - S * bw * bw;
        double lam[3], Q[9];
        sym3_eigen(c00, c01, c02, c11, c12, c22, lam, Q);
        int o0 = 0, o1 = 1, o2 = 2, tmp;                                   // descending order
        if (lam[o1] > lam[o0]) { tmp = o0; o0 = o1; o1 = tmp; }
        if (lam[o2] > lam[o0]) { tmp = o0; o0 = o2; o2 = tmp; }
        if (lam[o2] > lam[o1]) { tmp = o1; o1 = o2; o2 = tmp; }
        st->sing[0] = sqrt(fmax(lam[o0], 0.0));
        st->sing[1] = sqrt(fmax(lam[o1], 0.0));
        st->sing[2] = sqrt(fmax(lam[o2], 0.0));
        if (!(lam[o0] > 0.0) || lam[o1] <= 1e-10 * lam[o0]) st->status = TOI_ERR_DEGENERATE_GEOMETRY;
        // plane normal = e1 x e2 of the two dominant directions (right-handed third axis)
        const double e1x = Q[o0], e1y = Q[3 + o0], e1z = Q[6 + o0];
        const double e2x = Q[o1], e2y = Q[3 + o1], e2z = Q[6 + o1];
        double nx = e1y * e2z - e1z * e2y, ny = e1z * e2x - e1x * e2z, nz = e1x * e2y - e1y * e2x;
        const double inv = 1.0 / sqrt(nx * nx + ny * ny + nz * nz);
        nx *= inv; ny *= inv; nz *= inv;
        if (nz < 0.0) { nx = -nx; ny = -ny; nz = -nz; }                    // G4: V33 > 0
        const double k1 = 1.0 + nz;
        V[0] = 1.0 - nx * nx / k1; V[1] = -nx * ny / k1;      V[2] = -nx;
        V[3] = -nx * ny / k1;      V[4] = 1.0 - ny * ny / k1; V[5] = -ny;
        V[6] = nx;                 V[7] = ny;                 V[8] = nz;
    }
    for (int k = 0; k < 9; ++k) st->V[k] = V[k];
    st->omega = fabs(V[0] * V[4] - V[3] * V[1]);                           // Eq. 8
    if (!(V[8] >= 1e-6)) st->status = TOI_ERR_DEGENERATE_GEOMETRY;
}

__global__ void k_cell_indices(Geometry g, const double *__restrict__ uvw, const SnapState *__restrict__ st,
                               int32_t *__restrict__ iu_out, int32_t *__restrict__ iv_out)
{
    const long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= (long long)g.n_b * g.n_c) return;
    const int j = (int)(q / g.n_c), c = (int)(q % g.n_c);
    double rho1, rho2;
    int iu, iv;
    float xu, xv;
    rotate_baseline(st->V, uvw + 3 * j, rho1, rho2);
    sample_cell(rho1, rho2, g.s[c], g.kappa, iu, iv, xu, xv);
    iu_out[q] = iu;
    iv_out[q] = iv;
}

}  // namespace

void launch_planefit(const Geometry &g, const double *d_uvw, double S1, double S2, const double *d_V_inject,
                     SnapState *st, cudaStream_t stream)
{
    launch_pdl(k_planefit, dim3(1), dim3(kFitThreads), 0, stream, g.n_b, g.n_c, d_uvw, S1, S2, d_V_inject, st);
}

void launch_cell_indices(const Geometry &g, const double *d_uvw, const SnapState *st, int32_t *d_iu,
                         int32_t *d_iv, cudaStream_t stream)
{
    const long long S = (long long)g.n_b * g.n_c;
    const int threads = 256;
    k_cell_indices<<<(unsigned)((S + threads - 1) / threads), threads, 0, stream>>>(g, d_uvw, st, d_iu, d_iv);
}

}  // namespace toi
