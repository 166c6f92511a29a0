/*
 * toi_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * A plain, slow, fp64 CPU statement of what the TOI (2-D mode) snapshot imager of
 * arxiv 2512.06254 computes, written from /root/reference/PAPER.md (cited as PAPER.md:LINE)
 * and the readings G1..G19 recorded in DESIGN.md section 3 (the paper is silent on the
 * gridding kernel, padding, grid correction, uniform weighting; those readings are listed
 * there).  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference legs may call this file.  It shares no code, header, table or constant
 * generator with paper_2512_06254_b200/csrc (the CUDA path) and includes nothing of it.
 *
 * Two tiers:
 *   Tier D  toi_oracle_image_dft*      the definition, PAPER.md:142-150 (Eq. 7, Eq. 8): a
 *                                      weighted direct Fourier sum on the transformed plane.
 *   Tier G  toi_oracle_image_gridded   the same image reached by convolutional gridding,
 *                                      inverse FFT, grid correction and crop, every step in
 *                                      fp64, in the order DESIGN.md section 3 fixes.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): Tier G against Tier D; Tier D against a
 * numpy restatement of Eq. 7 on tiny inputs; unit point source = 1 Jy peak; Hermitian input
 * => real image; V orthogonal, |rho| = |uvw|, omega = |V33|; plane fit against numpy SVD and
 * against exactly planar inputs with a known normal; FFT against numpy.fft.ifft2; psi
 * quadrature convergence; shift theorem; linearity; Parseval; thread-count independence.
 * Uniform weighting (G14) is NOT defined by the paper: "parity unpinned" beyond the
 * self-consistency invariants P10.
 *
 * Build: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC (oracle/__init__.py does it).
 * -ffp-contract=off matters: the cell-index expressions below are normative to the last bit.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#include <time.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_OK 0
#define ORC_ERR_ARG (-1)
#define ORC_ERR_NOMEM (-4)
#define ORC_ERR_DEGENERATE (-5)

#define ORC_C0 299792458.0 /* speed of light, m/s: metres -> wavelengths */
#define ORC_PI 3.14159265358979323846

typedef struct { double re, im; } orc_c128;
typedef struct { float re, im; } orc_c64;

/* ------------------------------------------------------------------------------------------
 * Step 1. s_c = nu_c / c0: the factor that turns a UVW row in metres into wavelengths for
 * channel c ("converted from metres to wavelengths for each frequency channel",
 * PAPER.md:275).
 * ---------------------------------------------------------------------------------------- */
void toi_oracle_chan_scale(int32_t n_c, const double *chan_freq_hz, double *s)
{
    for (int32_t c = 0; c < n_c; ++c) s[c] = chan_freq_hz[c] / ORC_C0;
}

/* ------------------------------------------------------------------------------------------
 * Cyclic Jacobi eigen-decomposition of a symmetric 3x3 matrix (textbook; Golub & Van Loan
 * 8.5).  A is overwritten by its diagonal form, E's COLUMNS are the eigenvectors.
 * ---------------------------------------------------------------------------------------- */
static void orc_jacobi3(double A[3][3], double E[3][3])
{
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) E[i][j] = (i == j) ? 1.0 : 0.0;
    for (int sweep = 0; sweep < 64; ++sweep) {
        double off = fabs(A[0][1]) + fabs(A[0][2]) + fabs(A[1][2]);
        double dia = fabs(A[0][0]) + fabs(A[1][1]) + fabs(A[2][2]);
        if (off <= 1e-300 || off <= 1e-22 * dia) break;
        for (int p = 0; p < 2; ++p)
            for (int q = p + 1; q < 3; ++q) {
                if (A[p][q] == 0.0) continue;
                double theta = (A[q][q] - A[p][p]) / (2.0 * A[p][q]);
                double t = (theta >= 0.0 ? 1.0 : -1.0) / (fabs(theta) + sqrt(theta * theta + 1.0));
                double c = 1.0 / sqrt(t * t + 1.0), s = t * c;
                /* A <- J^T A J with J the rotation in the (p,q) plane */
                for (int k = 0; k < 3; ++k) {
                    double akp = A[k][p], akq = A[k][q];
                    A[k][p] = c * akp - s * akq;
                    A[k][q] = s * akp + c * akq;
                }
                for (int k = 0; k < 3; ++k) {
                    double apk = A[p][k], aqk = A[q][k];
                    A[p][k] = c * apk - s * aqk;
                    A[q][k] = s * apk + c * aqk;
                }
                for (int k = 0; k < 3; ++k) {
                    double ekp = E[k][p], ekq = E[k][q];
                    E[k][p] = c * ekp - s * ekq;
                    E[k][q] = s * ekp + c * ekq;
                }
            }
    }
}

/* ------------------------------------------------------------------------------------------
 * Steps 2-3. Basis estimate (section 3.1).
 *   B  [S][3], rows b_q = s_c * uvw_j for every (baseline j, channel c) pair (G1: all rows x
 *      all channels, unweighted, flags ignored), never stored: it is re-formed on the fly.
 *   Bbar = column means of B; Btilde = B - Bbar; C = Btilde^T Btilde (plain triple loop).
 *   Eigen-decomposition of C (= squared singular values / right singular vectors of Btilde),
 *   lambda1 >= lambda2 >= lambda3; e1, e2 span the visibility plane.
 *   basis == 0 (default, reading G3): only the plane normal n = e1 x e2 (flipped so n_w >= 0,
 *      G4) is taken from the SVD; the in-plane axes are the minimal rotation of (u,v,w) that
 *      takes w onto n, so V -> I as the tilt -> 0:
 *        v1 = (1 - a^2/(1+c), -ab/(1+c), -a), v2 = (-ab/(1+c), 1 - b^2/(1+c), -b), v3 = (a,b,c).
 *   basis == 1 (literal reading of PAPER.md:117): rows of V are e1, e2 (sign rule: the
 *      largest-magnitude component of each is positive) and v3 = v1 x v2; if V33 < 0 then
 *      v2 and v3 are negated (G4 canonicalisation V33 > 0 takes precedence).
 *   omega = |V11 V22 - V21 V12| (Eq. 8).  sing[k] = sqrt(lambda_k).
 * Returns ORC_ERR_DEGENERATE if lambda2 <= 1e-10 lambda1 (collinear: no plane) or V33 < 1e-6.
 * Accumulators are long double so that the oracle is the closest thing to the exact sums.
 * ---------------------------------------------------------------------------------------- */
int toi_oracle_plane_fit(int32_t n_b, int32_t n_c, const double *uvw_m, const double *s,
                         int32_t basis, double *V /*[9] row-major*/, double *omega,
                         double *sing /*[3]*/)
{
    if (n_b < 1 || n_c < 1 || !uvw_m || !s || !V) return ORC_ERR_ARG;
    const double S = (double)n_b * (double)n_c;
    long double m0 = 0, m1 = 0, m2 = 0;
    for (int32_t j = 0; j < n_b; ++j)
        for (int32_t c = 0; c < n_c; ++c) {
            m0 += (long double)(s[c] * uvw_m[3 * j + 0]);
            m1 += (long double)(s[c] * uvw_m[3 * j + 1]);
            m2 += (long double)(s[c] * uvw_m[3 * j + 2]);
        }
    const double mean[3] = {(double)(m0 / S), (double)(m1 / S), (double)(m2 / S)};
    long double acc[3][3] = {{0}};
    for (int32_t j = 0; j < n_b; ++j)
        for (int32_t c = 0; c < n_c; ++c) {
            double bt[3];
            for (int k = 0; k < 3; ++k) bt[k] = s[c] * uvw_m[3 * j + k] - mean[k];
            for (int a = 0; a < 3; ++a)
                for (int b = 0; b < 3; ++b) acc[a][b] += (long double)(bt[a] * bt[b]);
        }
    double C[3][3], E[3][3];
    for (int a = 0; a < 3; ++a)
        for (int b = 0; b < 3; ++b) C[a][b] = (double)acc[a][b];
    orc_jacobi3(C, E);
    int idx[3] = {0, 1, 2};
    for (int a = 0; a < 2; ++a)
        for (int b = a + 1; b < 3; ++b)
            if (C[idx[b]][idx[b]] > C[idx[a]][idx[a]]) { int t = idx[a]; idx[a] = idx[b]; idx[b] = t; }
    double lam[3], e[3][3]; /* e[k] = k-th eigenvector as a row */
    for (int k = 0; k < 3; ++k) {
        lam[k] = C[idx[k]][idx[k]];
        for (int a = 0; a < 3; ++a) e[k][a] = E[a][idx[k]];
    }
    if (sing) for (int k = 0; k < 3; ++k) sing[k] = sqrt(lam[k] > 0.0 ? lam[k] : 0.0);
    if (!(lam[0] > 0.0) || lam[1] <= 1e-10 * lam[0]) return ORC_ERR_DEGENERATE;

    if (basis == 0) {
        double n[3] = {e[0][1] * e[1][2] - e[0][2] * e[1][1], e[0][2] * e[1][0] - e[0][0] * e[1][2],
                       e[0][0] * e[1][1] - e[0][1] * e[1][0]};
        double nn = sqrt(n[0] * n[0] + n[1] * n[1] + n[2] * n[2]);
        for (int k = 0; k < 3; ++k) n[k] /= nn;
        if (n[2] < 0.0) for (int k = 0; k < 3; ++k) n[k] = -n[k];
        const double a = n[0], b = n[1], c = n[2];
        V[0] = 1.0 - a * a / (1.0 + c); V[1] = -a * b / (1.0 + c);      V[2] = -a;
        V[3] = -a * b / (1.0 + c);      V[4] = 1.0 - b * b / (1.0 + c); V[5] = -b;
        V[6] = a;                       V[7] = b;                       V[8] = c;
    } else {
        for (int r = 0; r < 2; ++r) {
            int big = 0;
            for (int a = 1; a < 3; ++a) if (fabs(e[r][a]) > fabs(e[r][big])) big = a;
            double sg = e[r][big] < 0.0 ? -1.0 : 1.0;
            for (int a = 0; a < 3; ++a) V[3 * r + a] = sg * e[r][a];
        }
        V[6] = V[1] * V[5] - V[2] * V[4];
        V[7] = V[2] * V[3] - V[0] * V[5];
        V[8] = V[0] * V[4] - V[1] * V[3];
        if (V[8] < 0.0) for (int a = 3; a < 9; ++a) V[a] = -V[a];
    }
    if (omega) *omega = fabs(V[0] * V[4] - V[3] * V[1]);
    if (V[8] < 1e-6) return ORC_ERR_DEGENERATE;
    return ORC_OK;
}

/* ------------------------------------------------------------------------------------------
 * Step 4. R = B V^T on the UNCENTRED baselines, done in metres (scaling by s_c
 * commutes with the rotation; reading G2): rho_j = V uvw_j, evaluated left to right with
 * every operation individually rounded (normative for bit-exact cell indices, G5).
 * ---------------------------------------------------------------------------------------- */
void toi_oracle_rotate(int32_t n_b, const double *uvw_m, const double *V, double *rho /*[n_b][3]*/)
{
    for (int32_t j = 0; j < n_b; ++j) {
        const double u = uvw_m[3 * j + 0], v = uvw_m[3 * j + 1], w = uvw_m[3 * j + 2];
        for (int k = 0; k < 3; ++k)
            rho[3 * j + k] = ((V[3 * k + 0] * u) + (V[3 * k + 1] * v)) + (V[3 * k + 2] * w);
    }
}

/* kappa = G * beta_rad: grid cells per unit of r (wavelengths). beta is given in degrees
 * (Eq. 9).  Normative expression (G5). */
double toi_oracle_kappa(int32_t G, double cell_size_deg)
{
    return (double)G * (cell_size_deg * (ORC_PI / 180.0));
}

/* ------------------------------------------------------------------------------------------
 * Step 5. Per sample (j,c): continuous grid coordinates and centre cell (readings G6, G10).
 *   r1 = rho_j1 * s_c ; gu = -(r1 * kappa)   (the minus is Eq. 9's x = -beta(...))
 *   r2 = rho_j2 * s_c ; gv = +(r2 * kappa)
 *   iu = floor(gu + 1/2), iv = floor(gv + 1/2)  (tie -> up)
 *   on grid iff -G/2 + h <= iu, iv <= G/2 - 1 - h with h = (W-1)/2: the whole W x W footprint
 *   fits; otherwise the sample is dropped everywhere (no wrap-around).
 * ---------------------------------------------------------------------------------------- */
static inline void orc_sample_coord(const double *rho_j, double s_c, double kappa, double *gu,
                                    double *gv, int32_t *iu, int32_t *iv)
{
    double t1 = rho_j[0] * s_c;
    double t2 = rho_j[1] * s_c;
    *gu = -(t1 * kappa);
    *gv = +(t2 * kappa);
    *iu = (int32_t)floor(*gu + 0.5);
    *iv = (int32_t)floor(*gv + 0.5);
}

static inline int orc_on_grid(int32_t iu, int32_t iv, int32_t G, int32_t W)
{
    const int32_t h = (W - 1) / 2;
    return iu >= -G / 2 + h && iu <= G / 2 - 1 - h && iv >= -G / 2 + h && iv <= G / 2 - 1 - h;
}

void toi_oracle_cell_indices(int32_t n_b, int32_t n_c, const double *rho, const double *s,
                             int32_t G, double cell_size_deg, int32_t W, int32_t *iu_out,
                             int32_t *iv_out, uint8_t *on_grid_out)
{
    const double kappa = toi_oracle_kappa(G, cell_size_deg);
#pragma omp parallel for schedule(static)
    for (int32_t j = 0; j < n_b; ++j)
        for (int32_t c = 0; c < n_c; ++c) {
            double gu, gv;
            int32_t iu, iv;
            orc_sample_coord(rho + 3 * j, s[c], kappa, &gu, &gv, &iu, &iv);
            const int64_t q = (int64_t)j * n_c + c;
            iu_out[q] = iu;
            iv_out[q] = iv;
            if (on_grid_out) on_grid_out[q] = (uint8_t)orc_on_grid(iu, iv, G, W);
        }
}

/* ------------------------------------------------------------------------------------------
 * Step 6a. Data handling (readings G12, G13).  For the two parallel hands a, b:
 *   w_p = 0 if flagged, or if the weight is <= 0 or not finite; else weight_p (1 if no weights)
 *   w_I = w_a + w_b ;  z = w_a Vis_a + w_b Vis_b, where a pol with w_p = 0 is SKIPPED (never
 *   multiplied: data under a flag may be NaN).  pol_a == pol_b means a single hand.
 * ---------------------------------------------------------------------------------------- */
static inline void orc_sample_data(const orc_c64 *vis_q, const float *wgt_q, const uint8_t *flg_q,
                                   int32_t pol_a, int32_t pol_b, double *wI, double *zre, double *zim)
{
    double w_sum = 0.0, re = 0.0, im = 0.0;
    const int npol = (pol_a == pol_b) ? 1 : 2;
    for (int k = 0; k < npol; ++k) {
        const int p = k == 0 ? pol_a : pol_b;
        double w = wgt_q ? (double)wgt_q[p] : 1.0;
        if ((flg_q && flg_q[p]) || !(w > 0.0) || !isfinite(w)) continue;
        w_sum += w;
        re += w * (double)vis_q[p].re;
        im += w * (double)vis_q[p].im;
    }
    *wI = w_sum; *zre = re; *zim = im;
}

/* Gridding kernel (reading G9; the paper is silent): exponential of semicircle
 * phi(x) = exp(beta_k (sqrt(1 - (2x/W)^2) - 1)) for |x| <= W/2, else 0; beta_k = 2.30 W. */
static inline double orc_phi(double x, int32_t W)
{
    const double t = 2.0 * x / (double)W;
    const double a = 1.0 - t * t;
    if (a < 0.0) return 0.0;
    return exp(2.30 * (double)W * (sqrt(a) - 1.0));
}
double toi_oracle_phi(double x, int32_t W) { return orc_phi(x, W); }

/* Gauss-Legendre nodes/weights on [-1,1] by Newton iteration on P_n (textbook). */
static void orc_gauss_legendre(int n, double *x, double *w)
{
    for (int i = 0; i < (n + 1) / 2; ++i) {
        double z = cos(ORC_PI * (i + 0.75) / (n + 0.5)), pp = 1.0;
        for (int it = 0; it < 100; ++it) {
            double p1 = 1.0, p2 = 0.0;
            for (int k = 1; k <= n; ++k) {
                double p3 = p2; p2 = p1;
                p1 = ((2.0 * k - 1.0) * z * p2 - (k - 1.0) * p3) / k;
            }
            pp = n * (z * p1 - p2) / (z * z - 1.0);
            double dz = p1 / pp;
            z -= dz;
            if (fabs(dz) < 1e-16) break;
        }
        x[i] = -z; x[n - 1 - i] = z;
        w[i] = w[n - 1 - i] = 2.0 / ((1.0 - z * z) * pp * pp);
    }
}

/* Grid correction (reading G11): psi(n) = int_{-W/2}^{W/2} phi(x) cos(2 pi x n / G) dx, the
 * continuous Fourier transform of the gridding kernel at image pixel offset n, by Gauss-
 * Legendre with n_nodes points on each of 16 equal panels of [-W/2, W/2] (panels, because
 * phi has a square-root end-point behaviour that a single high-order rule resolves slowly). */
double toi_oracle_psi(int32_t n, int32_t G, int32_t W, int32_t n_nodes)
{
    if (n_nodes < 2) n_nodes = 64;
    if (n_nodes > 512) n_nodes = 512;
    double x[512], w[512];
    orc_gauss_legendre(n_nodes, x, w);
    const int panels = 16;
    const double half = 0.5 * (double)W, pw = (double)W / panels;
    long double sum = 0;
    for (int p = 0; p < panels; ++p) {
        const double a = -half + p * pw, mid = a + 0.5 * pw;
        for (int k = 0; k < n_nodes; ++k) {
            double xx = mid + 0.5 * pw * x[k];
            sum += (long double)(0.5 * pw * w[k] * orc_phi(xx, W) *
                                 cos(2.0 * ORC_PI * xx * (double)n / (double)G));
        }
    }
    return (double)sum;
}

/* ------------------------------------------------------------------------------------------
 * Own FFT (step 8).  Unnormalised transform with kernel exp(sign * 2 pi i k n / len) over one
 * line of stride `stride`.  Power-of-two lengths: iterative radix-2 Cooley-Tukey; any other
 * length: the O(len^2) definition.  Pinned against numpy.fft (test P12).
 * ---------------------------------------------------------------------------------------- */
static void orc_fft_line(orc_c128 *a, int64_t len, int sign, const orc_c128 *tw /*len entries: exp(sign 2 pi i k/len)*/,
                         orc_c128 *scratch)
{
    if ((len & (len - 1)) == 0) {
        for (int64_t i = 1, j = 0; i < len; ++i) { /* bit reversal */
            int64_t bit = len >> 1;
            for (; j & bit; bit >>= 1) j ^= bit;
            j ^= bit;
            if (i < j) { orc_c128 t = a[i]; a[i] = a[j]; a[j] = t; }
        }
        for (int64_t half = 1; half < len; half <<= 1) {
            const int64_t step = len / (2 * half);
            for (int64_t base = 0; base < len; base += 2 * half)
                for (int64_t k = 0; k < half; ++k) {
                    const orc_c128 w = tw[k * step];
                    orc_c128 *p = &a[base + k], *q = &a[base + k + half];
                    const double tr = q->re * w.re - q->im * w.im, ti = q->re * w.im + q->im * w.re;
                    q->re = p->re - tr; q->im = p->im - ti;
                    p->re += tr; p->im += ti;
                }
        }
    } else {
        for (int64_t n = 0; n < len; ++n) {
            long double sr = 0, si = 0;
            for (int64_t k = 0; k < len; ++k) {
                const orc_c128 w = tw[(k * n) % len];
                sr += (long double)(a[k].re * w.re - a[k].im * w.im);
                si += (long double)(a[k].re * w.im + a[k].im * w.re);
            }
            scratch[n].re = (double)sr; scratch[n].im = (double)si;
        }
        memcpy(a, scratch, (size_t)len * sizeof(orc_c128));
    }
    (void)sign;
}

/* In-place unnormalised 2-D transform of a row-major [n][n] array:
 * out[m][l] = sum_{r,k} in[r][k] exp(sign 2 pi i (k l + r m)/n).  sign = +1 is the inverse
 * transform the imager uses (Eq. 7 has exp(+i 2 pi ...)). */
int toi_oracle_fft2(orc_c128 *a, int32_t n, int32_t sign)
{
    if (!a || n < 1 || (sign != 1 && sign != -1)) return ORC_ERR_ARG;
    orc_c128 *tw = (orc_c128 *)malloc((size_t)n * sizeof(orc_c128));
    if (!tw) return ORC_ERR_NOMEM;
    for (int32_t k = 0; k < n; ++k) {
        const double ang = (double)sign * 2.0 * ORC_PI * (double)k / (double)n;
        tw[k].re = cos(ang); tw[k].im = sin(ang);
    }
    int fail = 0;
#pragma omp parallel
    {
        orc_c128 *col = (orc_c128 *)malloc((size_t)n * sizeof(orc_c128));
        orc_c128 *scr = (orc_c128 *)malloc((size_t)n * sizeof(orc_c128));
        if (!col || !scr) {
#pragma omp atomic write
            fail = 1;
        }
#pragma omp barrier
        if (!fail) {
#pragma omp for schedule(static)
            for (int32_t r = 0; r < n; ++r) orc_fft_line(a + (int64_t)r * n, n, sign, tw, scr);
#pragma omp for schedule(static)
            for (int32_t k = 0; k < n; ++k) {
                for (int32_t r = 0; r < n; ++r) col[r] = a[(int64_t)r * n + k];
                orc_fft_line(col, n, sign, tw, scr);
                for (int32_t r = 0; r < n; ++r) a[(int64_t)r * n + k] = col[r];
            }
        }
        free(col); free(scr);
    }
    free(tw);
    return fail ? ORC_ERR_NOMEM : ORC_OK;
}

/* ------------------------------------------------------------------------------------------
 * Configuration of one imaging call (mirrors the paper's inputs).
 * ---------------------------------------------------------------------------------------- */
typedef struct {
    int32_t n_b, n_c, n_p;   /* rows (baselines) of one time sample, channels, polarisations */
    int32_t pol_a, pol_b;    /* the two parallel hands (equal => single hand) */
    int32_t N;               /* image side (even) */
    double  cell_size_deg;   /* beta, degrees (Eq. 9) */
    int32_t weighting;       /* 0 natural, 1 uniform (G14) */
    int32_t G;               /* padded grid side, 0 -> 2N (G9) */
    int32_t W;               /* kernel support, 0 -> 7 (odd) */
    int32_t apply_jacobian;  /* 1: divide by omega (Eq. 7) */
    int32_t basis;           /* 0 minimal rotation (G3), 1 principal axes (literal) */
} orc_config;

typedef struct {
    double V[9], omega, sing[3], wsum;
    int64_t n_gridded, n_off_grid, n_flagged;
} orc_info;

static int orc_resolve(const orc_config *cfg, int32_t *G, int32_t *W)
{
    *G = cfg->G > 0 ? cfg->G : 2 * cfg->N;
    *W = cfg->W > 0 ? cfg->W : 7;
    if (cfg->n_b < 1 || cfg->n_c < 1 || cfg->n_p < 1 || cfg->N < 2 || (cfg->N & 1) || (*G & 1) ||
        *G < cfg->N || !(*W & 1) || *W < 1 || *W > 15 || *G < 2 * *W || !(cfg->cell_size_deg > 0.0) ||
        cfg->pol_a < 0 || cfg->pol_a >= cfg->n_p || cfg->pol_b < 0 || cfg->pol_b >= cfg->n_p)
        return ORC_ERR_ARG;
    return ORC_OK;
}

/* Common front end: s_c, V (fitted, or injected when V_in != NULL), rho. */
static int orc_front(const orc_config *cfg, const double *chan_freq_hz, const double *uvw_m,
                     const double *V_in, double **s_out, double **rho_out, orc_info *info)
{
    double *s = (double *)malloc((size_t)cfg->n_c * sizeof(double));
    double *rho = (double *)malloc((size_t)cfg->n_b * 3 * sizeof(double));
    if (!s || !rho) { free(s); free(rho); return ORC_ERR_NOMEM; }
    toi_oracle_chan_scale(cfg->n_c, chan_freq_hz, s);
    int rc = ORC_OK;
    if (V_in) {
        memcpy(info->V, V_in, 9 * sizeof(double));
        info->omega = fabs(V_in[0] * V_in[4] - V_in[3] * V_in[1]);
        info->sing[0] = info->sing[1] = info->sing[2] = 0.0;
    } else {
        rc = toi_oracle_plane_fit(cfg->n_b, cfg->n_c, uvw_m, s, cfg->basis, info->V, &info->omega, info->sing);
    }
    if (rc != ORC_OK) { free(s); free(rho); return rc; }
    toi_oracle_rotate(cfg->n_b, uvw_m, info->V, rho);
    *s_out = s; *rho_out = rho;
    return ORC_OK;
}

/* Step 6b. Uniform weighting (reading G14; NOT in the paper, which images with natural
 * weights): density D on the G x G gridding cells at the centre cell,
 * Hermitian-symmetrised: D[iv][iu] += w_I and D[-iv][-iu] += w_I; then f_q = 1 / D[cell_q].
 * D is stored centred: D[(iv + G/2) * G + (iu + G/2)].  Sequential in q (deterministic). */
static void orc_density(const orc_config *cfg, int32_t G, int32_t W, const double *rho, const double *s,
                        const orc_c64 *vis, const float *weights, const uint8_t *flags, double *D)
{
    const double kappa = toi_oracle_kappa(G, cfg->cell_size_deg);
    memset(D, 0, (size_t)G * G * sizeof(double));
    for (int32_t j = 0; j < cfg->n_b; ++j)
        for (int32_t c = 0; c < cfg->n_c; ++c) {
            double gu, gv, wI, zr, zi; int32_t iu, iv;
            orc_sample_coord(rho + 3 * j, s[c], kappa, &gu, &gv, &iu, &iv);
            if (!orc_on_grid(iu, iv, G, W)) continue;
            const int64_t q = ((int64_t)j * cfg->n_c + c) * cfg->n_p;
            orc_sample_data(vis + q, weights ? weights + q : NULL, flags ? flags + q : NULL,
                            cfg->pol_a, cfg->pol_b, &wI, &zr, &zi);
            if (!(wI > 0.0)) continue;
            D[(int64_t)(iv + G / 2) * G + (iu + G / 2)] += wI;
            D[(int64_t)(-iv + G / 2) * G + (-iu + G / 2)] += wI;
        }
}

/* ------------------------------------------------------------------------------------------
 * Tier G.  image[j][i] (row-major, N x N, fp64), i = column (t1 axis), j = row (t2 axis):
 *   t1(i) = -beta_rad (i - N/2), t2(j) = +beta_rad (j - N/2)   (Eq. 9, 0-based; G6)
 * Steps 1-9 of DESIGN.md section 3.  Optional outputs (may be NULL):
 *   grid_out   [G][G] complex128, CENTRED (cell (iv,iu) at [iv+G/2][iu+G/2]), before the FFT
 *   dens_out   [G][G] fp64, centred, uniform-weighting density (zeros for natural)
 *   iu_out, iv_out [n_b][n_c] int32 centre cells
 *   V_in       inject the transform instead of fitting it (index-parity protocol G5)
 * ---------------------------------------------------------------------------------------- */
/* Wall-clock seconds the last toi_oracle_image_gridded call spent in each stage: plane fit + rotation,
 * cell indices + weighting (density, counts, Wsum), gridding, FFT, correction + crop.  Read by
 * bench.py's cpu_baseline; instrumentation only -- no arithmetic depends on it. */
static double orc_stage_s[5];
static double orc_now(void)
{
#ifdef _OPENMP
    return omp_get_wtime();
#else
    return (double)clock() / CLOCKS_PER_SEC;
#endif
}
void toi_oracle_last_stage_seconds(double out[5]) { memcpy(out, orc_stage_s, sizeof orc_stage_s); }

int toi_oracle_image_gridded(const orc_config *cfg, const double *chan_freq_hz, const double *uvw_m,
                             const orc_c64 *vis, const float *weights, const uint8_t *flags,
                             const double *V_in, double *image, orc_info *info_out,
                             orc_c128 *grid_out, double *dens_out, int32_t *iu_out, int32_t *iv_out)
{
    int32_t G, W;
    double t_mark = orc_now(), t_now;
    memset(orc_stage_s, 0, sizeof orc_stage_s);
#define ORC_STAGE(k) (t_now = orc_now(), orc_stage_s[k] += t_now - t_mark, t_mark = t_now)
    if (!cfg || !chan_freq_hz || !uvw_m || !vis || !image) return ORC_ERR_ARG;
    int rc = orc_resolve(cfg, &G, &W);
    if (rc) return rc;
    const int32_t N = cfg->N, h = (W - 1) / 2;
    orc_info info; memset(&info, 0, sizeof info);
    double *s = NULL, *rho = NULL;
    rc = orc_front(cfg, chan_freq_hz, uvw_m, V_in, &s, &rho, &info);
    if (rc) { if (info_out) *info_out = info; return rc; }
    ORC_STAGE(0);
    const double kappa = toi_oracle_kappa(G, cfg->cell_size_deg);
    const int64_t S = (int64_t)cfg->n_b * cfg->n_c;

    int32_t *iu = (int32_t *)malloc((size_t)S * sizeof(int32_t));
    int32_t *iv = (int32_t *)malloc((size_t)S * sizeof(int32_t));
    uint8_t *on = (uint8_t *)malloc((size_t)S);
    orc_c128 *grid = (orc_c128 *)calloc((size_t)G * G, sizeof(orc_c128)); /* centred layout */
    double *D = cfg->weighting == 1 ? (double *)malloc((size_t)G * G * sizeof(double)) : NULL;
    if (!iu || !iv || !on || !grid || (cfg->weighting == 1 && !D)) {
        free(iu); free(iv); free(on); free(grid); free(D); free(s); free(rho); return ORC_ERR_NOMEM;
    }
    toi_oracle_cell_indices(cfg->n_b, cfg->n_c, rho, s, G, cfg->cell_size_deg, W, iu, iv, on);
    if (D) orc_density(cfg, G, W, rho, s, vis, weights, flags, D);

    /* counts and Wsum = sum_q f_q w_I,q over on-grid samples (G7), sequential in q */
    {
        long double wsum = 0;
        for (int64_t q = 0; q < S; ++q) {
            if (!on[q]) { info.n_off_grid++; continue; }
            double wI, zr, zi;
            const int64_t o = q * cfg->n_p;
            orc_sample_data(vis + o, weights ? weights + o : NULL, flags ? flags + o : NULL,
                            cfg->pol_a, cfg->pol_b, &wI, &zr, &zi);
            if (!(wI > 0.0)) { info.n_flagged++; continue; }
            info.n_gridded++;
            double f = 1.0;
            if (D) f = 1.0 / D[(int64_t)(iv[q] + G / 2) * G + (iu[q] + G / 2)];
            wsum += (long double)(f * wI);
        }
        info.wsum = (double)wsum;
    }
    ORC_STAGE(1);

    /* Step 7. scatter: grid[iv+dv][iu+du] += f z phi(iu+du-gu) phi(iv+dv-gv), |du|,|dv| <= h.
     * Threads own bands of grid rows; every thread walks the samples in q order, so each
     * cell's sum is in q order whatever the thread count (pin P14). */
    {
        int nthreads = 1;
#ifdef _OPENMP
        nthreads = omp_get_max_threads();
#endif
        /* band edges: equal share of footprint rows */
        int64_t *rowcount = (int64_t *)calloc((size_t)G + 1, sizeof(int64_t));
        int32_t *edge = (int32_t *)malloc((size_t)(nthreads + 1) * sizeof(int32_t));
        if (!rowcount || !edge) { free(rowcount); free(edge); rc = ORC_ERR_NOMEM; goto done; }
        int64_t total = 0;
        for (int64_t q = 0; q < S; ++q)
            if (on[q]) for (int dv = -h; dv <= h; ++dv) { rowcount[iv[q] + dv + G / 2]++; total++; }
        edge[0] = 0;
        { int64_t run = 0; int t = 1;
          for (int32_t r = 0; r < G && t < nthreads; ++r) {
              run += rowcount[r];
              while (t < nthreads && run * nthreads >= total * t) edge[t++] = r + 1;
          }
          for (; t <= nthreads; ++t) edge[t] = G;
          edge[nthreads] = G; }
#pragma omp parallel num_threads(nthreads)
        {
            int tid = 0;
#ifdef _OPENMP
            tid = omp_get_thread_num();
#endif
            const int32_t r0 = edge[tid], r1 = edge[tid + 1];
            for (int64_t q = 0; q < S && r0 < r1; ++q) {
                if (!on[q]) continue;
                const int32_t rc0 = iv[q] + G / 2;
                if (rc0 + h < r0 || rc0 - h >= r1) continue;
                const int32_t j = (int32_t)(q / cfg->n_c), c = (int32_t)(q % cfg->n_c);
                double gu, gv, wI, zr, zi; int32_t iuq, ivq;
                orc_sample_coord(rho + 3 * j, s[c], kappa, &gu, &gv, &iuq, &ivq);
                const int64_t o = q * cfg->n_p;
                orc_sample_data(vis + o, weights ? weights + o : NULL, flags ? flags + o : NULL,
                                cfg->pol_a, cfg->pol_b, &wI, &zr, &zi);
                if (!(wI > 0.0)) continue;
                double f = 1.0;
                if (D) f = 1.0 / D[(int64_t)(ivq + G / 2) * G + (iuq + G / 2)];
                double pu[16], pv[16];
                for (int d = -h; d <= h; ++d) {
                    pu[d + h] = orc_phi((double)(iuq + d) - gu, W);
                    pv[d + h] = orc_phi((double)(ivq + d) - gv, W);
                }
                for (int dv = -h; dv <= h; ++dv) {
                    const int32_t row = ivq + dv + G / 2;
                    if (row < r0 || row >= r1) continue;
                    orc_c128 *g = grid + (int64_t)row * G + (iuq - h + G / 2);
                    for (int du = 0; du < W; ++du) {
                        const double wt = pu[du] * pv[dv + h];
                        g[du].re += (f * zr) * wt;
                        g[du].im += (f * zi) * wt;
                    }
                }
            }
        }
        free(rowcount); free(edge);
    }
    ORC_STAGE(2);
    if (grid_out) memcpy(grid_out, grid, (size_t)G * G * sizeof(orc_c128));
    if (dens_out) { if (D) memcpy(dens_out, D, (size_t)G * G * sizeof(double)); else memset(dens_out, 0, (size_t)G * G * sizeof(double)); }
    if (iu_out) memcpy(iu_out, iu, (size_t)S * sizeof(int32_t));
    if (iv_out) memcpy(iv_out, iv, (size_t)S * sizeof(int32_t));

    /* Step 8. F[m][n] = sum_{kv,ku} grid(kv,ku) exp(+2 pi i (ku n + kv m)/G), signed indices.
     * Signed cell k lives at array index (k + G) mod G for the FFT; pixel offset n is read
     * back from index (n + G) mod G. */
    {
        orc_c128 *a = (orc_c128 *)malloc((size_t)G * G * sizeof(orc_c128));
        if (!a) { rc = ORC_ERR_NOMEM; goto done; }
        for (int32_t kv = -G / 2; kv < G / 2; ++kv)
            for (int32_t ku = -G / 2; ku < G / 2; ++ku)
                a[(int64_t)((kv + G) % G) * G + ((ku + G) % G)] = grid[(int64_t)(kv + G / 2) * G + (ku + G / 2)];
        rc = toi_oracle_fft2(a, G, +1);
        if (rc) { free(a); goto done; }
        ORC_STAGE(3);
        /* Step 9. image = Re F / (psi(i-N/2) psi(j-N/2) omega Wsum)  (G7, G8, G11) */
        double *ipsi = (double *)malloc((size_t)N * sizeof(double));
        if (!ipsi) { free(a); rc = ORC_ERR_NOMEM; goto done; }
        for (int32_t i = 0; i < N; ++i) ipsi[i] = toi_oracle_psi(i - N / 2, G, W, 64);
        const double norm = (cfg->apply_jacobian ? info.omega : 1.0) * info.wsum;
        for (int32_t jj = 0; jj < N; ++jj)
            for (int32_t ii = 0; ii < N; ++ii) {
                const int32_t m = jj - N / 2, n = ii - N / 2;
                const orc_c128 F = a[(int64_t)((m + G) % G) * G + ((n + G) % G)];
                image[(int64_t)jj * N + ii] = info.wsum > 0.0 ? F.re / (ipsi[ii] * ipsi[jj] * norm) : 0.0;
            }
        free(ipsi); free(a);
        ORC_STAGE(4);
    }
#undef ORC_STAGE
done:
    if (info_out) *info_out = info;
    free(iu); free(iv); free(on); free(grid); free(D); free(s); free(rho);
    return rc;
}

/* ------------------------------------------------------------------------------------------
 * Tier D.  Eq. 7 evaluated as written, for a list of pixels (i = column,
 * j = row):  I = sum_q f_q z_q exp[i 2 pi (r1_q t1(i) + r2_q t2(j))] / (omega Wsum),
 * r = rho s_c in wavelengths (NOT snapped to cells).  Samples the gridder drops (off-grid,
 * G10) are dropped here too so both tiers sum the same set; uniform f_q uses the same
 * density.  out_re/out_im [n_pix]; the image is out_re, out_im exists for pin P3.
 * ---------------------------------------------------------------------------------------- */
int toi_oracle_image_dft_pixels(const orc_config *cfg, const double *chan_freq_hz, const double *uvw_m,
                                const orc_c64 *vis, const float *weights, const uint8_t *flags,
                                const double *V_in, int64_t n_pix, const int32_t *pix_i, const int32_t *pix_j,
                                double *out_re, double *out_im, orc_info *info_out)
{
    int32_t G, W;
    if (!cfg || !chan_freq_hz || !uvw_m || !vis || !out_re || n_pix < 0) return ORC_ERR_ARG;
    int rc = orc_resolve(cfg, &G, &W);
    if (rc) return rc;
    orc_info info; memset(&info, 0, sizeof info);
    double *s = NULL, *rho = NULL;
    rc = orc_front(cfg, chan_freq_hz, uvw_m, V_in, &s, &rho, &info);
    if (rc) { if (info_out) *info_out = info; return rc; }
    const double kappa = toi_oracle_kappa(G, cfg->cell_size_deg);
    const double beta_rad = cfg->cell_size_deg * (ORC_PI / 180.0);
    const int64_t S = (int64_t)cfg->n_b * cfg->n_c;
    double *D = cfg->weighting == 1 ? (double *)malloc((size_t)G * G * sizeof(double)) : NULL;
    double *fz_re = (double *)malloc((size_t)S * sizeof(double));
    double *fz_im = (double *)malloc((size_t)S * sizeof(double));
    double *r1 = (double *)malloc((size_t)S * sizeof(double));
    double *r2 = (double *)malloc((size_t)S * sizeof(double));
    if ((cfg->weighting == 1 && !D) || !fz_re || !fz_im || !r1 || !r2) {
        free(D); free(fz_re); free(fz_im); free(r1); free(r2); free(s); free(rho); return ORC_ERR_NOMEM;
    }
    if (D) orc_density(cfg, G, W, rho, s, vis, weights, flags, D);
    long double wsum = 0;
    int64_t n_used = 0;
    for (int32_t j = 0; j < cfg->n_b; ++j)
        for (int32_t c = 0; c < cfg->n_c; ++c) {
            double gu, gv, wI, zr, zi; int32_t iu, iv;
            orc_sample_coord(rho + 3 * j, s[c], kappa, &gu, &gv, &iu, &iv);
            if (!orc_on_grid(iu, iv, G, W)) { info.n_off_grid++; continue; }
            const int64_t o = ((int64_t)j * cfg->n_c + c) * cfg->n_p;
            orc_sample_data(vis + o, weights ? weights + o : NULL, flags ? flags + o : NULL,
                            cfg->pol_a, cfg->pol_b, &wI, &zr, &zi);
            if (!(wI > 0.0)) { info.n_flagged++; continue; }
            info.n_gridded++;
            double f = 1.0;
            if (D) f = 1.0 / D[(int64_t)(iv + G / 2) * G + (iu + G / 2)];
            wsum += (long double)(f * wI);
            fz_re[n_used] = f * zr; fz_im[n_used] = f * zi;
            r1[n_used] = rho[3 * j + 0] * s[c];
            r2[n_used] = rho[3 * j + 1] * s[c];
            n_used++;
        }
    info.wsum = (double)wsum;
    const double norm = (cfg->apply_jacobian ? info.omega : 1.0) * info.wsum;
#pragma omp parallel for schedule(dynamic, 4)
    for (int64_t p = 0; p < n_pix; ++p) {
        const double t1 = -beta_rad * (double)(pix_i[p] - cfg->N / 2);
        const double t2 = +beta_rad * (double)(pix_j[p] - cfg->N / 2);
        long double sr = 0, si = 0;
        for (int64_t q = 0; q < n_used; ++q) {
            const double ph = 2.0 * ORC_PI * (r1[q] * t1 + r2[q] * t2);
            const double cs = cos(ph), sn = sin(ph);
            sr += (long double)(fz_re[q] * cs - fz_im[q] * sn);
            si += (long double)(fz_re[q] * sn + fz_im[q] * cs);
        }
        out_re[p] = info.wsum > 0.0 ? (double)(sr / norm) : 0.0;
        if (out_im) out_im[p] = info.wsum > 0.0 ? (double)(si / norm) : 0.0;
    }
    if (info_out) *info_out = info;
    free(D); free(fz_re); free(fz_im); free(r1); free(r2); free(s); free(rho);
    return ORC_OK;
}

int toi_oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void toi_oracle_set_num_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}
