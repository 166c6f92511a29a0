// k_fft.cu -- step a6 (+ a7), hand-written: the pruned inverse 2-D transform of the gridding grid
// (PAPER.md:301 names the inverse FFT as the heaviest stage).
//   F[m][n] = sum_{y, x} grid[y][x] exp(+2 pi i (x n + y m) / G)       (array indices; the grid is stored
//   centred, which multiplies F by (-1)^(n + m): undone where the image is written, as in k_correct_crop)
// Only the N columns n and N rows m the crop keeps are ever needed, and most of the grid is
// zero (three quarters of its tiles at config 2, about nine tenths at config 4).  Two kernels, both built on the shared-memory FFT of fft_smem.cuh:
//   k_fft_rows   one CTA per grid row: the row is read THROUGH THE TILE MAP of the sparse clear (tiles
//                the gridder did not mark are known to be zero and are not read: 36 MB instead of
//                134 MB at config 2) straight into the first stage's registers, transformed along x,
//                and only the N needed columns are written to the workspace, in blocks of 4 columns
//                (a row without a marked tile writes zeros and skips the transform);
//   k_fft_cols   one CTA per block of needed columns: read as one contiguous run, transformed
//                along y, and only the N needed rows leave the SM -- either as the finished image
//                pixel Re F (-1)^(n+m) / (psi psi omega Wsum) (correction, crop and normalisation of
//                step a7 fused: the transformed grid is never written back), or, for the Chebyshev
//                moments of the 3-D mode, as the cropped complex moment [N][N].
// cuFFT needs G x G reads and writes in both passes, a separate crop kernel, and cannot skip zeros.
// For G = 2^10 .. 2^14 with G >= 4N/3 and N a multiple of 16; other shapes stay on cuFFT.
#include "fft_smem.cuh"
#include "toi_internal.cuh"

namespace toi {
namespace {

// Workspace layout between the passes: only the N needed columns, in blocks of CB columns,
//   work[(n' / CB) G CB + y CB + n' % CB],  n' = n for n < N/2, n - (G - N) for n >= G - N/2
// so that the column pass reads the CB columns of a block as ONE contiguous run of G CB float2 (a
// strided read of 32-byte row segments opens a DRAM page per segment and ran at a fifth of the
// bandwidth); the scatter is on the write side, where nothing waits for it and L2 merges the
// segments of neighbouring rows.  CB >= 4: the row pass writes whole 32-byte sectors.
__host__ __device__ constexpr int cols_block(int log2g) { return log2g <= 11 ? 8 : 4; }

// where the row pass's last stage puts its results
template <int LOG2G>
struct ToWorkspace {
    float2 *dst;                                 // work + y CB
    int half, N_;
    __device__ __forceinline__ void operator()(int n, float2 *, float2 v) const
    {
        constexpr int G = 1 << LOG2G, CB = cols_block(LOG2G);
        const unsigned np = n < half ? n : n - (G - N_);
        // 32-bit element index: G N < 2^31
        if (n < half || n >= G - half) dst[(np / CB) * (unsigned)(G * CB) + np % CB] = v;
    }
};

// Persistent CTAs (the twiddle tables are filled once per CTA): CTA b takes rows b, b + gridDim.x, ...
// T threads per row, G / T elements each.
template <int LOG2G, int T, int MINB>
__global__ void __launch_bounds__(T, MINB)
k_fft_rows(const float2 *__restrict__ grid, float2 *__restrict__ work, const uint8_t *__restrict__ map, int N,
           const float2 *__restrict__ tw)
{
    using P = fft::Plan<LOG2G>;
    constexpr int G = 1 << LOG2G, kTiles = G / kTileW;
    extern __shared__ float2 s_dyn[];
    float2 *const s_tab = s_dyn, *const s_seq = s_dyn + P::kTabFloat2;
    const int t = threadIdx.x, half = N >> 1;
    fft::fill_tables<LOG2G>(s_tab, tw, t, T);      // plan constants: before the wait, under the previous kernel's tail
    pdl_wait();
    pdl_trigger();
    static_assert(kTiles <= 128, "a row's tile marks are carried as two 64-bit masks");
    for (int y = blockIdx.x; y < G; y += gridDim.x) {
        const uint8_t *mrow = map + (size_t)(y / kTileH) * tiles_per_row(G);
        const float2 *src = grid + (size_t)y * G;
        // the marks of this row's G / 128 tiles as bit masks (lane l looks at tiles l, l + 32, l + 64, l + 96)
        const int lane = t & 31;
        unsigned m[4];
#pragma unroll
        for (int w = 0; w < 4; ++w)
            m[w] = 32 * w < kTiles ? __ballot_sync(0xffffffffu, lane + 32 * w < kTiles && __ldg(mrow + lane + 32 * w) != 0) : 0u;
        const unsigned long long marks_lo = ((unsigned long long)m[1] << 32) | m[0], marks_hi = ((unsigned long long)m[3] << 32) | m[2];
        const ToWorkspace<LOG2G> to_work{work + (size_t)y * cols_block(LOG2G), half, N};
        if ((marks_lo | marks_hi) == 0ull) {     // an all-zero row transforms to zeros
            for (int n = t; n < half; n += T) {
                to_work(n, nullptr, make_float2(0.0f, 0.0f));
                to_work(G - half + n, nullptr, make_float2(0.0f, 0.0f));
            }
            continue;
        }
        __syncthreads();                         // the previous row's last stage has read s_seq; the tables are filled
        // stage A reads the row straight from the grid (consecutive threads, consecutive cells), through the tile marks
        const auto from_grid = [&](int b, int r) {
            const int x = b + r * P::L1, tile = x / kTileW;
            float2 v = make_float2(0.0f, 0.0f);
            if (((tile < 64 ? marks_lo : marks_hi) >> (tile & 63)) & 1ull) v = __ldcs(src + x);      // read once: the clear zeroes it next
            return v;
        };
        // the last stage hands its results straight to the workspace: only the needed columns, 8-byte
        // stores from consecutive threads to consecutive addresses
        fft::transform_from<LOG2G, T>(s_seq, t, s_tab, from_grid, to_work);
    }
}

// C columns (a part of a block of CB) per CTA pass, CT of them in flight at a time (CT groups of T threads);
// persistent CTAs, CTA b takes parts b, b + gridDim.x, ... so that the parts of a block are read at about
// the same time (the block's sectors then come from L2 for all but the first).
// Sequences sit kSkew float2 apart beyond their padded length, so that the C columns of one grid row
// fall on different banks when a row segment is stored.
constexpr int kSkew = 4;
// The sparse clear can ride along (grid != nullptr or dens != nullptr): the row pass has read the grid, so
// every warp of this pass first zeroes its share of the marked tiles (stores nobody waits for) and then
// turns to its columns -- instead of a k_clear_tiles launch of its own between the two passes.
struct ClearArgs {
    float2 *grid;
    float *dens;
    uint8_t *map;
    int G, tpr;
    long long n_tiles;
};
template <int LOG2G, int C, int CT, int T, int UA, bool IMAGE>
__global__ void __launch_bounds__(T * CT)
k_fft_cols(const float2 *__restrict__ work, int N, const float2 *__restrict__ tw, const double *__restrict__ ipsi,
           const SnapState *__restrict__ st, int apply_jacobian, float *__restrict__ image, float2 *__restrict__ moment,
           ClearArgs clr)
{
    using P = fft::Plan<LOG2G>;
    constexpr int CB = cols_block(LOG2G);
    constexpr int G = 1 << LOG2G, NT = T * CT, SEQ = P::kPadded + kSkew;
    static_assert(CB % C == 0 && (C * P::L1) % NT == 0 && C % CT == 0, "a part must divide evenly among the threads");
    extern __shared__ float2 s_dyn[];
    float2 *const s_tab = s_dyn, *const s_seq = s_dyn + P::kTabFloat2;       // [C][SEQ]
    const int tid = threadIdx.x, half = N >> 1;
    fft::fill_tables<LOG2G>(s_tab, tw, tid, NT);   // plan constants: before the wait, under the previous kernel's tail
    pdl_wait();
    pdl_trigger();
    if (clr.map != nullptr) {
        const long long n_warps = (long long)gridDim.x * (NT / 32);
        for (long long w = (long long)blockIdx.x * (NT / 32) + (tid >> 5); w * kClearTilesPerWarp < clr.n_tiles; w += n_warps)
            clear_tiles_warp(clr.grid, clr.dens, clr.G, clr.map, clr.tpr, clr.n_tiles, w * kClearTilesPerWarp, tid & 31);
    }
    const double wsum = st->wsum;
    const bool ok = st->status == TOI_OK && wsum > 0.0;
    const double inv_norm = ok ? 1.0 / ((apply_jacobian ? st->omega : 1.0) * wsum) : 0.0;
    const int grp = tid / T, t = tid % T;
    for (int first = blockIdx.x * C; first < N; first += gridDim.x * C) {
        // my C columns: array indices n0 .. n0 + C - 1, inside [0, N/2) or [G - N/2, G)
        const int n0 = first < half ? first : G - half + (first - half);
        const float2 *src = work + (size_t)(first / CB) * ((size_t)G * CB) + first % CB;
        __syncthreads();                         // the previous pass has read s_seq; the tables are filled
        // stage A by all threads over (b, column), column fastest: its inputs come straight from the workspace,
        // a warp reads 32 consecutive float2 when C = CB
#pragma unroll UA
        for (int e = tid; e < C * P::L1; e += NT) {
            const int c = e % C, b = e / C;
            const float2 *col = src + c;
            fft::stage_a_butterfly<LOG2G>(s_seq + c * SEQ + fft::pad16(b), b, s_tab,
                                          [&](int bb, int r) { return __ldcs(col + (size_t)(bb + r * P::L1) * CB); });
        }
        __syncthreads();
#pragma unroll 1
        for (int c = grp; c < C; c += CT) fft::stage_b<LOG2G, T>(s_seq + c * SEQ, t, s_tab);
        __syncthreads();
#pragma unroll 1
        for (int c = grp; c < C; c += CT) fft::stage_c<LOG2G, T>(s_seq + c * SEQ, t, fft::SmemOut{});
        __syncthreads();                         // output k of column c now sits at phys_out(k)
        if (IMAGE) {
            // step a7 fused: image[j][i] = Re F[m][n] (-1)^(n+m) / (psi(n) psi(m) omega Wsum), n = i - N/2, m = j - N/2
            const int i0 = (n0 < half ? n0 : n0 - G) + half;     // image column of my first column
            for (int idx = tid; idx < C * N; idx += NT) {
                const int c = idx % C, j = idx / C;
                const int m = j - half, i = i0 + c, n = i - half;
                float out = 0.0f;
                if (ok) {
                    const float re = s_seq[c * SEQ + fft::phys_out<LOG2G>(m < 0 ? m + G : m)].x;
                    const float f = (float)(ipsi[i] * ipsi[j] * inv_norm);
                    out = ((n + m) & 1) ? -(re * f) : re * f;
                }
                image[(size_t)j * N + i] = out;
            }
        } else {
            // the complex transform of the pixels the crop keeps, moment[j][i] = F[m][n] (3-D mode: k_cheb_combine reads it)
            const int i0 = (n0 < half ? n0 : n0 - G) + half;
            for (int idx = tid; idx < C * N; idx += NT) {
                const int c = idx % C, j = idx / C;
                const int m = j - half;
                moment[(size_t)j * N + i0 + c] = s_seq[c * SEQ + fft::phys_out<LOG2G>(m < 0 ? m + G : m)];
            }
        }
    }
}

template <int LOG2G, int T, int MINB>
void rows_launch(const float2 *grid, float2 *work, const uint8_t *map, int N, const float2 *tw, int n_sms,
                 cudaStream_t stream)
{
    using P = fft::Plan<LOG2G>;
    constexpr int G = 1 << LOG2G;
    constexpr size_t smem = (size_t)(P::kTabFloat2 + P::kPadded) * sizeof(float2);
    static const cudaError_t once = cudaFuncSetAttribute(k_fft_rows<LOG2G, T, MINB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    (void)once;
    int per_sm = (int)((224 * 1024) / (smem + 1024));
    if (per_sm > MINB) per_sm = MINB;
    if (per_sm < 1) per_sm = 1;
    int ctas = per_sm * n_sms;
    if (ctas > G) ctas = G;
    launch_pdl(k_fft_rows<LOG2G, T, MINB>, dim3(ctas), dim3(T), smem, stream, grid, work, map, N, tw);
}

template <int LOG2G, int C, int CT, int T, int UA>
void cols_launch(const float2 *work, int N, const float2 *tw, const double *ipsi, const SnapState *st, int apply_jacobian,
                 float *image, float2 *moment, const ClearArgs &clr, int n_sms, cudaStream_t stream)
{
    using P = fft::Plan<LOG2G>;
    constexpr size_t smem = (size_t)(P::kTabFloat2 + C * (P::kPadded + kSkew)) * sizeof(float2);
    int per_sm = (int)((224 * 1024) / (smem + 1024));
    if (per_sm * T * CT > 1024) per_sm = 1024 / (T * CT);
    if (per_sm < 1) per_sm = 1;
    int ctas = per_sm * n_sms;
    if (ctas > N / C) ctas = N / C;
    if (image) {
        static const cudaError_t once = cudaFuncSetAttribute(k_fft_cols<LOG2G, C, CT, T, UA, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        (void)once;
        launch_pdl(k_fft_cols<LOG2G, C, CT, T, UA, true>, dim3(ctas), dim3(T * CT), smem, stream, work, N, tw, ipsi, st, apply_jacobian, image, moment, clr);
    } else {
        static const cudaError_t once = cudaFuncSetAttribute(k_fft_cols<LOG2G, C, CT, T, UA, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        (void)once;
        launch_pdl(k_fft_cols<LOG2G, C, CT, T, UA, false>, dim3(ctas), dim3(T * CT), smem, stream, work, N, tw, ipsi, st, apply_jacobian, image, moment, clr);
    }
}

int log2_exact(int G)
{
    for (int l = 0; l < 31; ++l)
        if ((1 << l) == G) return l;
    return -1;
}

}  // namespace

// shapes the hand-written transform takes: G = 2^10 .. 2^14, pruned (4 N <= 3 G), N a multiple of 16
bool fft_custom_supported(int N, int G)
{
    const int l = log2_exact(G);
    return l >= 10 && l <= 14 && 4 * N <= 3 * G && N % 16 == 0;
}

// W^m = exp(+2 pi i m / G), m = 0 .. G - 1, computed in fp64
void fft_twiddle_table(int G, float2 *host_out)
{
    const double two_pi = 6.283185307179586476925286766559;
    for (int m = 0; m < G; ++m) {
        const double a = two_pi * (double)m / (double)G;
        host_out[m] = make_float2((float)cos(a), (float)sin(a));
    }
}

// pass 1: rows of `grid` (read through the tile map) -> needed columns of `work`
void launch_fft_rows(int N, int G, const float2 *d_grid, float2 *d_work, const uint8_t *d_map, const float2 *d_tw,
                     int n_sms, cudaStream_t stream)
{
    switch (log2_exact(G)) {
    case 10: rows_launch<10, 64, 8>(d_grid, d_work, d_map, N, d_tw, n_sms, stream); break;
    case 11: rows_launch<11, 128, 4>(d_grid, d_work, d_map, N, d_tw, n_sms, stream); break;
    case 12: rows_launch<12, 256, 3>(d_grid, d_work, d_map, N, d_tw, n_sms, stream); break;
    case 13: rows_launch<13, 256, 2>(d_grid, d_work, d_map, N, d_tw, n_sms, stream); break;
    default: rows_launch<14, 512, 1>(d_grid, d_work, d_map, N, d_tw, n_sms, stream); break;
    }
}

// pass 2: the needed columns of `work`; d_image != nullptr: the finished image (step a7 fused), else the
// complex values of the N x N pixels the crop keeps into d_moment[j][i].  d_clear_map != nullptr: the sparse
// clear of d_clear_grid / d_clear_density (either may be null) runs inside this pass (k_clear.cu otherwise)
void launch_fft_cols(int N, int G, const float2 *d_work, const float2 *d_tw, const double *d_ipsi, const SnapState *st,
                     int apply_jacobian, float *d_image, float2 *d_moment, float2 *d_clear_grid, float *d_clear_density,
                     uint8_t *d_clear_map, int n_sms, cudaStream_t stream)
{
    ClearArgs clr;
    clr.grid = d_clear_grid; clr.dens = d_clear_density; clr.map = d_clear_map;
    clr.G = G; clr.tpr = tiles_per_row(G); clr.n_tiles = (long long)tiles_per_row(G) * tile_rows(G);
    switch (log2_exact(G)) {
    case 10: cols_launch<10, 8, 8, 64, 1>(d_work, N, d_tw, d_ipsi, st, apply_jacobian, d_image, d_moment, clr, n_sms, stream); break;
    case 11: cols_launch<11, 8, 4, 128, 1>(d_work, N, d_tw, d_ipsi, st, apply_jacobian, d_image, d_moment, clr, n_sms, stream); break;
    case 12: cols_launch<12, 4, 4, 128, 1>(d_work, N, d_tw, d_ipsi, st, apply_jacobian, d_image, d_moment, clr, n_sms, stream); break;
    case 13: cols_launch<13, 2, 2, 128, 1>(d_work, N, d_tw, d_ipsi, st, apply_jacobian, d_image, d_moment, clr, n_sms, stream); break;
    default: cols_launch<14, 1, 1, 512, 1>(d_work, N, d_tw, d_ipsi, st, apply_jacobian, d_image, d_moment, clr, n_sms, stream); break;
    }
}

}  // namespace toi
