// k_grid_sliding.cu -- step a5, the product gridder (TOI_GRIDDER_SLIDING):
//   grid[iv+dv][iu+du] += f z phi(iu+du-gu) phi(iv+dv-gv),  du, dv = -3..3
// ("place visibilities on a grid"; kernel, support and edge rule: DESIGN.md G9, G10).
//
// Design (sm_100a; none of it is the paper's -- DESIGN.md section 6):
//  * The samples of one baseline lie on a ray through the uv origin, monotone in channel, and move
//    a few hundredths of a cell per channel: consecutive channels share a 7x7 footprint for many
//    samples and the footprint then slides by ONE cell.  So a group of 7 lanes keeps the whole
//    7x7 complex footprint in registers (lane = column, 7 row accumulators of packed re/im) and
//    streams through a strip of consecutive channels.  Per sample each lane does one packed
//    multiply (z * phi_u[column]) and seven packed FMAs (fma.rn.f32x2 -> FFMA2, new on sm_100).
//  * When the centre cell moves by one column, only the retiring column (7 cells, one lane) is
//    flushed; the lane then owns the entering column (columns are owned by absolute column mod 7,
//    so nothing is shuffled).  When it moves by one row, the retiring row is flushed (one cell
//    per lane, 56 contiguous bytes) and the row accumulators shift by one register.  Flushes are
//    vector reductions red.global.add.v2.f32 (one per complex cell).  Per run of ~17 samples that
//    is 7 reductions instead of 17 * 98 scalar atomics.
//  * A warp carries four such groups (28 of 32 lanes) on four adjacent strips of one baseline.
//    All 32 lanes first pre-process 32 samples (fp64 cell index, flags/weights/polarisation
//    average, 14 kernel taps on the MUFU pipe) into a shared-memory record each; the groups
//    then consume their 8 records.  Tasks (baseline, block of 4 strips) come from an atomic
//    queue, so the grid is persistent: 2 CTAs x 8 warps per SM.
//  * fp32 summation is blocked by construction: register chains are bounded by the time a cell
//    stays inside a sliding window (tens to a few hundred samples), everything else is summed by
//    the L2 reduction units.
#include "toi_internal.cuh"

namespace toi {
namespace {

typedef unsigned long long u64;

constexpr int kGroups = 4;        // 7-lane groups per warp
constexpr int kBatch = 8;         // samples per group per pre-processing batch (4 * 8 = 32 lanes)
constexpr int kWarps = 8;         // warps per CTA
constexpr int kRecQuads = 7;      // record = 7 x 16 B: {zre, zim, iu, iv | pu0..3 | pu4..6,- |
                                  //                    pv0,pv0,pv1,pv1 | pv2.. | pv4.. | pv6,pv6,-,-}
constexpr int kModBias = 7 << 20; // makes (x + kModBias) % 7 a mathematical mod for |x| < 2^22

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
__device__ __forceinline__ u64 mul2(u64 a, u64 b)
{
    u64 d;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ void red_cell(float2 *cell, u64 v)
{
    const float2 f = unpack2(v);
    if (f.x != 0.0f || f.y != 0.0f)
        asm volatile("red.global.add.v2.f32 [%0], {%1, %2};" ::"l"(cell), "f"(f.x), "f"(f.y) : "memory");
}

__global__ void __launch_bounds__(kWarps * 32, 2)
k_grid_sliding(Geometry g, Inputs in, SnapState *__restrict__ st, const float *__restrict__ D,
               float2 *__restrict__ grid, int strip_len, int tasks_per_row, unsigned n_tasks)
{
    __shared__ float4 s_rec[kWarps][32 * kRecQuads];
    if (st->status != TOI_OK) return;
    const int lane = threadIdx.x & 31;
    float4 *rec = s_rec[threadIdx.x >> 5];

    // roles: every lane pre-processes one sample per batch; lanes 0..27 accumulate
    const int pre_k = lane >> 2, pre_g = lane & 3;
    const bool acc_lane = lane < 7 * kGroups;
    const int grp = lane / 7, m = lane - 7 * grp;
    const int G = g.G;

    double wsum = 0.0;
    unsigned n_grid = 0, n_off = 0, n_flag = 0;

    for (;;) {
        unsigned task = 0;
        if (lane == 0) task = atomicAdd(&st->task_counter, 1u);
        task = __shfl_sync(0xffffffffu, task, 0);
        if (task >= n_tasks) break;
        const int j = (int)(task / (unsigned)tasks_per_row);
        const int c_task = (int)(task % (unsigned)tasks_per_row) * (kGroups * strip_len);
        double rho1, rho2;
        rotate_baseline(st->V, in.uvw + 3 * j, rho1, rho2);
        const int c_lo = c_task + pre_g * strip_len;
        const int c_hi = min(c_lo + strip_len, g.n_c);
        const int c_end = min(c_task + kGroups * strip_len, g.n_c);   // of the whole task

        // sliding-window state of my group (uniform across its 7 lanes)
        u64 acc[kW];
#pragma unroll
        for (int d = 0; d < kW; ++d) acc[d] = 0ull;
        int cu = kOffGrid, cv = kOffGrid;    // closed window: any real cell mismatches
        int mydu = 0;                        // which tap column of the window this lane holds

        for (int b = 0; b < strip_len && c_task + b < c_end; b += kBatch) {
            // ---------------- pre-process one sample per lane ----------------
            {
                const int c = c_lo + b + pre_k;
                float4 q0 = make_float4(0.0f, 0.0f, __int_as_float(kOffGrid), __int_as_float(kOffGrid));
                float pu[kW], pv[kW];
#pragma unroll
                for (int d = 0; d < kW; ++d) pu[d] = pv[d] = 0.0f;
                if (c < c_hi) {
                    double gu, gv;
                    int iu, iv;
                    sample_cell(rho1, rho2, g.s[c], g.kappa, gu, gv, iu, iv);
                    if (!cell_on_grid(iu, iv, G)) {
                        ++n_off;
                    } else {
                        const long long o = ((long long)j * g.n_c + c) * g.n_p;
                        float wa, wb;
                        sample_weights(g, in, o, wa, wb);
                        const float wI = wa + wb;
                        q0.z = __int_as_float(iu);
                        q0.w = __int_as_float(iv);
                        if (!(wI > 0.0f)) {
                            ++n_flag;       // coordinates stay valid, z = 0: the window just slides
                        } else {
                            ++n_grid;
                            float2 z = sample_stokes(g, in, o, wa, wb);
                            float f = 1.0f;
                            if (D) f = 1.0f / __ldg(D + (size_t)wrap_index(iv, G) * G + wrap_index(iu, G));
                            wsum += (double)f * (double)wI;
                            q0.x = z.x * f;
                            q0.y = z.y * f;
                            kernel_taps((float)(gu - (double)iu), pu);
                            kernel_taps((float)(gv - (double)iv), pv);
                        }
                    }
                }
                float4 *r = rec + lane * kRecQuads;
                r[0] = q0;
                r[1] = make_float4(pu[0], pu[1], pu[2], pu[3]);
                r[2] = make_float4(pu[4], pu[5], pu[6], 0.0f);
                r[3] = make_float4(pv[0], pv[0], pv[1], pv[1]);
                r[4] = make_float4(pv[2], pv[2], pv[3], pv[3]);
                r[5] = make_float4(pv[4], pv[4], pv[5], pv[5]);
                r[6] = make_float4(pv[6], pv[6], 0.0f, 0.0f);
            }
            __syncwarp();
            // ---------------- accumulate: group grp consumes records k*4 + grp ----------------
            if (acc_lane) {
#pragma unroll 1
                for (int k = 0; k < kBatch; ++k) {
                    const float4 *r = rec + (k * kGroups + grp) * kRecQuads;
                    const float4 q0 = r[0];
                    const int iu = __float_as_int(q0.z), iv = __float_as_int(q0.w);
                    if (iu != cu || iv != cv) {
                        if (iu == kOffGrid) continue;               // padding / off-grid sample
                        const int du = iu - cu, dv = iv - cv;
                        if (cu != kOffGrid && du >= -1 && du <= 1 && dv >= -1 && dv <= 1) {
                            if (du != 0) {                          // slide one column
                                if (mydu == (du > 0 ? 0 : kW - 1)) {
                                    float2 *col = grid + wrap_index(cu - du * kH, G);
#pragma unroll
                                    for (int d = 0; d < kW; ++d) {
                                        red_cell(col + (size_t)wrap_index(cv - kH + d, G) * G, acc[d]);
                                        acc[d] = 0ull;
                                    }
                                }
                                cu += du;
                                mydu -= du;
                                mydu = mydu < 0 ? kW - 1 : (mydu >= kW ? 0 : mydu);
                            }
                            if (dv != 0) {                          // slide one row
                                float2 *row = grid + (size_t)wrap_index(cv - dv * kH, G) * G +
                                              wrap_index(cu - kH + mydu, G);
                                if (dv > 0) {
                                    red_cell(row, acc[0]);
#pragma unroll
                                    for (int d = 0; d < kW - 1; ++d) acc[d] = acc[d + 1];
                                    acc[kW - 1] = 0ull;
                                } else {
                                    red_cell(row, acc[kW - 1]);
#pragma unroll
                                    for (int d = kW - 1; d > 0; --d) acc[d] = acc[d - 1];
                                    acc[0] = 0ull;
                                }
                                cv += dv;
                            }
                        } else {                                    // first sample, or a jump
                            if (cu != kOffGrid) {
                                float2 *col = grid + wrap_index(cu - kH + mydu, G);
#pragma unroll
                                for (int d = 0; d < kW; ++d) {
                                    red_cell(col + (size_t)wrap_index(cv - kH + d, G) * G, acc[d]);
                                    acc[d] = 0ull;
                                }
                            }
                            cu = iu;
                            cv = iv;
                            mydu = (m - cu + kH + kModBias) % kW;   // column (cu-3+mydu) = m (mod 7)
                        }
                    }
                    const float pu = reinterpret_cast<const float *>(r + 1)[mydu];
                    const u64 t = mul2(pack2(q0.x, q0.y), pack2(pu, pu));
                    const ulonglong2 v01 = *reinterpret_cast<const ulonglong2 *>(r + 3);
                    const ulonglong2 v23 = *reinterpret_cast<const ulonglong2 *>(r + 4);
                    const ulonglong2 v45 = *reinterpret_cast<const ulonglong2 *>(r + 5);
                    const u64 v6 = *reinterpret_cast<const u64 *>(r + 6);
                    acc[0] = fma2(t, v01.x, acc[0]);
                    acc[1] = fma2(t, v01.y, acc[1]);
                    acc[2] = fma2(t, v23.x, acc[2]);
                    acc[3] = fma2(t, v23.y, acc[3]);
                    acc[4] = fma2(t, v45.x, acc[4]);
                    acc[5] = fma2(t, v45.y, acc[5]);
                    acc[6] = fma2(t, v6, acc[6]);
                }
            }
            __syncwarp();
        }
        // strip done: flush what is left of the window
        if (acc_lane && cu != kOffGrid) {
            float2 *col = grid + wrap_index(cu - kH + mydu, G);
#pragma unroll
            for (int d = 0; d < kW; ++d) red_cell(col + (size_t)wrap_index(cv - kH + d, G) * G, acc[d]);
        }
    }

#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        wsum += __shfl_xor_sync(0xffffffffu, wsum, d);
        n_grid += __shfl_xor_sync(0xffffffffu, n_grid, d);
        n_off += __shfl_xor_sync(0xffffffffu, n_off, d);
        n_flag += __shfl_xor_sync(0xffffffffu, n_flag, d);
    }
    if (lane == 0) {
        if (wsum != 0.0) atomicAdd(&st->wsum, wsum);
        if (n_grid) atomicAdd(&st->n_gridded, (unsigned long long)n_grid);
        if (n_off) atomicAdd(&st->n_off_grid, (unsigned long long)n_off);
        if (n_flag) atomicAdd(&st->n_flagged, (unsigned long long)n_flag);
    }
}

}  // namespace

void launch_grid_sliding(const Geometry &g, const Inputs &in, SnapState *st, const float *d_density,
                         float2 *d_grid, int n_sms, cudaStream_t stream)
{
    // strip length: a quarter of the row, rounded up to a batch, capped at 256 channels
    int strip = ((g.n_c + kGroups - 1) / kGroups + kBatch - 1) / kBatch * kBatch;
    if (strip > 256) strip = 256;
    const int tasks_per_row = (g.n_c + kGroups * strip - 1) / (kGroups * strip);
    const long long n_tasks = (long long)g.n_b * tasks_per_row;
    long long ctas = (n_tasks + kWarps - 1) / kWarps;
    if (ctas > 2LL * n_sms) ctas = 2LL * n_sms;   // persistent: 2 CTAs per SM pull from the queue
    k_grid_sliding<<<(unsigned)ctas, kWarps * 32, 0, stream>>>(g, in, st, d_density, d_grid, strip,
                                                               tasks_per_row, (unsigned)n_tasks);
}

}  // namespace toi
