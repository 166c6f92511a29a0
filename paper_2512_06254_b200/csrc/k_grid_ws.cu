// k_grid_ws.cu -- step a5, warp-specialised gridder: the sliding register window of grid_window.cuh
// with its two halves split between PRODUCER warps (fp64 cell index, weights / flags / parallel-hand
// average, 14 kernel taps -> 80-byte shared-memory records) and CONSUMER warps (the 8 x 8-cell
// register window: 4 record bodies per batch, window moves, red.global.add flushes):
//   grid[iv+dv][iu+du] += f z phi(iu+du-gu) phi(iv+dv-gv),  du, dv = -3..3
//
// Why: the fused kernel (k_grid_pair8.cu) holds 32 accumulator registers AND the pre-processing
// state in every warp (114-122 registers -> 16 warps/SM), runs both halves back to back in one warp
// (every dependent chain of one half waits for the other to finish) and is issue/latency bound at
// 62 % of the issue slots.  Here a producer warp holds no accumulators and a consumer warp no
// pre-processing state (both <= 80 registers -> 24 warps/SM), the two halves of a batch overlap in
// time, and each role's loop is small.  A producer/consumer pair owns a ring of kSlots record
// batches in shared memory; mbarriers (one "full", one "empty" per slot) hand the slots over; a
// control word per slot tells the consumer to flush its windows (end of a task's strips) or stop.
// The producer requests its raw inputs (and, with a density map, the density value of the cell)
// two batches ahead, into two alternating register sets.
#include "grid_window.cuh"

namespace toi {
namespace {

constexpr int kPairs = 5;            // producer/consumer warp pairs per CTA: warps 0..4 produce, 5..9 consume
constexpr int kSlots = 4;            // record batches in flight per pair
constexpr int kCtasPerSm = 2;        // 2 x 10 warps = 20 warps/SM, <= 96 registers per thread
constexpr unsigned kCtlFlush = 1u, kCtlStop = 2u;

struct PairRing {
    uint4 rec[kSlots][kWarpQuads];
    unsigned long long full[kSlots], empty[kSlots];
    unsigned ctl[kSlots];
    unsigned pad_[16 - kSlots];      // keep the next pair's records 16-byte aligned
};

__device__ __forceinline__ unsigned smem_addr(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
// mbarriers by their 32-bit shared address
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" : : "r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" : : "r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity)
{
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@!p bra WAIT_%=;\n\t"
        "}"
        : : "r"(bar), "r"(parity) : "memory");
}

constexpr size_t kRingBytes = sizeof(PairRing) * kPairs;     // dynamic shared memory per CTA

// Geometry of one sample, computed when its raw inputs are requested (two batches before use).
struct Ahead {
    Raw raw;
    Cell cell;
};

template <int MODE, int OPT, bool CHEB>
__global__ void __launch_bounds__(2 * kPairs * 32, kCtasPerSm)
k_grid_ws(Geometry g, Inputs in, SnapState *__restrict__ st, const float *__restrict__ D,
          float2 *__restrict__ grid, uint8_t *__restrict__ tiles, int strip_len, int tasks_per_row,
          unsigned n_tasks, ChebArgs cheb)
{
    extern __shared__ __align__(16) unsigned char s_dyn[];
    PairRing *const s_ring = reinterpret_cast<PairRing *>(s_dyn);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int pair = warp % kPairs;
    const bool producer = warp < kPairs;
    PairRing &ring = s_ring[pair];
    const unsigned bar_full = smem_addr(ring.full), bar_empty = smem_addr(ring.empty);   // + 8 * slot
    if (lane < kSlots && warp < kPairs) {
        mbar_init(bar_full + 8u * lane, 1u);
        mbar_init(bar_empty + 8u * lane, 1u);
    }
    __syncthreads();
    if (st->status != TOI_OK) return;
    const int grp = lane >> 2, L = lane & 3;
    const int G = g.G;

    if (producer) {
        // ======================= producer: one sample per lane and batch =======================
        const bool has_w = OPT >= 0 ? (OPT & kHasW) != 0 : in.weights != nullptr;
        const bool has_f = OPT >= 0 ? (OPT & kHasF) != 0 : in.flags != nullptr;
        const bool has_d = OPT >= 0 ? (OPT & kHasD) != 0 : D != nullptr;
        const int pre_k = L;
        const int my_quad = group_quad(grp) + pre_k * kRecQuads;
        const float *const Dc = has_d ? D + centre_index(0, 0, G) : nullptr;
        double wsum = 0.0;
        unsigned n_grid = 0, n_off = 0, n_flag = 0;
        // Chebyshev passes repeat the samples: Wsum / n_gridded once per slab, the rejects once per snapshot
        const bool count = !CHEB || (cheb.count & 1) != 0, count_rej = !CHEB || (cheb.count & 2) != 0;
        unsigned slot = 0, phase = 0;          // ring position of the next batch to hand over

        // dynamic task queue; the NEXT task is requested while the current one is processed
        unsigned task_ahead = 0;
        if (lane == 0) task_ahead = atomicAdd(&st->task_counter, 1u);
        for (;;) {
            const unsigned task = __shfl_sync(0xffffffffu, task_ahead, 0);
            if (task >= n_tasks) break;
            if (lane == 0) task_ahead = atomicAdd(&st->task_counter, 1u);
            const int j = (int)(task / (unsigned)tasks_per_row);
            const int c_task = (int)(task % (unsigned)tasks_per_row) * (kGroups * strip_len);
            double rho1, rho2;
            rotate_baseline(st->V, in.uvw + 3 * j, rho1, rho2);
            const double rho3 = CHEB ? rotate_row3(st->V, in.uvw + 3 * j) : 0.0;
            const int c_lo = c_task + grp * strip_len + pre_k;        // my channel in batch 0
            const int c_hi = min(c_task + (grp + 1) * strip_len, g.n_c);
            const long long q_row = (long long)j * g.n_c;
            const int n_batches = (min(strip_len, g.n_c - c_task) + kBatch - 1) / kBatch;

            // Sparse clear (k_clear.cu): mark the tiles my strip's windows can reach.  The samples of a
            // strip lie on a ray, monotone in channel (the plan passes `tiles` only when the channel
            // scales are monotone), so the windows stay inside the box spanned by the strip's two end
            // samples, widened by the 4 cells a window reaches beyond its sample's centre on either side.
            if (tiles != nullptr) {
                const int c_first = c_task + grp * strip_len;
                const bool some = c_first < c_hi;
                const double s_end = __ldg(g.s + ((L & 1) ? max(c_hi - 1, 0) : min(c_first, g.n_c - 1)));
                const double lim = (double)G;                         // far outside the grid; also absorbs NaN
                const double eu = fmin(fmax(-__dmul_rn(__dmul_rn(rho1, s_end), g.kappa), -lim), lim);
                const double ev = fmin(fmax(__dmul_rn(__dmul_rn(rho2, s_end), g.kappa), -lim), lim);
                const int iu = __double2int_rd(eu + 0.5), iv = __double2int_rd(ev + 0.5);
                const int ju = __shfl_xor_sync(0xffffffffu, iu, 1), jv = __shfl_xor_sync(0xffffffffu, iv, 1);
                if (some && L == 0) {
                    const int h = G >> 1, tpr = tiles_per_row(G);
                    const int x0 = max(min(iu, ju) - 4 + h, 0) / kTile, x1 = min(max(iu, ju) + 4 + h, G - 1) / kTile;
                    const int y0 = max(min(iv, jv) - 4 + h, 0) / kTile, y1 = min(max(iv, jv) + 4 + h, G - 1) / kTile;
                    for (int ty = y0; ty <= y1; ++ty)
                        for (int tx = x0; tx <= x1; ++tx)
                            if (tiles[ty * tpr + tx] == 0) tiles[ty * tpr + tx] = 1;   // L1 hit instead of a store, mostly
                }
            }

            float wpart = 0.0f;
            // request the raw inputs of batch `bb` and locate its sample (cell, window base, sub-cell
            // offsets, density value): everything that depends only on (baseline, channel)
            auto s_of = [&](int bb) {       // channel scale of my sample in batch bb (requested a batch before use)
                const int c = c_lo + bb * kBatch;
                return (bb < n_batches && c < c_hi) ? __ldg(g.s + c) : 0.0;
            };
            auto fetch = [&](int bb, Ahead &a, double s_c) {
                const int c = c_lo + bb * kBatch;
                a.cell.key = kNoKey; a.cell.sh = 0u; a.cell.xu = a.cell.xv = 0.0f; a.cell.dens = 1.0f;
                if (bb < n_batches && c < c_hi) {
                    load_raw<MODE, false>(g, in, has_w, has_f, q_row + c, c, a.raw);
                    int iu, iv;
                    sample_cell(rho1, rho2, s_c, g.kappa, iu, iv, a.cell.xu, a.cell.xv);
                    if (cell_on_grid(iu, iv, G)) {
                        const int bu = (iu - kH) & ~1, bv = (iv - kH) & ~1;
                        a.cell.key = cell_key(bu, bv);
                        a.cell.sh = (unsigned)((iu - kH) & 1) | ((unsigned)((iv - kH) & 1) << 1);
                        if (has_d) a.cell.dens = __ldg(Dc + ((long long)iv * G + iu));
                    } else {
                        a.cell.xu = a.cell.xv = 0.0f;          // taps stay finite whatever the coordinates were
                        if (count_rej) ++n_off;
                    }
                }
            };
            // turn the sample in `a` (batch bb) into its record, hand the batch over, refill `a`
            double s_next;                   // scale of the sample the NEXT emit will fetch
            auto emit = [&](int bb, Ahead &a, int refill) {
                const int c = c_lo + bb * kBatch;
                // a flagged sample keeps its own cell as key (z = 0): it moves the window exactly as
                // its unflagged neighbours do; a record that contributes nothing has z = 0, finite taps
                const unsigned key = a.cell.key;
                const bool on = key != kNoKey;
                constexpr unsigned fmask_b = MODE == 2 ? 0x0000ff00u : 0xff000000u;
                const float wa = (on && weight_ok(a.raw.wa) && !(a.raw.fl & 0x000000ffu)) ? a.raw.wa : 0.0f;
                const float wb = (on && weight_ok(a.raw.wb) && !(a.raw.fl & fmask_b)) ? a.raw.wb : 0.0f;
                const float wI = wa + wb;
                float tk = 1.0f;
                bool mine = true;
                if (CHEB && wI > 0.0f) {
                    // Eq. 19: slab of this sample and its position s_q in it (G24); T_k(s_q) by the
                    // three-term recurrence in fp64 (T_k amplifies rounding by ~k^2)
                    const double r3 = __dmul_rn(rho3, __ldg(g.s + min(c, g.n_c - 1)));
                    int pq = 0;
                    double sq = 0.0;
                    if (cheb.d > 0.0) {
                        pq = min((int)floor((r3 - cheb.r3_min) / (2.0 * cheb.d)), cheb.n_slab - 1);
                        sq = (r3 - (cheb.r3_min + (2.0 * (double)pq + 1.0) * cheb.d)) / cheb.d;
                    }
                    mine = pq == cheb.p;
                    double t0 = 1.0, t1 = sq;
                    for (int kk = 1; kk < cheb.k; ++kk) {
                        const double t2 = fma(2.0 * sq, t1, -t0);
                        t0 = t1; t1 = t2;
                    }
                    tk = (float)(cheb.k == 0 ? 1.0 : t1);
                }
                const bool valid = wI > 0.0f && mine;
                if (on && !(wI > 0.0f) && count_rej) ++n_flag;
                if (valid && count) ++n_grid;
                // z = w_a Vis_a + w_b Vis_b; a zero-weight hand is skipped (its data may be NaN)
                float zx = 0.0f, zy = 0.0f;
                if (wa > 0.0f) { zx = wa * a.raw.a.x; zy = wa * a.raw.a.y; }
                if (wb > 0.0f) { zx = fmaf(wb, a.raw.b.x, zx); zy = fmaf(wb, a.raw.b.y, zy); }
                if (CHEB) { zx *= tk; zy *= tk; }
                if (!valid) zx = zy = 0.0f;
                float f = 1.0f;
                if (has_d) {
                    // the density of a cell whose samples are all flagged is 0: never invert it
                    const float dens = valid ? a.cell.dens : 1.0f;
                    asm volatile("rcp.approx.ftz.f32 %0, %1;" : "=f"(f) : "f"(dens));
                }
                if (!CHEB || count) wpart = fmaf(f, valid ? wI : 0.0f, wpart);
                const float xu = a.cell.xu, xv = a.cell.xv;
                const bool su = (a.cell.sh & 1u) != 0u, sv = (a.cell.sh & 2u) != 0u;
                // ---- this sample's raw inputs and cell are used up: request batch `refill`'s ----
                fetch(refill, a, s_next);
                s_next = s_of(refill + 1);
                float pu[kW], pv[kW];
                kernel_taps2(xu, xv, pu, pv);
                // the 7 taps sit at window offset 0 or 1 on each axis; the free end is zero
                unsigned wu[kR], wv[kR];
#pragma unroll
                for (int i = 0; i < kR; ++i) {
                    const float lo_u = i < kW ? pu[i] : 0.0f, hi_u = i > 0 ? pu[i - 1] : 0.0f;
                    const float lo_v = i < kW ? pv[i] : 0.0f, hi_v = i > 0 ? pv[i - 1] : 0.0f;
                    wu[i] = __float_as_uint(su ? hi_u : lo_u);
                    wv[i] = __float_as_uint(sv ? hi_v : lo_v);
                }
                mbar_wait(bar_empty + 8u * slot, phase ^ 1u);    // the consumer is done with this slot
                uint4 *my_rec = ring.rec[slot] + my_quad;
                my_rec[1] = make_uint4(wv[1], wv[2], wv[3], wv[4]);
                my_rec[2] = make_uint4(wv[5], wv[6], wv[7], 0u);
                my_rec[3] = make_uint4(wu[0], wu[1], wu[2], wu[3]);
                my_rec[4] = make_uint4(wu[4], wu[5], wu[6], wu[7]);
                my_rec[0] = make_uint4(__float_as_uint(zx * f), __float_as_uint(zy * f), key, wv[0]);
                if (lane == 0) ring.ctl[slot] = bb == n_batches - 1 ? kCtlFlush : 0u;
                __syncwarp();
                if (lane == 0) mbar_arrive(bar_full + 8u * slot);
                if (++slot == kSlots) { slot = 0; phase ^= 1u; }
            };

            Ahead a0, a1;
            a0.raw.a = a0.raw.b = a1.raw.a = a1.raw.b = make_float2(0.0f, 0.0f);
            a0.raw.wa = a0.raw.wb = a1.raw.wa = a1.raw.wb = 0.0f;
            a0.raw.fl = a1.raw.fl = 0u;
            fetch(0, a0, s_of(0));
            fetch(1, a1, s_of(1));
            s_next = s_of(2);
            for (int bb = 0; bb < n_batches; bb += 2) {
                emit(bb, a0, bb + 2);
                if (bb + 1 < n_batches) emit(bb + 1, a1, bb + 3);
            }
            wsum += (double)wpart;
        }
        // no task left: one empty batch that tells the consumer to stop
        {
            mbar_wait(bar_empty + 8u * slot, phase ^ 1u);
            uint4 *my_rec = ring.rec[slot] + my_quad;
            const uint4 zero = make_uint4(0u, 0u, 0u, 0u);
            my_rec[1] = zero; my_rec[2] = zero; my_rec[3] = zero; my_rec[4] = zero;
            my_rec[0] = make_uint4(0u, 0u, kNoKey, 0u);
            if (lane == 0) ring.ctl[slot] = kCtlFlush | kCtlStop;
            __syncwarp();
            if (lane == 0) mbar_arrive(bar_full + 8u * slot);
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
    } else {
        // ======================= consumer: group of 4 lanes = one strip's window =======================
        const float2 *const gc = grid + centre_index(0, 0, G);   // cell (0, 0)
        const long long rs = (long long)G * 8;                   // row stride in bytes
        const unsigned goff = (unsigned)group_quad(grp) * 16u;   // my group's records inside a slot
        const unsigned rec0 = smem_addr(ring.rec[0]) + goff, ctl0 = smem_addr(ring.ctl);
        unsigned slot = 0, phase = 0;
        // one pass of the outer loop = the strips of one task: the accumulators are cleared and the
        // window closed OUTSIDE the batch loop (a plain write to an accumulator inside it makes ptxas
        // rename the accumulators and copy them at every batch)
        for (;;) {
            u64 accA[kR], accB[kR];
#pragma unroll
            for (int d = 0; d < kR; ++d) accA[d] = accB[d] = 0ull;
            unsigned ckey = kNoKey;              // closed window; else the packed base cell (bu, bv)
            unsigned tapA = 0u;                  // window column held by my slot L; slot L + 4 holds tapA ^ 4
            unsigned offA = 48u, offB = 48u + 16u;   // offsets of my two taps in record 0 of my group
            unsigned ctl;
            for (;;) {
                mbar_wait(bar_full + 8u * slot, phase);
                asm volatile("ld.shared.u32 %0, [%1];" : "=r"(ctl) : "r"(ctl0 + 4u * slot) : "memory");
                const unsigned rgs = rec0 + slot * (unsigned)(kWarpQuads * 16);
                unsigned rpa = rgs + offA, rpb = rgs + offB;
                consume_batch(accA, accB, tapA, ckey, rpa, rpb, rgs, gc, (unsigned)rs, G, L);
                offA = rpa - rgs; offB = rpb - rgs;
                __syncwarp();
                if (lane == 0) mbar_arrive(bar_empty + 8u * slot);
                if (++slot == kSlots) { slot = 0; phase ^= 1u; }
                if (ctl & kCtlFlush) break;
            }
            // the strips of this task are done: flush what is left of the window
            if (ckey != kNoKey) flush_sets(accA, accB, tapA, ckey, gc, rs, G);
            if (ctl & kCtlStop) break;
        }
    }
}

template <int MODE>
void launch_mode(int opt, dim3 grid, dim3 block, cudaStream_t stream, const Geometry &g, const Inputs &in,
                 SnapState *st, const float *D, float2 *d_grid, uint8_t *tiles, int strip, int tasks_per_row,
                 unsigned n_tasks)
{
    // 3 CTAs x 31 KB of rings per SM: ask for the large shared-memory carve-out
#define TOI_LAUNCH(O)                                                                                                     \
    {                                                                                                                     \
        static const cudaError_t once = cudaFuncSetAttribute(k_grid_ws<MODE, O, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kRingBytes); \
        (void)once;                                                                                                       \
        k_grid_ws<MODE, O, false><<<grid, block, kRingBytes, stream>>>(g, in, st, D, d_grid, tiles, strip, tasks_per_row, n_tasks, ChebArgs()); \
    }
    switch (opt) {
    case kHasW | kHasF | kHasD: TOI_LAUNCH(kHasW | kHasF | kHasD); break;
    case kHasW | kHasF: TOI_LAUNCH(kHasW | kHasF); break;
    case kHasD: TOI_LAUNCH(kHasD); break;
    case 0: TOI_LAUNCH(0); break;
    default: TOI_LAUNCH(-1); break;
    }
#undef TOI_LAUNCH
}

struct Shape {
    int strip, tasks_per_row;
    long long n_tasks, ctas;
};

// strip length (channels per group per task): 8 strips per task; aim at >= 6 tasks per producer
// warp, within [16, 128] channels and a multiple of the 4-sample batch
Shape task_shape(const Geometry &g, int n_sms)
{
    Shape s;
    const long long pairs = (long long)kCtasPerSm * n_sms * kPairs;
    const long long want = ((long long)g.n_b * g.n_c) / (kGroups * 6 * pairs);
    s.strip = pick_strip(g.n_c, kGroups, kBatch, want, 16, 128);
    s.tasks_per_row = (g.n_c + kGroups * s.strip - 1) / (kGroups * s.strip);
    s.n_tasks = (long long)g.n_b * s.tasks_per_row;
    s.ctas = (s.n_tasks + kPairs - 1) / kPairs;
    if (s.ctas > (long long)kCtasPerSm * n_sms) s.ctas = (long long)kCtasPerSm * n_sms;   // persistent CTAs pull from the queue
    return s;
}

}  // namespace

// G <= 32768 (toi_plan_create checks): a window base must fit the packed 16-bit key.
void launch_grid_ws(const Geometry &g, const Inputs &in, SnapState *st, const float *d_density,
                    float2 *d_grid, uint8_t *tiles, int n_sms, cudaStream_t stream)
{
    const Shape s = task_shape(g, n_sms);
    const dim3 grid((unsigned)s.ctas), block(2 * kPairs * 32);
    const uintptr_t aw = (uintptr_t)in.weights, af = (uintptr_t)in.flags, av = (uintptr_t)in.vis;
    const int opt = (in.weights ? kHasW : 0) | (in.flags ? kHasF : 0) | (d_density ? kHasD : 0);
    if (g.n_p == 4 && g.pol_a == 0 && g.pol_b == 3 && (aw & 15) == 0 && (af & 3) == 0)
        launch_mode<4>(opt, grid, block, stream, g, in, st, d_density, d_grid, tiles, s.strip, s.tasks_per_row, (unsigned)s.n_tasks);
    else if (g.n_p == 2 && g.pol_a == 0 && g.pol_b == 1 && (av & 15) == 0 && (aw & 7) == 0 && (af & 1) == 0)
        launch_mode<2>(opt, grid, block, stream, g, in, st, d_density, d_grid, tiles, s.strip, s.tasks_per_row, (unsigned)s.n_tasks);
    else
        launch_mode<0>(-1, grid, block, stream, g, in, st, d_density, d_grid, tiles, s.strip, s.tasks_per_row, (unsigned)s.n_tasks);
}

// One Chebyshev-moment pass of the near-coplanar mode.
void launch_grid_ws_cheb(const Geometry &g, const Inputs &in, SnapState *st, const float *d_density,
                         float2 *d_grid, uint8_t *tiles, int n_sms, const ChebArgs &cheb, cudaStream_t stream)
{
    const Shape s = task_shape(g, n_sms);
    const dim3 grid((unsigned)s.ctas), block(2 * kPairs * 32);
    const uintptr_t aw = (uintptr_t)in.weights, af = (uintptr_t)in.flags, av = (uintptr_t)in.vis;
#define TOI_LAUNCH_CHEB(M)                                                                                                \
    do {                                                                                                                   \
        static const cudaError_t once = cudaFuncSetAttribute(k_grid_ws<M, -1, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kRingBytes); \
        (void)once;                                                                                                       \
        k_grid_ws<M, -1, true><<<grid, block, kRingBytes, stream>>>(g, in, st, d_density, d_grid, tiles, s.strip, s.tasks_per_row, (unsigned)s.n_tasks, cheb); \
    } while (0)
    if (g.n_p == 4 && g.pol_a == 0 && g.pol_b == 3 && (aw & 15) == 0 && (af & 3) == 0)
        TOI_LAUNCH_CHEB(4);
    else if (g.n_p == 2 && g.pol_a == 0 && g.pol_b == 1 && (av & 15) == 0 && (aw & 7) == 0 && (af & 1) == 0)
        TOI_LAUNCH_CHEB(2);
    else
        TOI_LAUNCH_CHEB(0);
#undef TOI_LAUNCH_CHEB
}

}  // namespace toi
