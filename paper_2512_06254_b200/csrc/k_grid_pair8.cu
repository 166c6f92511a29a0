// k_grid_pair8.cu -- step a5, the product gridder (TOI_GRIDDER_SLIDING): sliding register window,
// two columns per lane, window aligned to EVEN cells:
//   grid[iv+dv][iu+du] += f z phi(iu+du-gu) phi(iv+dv-gv),  du, dv = -3..3
// ("place visibilities on a grid"; kernel, support and edge rule: DESIGN.md G9, G10).
//
// k_grid_pair.cu (groups of 4 lanes, lane = two of eight column slots, 8 groups per warp) spends 39 %
// of its instructions in the window-move blocks: with 8 groups per warp, 4 record bodies in 10 take
// one for at least one group.  Here the window is 8 x 8 cells with its top-left corner on EVEN cell
// coordinates, base = (centre - 3) & ~1.  A sample's 7 x 7 footprint starts at offset 0 or 1 in
// that window -- the pre-processing lane places its taps accordingly and pads with a zero -- so
// the window moves only when the base changes, i.e. every TWO cells of travel instead of every
// cell, and then by two rows or columns at once (same instruction count as by one).  All eight
// column slots are live (slot = column mod 8: lane c mod 4, set (c mod 8) / 4), 8 row accumulators
// per slot.  Per record and lane: 2 FMUL2 + 16 FFMA2.  The window may overhang the grid by one
// row / column of zeros: the plan allocates a guard band around the grid for those flushes.
// Pre-processing: all 32 lanes turn 32 samples (4 consecutive channels of each of the 8 strips) into
// 80-byte shared-memory records; raw inputs (and, with a density map, the cell and its density
// value) are requested one batch ahead.  Accumulator writes inside the window-move blocks are
// predicated on a predicate ptxas cannot see through (`pad == 0`), which keeps it from renaming the
// accumulators and paying 10 MOVs per record on the fast path.

#include "grid_window.cuh"


namespace toi {
namespace {

// The task queue: rows [0, j1) are cut into tasks of 8 strips of strip1 channels, the remaining rows
// into tasks of 8 strips of strip2 (about half as long).  Tasks are claimed in ascending order, so
// the kernel's last ~fifth of work comes in small pieces: warps then finish within half a small
// task of one another instead of half a large one (the tail was 7 % of the warp-time, ncu
// sm__warps_active 14.9 of 16), at the price of one more window flush per strip there.
struct TaskShape {
    int strip1, tpr1, strip2, tpr2;
    unsigned t1, j1, n_tasks;       // tasks of the first kind, rows they cover, all tasks
};

// An atomic add (inline PTX included) is compiled by ptxas into its warp-aggregated form: elect a lane,
// add the population count, broadcast the result with a shuffle -- which waits for the atomic's round
// trip to L2 on the spot (2 % of the kernel's warp time).  atom.inc with a bound no task count reaches
// is not rewritten: its result stays in flight until the next task needs it.
__device__ __forceinline__ unsigned claim_task(unsigned *counter)
{
    unsigned t;
    asm volatile("atom.global.inc.u32 %0, [%1], 0x7fffffff;" : "=r"(t) : "l"(counter) : "memory");
    return t;
}

constexpr int kWarps = 8;         // warps per CTA
constexpr int ctas_per_sm(bool) { return 2; }          // 16 warps/SM at <= 128 registers (4 x 4 warps measured 1 % slower)


// CHEB: one Chebyshev-moment pass of the near-coplanar mode (struct ChebArgs): only the samples of
// slab cheb.p contribute, each multiplied by T_k(s_q); never combined with PIPE (the current sample's
// channel scale is needed for r3).
template <int MODE, int OPT, bool PIPE, bool CHEB>
__global__ void __launch_bounds__(kWarps * 32, ctas_per_sm(PIPE))
k_grid_pair8(Geometry g, Inputs in, SnapState *__restrict__ st, const float *__restrict__ D,
            float2 *__restrict__ grid, uint8_t *__restrict__ tiles, TaskShape shape, ChebArgs cheb)
{
    static_assert(!(PIPE && CHEB), "the Chebyshev pass computes the cell in place");
    __shared__ uint4 s_rec[kWarps * kWarpQuads];
    for (int i = threadIdx.x; i < kWarps * kWarpQuads; i += kWarps * 32) s_rec[i] = make_uint4(0u, 0u, 0u, 0u);
    __syncthreads();
    pdl_wait();
    pdl_trigger();
    if (st->status != TOI_OK) return;
    const bool has_w = OPT >= 0 ? (OPT & kHasW) != 0 : in.weights != nullptr;
    const bool has_f = OPT >= 0 ? (OPT & kHasF) != 0 : in.flags != nullptr;
    const bool has_d = OPT >= 0 ? (OPT & kHasD) != 0 : D != nullptr;
    const int lane = threadIdx.x & 31;
    uint4 *rec = s_rec + (threadIdx.x >> 5) * kWarpQuads;

    // every lane pre-processes one sample per batch (strip grp, channel pre_k of the batch) AND
    // accumulates: group grp = lane / 4 = strip, L = lane % 4 = its two column slots L and L + 4
    const int grp = lane >> 2, L = lane & 3;
    const int pre_k = L;
    uint4 *my_rec = rec + group_quad(grp) + pre_k * kRecQuads;
    const unsigned rgs = (unsigned)__cvta_generic_to_shared(rec + group_quad(grp));
    const int G = g.G;
    const float2 *const gc = grid + centre_index(0, 0, G);   // cell (0, 0)
    const long long rs = (long long)G * 8;                   // row stride in bytes
    const float *const Dc = has_d ? D + centre_index(0, 0, G) : nullptr;

    double wsum = 0.0;
    unsigned n_grid = 0, n_off = 0, n_flag = 0;
    // Chebyshev passes repeat the samples: Wsum / n_gridded once per slab, the rejects once per snapshot
    const bool count = !CHEB || (cheb.count & 1) != 0, count_rej = !CHEB || (cheb.count & 2) != 0;

    // dynamic task queue; the NEXT task is requested while the current one is processed (the atomic's
    // round trip to L2 was 4 % of the kernel when taken in place)
    unsigned task_ahead = 0;
    if (lane == 0) task_ahead = claim_task(&st->task_counter);
    for (;;) {
        const unsigned task = __shfl_sync(0xffffffffu, task_ahead, 0);
        if (task >= shape.n_tasks) break;
        if (lane == 0) task_ahead = claim_task(&st->task_counter);
        const bool big = task < shape.t1;
        const unsigned t_in = big ? task : task - shape.t1, tpr = (unsigned)(big ? shape.tpr1 : shape.tpr2);
        const int strip_len = big ? shape.strip1 : shape.strip2;
        const int j = (int)((big ? 0u : shape.j1) + t_in / tpr);
        const int c_task = (int)(t_in % tpr) * (kGroups * strip_len);
        const int c_lo = c_task + grp * strip_len + pre_k;        // my channel in batch 0
        const int c_hi = min(c_task + (grp + 1) * strip_len, g.n_c);
        const long long q_row = (long long)j * g.n_c;

        // The task's first loads go out before anything waits: raw inputs of batch 0 (DRAM), channel
        // scales, then the baseline (L2).  Taken one after the other -- baseline, rotation, tile marks,
        // raw inputs -- their latencies added up to 15 % of the kernel's warp time.
        Raw nxt;
        nxt.a = nxt.b = make_float2(0.0f, 0.0f); nxt.wa = nxt.wb = 0.0f; nxt.fl = 0u; nxt.s = 0.0;
        double s_first = 0.0, s_ahead = 0.0;
        auto first_loads = [&]() {
            if (c_lo < c_hi) {
                load_raw<MODE, !PIPE>(g, in, has_w, has_f, q_row + c_lo, c_lo, nxt);
                if (PIPE) {
                    s_first = __ldg(g.s + c_lo);
                    if (c_lo + kBatch < c_hi) s_ahead = __ldg(g.s + c_lo + kBatch);
                }
            }
        };
        if (!CHEB) first_loads();
        __syncwarp();                        // keeps ptxas from hoisting the baseline's loads (and their first use) above these
        double rho1, rho2;
        rotate_baseline(st->V, in.uvw + 3 * j, rho1, rho2);
        const double rho3 = CHEB ? rotate_row3(st->V, in.uvw + 3 * j) : 0.0;
        if (CHEB && tiles != nullptr && !count_rej && cheb.d > 0.0) {
            // r3 = rho3 s_c is monotone along the task's channels (monotone channel scales: the plan passes
            // `tiles` only then), and so is the slab index: a task whose end samples both fall on one side
            // of slab cheb.p holds none of its samples.  (Not in the pass that counts the rejects.)
            const double ra = __dmul_rn(rho3, __ldg(g.s + c_task));
            const double rb = __dmul_rn(rho3, __ldg(g.s + min(c_task + kGroups * strip_len, g.n_c) - 1));
            const int pa = min((int)floor((fmin(ra, rb) - cheb.r3_min) / (2.0 * cheb.d)), cheb.n_slab - 1);
            const int pb = min((int)floor((fmax(ra, rb) - cheb.r3_min) / (2.0 * cheb.d)), cheb.n_slab - 1);
            if (cheb.p < pa || cheb.p > pb) continue;
        }
        if (CHEB) first_loads();

        // Sparse clear (k_clear.cu): mark the tiles my strip's windows can reach.  The samples of a
        // strip lie on a ray, monotone in channel (the plan passes `tiles` only when the channel
        // scales are monotone), so the windows stay inside the box spanned by the strip's two end
        // samples, widened by the 4 cells a window reaches beyond its sample's centre on either side.
        // Plain stores, nothing read back: testing an entry first made every mark a dependent load
        // (5 % of the kernel's warp time waiting for them).
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
                const int x0 = max(min(iu, ju) - 4 + h, 0) / kTileW, x1 = min(max(iu, ju) + 4 + h, G - 1) / kTileW;
                const int y0 = max(min(iv, jv) - 4 + h, 0) / kTileH, y1 = min(max(iv, jv) + 4 + h, G - 1) / kTileH;
                for (int ty = y0; ty <= y1; ++ty)
                    for (int tx = x0; tx <= x1; ++tx) tiles[ty * tpr + tx] = 1;
            }
        }

        // sliding-window state of my group (ckey uniform across its 4 lanes)
        u64 accA[kR], accB[kR];
#pragma unroll
        for (int d = 0; d < kR; ++d) accA[d] = accB[d] = 0ull;
        unsigned ckey = kNoKey;              // closed window; else the packed base cell (bu, bv)
        unsigned tapA = 0u;                  // window column held by my slot L; slot L + 4 holds tapA ^ 4
        unsigned rpa = rgs + 48, rpb = rgs + 48 + 16;        // shared addresses of my two taps in record 0
        float wpart = 0.0f;

        auto locate = [&](double s_c, Cell &cl) {
            int iu, iv;
            sample_cell(rho1, rho2, s_c, g.kappa, iu, iv, cl.xu, cl.xv);
            cl.key = kNoKey;
            cl.sh = 0u;
            cl.dens = 1.0f;
            if (cell_on_grid(iu, iv, G)) {
                const int bu = (iu - kH) & ~1, bv = (iv - kH) & ~1;
                cl.key = cell_key(bu, bv);
                cl.sh = (unsigned)((iu - kH) & 1) | ((unsigned)((iv - kH) & 1) << 1);
                if (has_d) cl.dens = __ldg(Dc + (iv * G + iu));      // |iv G + iu| < G^2 / 2 <= 2^29 (G <= 32768)
            } else {
                cl.xu = cl.xv = 0.0f;          // taps stay finite whatever the coordinates were
                if (count_rej) ++n_off;
            }
        };
        // software pipeline: raw inputs and cell (+ density) of batch b + 1 are requested while
        // batch b is processed; the channel scale s_c runs two batches ahead
        Cell cnxt;
        cnxt.key = kNoKey; cnxt.sh = 0u; cnxt.xu = cnxt.xv = 0.0f; cnxt.dens = 1.0f;
        if (PIPE && c_lo < c_hi) locate(s_first, cnxt);

        for (int b = 0; b < strip_len && c_task + b < g.n_c; b += kBatch) {
            // ---------------- pre-process one sample per lane ----------------
            {
                const int c = c_lo + b;
                const Raw cur = nxt;
                Cell cell = cnxt;
                if (c + kBatch < c_hi && b + kBatch < strip_len) {
                    load_raw<MODE, !PIPE>(g, in, has_w, has_f, q_row + c + kBatch, c + kBatch, nxt);
                    if (PIPE) {
                        locate(s_ahead, cnxt);
                        if (c + 2 * kBatch < c_hi) s_ahead = __ldg(g.s + c + 2 * kBatch);
                    }
                }
                if (!PIPE && c < c_hi) locate(cur.s, cell);
                unsigned key = kNoKey;
                bool valid = false;
                float wI = 0.0f, zx = 0.0f, zy = 0.0f, pv0 = 0.0f;
                if (c < c_hi && cell.key != kNoKey) {
                    // a flagged sample keeps its own cell as key (z = 0, zero taps): it moves the
                    // window exactly as its unflagged neighbours do and never takes the slow path
                    key = cell.key;
                    constexpr unsigned fmask_b = MODE == 2 ? 0x0000ff00u : 0xff000000u;
                    const float wa = (weight_ok(cur.wa) && !(cur.fl & 0x000000ffu)) ? cur.wa : 0.0f;
                    const float wb = (weight_ok(cur.wb) && !(cur.fl & fmask_b)) ? cur.wb : 0.0f;
                    wI = wa + wb;
                    float tk = 1.0f;
                    bool mine = true;
                    if (CHEB && wI > 0.0f) {
                        // Eq. 19: slab of this sample and its position s_q in it (G24); T_k(s_q) by the
                        // three-term recurrence in fp64 (T_k amplifies rounding by ~k^2)
                        const double r3 = __dmul_rn(rho3, cur.s);
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
                    if (!(wI > 0.0f)) {
                        if (count_rej) ++n_flag;
                    } else if (mine) {
                        if (count) ++n_grid;
                        valid = true;
                        // z = w_a Vis_a + w_b Vis_b; a zero-weight hand is skipped (its data may be NaN)
                        if (wa > 0.0f) { zx = wa * cur.a.x; zy = wa * cur.a.y; }
                        if (wb > 0.0f) { zx = fmaf(wb, cur.b.x, zx); zy = fmaf(wb, cur.b.y, zy); }
                        if (CHEB) { zx *= tk; zy *= tk; }
                        float pu[kW], pv[kW];
                        kernel_taps2(cell.xu, cell.xv, pu, pv);
                        // the 7 taps sit at window offset 0 or 1 on each axis; the free end is zero
                        const bool su = (cell.sh & 1u) != 0u, sv = (cell.sh & 2u) != 0u;
                        unsigned wu[kR], wv[kR];
#pragma unroll
                        for (int i = 0; i < kR; ++i) {
                            const float lo_u = i < kW ? pu[i] : 0.0f, hi_u = i > 0 ? pu[i - 1] : 0.0f;
                            const float lo_v = i < kW ? pv[i] : 0.0f, hi_v = i > 0 ? pv[i - 1] : 0.0f;
                            wu[i] = __float_as_uint(su ? hi_u : lo_u);
                            wv[i] = __float_as_uint(sv ? hi_v : lo_v);
                        }
                        pv0 = __uint_as_float(wv[0]);
                        my_rec[1] = make_uint4(wv[1], wv[2], wv[3], wv[4]);
                        my_rec[2] = make_uint4(wv[5], wv[6], wv[7], 0u);
                        my_rec[3] = make_uint4(wu[0], wu[1], wu[2], wu[3]);
                        my_rec[4] = make_uint4(wu[4], wu[5], wu[6], wu[7]);
                    }
                }
                // a record without a sample (flagged, off the grid, padding) keeps the taps its slot held
                // before -- finite: the slots start at zero and only ever hold taps -- and has z = 0
                float f = 1.0f;
                if (has_d) {
                    // the density of a cell whose samples are all flagged is 0: never invert it
                    const float dens = valid ? cell.dens : 1.0f;
                    asm volatile("rcp.approx.ftz.f32 %0, %1;" : "=f"(f) : "f"(dens));
                }
                if (!CHEB || (count && valid)) wpart = fmaf(f, wI, wpart);
                my_rec[0] = make_uint4(__float_as_uint(zx * f), __float_as_uint(zy * f), key, __float_as_uint(pv0));
            }
            __syncwarp();
            // ---------------- accumulate: every group consumes its 4 records ----------------
            consume_batch(accA, accB, tapA, ckey, rpa, rpb, rgs, gc, (unsigned)rs, G, L);
            __syncwarp();
        }
        // strip done: flush what is left of the window
        if (ckey != kNoKey) flush_sets(accA, accB, tapA, ckey, gc, rs, G);
        wsum += (double)wpart;
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

template <int MODE>
void launch_mode(int opt, dim3 grid, dim3 block, cudaStream_t stream, const Geometry &g, const Inputs &in,
                 SnapState *st, const float *D, float2 *d_grid, uint8_t *tiles, const TaskShape &shape)
{
#define TOI_LAUNCH(O, P) launch_pdl(k_grid_pair8<MODE, O, P, false>, grid, block, 0, stream, g, in, st, D, d_grid, tiles, shape, ChebArgs())
    switch (opt) {
    case kHasW | kHasF | kHasD: TOI_LAUNCH(kHasW | kHasF | kHasD, true); break;
    case kHasW | kHasF: TOI_LAUNCH(kHasW | kHasF, false); break;
    case kHasD: TOI_LAUNCH(kHasD, true); break;
    case 0: TOI_LAUNCH(0, false); break;
    default:
        if (D) TOI_LAUNCH(-1, true); else TOI_LAUNCH(-1, false);
        break;
    }
#undef TOI_LAUNCH
}

}  // namespace

namespace {

// strip length (channels per group per task): 8 strips per task; aim at >= 6 tasks per resident
// warp, within [16, 128] channels and a multiple of the 4-sample batch; the last fifth of the rows
// gets strips of about half that length (struct TaskShape)
TaskShape task_shape(const Geometry &g, int n_sms, int ctas_per_sm_, long long *ctas)
{
    TaskShape sh;
    const long long warps = (long long)ctas_per_sm_ * n_sms * kWarps;
    const long long want = ((long long)g.n_b * g.n_c) / (kGroups * 6 * warps);
    sh.strip1 = pick_strip(g.n_c, kGroups, kBatch, want, 16, 128);
    sh.tpr1 = (g.n_c + kGroups * sh.strip1 - 1) / (kGroups * sh.strip1);
    sh.strip2 = pick_strip(g.n_c, kGroups, kBatch, sh.strip1 / 2, 16, 128);
    sh.tpr2 = (g.n_c + kGroups * sh.strip2 - 1) / (kGroups * sh.strip2);
    sh.j1 = sh.strip2 < sh.strip1 ? (unsigned)(g.n_b - g.n_b / 5) : (unsigned)g.n_b;
    sh.t1 = sh.j1 * (unsigned)sh.tpr1;
    const long long n_tasks = (long long)sh.t1 + (long long)(g.n_b - (int)sh.j1) * sh.tpr2;
    sh.n_tasks = (unsigned)n_tasks;
    *ctas = (n_tasks + kWarps - 1) / kWarps;
    if (*ctas > (long long)ctas_per_sm_ * n_sms) *ctas = (long long)ctas_per_sm_ * n_sms;   // persistent CTAs pull from the queue
    return sh;
}

}  // namespace

// G <= 32768 (toi_plan_create checks): a window base must fit the packed 16-bit key.
void launch_grid_pair8(const Geometry &g, const Inputs &in, SnapState *st, const float *d_density,
                       float2 *d_grid, uint8_t *tiles, int n_sms, cudaStream_t stream)
{
    long long ctas = 0;
    const TaskShape shape = task_shape(g, n_sms, ctas_per_sm(d_density != nullptr), &ctas);
    const dim3 grid((unsigned)ctas), block(kWarps * 32);
    const uintptr_t aw = (uintptr_t)in.weights, af = (uintptr_t)in.flags, av = (uintptr_t)in.vis;
    const int opt = (in.weights ? kHasW : 0) | (in.flags ? kHasF : 0) | (d_density ? kHasD : 0);
    if (g.n_p == 4 && g.pol_a == 0 && g.pol_b == 3 && (aw & 15) == 0 && (af & 3) == 0)
        launch_mode<4>(opt, grid, block, stream, g, in, st, d_density, d_grid, tiles, shape);
    else if (g.n_p == 2 && g.pol_a == 0 && g.pol_b == 1 && (av & 15) == 0 && (aw & 7) == 0 && (af & 1) == 0)
        launch_mode<2>(opt, grid, block, stream, g, in, st, d_density, d_grid, tiles, shape);
    else
        launch_mode<0>(-1, grid, block, stream, g, in, st, d_density, d_grid, tiles, shape);
}

// One Chebyshev-moment pass of the near-coplanar mode.
void launch_grid_pair8_cheb(const Geometry &g, const Inputs &in, SnapState *st, const float *d_density,
                            float2 *d_grid, uint8_t *tiles, int n_sms, const ChebArgs &cheb, cudaStream_t stream)
{
    long long ctas = 0;
    const TaskShape shape = task_shape(g, n_sms, ctas_per_sm(false), &ctas);
    const dim3 grid((unsigned)ctas), block(kWarps * 32);
    const uintptr_t aw = (uintptr_t)in.weights, af = (uintptr_t)in.flags, av = (uintptr_t)in.vis;
#define TOI_LAUNCH_CHEB(M) launch_pdl(k_grid_pair8<M, -1, false, true>, grid, block, 0, stream, g, in, st, d_density, d_grid, tiles, shape, cheb)
    if (g.n_p == 4 && g.pol_a == 0 && g.pol_b == 3 && (aw & 15) == 0 && (af & 3) == 0)
        TOI_LAUNCH_CHEB(4);
    else if (g.n_p == 2 && g.pol_a == 0 && g.pol_b == 1 && (av & 15) == 0 && (aw & 7) == 0 && (af & 1) == 0)
        TOI_LAUNCH_CHEB(2);
    else
        TOI_LAUNCH_CHEB(0);
#undef TOI_LAUNCH_CHEB
}

}  // namespace toi
