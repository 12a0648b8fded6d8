// debye_aux.cuh -- setup (S0/S1), pack (S0) and final+epilogue (S7) kernels of libdebye.
#pragma once
#include <cuda_runtime.h>
#include <cstdint>
#include <cmath>
#include "debye_plan.cuh"
#include "debye_pairs.cuh"

namespace debye {

#define DEBYE_SETUP_THREADS 1024
#define DEBYE_SETUP_MAXQ 4096

// S0 + S1.  One CTA: type histogram, segment offsets, stable counting-sort permutation, q-grid analysis and the
// unit prefix per type pair.  Stable = atoms of one type keep their input order, so the sorted layout (and with
// it every rounding in the pair sums) is a pure function of the input.
// perm[p] = original index of the atom at sorted position p.
// Sort: warp w owns the contiguous chunk [w C, (w+1) C) of the atoms, C a multiple of 32.  Pass 1 counts types per warp
// (one __match_any_sync per 32 atoms, no atomics: only warp w touches wcnt[w]); a 32 x 32 prefix gives every
// (warp, type) its first output slot; pass 2 walks the chunk again and places the atoms.  Two block barriers in total.
// If pack_here != 0 the CTA also gathers the coordinates (small N x B: saves the pack launch).
__global__ void __launch_bounds__(DEBYE_SETUP_THREADS) debye_setup_kernel(DevPlan *plan, const int32_t *__restrict__ type, const float *__restrict__ q,
                                                                            int32_t *__restrict__ perm, int N, int T, int M, int B, int alt_offered /* a recurrence launch sized for M - 1 indices exists */,
                                                                            int hint_class /* -3: no hint; -4: piecewise uniform (hint_pieces); else the grid class the caller promised (debye_grid_class) */,
                                                                            int hint_pieces /* hint_class == -4: (number of pieces << 8) | K / 8 as debye_find_pieces gives them; hint_class == -3:
                                                                                               the centred-form launch on offer for a uniform grid with a general start, 0 if none */,
                                                                            const float *__restrict__ xyz, float4 *__restrict__ sorted, int pack_here, const float *__restrict__ weight,
                                                                            int shard_rank, int shard_world)
{
    pdl_trigger();                         // first kernel of the call: lets the next grid be staged (it waits for our completion)
    constexpr int NWARP = DEBYE_SETUP_THREADS / 32;
    constexpr int SORT_UNROLL = 8;
    __shared__ int wcnt[NWARP][DEBYE_MAX_TYPES_I];      // pass 1: atoms of type t in warp w's chunk; pass 2: running output slot
    __shared__ int seg[DEBYE_MAX_TYPES_I + 1];
    __shared__ float red[NWARP], red2[NWARP], qmax_s[NWARP];
    __shared__ int hint_bad_s, s_cls, s_runs_ok, s_nruns;
    __shared__ int32_t s_run_start[DEBYE_MAX_PIECES + 1];
    __shared__ float q_sh[DEBYE_SETUP_MAXQ];            // q, for the piece finding (DEBYE_MAX_Q of include/debye.h)
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int chunk = ((N + NWARP - 1) / NWARP + 31) / 32 * 32;
    const int c0 = warp * chunk, c1 = min(N, c0 + chunk);
    wcnt[warp][lane] = 0;
    __syncwarp();
    for (int s0 = c0; s0 < c1; s0 += 32 * SORT_UNROLL) {
        int tt[SORT_UNROLL];
#pragma unroll
        for (int x = 0; x < SORT_UNROLL; ++x) { const int i = s0 + 32 * x + lane; tt[x] = (i < c1) ? type[i] : -1; }   // loads in flight together
        // the SORT_UNROLL rankings first (independent of one another: pipelined), then the dependent counter updates
        unsigned pm[SORT_UNROLL];
#pragma unroll
        for (int x = 0; x < SORT_UNROLL; ++x) pm[x] = __match_any_sync(0xffffffffu, tt[x]);
#pragma unroll
        for (int x = 0; x < SORT_UNROLL; ++x) {
            const int t = tt[x];
            if (t >= 0 && (pm[x] & ((1u << lane) - 1)) == 0) wcnt[warp][t] += __popc(pm[x]);
            __syncwarp();
        }
    }
    // ---- q grid analysis (independent of the sort; its reduction shares the barriers below) ---------------------------
    const double q0 = (double)q[0];
    const double dq = debye_grid_dq(q0, (double)q[M - 1], M);
    float dev = 0.f, qsm = 3.0e38f, qmax = 0.f;
    for (int k = tid; k < M; k += blockDim.x) {
        const double qk = (double)q[k];
        dev = fmaxf(dev, debye_grid_dev(qk, k, q0, dq));
        const float aq = fabsf((float)qk);
        if (aq > 0.f) qsm = fminf(qsm, aq);
        qmax = fmaxf(qmax, aq);
    }
    for (int o = 16; o > 0; o >>= 1) { dev = fmaxf(dev, __shfl_xor_sync(0xffffffffu, dev, o)); qsm = fminf(qsm, __shfl_xor_sync(0xffffffffu, qsm, o)); qmax = fmaxf(qmax, __shfl_xor_sync(0xffffffffu, qmax, o)); }
    if (lane == 0) { red[warp] = dev; red2[warp] = qsm; qmax_s[warp] = qmax; }
    __syncthreads();
    // ---- type totals and segment offsets (warp 0: lane t owns type t), plan header, q verdict (thread 32) --------------
    if (warp == 0) {
        int tot = 0;
        for (int w = 0; w < NWARP; ++w) tot += wcnt[w][lane];
        if (lane >= T) tot = 0;
        int incl = tot;
        for (int o = 1; o < 32; o <<= 1) { int v = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += v; }
        seg[lane] = incl - tot;
        if (lane == 31) seg[32] = incl;
        plan->seg_off[lane] = incl - tot;
        plan->n_a[lane] = tot;
        if (lane == 31) plan->seg_off[32] = incl;
    }
    float d = 0.f, s = 3.0e38f, mx = 0.f;          // thread 32: the grid's deviation from the line, smallest non-zero |q|, largest |q|
    int cls = -2;
    if (tid == 32) {
        for (int w = 0; w < NWARP; ++w) { d = fmaxf(d, red[w]); s = fminf(s, red2[w]); mx = fmaxf(mx, qmax_s[w]); }
        cls = debye_grid_class(q0, dq, d, mx);
        s_cls = cls;
    }
    __syncthreads();
    // Piecewise-uniform grid (the centred product form, V_CENT): promised by the hint, or -- no hint -- a uniform grid with a general
    // start for which a centred launch is on offer.  The same segmentation as the host's (debye_plan.cuh), from a copy of q in
    // shared memory: runs by one thread, the 1.5-ulp test of every point by all threads, pieces by one thread; it has to give the
    // piece count and accumulator count the launch was sized for.  (A serial scan of global memory took 0.5 ms for 2000 points.)
    // ... or a grid from 0 or dq with more than 256 chain indices (more than two chunks: the recurrence would run its chain form).
    const bool need_pieces = hint_class == -4 || (hint_class == -3 && hint_pieces != 0 && (s_cls == -1 || (s_cls >= 0 && M - (s_cls == 0 ? 1 : 0) > 256)));
    bool pieces_ok = false;
    if (need_pieces) {
        for (int k = tid; k < M; k += blockDim.x) q_sh[k] = q[k];
        __syncthreads();
        if (tid == 32) s_runs_ok = debye_find_runs(q_sh, M, s_run_start, s_nruns) ? 1 : 0;
        __syncthreads();
        int ok = s_runs_ok;
        if (ok) {
            for (int k = tid; k < M; k += blockDim.x) {
                int r = 0;
                while (s_run_start[r + 1] <= k) ++r;
                if (!debye_run_point_ok(q_sh, s_run_start[r], s_run_start[r + 1], k)) ok = 0;
            }
        }
        ok = __syncthreads_and(ok);
        if (tid == 32)
            pieces_ok = ok && debye_pieces_from_runs(q_sh, s_run_start, s_nruns, plan->pieces) && plan->pieces.n == (hint_pieces >> 8) &&
                        plan->pieces.K == 8 * (hint_pieces & 255);
    }
    if (tid == 32) {
        const int uni = cls != -2;
        // zero start: q0 == 0 exactly (koff = 0) or q0 == dq to 1e-6 (koff = 1, the paper's own grid q_k = k dq, k >= 1)
        const int koff = cls >= 0 ? cls : -1;
        hint_bad_s = (hint_class != -3 && hint_class != cls) ? 1 : 0;
        if (!pieces_ok) plan->pieces.n = 0;
        if (hint_class == -4) hint_bad_s = pieces_ok ? 0 : 1;
        plan->hint_bad = hint_bad_s;
        plan->recur_alt = (koff == 0 && alt_offered) ? 1 : 0;
        plan->N = N; plan->T = T; plan->M = M; plan->B = B; plan->n_tp = T * (T + 1) / 2;
        plan->weighted = weight ? 1 : 0;
        plan->shard_rank = shard_rank; plan->shard_world = shard_world;
        plan->uniform = uni;
        plan->zero_start = koff;
        plan->q0 = q0;
        plan->dq = dq;
        plan->q_small = (s < 3.0e38f) ? s : 0.f;
        int va = (hint_class == -4) ? V_CENT : (uni ? V_RECUR : V_MUFU);
        // no hint, uniform grid with a general start: the centred product form if the launch on offer fits its pieces (it does:
        // one run of M points is cut into equal pieces, which the host derived from M), else the chain form
        if (hint_class == -3 && pieces_ok) va = V_CENT;
        plan->variant_auto = va;
    }
    __syncthreads();
    // ---- unit prefix per type pair (thread 0, n_tp <= 528 steps) while the other warps sort -----------------------------
    if (tid == 0) {
        // units per type pair; the side with less padding waste becomes the row (i) side
        int64_t pre = 0;
        int tp = 0;
        for (int a = 0; a < T; ++a)
            for (int b2 = a; b2 < T; ++b2, ++tp) {
                const int na = seg[a + 1] - seg[a], nb = seg[b2 + 1] - seg[b2];
                int64_t units;
                int ti = a, tj = b2;
                if (a == b2) {
                    const int rows = debye_diag_rows(na);
                    units = rows > 0 ? debye_diag_row_prefix(na, rows) : 0;
                } else {
                    const int64_t ra = (na + DEBYE_IB - 1) / DEBYE_IB, rb = (nb + DEBYE_IB - 1) / DEBYE_IB;
                    const int64_t ua = ra * nb, ub = rb * na;          // rows x j atoms
                    if (ub < ua) { ti = b2; tj = a; units = ub; } else units = ua;
                    if (na == 0 || nb == 0) units = 0;
                }
                plan->tp_ti[tp] = ti; plan->tp_tj[tp] = tj; plan->tp_prefix[tp] = pre;
                pre += units;
            }
        plan->tp_prefix[tp] = pre;
        // a wrong grid hint leaves no work: the pairs kernels return at once and the final kernel writes NaN
        plan->U1 = hint_bad_s ? 0 : pre;
    }
    // first output slot of (warp, type): exclusive prefix over the warps, per type (thread (w, t) = (warp, lane))
    int first = seg[lane];
    for (int w = 0; w < warp; ++w) first += wcnt[w][lane];
    __syncthreads();
    wcnt[warp][lane] = first;
    __syncwarp();
    // One structure packed here: the thread that places atom i also moves its coordinates (loaded together with the type labels,
    // coalesced in i, their latency under the ranking) -- no second pass through perm (the gather took 4 of the kernel's ~13 us
    // at 10 000 atoms: three batches of two dependent global loads).
    const bool fuse_pack = pack_here && B == 1;
    for (int s0 = c0; s0 < c1; s0 += 32 * SORT_UNROLL) {
        int tt[SORT_UNROLL];
        float cx[SORT_UNROLL][4];
#pragma unroll
        for (int x = 0; x < SORT_UNROLL; ++x) { const int i = s0 + 32 * x + lane; tt[x] = (i < c1) ? type[i] : -1; }
        if (fuse_pack) {
#pragma unroll
            for (int x = 0; x < SORT_UNROLL; ++x) {
                const int i = s0 + 32 * x + lane;
                if (i < c1) { const float *sx = xyz + (int64_t)i * 3; cx[x][0] = sx[0]; cx[x][1] = sx[1]; cx[x][2] = sx[2]; cx[x][3] = weight ? weight[i] : 1.0f; }
                else { cx[x][0] = cx[x][1] = cx[x][2] = cx[x][3] = 0.f; }
            }
        }
        unsigned pm[SORT_UNROLL];
#pragma unroll
        for (int x = 0; x < SORT_UNROLL; ++x) pm[x] = __match_any_sync(0xffffffffu, tt[x]);
#pragma unroll
        for (int x = 0; x < SORT_UNROLL; ++x) {
            const int t = tt[x];
            const unsigned peers = pm[x];
            const int rank = __popc(peers & ((1u << lane) - 1));
            if (t >= 0) {
                const int slot = wcnt[warp][t] + rank;
                perm[slot] = s0 + 32 * x + lane;
                if (fuse_pack) sorted[slot] = make_float4(cx[x][0], cx[x][1], cx[x][2], cx[x][3]);
            }
            __syncwarp();
            if (t >= 0 && rank == 0) wcnt[warp][t] += __popc(peers);
            __syncwarp();
        }
    }
    if (pack_here && !fuse_pack) {
        __syncthreads();                       // perm was written by this CTA: visible after the barrier
        const int total = N * B;                 // <= DEBYE_PACK_IN_SETUP
#pragma unroll 4
        for (int g = tid; g < total; g += DEBYE_SETUP_THREADS) {
            const int b = g / N, p = g - b * N;
            const int i = perm[p];
            const float *sx = xyz + ((int64_t)b * N + i) * 3;
            sorted[g] = make_float4(sx[0], sx[1], sx[2], weight ? weight[i] : 1.0f);
        }
    }
}

// S0: gather coordinates into type-sorted float4 (x, y, z, w_j), all conformers; w_j = 1 without weights (the kernels never
// need the type of an atom: tiles are type-homogeneous).
__global__ void debye_pack_kernel(const DevPlan *__restrict__ plan, const float *__restrict__ xyz, const int32_t *__restrict__ type, const int32_t *__restrict__ perm,
                                  float4 *__restrict__ sorted, int N, int B, const float *__restrict__ weight)
{
    pdl_wait();
    pdl_trigger();
    const int64_t total = (int64_t)N * B;
    for (int64_t g = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; g < total; g += (int64_t)gridDim.x * blockDim.x) {
        const int b = (int)(g / N), p = (int)(g % N);
        const int i = perm[p];
        const float *s = xyz + ((int64_t)b * N + i) * 3;
        sorted[g] = make_float4(s[0], s[1], s[2], weight ? weight[i] : 1.0f);
    }
}

// Weighted calls only: per type, sum of w_j and of w_j^2 in FP64 in a fixed order (one warp per type: lane-strided partial
// sums over the type's segment of the sorted array, then an xor-shuffle tree).  Grid = T blocks of 32 threads.
__global__ void debye_weight_sums_kernel(DevPlan *plan, const float4 *__restrict__ sorted)
{
    pdl_wait();
    const int t = blockIdx.x, lane = threadIdx.x;
    const int lo = plan->seg_off[t], hi = plan->seg_off[t + 1];
    double s1 = 0.0, s2 = 0.0;
    for (int i = lo + lane; i < hi; i += 32) { const double w = (double)sorted[i].w; s1 += w; s2 += w * w; }
    for (int o = 16; o > 0; o >>= 1) { s1 += __shfl_xor_sync(0xffffffffu, s1, o); s2 += __shfl_xor_sync(0xffffffffu, s2, o); }
    if (lane == 0) { plan->sw[t] = s1; plan->sw2[t] = s2; }
}

// number of unordered pairs of type pair (a, b)
__device__ __forceinline__ double pair_count(int na, int nb, bool diag) { return diag ? 0.5 * (double)na * (double)(na - 1) : (double)na * (double)nb; }

// S7 in two launches.
// (a) debye_reduce_kernel: fixed-order FP64 sum of the per-CTA records of every (conformer, type pair, q-chunk) X:
//         sums[X][l] = sum over the CTAs c that worked on X, in CTA order, of records[(c + X) K + l].
//     Block = (X, group of 32 slots); thread (lane, sl) adds the sl-th of NS equal slices of the CTA range for slot
//     32 g + lane (coalesced over the slots); the slices are then added in slice order.  The slicing is a fixed function
//     of (U, G), so every order is fixed and the result is bitwise reproducible.
// (b) debye_epilogue_kernel: per output q_k and type pair the slot (chunk, l) of the sum -- or, for the product form of
//     the recurrence, the telescoped chain of slots  B_{Sj+k0} = Out[j][k0] + B_{Sj-k0}  (debye_pairs.cuh) -- then
//         I(q_k) = sum_a n_a F_a^2 + 2 sum_{a<=b} F_a F_b S_ab(q_k),  S_ab = (1/q_k) sum sin(q_k r)/r  (q_k != 0), #pairs (q_k == 0).
//     Block = (conformer, tile of 8 q indices); thread (kk, g) handles q index k0 + kk and the type pairs g, g + 32, ...
//     in increasing order; the partial sums are added in g order.  mode 0: write I_out[b][k]; mode 1: S_out[b][tp][k].
#define DEBYE_RED_NS 8
#define DEBYE_RED_THREADS (32 * DEBYE_RED_NS)
#define DEBYE_FINAL_Q 8
#define DEBYE_FINAL_G 32
#define DEBYE_FINAL_THREADS (DEBYE_FINAL_Q * DEBYE_FINAL_G)
struct FinalSet { int variant, K, n_chunks, G, alt_gate; };   // parameters of one pairs launch (alt_gate as in the pairs kernel)
struct FinalSets { FinalSet s[4]; int n; };                    // up to: recurrence (M - 1 indices), recurrence, centred, MUFU
// which pairs launch did the work: the same device-side decisions the pairs kernels took
__device__ __forceinline__ int final_pick(const DevPlan *plan, const FinalSets &sets, int is_auto)
{
    for (int i = 0; i < sets.n; ++i) {
        const FinalSet &c = sets.s[i];
        if ((!is_auto || plan->variant_auto == c.variant) && (c.alt_gate < 0 || plan->recur_alt == c.alt_gate)) return i;
    }
    return 0;
}
__global__ void __launch_bounds__(DEBYE_RED_THREADS) debye_reduce_kernel(const DevPlan *__restrict__ plan, const double *__restrict__ records,
                                                                           double *__restrict__ sums, int is_auto, const FinalSets sets)
{
    __shared__ double part[DEBYE_RED_NS][32];
    pdl_wait();
    pdl_trigger();
    const int pick = final_pick(plan, sets, is_auto);
    const int K = sets.s[pick].K, n_chunks = sets.s[pick].n_chunks, G = sets.s[pick].G;
    const int Bn = plan->B, n_tp = plan->n_tp;
    const int groups = (K + 31) / 32;
    const int64_t nX = (int64_t)Bn * n_tp * n_chunks;
    if ((int64_t)blockIdx.x >= nX * groups) return;             // the grid is sized for the largest of the offered launches
    const int64_t X = blockIdx.x / groups;
    const int lane = threadIdx.x & 31, sl = threadIdx.x >> 5;
    const int l = (int)(blockIdx.x % groups) * 32 + lane;
    const int ch = (int)(X % n_chunks), tp = (int)((X / n_chunks) % n_tp), b = (int)(X / ((int64_t)n_chunks * n_tp));
    const int64_t U1 = plan->U1, Uc = U1 * n_chunks, U = Uc * Bn;
    const int64_t units = plan->tp_prefix[tp + 1] - plan->tp_prefix[tp];
    double s = 0.0;
    if (l < K && units > 0 && U > 0) {
        const DebyeRanges ranges(U, G);
        const int64_t ub = (int64_t)b * Uc + plan->tp_prefix[tp] * n_chunks + (int64_t)ch * units;
        const int64_t ue = ub + units - 1;
        if (U >= G) {           // every CTA owns at least one unit: all CTAs between the owners took part
            const int c_lo = ranges.owner(ub), c_hi = ranges.owner(ue);
            const int n = c_hi - c_lo + 1, per = (n + DEBYE_RED_NS - 1) / DEBYE_RED_NS;
            const int cb = c_lo + sl * per, ce = min(c_hi + 1, cb + per);
            const double *rp = records + ((int64_t)cb + X) * K + l;
            int c = cb;
            for (; c + 4 <= ce; c += 4, rp += 4 * (int64_t)K) {
                const double r0 = rp[0], r1 = rp[K], r2 = rp[2 * (int64_t)K], r3 = rp[3 * (int64_t)K];
                s += r0; s += r1; s += r2; s += r3;
            }
            for (; c < ce; ++c, rp += K) s += rp[0];
        } else if (sl == 0) {   // fewer units than CTAs: each unit has its own CTA
            for (int64_t u = ub; u <= ue; ++u) s += records[((int64_t)ranges.owner(u) + X) * K + l];
        }
    }
    part[sl][lane] = s;
    __syncthreads();
    if (sl == 0 && l < K) {
        double tot = 0.0;
#pragma unroll
        for (int x = 0; x < DEBYE_RED_NS; ++x) tot += part[x][lane];
        sums[X * K + l] = tot;
    }
}

__global__ void __launch_bounds__(DEBYE_FINAL_THREADS) debye_epilogue_kernel(const DevPlan *__restrict__ plan, const double *__restrict__ sums,
                                                                               const float *__restrict__ fftab, const float *__restrict__ q, double *__restrict__ out,
                                                                               int is_auto, const FinalSets sets, int mode)
{
    __shared__ double part[DEBYE_FINAL_G][DEBYE_FINAL_Q];
    pdl_wait();
    const int M = plan->M, T = plan->T, n_tp = plan->n_tp;
    const int ktiles = (M + DEBYE_FINAL_Q - 1) / DEBYE_FINAL_Q;
    const int kk = threadIdx.x % DEBYE_FINAL_Q, g = threadIdx.x / DEBYE_FINAL_Q;
    const int b = blockIdx.x / ktiles, k = (blockIdx.x % ktiles) * DEBYE_FINAL_Q + kk;
    const int pick = final_pick(plan, sets, is_auto);
    const int variant = sets.s[pick].variant, K = sets.s[pick].K, n_chunks = sets.s[pick].n_chunks;
    const bool bad = (variant == V_RECUR && !plan->uniform) || plan->hint_bad;   // forced recurrence on a non-uniform grid, or a wrong grid hint -> NaN
    const double nan = __longlong_as_double(0x7ff8000000000000LL);
    const double scale = (variant == V_RECUR) ? 0.5 : 1.0;            // the recurrence kernel accumulates 2 sin(q r)/r
    // centred product form: piece of output k and its local index (pieces are in increasing k)
    int piece = 0, mloc = 0;
    if (variant == V_CENT && !bad && k < M) {
        const int np = plan->pieces.n;
        while (piece + 1 < np && plan->pieces.off[piece + 1] <= k) ++piece;
        mloc = k - plan->pieces.off[piece];
    }
    // recurrence on a grid (k + koff) dq with at most 2 chunks ran in product form (the same test as in the pairs kernel)
    const bool product = variant == V_RECUR && plan->zero_start >= 0 && n_chunks <= 2;
    double I = 0.0;
    if (k < M) {
        // chain / grid index of output k (convention at slot_of); -1 only for q = 0, which never reads a sum
        const int idx = product ? k + plan->zero_start - 1 : k;
        const double qk = (double)q[k];
        // type pair index -> (a, b2): walk rows of the upper triangle
        int a = 0, rowstart = 0;
        for (int tp = g; tp < n_tp; tp += DEBYE_FINAL_G) {
            while (tp >= rowstart + (T - a)) { rowstart += T - a; ++a; }
            const int b2 = a + (tp - rowstart);
            double S;
            const int64_t units = plan->tp_prefix[tp + 1] - plan->tp_prefix[tp];
            if (bad) S = nan;
            else if (qk == 0.0 || units == 0) {
                // sum over the pairs of w_i w_j sinc(0): the pair count, or with weights sw_a sw_b resp. (sw_a^2 - sw2_a) / 2
                double cnt = pair_count(plan->n_a[a], plan->n_a[b2], a == b2);
                if (plan->weighted && units != 0) cnt = (a == b2) ? 0.5 * (plan->sw[a] * plan->sw[a] - plan->sw2[a]) : plan->sw[a] * plan->sw[b2];
                // tile split over GPUs: the closed-form terms are nobody's tile, rank 0 contributes them
                S = (plan->shard_rank == 0) ? cnt : 0.0;
            }
            else {
                const double *sp = sums + ((int64_t)b * n_tp + tp) * n_chunks * (int64_t)K;
                double s = 0.0;
                if (variant == V_CENT) {
                    // sum_pairs sin(q r)/r = scale (P + sgn Q), resp. scale x the level-0 slot (debye_pairs.cuh cent_slot_of)
                    int lp, lq; double sgn, sc;
                    cent_slot_of(K, mloc, lp, lq, sgn, sc);
                    const double *pp = sp + (int64_t)piece * K;
                    s = sc * (lq >= 0 ? pp[lp] + sgn * pp[lq] : pp[lp]);
                } else if (product) {
                    // kappa = idx + 1 = S j + kres with kres in 1..S:  B_kappa = Out[slot(kappa)] + B_{S j - kres}
                    const int Sres = 8 * n_chunks;
                    for (int kap = idx + 1; kap > 0;) {
                        const int j = (kap - 1) / Sres, kres = kap - Sres * j;
                        s += sp[(int64_t)((kres - 1) >> 3) * K + 8 * j + ((kres - 1) & 7)];
                        kap = Sres * j - kres;
                    }
                } else {
                    int ch = 0, l = 0;
                    slot_of(variant, K, n_chunks, idx, ch, l);
                    s = sp[(int64_t)ch * K + l];
                }
                S = scale * s / qk;
            }
            if (mode == 0) I += 2.0 * (double)fftab[a * M + k] * (double)fftab[b2 * M + k] * S;
            else out[((int64_t)b * n_tp + tp) * M + k] = S;
        }
    }
    if (mode != 0) return;
    part[g][kk] = I;
    __syncthreads();
    if (g == 0 && k < M) {
        double tot = 0.0;
        for (int a = 0; a < T; ++a) { const double fa = (double)fftab[a * M + k]; tot += (plan->weighted ? plan->sw2[a] : (double)plan->n_a[a]) * fa * fa; }
#pragma unroll
        for (int x = 0; x < DEBYE_FINAL_G; ++x) tot += part[x][kk];
        out[(int64_t)b * M + k] = tot;
    }
}

// Tile split of one structure over GPUs, the step after the exchange: S_parts[p][b][tp][k] are the partial
// structure factors of n_parts ranks (debye_partials_shard, gathered into one buffer).  One thread per (conformer, q index):
// S_ab = sum over parts in part order (fixed order: bitwise reproducible for a given number of ranks), then the same
// epilogue as debye_final_kernel, I = sum_a n_a F_a^2 + 2 sum_{a<=b} F_a F_b S_ab with type pairs in increasing order.
__global__ void __launch_bounds__(128) debye_combine_kernel(const double *__restrict__ S_parts, int n_parts, const int32_t *__restrict__ n_a,
                                                              const float *__restrict__ fftab, int B, int T, int M, double *__restrict__ out)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x, b = blockIdx.y;
    if (k >= M) return;
    const int n_tp = T * (T + 1) / 2;
    const int64_t part_stride = (int64_t)B * n_tp * M;
    double tot = 0.0;
    for (int a = 0; a < T; ++a) { const double fa = (double)fftab[a * M + k]; tot += (double)n_a[a] * fa * fa; }
    int tp = 0;
    for (int a = 0; a < T; ++a) {
        const double fa = (double)fftab[a * M + k];
        for (int b2 = a; b2 < T; ++b2, ++tp) {
            const double *sp = S_parts + ((int64_t)b * n_tp + tp) * M + k;
            double S = 0.0;
            for (int p = 0; p < n_parts; ++p) S += sp[p * part_stride];
            tot += 2.0 * fa * (double)fftab[b2 * M + k] * S;
        }
    }
    out[(int64_t)b * M + k] = tot;
}

}  // namespace debye
