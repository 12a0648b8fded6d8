// debye_small.cuh -- ONE launch for one small structure (N <= 2048 atoms, T <= 8 types, at most 128 chain indices).
//
// PAPER.md:88 ("N < W ... pN >= W workers, inner loop split p ways"), PAPER.md:25 (a refinement calls the profile 10^5+
// times), PAPER.md:104 (for small proteins the overheads, not the pairs, dominate).  A 1000-atom profile is ~2 us of
// arithmetic; run as setup + pairs + reduce + epilogue it takes four launches and their global-memory latency chains.
// Here every CTA
//   1. sorts the atoms by type in shared memory itself (the same stable counting sort as debye_setup_kernel; every CTA
//      gets the same permutation) and keeps the packed float4 atoms of the WHOLE structure there: no tile staging;
//   2. classifies the q grid (must be the grid the caller's hint promised: q_k = (k + koff) dq, koff in {0, 1});
//   3. runs its share of the unit line (debye_plan.cuh) through the product-form loop (prod_tile, debye_pairs.cuh) and
//      writes one FP64 record per type pair it touched;
//   4. waits at a grid-wide barrier (cooperative launch: the grid is at most one resident wave); then CTA k computes
//      output q_k: one thread per (type pair, element of the telescoped chain) sums that slot's records in CTA order,
//      the chain and the form-factor epilogue follow (what debye_reduce_kernel + debye_epilogue_kernel do).
//      Measured on B200 against a last-CTA-done reduction (ticket counter, one CTA does the whole final stage): 29 us
//      against 33 us per 1000-atom profile; the four-launch general path takes 40 us.
// Fixed unit ranges, fixed-order flush, records summed in CTA order: bitwise reproducible.
#pragma once
#include <cuda_runtime.h>
#include <cstdint>
#include <cstdio>
#include <cooperative_groups.h>
#include "debye_plan.cuh"
#include "debye_pairs.cuh"

namespace debye {

#define DEBYE_SMALL_NMAX 2048
#define DEBYE_SMALL_TMAX 8
#define DEBYE_SMALL_TP (DEBYE_SMALL_TMAX * (DEBYE_SMALL_TMAX + 1) / 2)
#define DEBYE_KMAX_LEVELS 17      // chain elements of one output: at most ceil(129 / 8)
#define DEBYE_SMALL_GMAX 256      // largest grid (one CTA per SM at most; the hosts cap it)
// Cost balance of the unit line: starting a row segment (pipeline fill, masked head, its share of a flush) costs about as much as
// DEBYE_SMALL_WROW units (one j atom x 128 i atoms), measured on B200 with 1000 atoms / 5 types: 26 units in one segment 6.1 us,
// in five segments 12.0 us.  Every row therefore counts DEBYE_SMALL_WROW virtual units in front of its real ones when the line
// is cut into equal ranges, so a CTA whose range crosses many short rows gets fewer real units.  0: plain unit count.
#ifndef DEBYE_SMALL_WROW
#define DEBYE_SMALL_WROW 16
#endif
// diagonal type pair with n atoms: weighted units before row r
__host__ __device__ inline int debye_small_diag_prefix(int n, int r) { return (int)debye_diag_row_prefix(n, r) + DEBYE_SMALL_WROW * r; }

struct SmallPlan {
    int32_t n_a[DEBYE_SMALL_TMAX], seg_off[DEBYE_SMALL_TMAX + 1];
    int32_t tp_ti[DEBYE_SMALL_TP], tp_tj[DEBYE_SMALL_TP], tp_prefix[DEBYE_SMALL_TP + 1];
    int32_t koff, bad;
    double dq;
};

// dynamic shared memory: the packed atoms during the pairs phase, part[n_tp][levels] + S[n_tp] of one output during the final phase
__host__ __device__ inline size_t debye_small_dyn_smem(int N, int T, int K)
{
    (void)K;
    // final phase: part[n_tp][levels] + S[n_tp], then the slice sums [levels][slices]; the CTA ranges of the n_tp type pairs cover
    // at most grid + n_tp CTAs (neighbours share a CTA), so slices <= (grid + n_tp) / 8 + n_tp, grid <= DEBYE_SMALL_GMAX
    const size_t n_tp = (size_t)(T * (T + 1) / 2);
    const size_t a = (size_t)((N + 7) / 8 * 8 + 8) * 16,
                 s = n_tp * (DEBYE_KMAX_LEVELS + 1) * 8 + ((DEBYE_SMALL_GMAX + n_tp) / 8 + n_tp + 1) * DEBYE_KMAX_LEVELS * 8;
    return a > s ? a : s;
}

template <int K>
__global__ void __launch_bounds__(DEBYE_IB, recur_min_ctas(K)) debye_small_kernel(const float *__restrict__ xyz, const int32_t *__restrict__ type, const int N, const int T,
                                                                                   const float *__restrict__ fftab, const float *__restrict__ q, const int M, const int hint_class,
                                                                                   double *__restrict__ records, double *__restrict__ out,
                                                                                   const int mode, int32_t *__restrict__ n_out)
{
    constexpr int NW = DEBYE_IB / 32;
    extern __shared__ __align__(16) unsigned char dyn[];
    float4 *atoms = reinterpret_cast<float4 *>(dyn);
    __shared__ SmallPlan sp;
    __shared__ int wcnt[NW][DEBYE_SMALL_TMAX];
    __shared__ int s_dev, s_qmax;
    __shared__ float tbuf[NW][32][33];
    __shared__ double wsum[NW][K];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int G = gridDim.x, c = blockIdx.x;
    const int n_tp = T * (T + 1) / 2;
#ifdef DEBYE_SMALL_TRACE
    unsigned long long tr[8];
#define TR(i) asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(tr[i]))
#else
#define TR(i)
#endif
    TR(0);
#ifdef DEBYE_SMALL_TRACE
    tr[6] = tr[7] = 0;
#endif

    // ---- 1. stable counting sort by type, packed atoms into shared memory -------------------------------------------
    const int chunk = ((N + NW - 1) / NW + 31) / 32 * 32;                     // <= DEBYE_SMALL_NMAX / NW
    const int c0 = min(N, warp * chunk), c1 = min(N, c0 + chunk);
    if (lane < DEBYE_SMALL_TMAX) wcnt[warp][lane] = 0;
    if (tid == 0) { s_dev = 0; s_qmax = 0; }
    __syncwarp();
    // a warp's chunk is at most 512 atoms: all its type labels are loaded at once (16 loads in flight per lane, one latency)
    constexpr int SORT_IT = DEBYE_SMALL_NMAX / (NW * 32);
    int tt[SORT_IT];
    float cx[SORT_IT][3];             // ... and so are its coordinates and the q grid: one global-memory latency for the prologue
#pragma unroll
    for (int x = 0; x < SORT_IT; ++x) { const int i = c0 + 32 * x + lane; tt[x] = (i < c1) ? type[i] : -1; }
#pragma unroll
    for (int x = 0; x < SORT_IT; ++x) {
        const int i = c0 + 32 * x + lane;
        if (c0 + 32 * x < c1) { const float *sx = xyz + (size_t)(i < c1 ? i : 0) * 3; cx[x][0] = sx[0]; cx[x][1] = sx[1]; cx[x][2] = sx[2]; }
        else { cx[x][0] = cx[x][1] = cx[x][2] = 0.f; }
    }
    const float q_first = q[0], q_last = q[M - 1], q_mine = (tid < M) ? q[tid] : 0.f;      // M <= 129 <= blockDim + 1: see below
#pragma unroll
    for (int x = 0; x < SORT_IT; ++x) {
        if (c0 + 32 * x < c1) {
            const int t = tt[x];
            const unsigned peers = __match_any_sync(0xffffffffu, t);
            if (t >= 0 && (peers & ((1u << lane) - 1)) == 0) wcnt[warp][t] += __popc(peers);
            __syncwarp();
        }
    }
    // ---- 2. q grid (independent of the sort; shares its barrier) ------------------------------------------------------
    const double q0 = (double)q_first;
    const double dq = debye_grid_dq(q0, (double)q_last, M);
    {
        float dev = 0.f, qmax = 0.f;
        if (tid < M) { dev = debye_grid_dev((double)q_mine, tid, q0, dq); qmax = fabsf(q_mine); }
        for (int k = tid + DEBYE_IB; k < M; k += DEBYE_IB) {        // only M = 129 gets here
            const double qk = (double)q[k];
            dev = fmaxf(dev, debye_grid_dev(qk, k, q0, dq));
            qmax = fmaxf(qmax, fabsf((float)qk));
        }
        for (int o = 16; o > 0; o >>= 1) { dev = fmaxf(dev, __shfl_xor_sync(0xffffffffu, dev, o)); qmax = fmaxf(qmax, __shfl_xor_sync(0xffffffffu, qmax, o)); }
        __syncthreads();                                    // s_dev / s_qmax initialised, wcnt complete
        if (lane == 0) { atomicMax(&s_dev, __float_as_int(dev)); atomicMax(&s_qmax, __float_as_int(qmax)); }   // non-negative floats order like ints
    }
    __syncthreads();
    if (tid == 0) {
        int pre = 0;
        for (int t = 0; t < DEBYE_SMALL_TMAX; ++t) {
            int tot = 0;
            if (t < T) for (int w = 0; w < NW; ++w) tot += wcnt[w][t];
            sp.n_a[t] = tot; sp.seg_off[t] = pre; pre += tot;
        }
        sp.seg_off[DEBYE_SMALL_TMAX] = pre;
        const int cls = debye_grid_class(q0, dq, __int_as_float(s_dev), __int_as_float(s_qmax));
        sp.koff = cls;
        sp.bad = (cls != hint_class || cls < 0) ? 1 : 0;    // the host sized K for the promised grid
        sp.dq = dq;
        // units per type pair; the side with less padding waste becomes the row (i) side (as debye_setup_kernel)
        int upre = 0, tp = 0;
        for (int a = 0; a < T; ++a)
            for (int b2 = a; b2 < T; ++b2, ++tp) {
                const int na = sp.n_a[a], nb = sp.n_a[b2];
                int units, ti = a, tj = b2;
                if (a == b2) {
                    const int rows = debye_diag_rows(na);
                    units = rows > 0 ? debye_small_diag_prefix(na, rows) : 0;
                } else {
                    const int ra = (na + DEBYE_IB - 1) / DEBYE_IB, rb = (nb + DEBYE_IB - 1) / DEBYE_IB;
                    const int ua = ra * nb, ub = rb * na;                  // the side with less padding becomes the row side ...
                    if (ub < ua) { ti = b2; tj = a; units = rb * (na + DEBYE_SMALL_WROW); } else units = ra * (nb + DEBYE_SMALL_WROW);   // ... weighted
                    if (na == 0 || nb == 0) units = 0;
                }
                sp.tp_ti[tp] = ti; sp.tp_tj[tp] = tj; sp.tp_prefix[tp] = upre;
                upre += units;
            }
        sp.tp_prefix[tp] = upre;
    }
    __syncthreads();
    {   // first output slot of (warp, type): the type's segment plus the counts of the warps before this one
        int first = 0;
        if (lane < DEBYE_SMALL_TMAX) { first = sp.seg_off[lane]; for (int w = 0; w < warp; ++w) first += wcnt[w][lane]; }
        __syncthreads();
        if (lane < DEBYE_SMALL_TMAX) wcnt[warp][lane] = first;
        __syncwarp();
    }
#pragma unroll
    for (int x = 0; x < SORT_IT; ++x) {
        if (c0 + 32 * x < c1) {
            const int t = tt[x];
            const unsigned peers = __match_any_sync(0xffffffffu, t);
            const int rank = __popc(peers & ((1u << lane) - 1));
            if (t >= 0) atoms[wcnt[warp][t] + rank] = make_float4(cx[x][0], cx[x][1], cx[x][2], 1.0f);
            __syncwarp();
            if (t >= 0 && rank == 0) wcnt[warp][t] += __popc(peers);
            __syncwarp();
        }
    }
    __syncthreads();

    TR(1);
    // ---- 3. this CTA's share of the unit line -----------------------------------------------------------------------------
    const int U = sp.bad ? 0 : sp.tp_prefix[n_tp];
    const int koff = sp.koff;
    RecurConst rc;
    {
        const double w1_d = dq * 0.15915494309189535;
        rc.w1 = (float)w1_d; rc.w1_lo = (float)(w1_d - (double)rc.w1);
        rc.wS = rc.wS_lo = rc.w4 = rc.w4_lo = 0.f; rc.cut2 = 0.f;
        rc.smult = 8.0f; rc.n_chunks = 1;
    }
    u64 acc[K / 2];
#pragma unroll
    for (int i = 0; i < K / 2; ++i) acc[i] = 0;
    double run = 0.0;                 // thread k < K owns the FP64 running sum of slot k
    auto flush = [&]() {              // as in debye_pairs_kernel: per-warp transpose, lane order, then warp order
#pragma unroll
        for (int s = 0; s < (K + 31) / 32; ++s) {
#pragma unroll
            for (int t = 0; t < 32; t += 2) {
                const int l = 32 * s + t;
                if (l < K) {
                    float lo, hi;
                    upk2(acc[l / 2], lo, hi);
                    tbuf[warp][t][lane] = lo;
                    tbuf[warp][t + 1][lane] = hi;
                    acc[l / 2] = 0;
                }
            }
            __syncwarp();
            if (32 * s + lane < K) {
                // four interleaved partial sums (lanes j = x mod 4), then (0 + 1) + (2 + 3): a fixed order with a quarter of the
                // dependent FP64 additions of the plain lane-order sum -- this kernel flushes once per type pair it touches
                double p0 = 0.0, p1 = 0.0, p2 = 0.0, p3 = 0.0;
#pragma unroll
                for (int j = 0; j < 32; j += 4) {
                    p0 += (double)tbuf[warp][lane][j]; p1 += (double)tbuf[warp][lane][j + 1];
                    p2 += (double)tbuf[warp][lane][j + 2]; p3 += (double)tbuf[warp][lane][j + 3];
                }
                wsum[warp][32 * s + lane] = (p0 + p1) + (p2 + p3);
            }
            __syncwarp();
        }
        __syncthreads();
        if (tid < K) run += (wsum[0][tid] + wsum[1][tid]) + (wsum[2][tid] + wsum[3][tid]);
        __syncthreads();
    };
    if (U > 0) {
        int u = (int)debye_range_begin(U, c, G);
        const int u1 = (c + 1 == G) ? U : (int)debye_range_begin(U, c + 1, G);
        int curX = -1, pending = 0;
        while (u < u1) {
            int lo = 0, hi = n_tp;                    // largest tp with tp_prefix[tp] <= u
            while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (sp.tp_prefix[mid] <= u) lo = mid; else hi = mid; }
            const int tp = lo, v = u - sp.tp_prefix[tp];
            const int ti = sp.tp_ti[tp], tj = sp.tp_tj[tp];
            const bool diag = (ti == tj);
            const int n_i = sp.n_a[ti], n_j = sp.n_a[tj];
            int row, jo, row_units;          // jo < 0: inside the row's virtual units (DEBYE_SMALL_WROW)
            if (!diag) { row = v / (n_j + DEBYE_SMALL_WROW); jo = v % (n_j + DEBYE_SMALL_WROW) - DEBYE_SMALL_WROW; row_units = n_j; }
            else {
                int rl = 0, rh = debye_diag_rows(n_i);
                while (rh - rl > 1) { const int mid = (rl + rh) >> 1; if (debye_small_diag_prefix(n_i, mid) <= v) rl = mid; else rh = mid; }
                row = rl; jo = v - debye_small_diag_prefix(n_i, row) - DEBYE_SMALL_WROW; row_units = n_i - 1 - row * DEBYE_IB;
            }
            // every CTA whose range touches the type pair -- even in virtual units only -- owns a record of it (the final stage
            // reads the records of all CTAs between the owners of the type pair's first and last unit)
            if (tp != curX) {
                if (curX >= 0) { if (pending) flush(); pending = 0; if (tid < K) { records[((int64_t)c + curX) * K + tid] = run; run = 0.0; } }
                curX = tp;
            }
            if (jo < 0) {                    // skip the virtual units; the range may end inside them
                u += -jo; jo = 0;
                if (u >= u1) break;
            }
            const int len = min(u1 - u, row_units - jo);
            const int i_local = row * DEBYE_IB + tid;
            const bool ivalid = i_local < n_i;
            const float4 pi = atoms[sp.seg_off[ti] + (ivalid ? i_local : 0)];
            const int j_first = diag ? (row * DEBYE_IB + 1 + jo) : jo;      // index within the j type segment
            const float4 *src = atoms + sp.seg_off[tj] + j_first;
            int jj0 = 0;
            if (diag) jj0 = max(0, row * DEBYE_IB + warp * 32 + 1 - j_first);
            const int w_last_i = row * DEBYE_IB + warp * 32 + 31;
            const int jfree = (w_last_i >= n_i) ? 0x7fffffff : (diag ? max(0, w_last_i + 1 - j_first) : 0);
#ifdef DEBYE_SMALL_TRACE
            unsigned long long ta, tb; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(ta));
#endif
            if (row * DEBYE_IB + warp * 32 < n_i) prod_tile<K, RM_P1, false>(acc, src, jj0, len, pi, ivalid, diag, i_local, j_first, rc, jfree);
#ifdef DEBYE_SMALL_TRACE
            asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(tb)); tr[6] += tb - ta; tr[7] += 1;
#endif
            pending += len;
            if (pending >= DEBYE_FLUSH_J) { flush(); pending = 0; }
            u += len;
        }
        if (curX >= 0) { if (pending) flush(); if (tid < K) records[((int64_t)c + curX) * K + tid] = run; }
    }

    // ---- 4. grid-wide barrier (cooperative launch: all CTAs are resident), then CTA k computes output q_k -------------------
    // CTA range of every type pair (the same for every CTA; computed before the barrier, where it overlaps the stragglers)
    __shared__ int s_clo[DEBYE_SMALL_TP], s_chi[DEBYE_SMALL_TP];
    const bool bad = sp.bad != 0;
    if (tid < n_tp) {
        int lo_c = 0, hi_c = -1;
        if (U > 0) {
            const DebyeRanges ranges(U, G);
            const int units = sp.tp_prefix[tid + 1] - sp.tp_prefix[tid];
            if (units > 0) { lo_c = ranges.owner(sp.tp_prefix[tid]); hi_c = ranges.owner(sp.tp_prefix[tid] + units - 1); }
        }
        s_clo[tid] = lo_c; s_chi[tid] = hi_c;
    }
    // slices of 8 CTAs per type pair (final stage): s_soff[tp] = slices before type pair tp
    __shared__ int s_soff[DEBYE_SMALL_TP + 1], s_maxg;
    __syncthreads();
    if (tid == 0) {
        int pre = 0, mg = 1;
        for (int tp = 0; tp < n_tp; ++tp) {
            const int g8 = (s_chi[tp] >= s_clo[tp]) ? (s_chi[tp] - s_clo[tp]) / 8 + 1 : 0;
            s_soff[tp] = pre; pre += g8;
            if (g8 > mg) mg = g8;
        }
        s_soff[n_tp] = pre; s_maxg = mg;                    // most slices of one type pair
    }
    // What output k needs beyond the records -- q_k, the table column F[.][k], the slots of its telescoped chain -- does not
    // depend on the pairs phase: it is fetched BEFORE the grid barrier for the CTA's first output (two global-memory latencies
    // off the critical path of the final stage, which every CTA with an output runs after the slowest CTA's arrival).
    __shared__ int s_slot[DEBYE_KMAX_LEVELS], s_nlev;
    __shared__ float s_F[DEBYE_SMALL_TMAX], s_qk;
    auto prep = [&](const int k) {
        if (tid < DEBYE_SMALL_TMAX) s_F[tid] = (tid < T && mode == 0) ? fftab[tid * M + k] : 0.f;
        if (tid == 32) s_qk = q[k];
        if (tid == 64) {                                  // the telescoped chain  B_kappa = Out[slot(kappa)] + B_{8 j - kres}  (debye_pairs.cuh)
            int n = 0;
            for (int kap = k + koff; kap > 0;) {
                const int j = (kap - 1) >> 3, kres = kap - 8 * j;
                s_slot[n++] = 8 * j + kres - 1;
                kap = 8 * j - kres;
            }
            s_nlev = n;
        }
    };
    if (c < M) prep(c);
    TR(2);
    __threadfence();
    cooperative_groups::this_grid().sync();
    TR(3);
    double *part = reinterpret_cast<double *>(dyn);       // the atoms are no longer needed: part[n_tp][nlev], Sq[n_tp]
    const double nan = __longlong_as_double(0x7ff8000000000000LL);
    for (int k = c; k < M; k += G) {                      // one CTA per q index (both modes)
        if (k != c) {
            __syncthreads();                              // part / s_slot / s_F of the previous k are no longer read
            prep(k);
            __syncthreads();
        }
        const double qk = (double)s_qk;
        const int nlev = s_nlev;
        // The records of a type pair's CTAs are added in CTA order in slices of 8 (one thread per (chain element, slice): eight
        // loads in flight, the records sit in L2), then the slices in slice order (one thread per (type pair, chain element)).
        // One thread per (type pair, chain element) walking the whole CTA range took 5 us for the outputs with five chain
        // elements (measured, 1000 atoms) -- and the slowest CTA of the final stage ends the kernel.
        const int ntask = n_tp * nlev;
        double *Sq = part + ntask;
        double *ssum = Sq + n_tp;                                   // [nlev][slices]
        const int nsl = s_soff[n_tp];
        // ... unless the (type pair, chain element) tasks already fill the CTA and no type pair spans many CTAs (many types): in
        // global-memory latencies, passes x slices of the longest walk against passes over the slices + 1
        const bool by_slices = (nsl * nlev + DEBYE_IB - 1) / DEBYE_IB + 1 < (ntask + DEBYE_IB - 1) / DEBYE_IB * s_maxg;
        if (!bad && U >= G && by_slices) {
            for (int item = tid; item < nsl * nlev; item += DEBYE_IB) {
                const int e = item / nsl, sidx = item - e * nsl, l = s_slot[e];
                int tp = 0;
                while (s_soff[tp + 1] <= sidx) ++tp;                // <= 36 steps
                int cc = s_clo[tp] + 8 * (sidx - s_soff[tp]);
                const int ce = min(s_chi[tp] + 1, cc + 8);
                const double *rp = records + ((int64_t)cc + tp) * K + l;
                double r[8];
#pragma unroll
                for (int x = 0; x < 8; ++x) r[x] = (cc + x < ce) ? __ldcg(rp + x * K) : 0.0;
                double sum = 0.0;
#pragma unroll
                for (int x = 0; x < 8; ++x) sum += r[x];
                ssum[item] = sum;
            }
        }
        __syncthreads();
        for (int task = tid; task < ntask; task += DEBYE_IB) {
            const int tp = task / nlev, e = task - tp * nlev, l = s_slot[e];
            double sum = 0.0;
            if (!bad && U > 0) {
                if (U >= G && by_slices) {
                    for (int x = s_soff[tp]; x < s_soff[tp + 1]; ++x) sum += ssum[e * nsl + x];
                } else if (U >= G) {                      // this thread walks the type pair's CTA range: slices of 8 in CTA order
                    int cc = s_clo[tp];
                    const int c_hi = s_chi[tp];
                    const double *rp = records + ((int64_t)cc + tp) * K + l;
                    for (; cc <= c_hi; cc += 8, rp += 8 * K) {
                        double r[8];
#pragma unroll
                        for (int x = 0; x < 8; ++x) r[x] = (cc + x <= c_hi) ? __ldcg(rp + x * K) : 0.0;
                        double s8 = 0.0;
#pragma unroll
                        for (int x = 0; x < 8; ++x) s8 += r[x];
                        sum += s8;
                    }
                } else {                                  // fewer units than CTAs: each unit has its own CTA
                    const DebyeRanges ranges(U, G);
                    for (int uu = sp.tp_prefix[tp]; uu < sp.tp_prefix[tp + 1]; ++uu) sum += __ldcg(records + ((int64_t)ranges.owner(uu) + tp) * K + l);
                }
            }
            part[task] = sum;
        }
        __syncthreads();
        if (tid < n_tp) {
            const int tp = tid;
            const int a = min(sp.tp_ti[tp], sp.tp_tj[tp]), b2 = max(sp.tp_ti[tp], sp.tp_tj[tp]);
            const int units = sp.tp_prefix[tp + 1] - sp.tp_prefix[tp];
            double S;
            if (bad) S = nan;
            else if (qk == 0.0 || units == 0) S = (a == b2) ? 0.5 * (double)sp.n_a[a] * (double)(sp.n_a[a] - 1) : (double)sp.n_a[a] * (double)sp.n_a[b2];
            else {
                double sum = 0.0;
                for (int e = 0; e < nlev; ++e) sum += part[tp * nlev + e];
                S = 0.5 * sum / qk;
            }
            // mode 0: the type pair's term of I(q_k) (one thread per type pair: a single thread multiplying all of them out ran a
            // dependent FP64 chain of 1.8 us, measured with 15 type pairs)
            if (mode == 0) Sq[tp] = 2.0 * (double)s_F[a] * (double)s_F[b2] * S; else out[tp * M + k] = S;
        }
        if (mode == 0) {
            __syncthreads();
            if (tid == 0) {
                double F[DEBYE_SMALL_TMAX];                 // the table column of this q: all loads in flight together
#pragma unroll
                for (int a = 0; a < DEBYE_SMALL_TMAX; ++a) F[a] = (double)s_F[a];               // 0 beyond T
                double tot = 0.0;
#pragma unroll
                for (int a = 0; a < DEBYE_SMALL_TMAX; ++a) tot += (double)sp.n_a[a] * F[a] * F[a];        // n_a = 0 beyond T
                for (int tp = 0; tp < n_tp; ++tp) tot += Sq[tp];                                         // type pairs in increasing order
                out[k] = tot;
            }
        }
    }
    if (mode != 0 && c == 0 && n_out && tid < T) n_out[tid] = sp.n_a[tid];
#ifdef DEBYE_SMALL_TRACE
    TR(5);
    if (tid == 0) if (tid == 0 && (c == 0 || c == G - 1)) printf("cta %d of %d: sort %llu pairs %llu (prod_tile %llu in %llu calls) barrier %llu final %llu total %llu ns\n", c, G, tr[1] - tr[0], tr[2] - tr[1], tr[6], tr[7], tr[3] - tr[2], tr[5] - tr[3], tr[5] - tr[0]);
#endif

}

}  // namespace debye
