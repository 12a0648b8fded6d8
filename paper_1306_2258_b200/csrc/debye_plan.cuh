// debye_plan.cuh -- device-resident plan shared by the setup, pairs and final kernels of libdebye.
//
// Work decomposition (S1 of SURVEY.md section 8(a); "only values for j <= k are computed"):
//   atoms are sorted by type; for every unordered type pair tp = (a <= b) the pairs form a rectangle
//   (a < b) or a strict upper triangle (a == b).  A "row" is a block of IB consecutive i atoms (one per
//   thread of a CTA); a "unit" is one j atom against one row (IB pairs x K q-values).  Units are linearised
//   as  conformer -> type pair -> q-chunk -> row -> j  and the persistent grid splits that line into G equal
//   contiguous ranges, so the assignment is static (bitwise reproducible) and balanced to one j atom.
#pragma once
#include <cstdint>
#include <cmath>

#define DEBYE_MAX_TYPES_I 32
#define DEBYE_MAX_TP (DEBYE_MAX_TYPES_I * (DEBYE_MAX_TYPES_I + 1) / 2)
#define DEBYE_IB 128          // i atoms per row == threads per pairs CTA
#define DEBYE_JT 512          // j atoms per shared-memory tile (8 KB, one cp.async.bulk); 2 buffers per CTA
#define DEBYE_TILE_PAD 8      // readable (finite) entries behind each buffer: the recurrence reads two groups ahead

enum DebyeVariant : int32_t { V_NONE = 0, V_F64 = 1, V_MUFU = 2, V_RECUR = 3, V_ACCURATE = 4, V_CENT = 5 };

// Piecewise-uniform grids (V_CENT, the centred product form of debye_pairs.cuh): q is a sequence of at most DEBYE_MAX_PIECES
// pieces, piece p = the points off[p] .. off[p] + cnt[p] - 1 with q = q0[p] + m dq[p] (m the local index), cnt[p] <= K <= 128.
#define DEBYE_MAX_PIECES 32
#define DEBYE_PIECE_KCAP 128
struct DebyePieces {
    int32_t n, K;                 // number of pieces; accumulators per thread (a multiple of 8 >= the longest piece)
    int32_t off[DEBYE_MAX_PIECES], cnt[DEBYE_MAX_PIECES];
    double q0[DEBYE_MAX_PIECES], dq[DEBYE_MAX_PIECES];
};

struct DevPlan {
    int32_t N, T, M, B;
    int32_t n_tp;                 // T(T+1)/2
    int32_t uniform;              // q is a uniform grid q0 + m dq (checked on the device)
    int32_t zero_start;           // uniform and q0 = koff dq with koff in {0, 1} (0 only if q0 == 0 exactly): koff; else -1
    int32_t recur_alt;            // recurrence: run the launch sized for M - 1 chain indices (koff == 0 and the host offered one)
    int32_t variant_auto;         // variant chosen on the device when the caller gave no DEBYE_SINC_* flag
    double q0, dq;                // least-squares-free fit: q0 = q[0], dq = (q[M-1]-q[0])/(M-1)
    float q_small;                // smallest non-zero |q|
    int32_t hint_bad;             // the caller's grid hint (DEBYE_QHINT_*) contradicts q: nothing is computed, the output is NaN
    int32_t weighted;             // per-atom weights given (debye_profile_weighted): sorted[].w holds w_j, else 1
    int32_t shard_rank, shard_world;   // tile split of ONE structure over GPUs (debye_partials_shard): pairs CTA c works iff
                                  // c % shard_world == shard_rank; the other CTAs leave their (zeroed) records alone
    int64_t U1;                   // units per conformer and per q-chunk
    DebyePieces pieces;           // piecewise-uniform grid (only filled in when the caller's hint promised one)
    double sw[DEBYE_MAX_TYPES_I];             // weighted calls: sum of w_j over the atoms of each type ...
    double sw2[DEBYE_MAX_TYPES_I];            // ... and of w_j^2 (self terms; q = 0 pair sums)
    int32_t seg_off[DEBYE_MAX_TYPES_I + 1];   // sorted-array offset of each type segment
    int32_t n_a[DEBYE_MAX_TYPES_I];           // atoms per type
    int32_t tp_ti[DEBYE_MAX_TP];              // type on the i (row) side
    int32_t tp_tj[DEBYE_MAX_TP];              // type on the j (column) side; == tp_ti on the diagonal
    int64_t tp_prefix[DEBYE_MAX_TP + 1];      // units before type pair tp (one chunk, one conformer)
};

// ---- q-grid classification, identical on the host (debye_q_hint) and on the device (debye_setup_kernel) -----------------
// class: -2 not uniform; -1 uniform, general start; 0 uniform with q[0] == 0; 1 uniform with q[0] == dq (the paper's grid).
// `dev` = max_k |q[k] - fma(k, dq, q0)| / max(|q[k]|, |dq|) rounded to float per element, `qmax` = max_k |q[k]|: maxima, so the
// order in which they are taken (serial on the host, tree on the device) does not matter; fma keeps host and device
// arithmetic identical.
__host__ __device__ inline double debye_grid_dq(double q0, double qlast, int M) { return (M > 1) ? (qlast - q0) / (double)(M - 1) : (q0 != 0.0 ? q0 : 1.0); }
__host__ __device__ inline float debye_grid_dev(double qk, int k, double q0, double dq)
{
    const double scale = fmax(fabs(qk), fabs(dq));
    return (float)(fabs(qk - fma((double)k, dq, q0)) / (scale > 1e-300 ? scale : 1e-300));
}
__host__ __device__ inline int debye_grid_class(double q0, double dq, float dev, float qmax)
{
    // Uniform if every q[k] is within 1.5 float ulps OF ITSELF (not of the largest |q|) of the line through the end points:
    // the recurrence evaluates the line, so whatever is accepted here is a relative error of q_k, i.e. of the phase q_k r.
    // A grid rounded once from the exact line deviates by at most 1 ulp (its own rounding plus that of the end points).
    (void)qmax;
    const bool uni = (dq != 0.0) && (dev <= 1.8e-7f);
    if (!uni) return -2;
    if (q0 == 0.0) return 0;
    if (fabs(q0 / dq - 1.0) <= 1e-6) return 1;
    return -1;
}

// Piecewise-uniform grids in three steps, the same arithmetic on the host (debye_q_hint: all three serially) and on the device
// (debye_setup_kernel: q staged in shared memory, step 2 by all threads), double arithmetic with fma and IEEE division only, so
// both get the same pieces from the same floats:
//   1. debye_find_runs: greedy maximal runs of equal steps (a loose test: the step into q[e] within 4 float ulps of the run's
//      first step, each difference carrying up to 2);
//   2. debye_run_point_ok for every point: the 1.5-ulp criterion of debye_grid_class against the line through the end points
//      of the point's run;
//   3. debye_pieces_from_runs: runs longer than DEBYE_PIECE_KCAP cut into equal pieces.
// false anywhere: not piecewise uniform, or more than DEBYE_MAX_PIECES pieces.
__host__ __device__ inline bool debye_find_runs(const float *q, int M, int32_t *run_start /* [DEBYE_MAX_PIECES + 1] */, int &n_runs)
{
    n_runs = 0;
    int s = 0;
    while (s < M) {
        if (n_runs == DEBYE_MAX_PIECES) return false;
        run_start[n_runs++] = s;
        int e = s + 1;
        if (e < M) {
            const double d0 = (double)q[s + 1] - (double)q[s];
            const double a0 = fmax(fmax(fabs((double)q[s]), fabs((double)q[s + 1])), fabs(d0));   // d0 carries the rounding of the run's first two points
            e = s + 2;
            while (e < M) {
                const double a = fmax(fmax(fabs((double)q[e]), fabs((double)q[e - 1])), a0);
                if (fabs(((double)q[e] - (double)q[e - 1]) - d0) > 4.8e-7 * a) break;
                ++e;
            }
        }
        s = e;
    }
    run_start[n_runs] = M;
    return true;
}
__host__ __device__ inline double debye_run_dq(const float *q, int s, int e) { return (e - s > 1) ? ((double)q[e - 1] - (double)q[s]) / (double)(e - 1 - s) : 0.0; }
// point k of the run [s, e): within 1.5 float ulps (1.8e-7 of max(|q_k|, |dq|)) of q[s] + (k - s) dq; no division per point
__host__ __device__ inline bool debye_run_point_ok(const float *q, int s, int e, int k)
{
    const double dq = debye_run_dq(q, s, e), qk = (double)q[k];
    const double scale = fmax(fabs(qk), fabs(dq));
    return fabs(qk - fma((double)(k - s), dq, (double)q[s])) <= 1.8e-7 * scale;
}
__host__ __device__ inline bool debye_pieces_from_runs(const float *q, const int32_t *run_start, int n_runs, DebyePieces &P)
{
    P.n = 0; P.K = 8;
    int maxcnt = 0;
    for (int r = 0; r < n_runs; ++r) {
        const int s = run_start[r], e = run_start[r + 1];
        const double dq = debye_run_dq(q, s, e);
        const int n = e - s, np = (n + DEBYE_PIECE_KCAP - 1) / DEBYE_PIECE_KCAP, per = (n + np - 1) / np;
        for (int x = 0; x < np; ++x) {
            if (P.n == DEBYE_MAX_PIECES) return false;
            const int o = x * per, c = (per < n - o) ? per : n - o;
            P.off[P.n] = s + o; P.cnt[P.n] = c; P.q0[P.n] = fma((double)o, dq, (double)q[s]); P.dq[P.n] = dq;
            ++P.n;
            if (c > maxcnt) maxcnt = c;
        }
    }
    P.K = (maxcnt + 7) / 8 * 8;
    if (P.K < 8) P.K = 8;
    return true;
}
// all three steps serially (the host's debye_q_hint)
__host__ __device__ inline bool debye_find_pieces(const float *q, int M, DebyePieces &P)
{
    int32_t run_start[DEBYE_MAX_PIECES + 1];
    int n_runs = 0;
    P.n = 0; P.K = 8;
    if (!debye_find_runs(q, M, run_start, n_runs)) return false;
    for (int r = 0; r < n_runs; ++r)
        for (int k = run_start[r]; k < run_start[r + 1]; ++k)
            if (!debye_run_point_ok(q, run_start[r], run_start[r + 1], k)) return false;
    return debye_pieces_from_runs(q, run_start, n_runs, P);
}

// ---- programmatic dependent launch (PDL) ------------------------------------------------------------------------
// Every kernel after the setup kernel is launched with cudaLaunchAttributeProgrammaticStreamSerialization and starts with
// pdl_wait(): its CTAs may be scheduled while the previous kernel of the call is still running and block here until that
// kernel has completed and its writes are visible.  Because EVERY kernel waits before it does anything (the instantiations
// that exit at once included), completion is transitive along the chain.  The setup and pack kernels call pdl_trigger() at
// their start so the next grid is staged early; the pairs kernels do not (a staged grid would hold registers that their own
// later waves need).
#ifdef __CUDACC__
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
#endif

// ---- unit decoding helpers (used identically by the pairs kernel and the final kernel) -------------------
__host__ __device__ inline int64_t debye_range_begin(int64_t U, int32_t c, int32_t G)
{
    // floor(U * c / G) without overflow for U < 2^52, G < 2^12
    return (U / G) * c + ((U % G) * c) / G;
}

// the same with the one 64-bit division hoisted and the other done in 32 bits (G < 2^16; final kernel: many evaluations
// for one (U, G))
struct DebyeRanges {
    int64_t U, qd; uint32_t rm, G;
    __host__ __device__ DebyeRanges(int64_t U_, int32_t G_) : U(U_), qd(U_ / G_), rm((uint32_t)(U_ - (U_ / G_) * G_)), G((uint32_t)G_) {}
    __host__ __device__ int64_t begin(int32_t c) const { return qd * c + (int64_t)((rm * (uint32_t)c) / G); }
    // CTA that owns unit u:  largest c with begin(c) <= u
    __host__ __device__ int32_t owner(int64_t u) const
    {
        int64_t c = (int64_t)(((double)u * (double)G) / (double)U);   // estimate, made exact by the two loops below
        if (c >= (int64_t)G) c = (int64_t)G - 1;
        if (c < 0) c = 0;
        while (c + 1 < (int64_t)G && begin((int32_t)(c + 1)) <= u) ++c;
        while (c > 0 && begin((int32_t)c) > u) --c;
        return (int32_t)c;
    }
};

// CTA that owns unit u:  largest c with range_begin(c) <= u
__host__ __device__ inline int32_t debye_owner(int64_t U, int32_t G, int64_t u) { return DebyeRanges(U, G).owner(u); }

// diagonal type pair with n atoms: units before row r, r(n-1) - IB r(r-1)/2
__host__ __device__ inline int64_t debye_diag_row_prefix(int64_t n, int64_t r)
{
    return r * (n - 1) - (int64_t)DEBYE_IB * (r * (r - 1) / 2);
}
__host__ __device__ inline int32_t debye_diag_rows(int32_t n) { return n >= 2 ? (n - 2) / DEBYE_IB + 1 : 0; }
