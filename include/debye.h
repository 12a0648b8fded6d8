/* debye.h -- C ABI of libdebye: Debye all-pairs sinc summation on NVIDIA B200 (sm_100a).
 *
 * What is computed (arxiv 1306.2258, Eq. 2; per-type form factors per BASELINE.json north_star):
 *
 *     I(q_m) = sum_{i=0}^{N-1} sum_{j=0}^{N-1} F[t_i][m] F[t_j][m] sinc(q_m |x_i - x_j|),   sinc(0) = 1,
 *
 * i.e. both sums include j == i (self terms counted once each), pairs i != j are evaluated once for i < j
 * and doubled ("only values for j <= k are computed").  Internally the library accumulates per
 * type pair S_ab(q_m) = sum_{i<j, {t_i,t_j}={a,b}} sin(q_m r_ij)/r_ij in FP32 (FP64 with DEBYE_FP64), reduces
 * in FP64 in a fixed order, and applies  I = sum_a n_a F_a^2 + 2 sum_{a<=b} F_a F_b S_ab / q_m  in an epilogue.
 *
 * Conventions
 *   - Every call returns a status (DEBYE_OK == 0).  No exceptions, no errno, nothing printed.
 *   - "dev" pointers are CUDA device pointers owned by the caller; "host" pointers are ordinary host memory.
 *   - Device-pointer calls are asynchronous on `stream`, never synchronise the host and never read device
 *     data on the host.  Scratch memory comes from a library-owned per-device cache that only grows
 *     (cudaMalloc on growth, which may synchronise the first time a larger problem is seen) or from a
 *     caller-supplied workspace (debye_set_workspace).  That scratch is one per device: a call on another stream than
 *     the previous call first makes its stream wait (cudaStreamWaitEvent, no host synchronisation) for the event the
 *     previous call recorded behind its last kernel, so calls on different streams serialise on the device instead
 *     of overwriting each other's records.  A plan (debye_plan_create) owns its scratch: plans on different streams run
 *     concurrently; one plan used on several streams serialises the same way.  Calls may come from several host threads
 *     (a mutex covers the shared scratch); one plan must not be executed from two host threads at once.
 *   - Results are bitwise reproducible run to run for the same inputs, flags, GPU model and library build.
 *   - Not checked (undefined behaviour if violated): 0 <= type[i] < T; finite inputs (NaN/Inf propagate).
 *   - fftab values may be negative (neutron scattering lengths); q may contain 0 and be in any
 *     order; q and -q give the same result.
 *   - There is no CPU fallback and no other backend: without a CUDA device every compute call returns
 *     DEBYE_ECUDA.
 */
#ifndef DEBYE_H
#define DEBYE_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct CUstream_st *debye_stream_t; /* == cudaStream_t; NULL is the legacy default stream */

enum {
    DEBYE_OK = 0,
    DEBYE_EINVAL = 1,       /* null pointer, N < 1, M < 1, T < 1, T > DEBYE_MAX_TYPES, M > DEBYE_MAX_Q, B < 1,
                               contradictory flags */
    DEBYE_EUNSUPPORTED = 2, /* size beyond what the build supports (N > 2^24) */
    DEBYE_ENOMEM = 3,       /* workspace allocation failed / supplied workspace too small */
    DEBYE_ECUDA = 4         /* a CUDA runtime call failed; see debye_last_cuda_error() */
};

#define DEBYE_MAX_TYPES 32
#define DEBYE_MAX_Q 4096

/* flags (bitwise or).  At most one of the DEBYE_SINC_* bits; none = automatic choice (made on the device,
 * no host sync): the recurrence kernel when q is a uniform grid from 0 or dq (telescoped product form), the centred
 * product form when it is uniform with another start, has more than 256 non-zero points or -- with the hint of debye_q_hint --
 * is a sequence of a few uniform pieces, else the MUFU kernel. */
enum {
    DEBYE_FP64 = 1u << 0,         /* double-precision pair arithmetic (libdevice sin), tolerance 1e-10 mode     */
    DEBYE_SINC_MUFU = 1u << 2,    /* FP32, one range-reduced MUFU.SIN per term; any q grid                      */
    DEBYE_SINC_RECUR = 1u << 3,   /* FP32, Chebyshev angle-addition recurrence across a uniform q grid          *
                                   * q_m = q_0 + m dq.  If q is not uniform (checked on the device) the output  *
                                   * is filled with NaN.                                                         */
    DEBYE_SINC_ACCURATE = 1u << 4, /* FP32, libdevice sinf per term (slow reference variant); any q grid;       *
                                   * plain calls only: DEBYE_EUNSUPPORTED with weights or in a tile split      */
    /* Optional grid hint, as returned by debye_q_hint() from a HOST copy of q.  Without it the library cannot know the
     * shape of the grid when it launches (q is device memory and calls never synchronise), so it launches every pairs
     * instantiation that could be needed and the device runs exactly one; with it, only that one is launched (two or
     * three launches fewer: ~12 us per call).  The device checks the hint against q; if it is wrong nothing is computed
     * and the output is filled with NaN. */
    DEBYE_QHINT = 1u << 8,          /* a hint is present                                                        */
    DEBYE_QHINT_UNIFORM = 1u << 9,  /* q[k] = q[0] + k dq, dq = (q[M-1] - q[0])/(M-1): every q[k] within 1.5 float
                                     * ulps (1.8e-7 relative to max(|q[k]|, |dq|)) of that line                  */
    DEBYE_QHINT_START0 = 1u << 10,  /* ... and q[0] == 0                                                        */
    DEBYE_QHINT_STARTDQ = 1u << 11, /* ... and q[0] == dq (the paper's grid q_k = k dq, k >= 1)   */
    /* Piecewise-uniform grid: q is a sequence of at most 32 uniform pieces (a SAXS range followed by a coarser WAXS range, a
     * grid with a dropped point, a uniform grid with a general start cut into pieces of at most 128 points).  Such grids run
     * the CENTRED PRODUCT FORM (one FP32 lane-operation per term) instead of one MUFU.SIN per term.
     * The host sizes the launch from the pieces, so this hint carries their number and the accumulators per thread in bits
     * 16-20 (pieces - 1, at most 32 pieces) and 21-25 (K / 8 - 1): take it from debye_q_hint / debye_q_hint_pieces, never build it by hand.
     * Excludes DEBYE_QHINT_UNIFORM / _START*.  The device repeats the segmentation and fills the output with NaN if the
     * hint does not match q. */
    DEBYE_QHINT_PIECES = 1u << 12,
    /* Force the centred product form (any piecewise-uniform grid, also a plain uniform one): needs DEBYE_QHINT_PIECES
     * (debye_q_hint_pieces), DEBYE_EUNSUPPORTED without it.  Automatic mode takes it whenever the hint says pieces. */
    DEBYE_SINC_CENTRED = 1u << 5
};
#define DEBYE_QHINT_NPIECES_SHIFT 16
#define DEBYE_QHINT_PIECEK_SHIFT 21

/* One structure.  PAPER.md:82, 88: inputs are N atom positions and the form factors at Q q-values, output
 * is I(q)[Q].
 *   xyz    dev  [N][3] float32, row-major (x,y,z), Angstrom
 *   type   dev  [N] int32, 0 <= type[i] < T
 *   fftab  dev  [T][M] float32 row-major, fftab[t][m] = f_t(q_m)
 *   q      dev  [M] float32, 1/Angstrom
 *   I_out  dev  [M] float64, written (not accumulated)
 * Errors: DEBYE_EINVAL / EUNSUPPORTED / ENOMEM / ECUDA as above; on error nothing is launched. */
int debye_profile(const float *xyz, const int32_t *type, int32_t N, const float *fftab, int32_t T,
                  const float *q, int32_t M, double *I_out, uint32_t flags, debye_stream_t stream);

/* B conformers of one molecule in one launch sequence (the profile is "recomputed hundreds
 * of thousands of times"; ensembles).  type / fftab / q are shared; the type sort is computed once.
 *   xyz    dev  [B][N][3] float32          I_out  dev  [B][M] float64 row-major */
int debye_profile_batch(const float *xyz, const int32_t *type, int32_t N, int32_t B, const float *fftab,
                        int32_t T, const float *q, int32_t M, double *I_out, uint32_t flags,
                        debye_stream_t stream);

/* Same results through HOST buffers: copies the inputs to the device (cudaMemcpyAsync on `stream`), runs the
 * device path, copies I_out back and synchronises `stream` before returning.  All pointers are host pointers
 * (pinned or pageable).  This is the end-to-end entry bench.py times ("e2e"). */
int debye_profile_host(const float *xyz, const int32_t *type, int32_t N, const float *fftab, int32_t T,
                       const float *q, int32_t M, double *I_out, uint32_t flags, debye_stream_t stream);
int debye_profile_batch_host(const float *xyz, const int32_t *type, int32_t N, int32_t B, const float *fftab,
                             int32_t T, const float *q, int32_t M, double *I_out, uint32_t flags,
                             debye_stream_t stream);

/* Per-atom weights (the paper's form factors are per atom because the excluded
 * volume and the hydration layer depend on the atom's environment).  This is the one-parameter family
 *     f_j(q_m) = weight[j] * fftab[type[j]][m],
 * which keeps the per-type-pair accumulation: the inner loop gains one multiply per pair (1/r times w_j), the i atom's
 * weight is applied when its accumulators are reduced, and the epilogue uses sum w and sum w^2 per type.
 *   weight dev (host for the _host entry) [N] float32, any sign; shared by all conformers of a batch.
 * One extra kernel launch (per-type weight sums).  Everything else as debye_profile / debye_profile_batch. */
int debye_profile_weighted(const float *xyz, const int32_t *type, const float *weight, int32_t N, const float *fftab,
                           int32_t T, const float *q, int32_t M, double *I_out, uint32_t flags, debye_stream_t stream);
int debye_profile_batch_weighted(const float *xyz, const int32_t *type, const float *weight, int32_t N, int32_t B,
                                 const float *fftab, int32_t T, const float *q, int32_t M, double *I_out,
                                 uint32_t flags, debye_stream_t stream);
int debye_profile_weighted_host(const float *xyz, const int32_t *type, const float *weight, int32_t N,
                                const float *fftab, int32_t T, const float *q, int32_t M, double *I_out,
                                uint32_t flags, debye_stream_t stream);

/* The paper's general case: one form-factor row per ATOM (the form factors "cannot be factored out of the
 * equation, because the non-uniform density of the water layer atoms around the molecule creates an intractable number of
 * possible f_k f_j combinations"; the GPU holds "all N positions of atoms and at least one set of QN associated
 * form factors for a specific q value", i.e. a Q x N table),
 *     I(q_m) = sum_i sum_j ff[i][m] ff[j][m] sinc(q_m |x_i - x_j|)      (Eq. 2; pairs once for i < j and doubled).
 * Without types there is no per-type-pair factoring: the inner loop is distance once per pair and chunk of 32 q, then per
 * q one range-reduced MUFU.SIN, a multiply by 1/r and an FMA with ff[j][m] from shared memory (XU-pipe bound); pairs with
 * q r <= 0.004 take an accurate series.  FP32 partial sums are multiplied by ff[i][m] and reduced in FP64 in a fixed order.
 *   xyz dev [N][3] float32, ff dev [N][M] float32 row-major (any sign), q dev [M] float32 (any grid; q and -q agree),
 *   I_out dev [M] float64 (written).  flags: 0 or DEBYE_SINC_MUFU (the FP32 path above), or DEBYE_FP64 (double-precision
 *   pair arithmetic, 1e-10 mode), optionally with a grid hint (DEBYE_QHINT_*, debye_q_hint); anything else is DEBYE_EINVAL.
 *   With a hint that promises q_k = (k + koff) dq, koff in {0, 1}, and at most 256 such q -- and neither DEBYE_SINC_MUFU nor
 *   DEBYE_FP64 -- the RECURRENCE runs instead (debye_peratom_recur.cuh): per pair the Chebyshev recurrence generates
 *   2 sin(q_k r)/r across the grid and each value is accumulated with one packed FMA against ff[j][k] from shared memory: 2 FP32
 *   lane-operations per term instead of ~9 instructions and a MUFU.SIN, four launches (re-layout of ff + grid check, self
 *   terms, pairs, final), scratch N x (16 + 4 K n_chunks) bytes more -- or, for at most 2048 atoms and at most 128 such q, ONE
 *   fused cooperative launch (debye_peratom_small.cuh: 27 us per 1000-atom profile).  The device checks the hint; a wrong one
 *   gives NaN.
 *   DEBYE_SINC_RECUR demands the recurrence: DEBYE_EUNSUPPORTED if the hinted grid is not one it takes.  Asynchronous on
 *   `stream`, same workspace rules and error codes as debye_profile (direct path scratch: at most 1.3 MB + 1 KB x M; a
 *   caller-supplied workspace that is too small gives DEBYE_ENOMEM).  The direct path takes q in chunks of 16..32 values fitted to M.  When the rows are copies of a type table (ff[i] = fftab[type[i]])
 *   the result equals debye_profile's to rounding -- and debye_profile is several times faster. */
int debye_profile_peratom(const float *xyz, const float *ff, int32_t N, const float *q, int32_t M, double *I_out,
                          uint32_t flags, debye_stream_t stream);
/* B conformers of one molecule with per-atom form factors (ensembles, refinement: PAPER.md:25, 46): xyz dev [B][N][3], the table
 * ff dev [N][M] is shared, I_out dev [B][M].  With a grid hint q_k = (k + koff) dq (at most 2 x 128 chain indices; automatic mode
 * or DEBYE_SINC_RECUR) all conformers run as ONE launch sequence -- the table is re-laid once, the unit line is conformer ->
 * chunk -> row -> j, which keeps the GPU full for small molecules; any other grid or variant runs the single-structure
 * sequence once per conformer on `stream`.  Every conformer's profile is what debye_profile_peratom gives for it to rounding
 * (the CTA ranges differ).  Errors as debye_profile_peratom; B outside [1, 65535] is DEBYE_EINVAL. */
int debye_profile_peratom_batch(const float *xyz, const float *ff, int32_t N, int32_t B, const float *q, int32_t M,
                                double *I_out, uint32_t flags, debye_stream_t stream);
/* The same through HOST buffers (copies in, runs the device path, copies I_out back, synchronises `stream`). */
int debye_profile_peratom_host(const float *xyz, const float *ff, int32_t N, const float *q, int32_t M, double *I_out,
                               uint32_t flags, debye_stream_t stream);

/* Plans: repeated profiles of ONE molecule whose coordinates change between calls (refinement, ensembles evaluated one
 * by one: the profile "must be recomputed hundreds of thousands of times").  debye_plan_create runs the
 * setup step once (type sort, schedule, analysis of the q grid), copies q and the weights into the plan, and synchronises
 * `stream` once to learn the shape of the grid, so that debye_plan_execute launches exactly pack + one pairs instantiation
 * + final, never synchronises, and gives bit for bit the result of debye_profile[_batch][_weighted] with the same inputs.
 *   type dev [N], q dev [M], weight dev [N] or NULL (read during create only); xyz dev [B][N][3], fftab dev [T][M],
 *   I_out dev [B][M].  A plan belongs to the device that was current at creation; destroy it with debye_plan_destroy once
 *   the work that uses it has completed.  Like every call, executions share the per-device workspace and must not overlap
 *   in time with other libdebye calls on the same device. */
typedef struct debye_plan debye_plan_t;
int debye_plan_create(debye_plan_t **plan, const int32_t *type, int32_t N, int32_t B, int32_t T, const float *q, int32_t M,
                      const float *weight, uint32_t flags, debye_stream_t stream);
int debye_plan_execute(debye_plan_t *plan, const float *xyz, const float *fftab, double *I_out, debye_stream_t stream);
void debye_plan_destroy(debye_plan_t *plan);

/* Per-type-pair partial structure factors (by-product of the path; lets a caller re-fit form factors without
 * redoing the pair sum):  S_out[b][p][m] = sum over pairs i<j with {t_i,t_j} = {a,b'} of sinc(q_m r_ij), for
 * p = a*(2T-a+1)/2 + (b'-a), a <= b' (row-major upper triangle);  n_out[t] = number of atoms of type t.
 *   S_out dev [B][T(T+1)/2][M] float64      n_out dev [T] int32 (may be NULL)
 * I(q_m) = sum_a n_a F_a^2 + 2 sum_p F_a F_b' S_out[p][m]. */
int debye_partials(const float *xyz, const int32_t *type, int32_t N, int32_t B, const float *q, int32_t T,
                   int32_t M, double *S_out, int32_t *n_out, uint32_t flags, debye_stream_t stream);

/* ONE structure (or batch) split over several GPUs by tiles of the upper triangle (the blocks of
 * the j <= k triangle are independent; PAPER.md:170-172 proposes several devices for one profile).  Every rank holds all
 * coordinates and calls debye_partials_shard with its own shard_rank in [0, shard_world): pairs CTA c of the static
 * schedule works iff c % shard_world == shard_rank (cyclic, which keeps the triangular load balanced), so
 *     sum over ranks of S_out == S_out of debye_partials     (same terms, same per-CTA FP32/FP64 sums; only the last FP64
 * additions are regrouped).  Terms that have a closed form (q_m == 0: pair counts) are contributed by rank 0 alone.
 * The one exchange step is an all-gather (or all-reduce) of S_out, [B][T(T+1)/2][M] float64 (<= 215 KB per conformer),
 * done by the caller (NCCL); debye_profile_from_partials then sums the gathered parts in part order and applies the
 * form-factor epilogue on the device:
 *     I_out[b][m] = sum_a n_a F_a^2 + 2 sum_{p=(a<=b')} F_a F_b' sum_{r < n_parts} S_parts[r][b][p][m].
 *   S_parts dev [n_parts][B][T(T+1)/2][M] float64, n_a dev [T] int32 (n_out of any rank), fftab dev [T][M], I_out dev [B][M].
 * Every rank must build the SAME static schedule, i.e. the same pairs grid (debye_launch_info: it follows from the SM count
 * and the kernel's occupancy): same GPU model and library build on every rank (sharding.assert_same_schedule checks it).
 * shard_world == 1 is debye_partials.  Unweighted only.  Errors: DEBYE_EINVAL for shard_rank outside [0, shard_world),
 * shard_world / n_parts outside [1, 4096], B > 65535 (from_partials), otherwise as debye_partials. */
int debye_partials_shard(const float *xyz, const int32_t *type, int32_t N, int32_t B, const float *q, int32_t T, int32_t M,
                         double *S_out, int32_t *n_out, uint32_t flags, int32_t shard_rank, int32_t shard_world,
                         debye_stream_t stream);
int debye_profile_from_partials(const double *S_parts, int32_t n_parts, const int32_t *n_a, const float *fftab, int32_t B,
                                int32_t T, int32_t M, double *I_out, debye_stream_t stream);

/* Grid hint flags for a q grid given as HOST memory (the same classification the device applies); OR them into `flags`.
 * Returns 0 (no hint) for q_host == NULL or M < 1. */
uint32_t debye_q_hint(const float *q_host, int32_t M);
/* The piecewise-uniform hint (DEBYE_QHINT | DEBYE_QHINT_PIECES | piece count | accumulator count) for ANY grid made of at most
 * 32 uniform pieces -- also a plain uniform grid, for which debye_q_hint prefers the telescoped product form or the chain --
 * or 0 if q is not such a grid.  debye_q_hint returns this hint by itself for grids that are not uniform as a whole. */
uint32_t debye_q_hint_pieces(const float *q_host, int32_t M);

/* Scratch bytes a call with these sizes needs (0 if the arguments are invalid): exact for the current CUDA device, a safe
 * upper bound (tens of MB) when there is none. */
size_t debye_workspace_bytes(int32_t N, int32_t B, int32_t T, int32_t M, uint32_t flags);
/* Optional caller-owned scratch for the current device (dev pointer, 256-byte aligned); NULL/0 returns to
 * the library-owned cache.  The caller keeps ownership and must keep it alive while calls are in flight. */
int debye_set_workspace(void *dev_ptr, size_t bytes);
/* Frees the library-owned workspace of every device (also done at process exit). */
void debye_shutdown(void);

/* One small structure WITHOUT ANY ALLOCATION, for callers that cannot call cudaMalloc (CUDA graph capture, tight serving
 * loops, harnesses that forbid it).  Same result as debye_profile on the same inputs and flags (the single cooperative launch
 * of the small-structure kernel: sort, pairs, FP64 reduction and epilogue), but the per-CTA FP64 records
 * live in a file-scope __device__ array of DEBYE_STATIC_SCRATCH_BYTES (292 KiB) that is part of the library's device image
 * (every GPU that uses the entry point holds it until the process exits) instead of the cudaMalloc'ed workspace.  The call
 * allocates nothing -- no cudaMalloc / cudaFree, no events, no workspace -- and never synchronises.
 *   xyz dev [N][3], type dev [N], fftab dev [T][M], q dev [M], I_out dev [M] float64: the caller's, as for debye_profile.
 *   flags MUST carry a grid hint DEBYE_QHINT | DEBYE_QHINT_UNIFORM | (DEBYE_QHINT_START0 or DEBYE_QHINT_STARTDQ), e.g. from
 *   debye_q_hint (the host may not read q; the device checks the hint and fills I_out with NaN if it is wrong);
 *   DEBYE_SINC_RECUR is accepted, the other variants are not (they need the allocated workspace).
 * Limits (what the array holds): N <= DEBYE_STATIC_MAX_ATOMS, T <= DEBYE_STATIC_MAX_TYPES, at most DEBYE_STATIC_MAX_Q
 * non-zero q values (M <= 129 with q[0] == 0, M <= 128 otherwise).  Anything beyond, or a missing / non-uniform hint, returns
 * DEBYE_EUNSUPPORTED and launches nothing; debye_profile_static_error() then names the limit that was exceeded (a message
 * for the calling thread's last debye_profile_static call, "" after a success).
 * SHARED SCRATCH: all calls on one GPU use the one array, which keeps the last call's records (the kernel writes every record
 * before it reads it: nothing needs clearing).  Calls on the same stream are ordered by the stream; calls that can overlap on
 * the GPU (different streams with no event between them) race and return wrong profiles: the caller orders them.  It does not
 * share anything with the other entry points and may overlap with those. */
#define DEBYE_STATIC_MAX_ATOMS 2048
#define DEBYE_STATIC_MAX_TYPES 8
#define DEBYE_STATIC_MAX_Q 128
#define DEBYE_STATIC_MAX_GRID 256                                   /* CTAs (one per SM at most)                      */
#define DEBYE_STATIC_SCRATCH_BYTES ((size_t)(256 + 36) * 128 * 8)   /* (CTAs + type pairs) records x 128 slots x 8 B */
int debye_profile_static(const float *xyz, const int32_t *type, int32_t N, const float *fftab, int32_t T, const float *q,
                         int32_t M, double *I_out, uint32_t flags, debye_stream_t stream);
const char *debye_profile_static_error(void);
/* The limits above at run time (any pointer may be NULL). */
void debye_profile_static_limits(int32_t *max_atoms, int32_t *max_types, int32_t *max_nonzero_q, size_t *scratch_bytes);

/* Introspection used by bench.py / tests (host-side, no GPU work):
 * number of library kernels one debye_profile[_batch] call with these arguments launches, and the grid /
 * chunking the pairs kernel would use (any out pointer may be NULL). */
int debye_launch_info(int32_t N, int32_t B, int32_t T, int32_t M, uint32_t flags, int32_t *n_launches,
                      int32_t *pairs_grid, int32_t *q_chunk, int32_t *n_chunks);

/* Measurement hook (bench.py's roofline leg): two caller-owned cudaEvent_t handles that every following call on
 * this device records, on the call's stream, immediately before and after the pairs kernel launch(es) -- the
 * dominant kernel -- so its device time can be read with cudaEventElapsedTime.  NULL, NULL switches it off. */
int debye_set_pairs_events(void *start_event, void *stop_event);

/* Diagnostics behind `bench.py --peaks` (the FP32 / MUFU issue peaks "are nominal; the build must
 * measure them"): micro-kernels of the instruction mixes the pairs kernels consist of, run on every SM of the current
 * device with ctas_per_sm (1..4) CTAs of 128 threads resident per SM; blocking (synchronise `stream`).
 *   test in [0, debye_pipe_bench_count()); debye_pipe_bench_name(test) describes it (NULL outside the range).
 *   *lane_ops_per_clk_per_sm: FP32-pipe (for the MUFU test: XU) lane-operations per SM clock cycle and SM, measured with
 *   clock64 inside the kernel, so independent of the clock the part happens to run at (nominal: 128, MUFU 16);
 *   *cycles_per_instr (may be NULL): cycles of one warp scheduler per warp instruction of the mix.
 * Errors: DEBYE_EINVAL bad arguments, DEBYE_EUNSUPPORTED if ctas_per_sm CTAs of that test do not fit on an SM.
 * debye_mufu_sin_error: error of MUFU.SIN (sin.approx.ftz.f32 of 2 pi t) against double sin on n points of (0, 1/2] turns:
 * maximum |e|, root mean square, and MEAN (a bias is a coherent error in every pair: DESIGN.md section 6).
 * debye_mufu_rsq_error: relative error of MUFU.RSQ (rsqrt.approx.ftz.f32) on n log-uniform points of [1, 4), same statistics;
 * its mean shifts every distance, i.e. the q axis, by that relative amount. */
int debye_pipe_bench_count(void);
const char *debye_pipe_bench_name(int test);
int debye_pipe_bench(int test, int ctas_per_sm, int iters, double *lane_ops_per_clk_per_sm, double *cycles_per_instr,
                     debye_stream_t stream);
int debye_mufu_sin_error(int n, double *max_abs, double *rms, double *mean, debye_stream_t stream);
int debye_mufu_rsq_error(int n, double *max_rel, double *rms, double *mean, debye_stream_t stream);

const char *debye_strerror(int status);
int debye_last_cuda_error(void); /* cudaError_t of the last failing runtime call on this thread, 0 if none */
int debye_version(void);         /* major*10000 + minor*100 + patch */

#ifdef __cplusplus
}
#endif
#endif /* DEBYE_H */
