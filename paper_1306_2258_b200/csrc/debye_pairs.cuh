// debye_pairs.cuh -- the all-pairs kernel of libdebye (steps S1-S6 of SURVEY.md section 8(a)).
//
// What one CTA does (PAPER.md:86-88 re-designed for sm_100a):
//   * owns a static contiguous range of "units" (one j atom x one row of 128 i atoms x K q-values), see
//     debye_plan.cuh; thread t keeps i atom t of the current row in registers (the paper's "private memory");
//   * streams the j atoms of the range through shared memory in 1 KB tiles with cp.async.bulk (TMA 1-D bulk
//     copy, SASS UBLKCP) completing on an mbarrier, double buffered (the paper's "local memory" blocks);
//   * because tiles are type-homogeneous, every pair of the range adds into the SAME K accumulators
//     S_ab(q_k) += sin(q_k r)/r  -- no form factor in the loop (north_star (c));
//   * FP32 accumulators are promoted to FP64 per flush: per-warp transpose through shared memory, each lane
//     sums 32 values in a fixed order, then a fixed-order sum over the 4 warps (north_star (f));
//   * per (conformer, type pair, q-chunk) the CTA writes one FP64 record; the final kernel adds records in
//     CTA order.
//
// Variants of the per-pair term evaluation (north_star (d), (e)):
//   V_RECUR    uniform grid q_k = qbase + k dq, theta = r dq.
//              PRODUCT FORM (grids q_k = (k + koff) dq, koff in {0, 1}, at most 2 q-chunks; all BASELINE configs and the
//              paper's own grid): with b_n = 2 sin(n theta)/r,
//                  2 cos(j S theta) * b_k0 = b_{S j + k0} - b_{S j - k0},
//              so per pair 8 seeds b_k0 (k0 = 1..8 of the chunk) times J weights W_j = 2 cos(j S theta) (W_0 := 1) give,
//              with ONE packed FMA lane per output, the sums Out[j][k0] = sum_pairs (b_{Sj+k0} - b_{Sj-k0}); the final stage
//              undoes the telescoping in FP64: B_{Sj+k0} = Out[j][k0] + B_{Sj-k0} (B_0 = 0, B_{-n} = -B_n).  1 FP32-pipe
//              lane-operation per term instead of the 2 (recurrence step + accumulate) of a chain, no MUFU in the loop,
//              and no small-angle problem: the weights carry only the even part of the angle.
//              CHAIN FORM (general start q_0, or more than 2 chunks): three-term (Chebyshev) recurrence
//              v_{k+S} = 2cos(S theta) v_k - v_{k-S} run as 4 packed chains (8 residues mod S = 8 n_chunks) with
//              fma.rn.f32x2 (SASS FFMA2), accumulated with add.rn.f32x2 (FADD2): 2 lane-operations per term.
//   V_MUFU     any grid: explicit range reduction in turns (magic-number rounding, exact FMA remainder), one
//              MUFU.SIN per term.
//   V_ACCURATE any grid: libdevice sinf per term (reference variant).
//   V_F64      any grid: double differences, sqrt, libdevice sin; FP64 accumulators.
//   Pairs closer than r_cut (theta below the level where MUFU's absolute error matters) and coincident atoms
//   take a warp-uniform slow path: Taylor series of sinc for |x| < 0.25, sinf otherwise.
#pragma once
#include <cuda_runtime.h>
#include <cstdint>
#include "debye_plan.cuh"

typedef unsigned long long u64;

namespace debye {

// ---- packed f32x2 helpers (Blackwell FFMA2/FADD2) ----------------------------------------------------------
__device__ __forceinline__ u64 pk2(float lo, float hi) { u64 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi)); return r; }
__device__ __forceinline__ void upk2(u64 v, float &lo, float &hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ u64 fma2(u64 a, u64 b, u64 c) { u64 d; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c)); return d; }
__device__ __forceinline__ u64 add2(u64 a, u64 b) { u64 d; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
__device__ __forceinline__ u64 sub2(u64 a, u64 b) { u64 d; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
__device__ __forceinline__ float sin_mufu(float x) { float y; asm("sin.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float rsqrt_mufu(float x) { float y; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

// sin(2 pi t) for t in turns, |t| < 2^22: magic-number round to nearest, exact remainder, MUFU.SIN
__device__ __forceinline__ float sin_turns(float t)
{
    const float MAGIC = 12582912.0f;             // 1.5 * 2^23
    float n = (t + MAGIC) - MAGIC;
    return sin_mufu((t - n) * 6.28318530717958648f);
}
// sin(2 pi r w) with the product's rounding error recovered by FMA (used where r*w can be hundreds of turns)
__device__ __forceinline__ float sin_turns_fma(float r, float w)
{
    const float MAGIC = 12582912.0f;
    float n = (fmaf(r, w, MAGIC)) - MAGIC;
    return sin_mufu(fmaf(r, w, -n) * 6.28318530717958648f);
}

// ---- accurate, UNBIASED trigonometry for the recurrence start-up ------------------------------------------------
// Measured on B200: MUFU.SIN has an absolute error of 3.4e-7 with a NON-ZERO MEAN (-1.1e-7 on
// (0, 0.5]).  A biased start value or a biased recurrence coefficient is a coherent phase / frequency error in every
// chain of every pair, and the cancellation in I(q) (condition number up to ~400 in cfg5) amplifies it to 7e-4.
// A relative frequency bias must stay below ~1e-9, so: frequencies are carried as hi + lo floats, the leading
// polynomial coefficient pi is split hi + lo, and everything else is round-to-nearest FMA arithmetic (unbiased).

// Fractional part of r * (w + w_lo) in turns, in [-1/2, 1/2], as the round-to-nearest of the EXACT value.
// The naive form  fma(r, w_lo, fma(r, w, -n))  rounds r*w - n first and then adds a correction r*w_lo that is below the
// resolution of the result, so the correction is (mostly) rounded away: every pair then runs its chain at the frequency w
// instead of w + w_lo, a coherent relative error of 1e-9 that cost up to 1.7e-4 at single q points of cfg5 (measured,
// DESIGN.md section 6).  Here the product is split error-free (p + e = r*w exactly), p - n is exact, and the two small
// parts e and r*w_lo are combined BEFORE the single final rounding, which is therefore unbiased.
__device__ __forceinline__ float reduce_turns(float r, float w, float w_lo)
{
    const float p = r * w;
    const float e = fmaf(r, w, -p);                  // exact
    return (p - rintf(p)) + fmaf(r, w_lo, e);
}
// The same for two frequencies w and mult * w (mult a power of two <= 2^12, so mult * p and mult * e are exact): shares the
// error-free product.  f1 <- frac(r (w + w_lo)),  fS <- frac(mult r (w + w_lo)).
__device__ __forceinline__ void reduce_turns_pair(float r, float w, float w_lo, float mult, float &f1, float &fS)
{
    const float p = r * w;
    const float l = fmaf(r, w_lo, fmaf(r, w, -p));   // everything below the rounding of p
    // rintf is one FRND on the conversion (XU) pipe, which is otherwise idle here; the magic-number form would cost two
    // FMA-pipe instructions per rounding
    f1 = (p - rintf(p)) + l;
    const float pS = p * mult;                       // exact
    fS = fmaf(l, mult, pS - rintf(pS));
}

// Folded sine / cosine of a reduced angle.  For |f| <= 1/2 let g = |f| and g' = min(g, 1/2 - g) in [0, 1/4] (the
// subtraction is exact); fold = (g > 1/4).  Returns s = 2 sin(pi g') and c = 2 cos(pi g'), from which
//     2 cos(2 pi f) = +/-(2 - s^2)           (minus when folded),
//     2 sin(2 pi f) = sign(f) s c            (folded or not),
// so the quantity that is squared is always the SMALL one: the phase error that a relative error rho of s causes in
// 2cos(2 pi f) is 2 rho tan(pi g') <= 2 rho, whereas without the fold it is 2 rho tan(pi f), unbounded towards f = 1/2;
// and on the half interval one fewer cosine coefficient is needed for a 500 times smaller approximation error.
// Measured (cfg5, dense q): unfolded polynomials on |f| <= 1/2 save 7 instructions per pair but give 1.6e-5 with a
// degree-9 sine and 2e-4 with a BETTER degree-11 sine -- the rounding of s next to 2 is what the tangent amplifies, not the
// approximation error -- against 6.5e-6 folded.
//   s = g' (2 pi + y (s1 + y (s2 + y (s3 + y s4)))),  c = 2 + y (d1 + y (d2 + y (d3 + y d4))),  y = g'^2.
// Near-minimax coefficients (iteratively reweighted least squares on 25 000 Chebyshev-spaced points of [0, 1/4] in fp64,
// fitting 2 sin(pi g) - 2 pi g on g^3..g^9 and 2 cos(pi g) - 2 on y..y^4): maximum relative error 9.3e-12 (s), maximum
// absolute error 1.1e-10 (c).  The linear coefficient is pinned to 2 pi, carried as hi + lo.
struct Folded { float s, c; bool fold; };
__device__ __forceinline__ Folded sincos_fold(const float f)
{
    Folded o;
    const float g = fabsf(f);
    o.fold = g > 0.25f;
    const float gp = fminf(g, 0.5f - g);
    const float y = gp * gp;
    float p = fmaf(y, 0.1619238643960947f, -1.198394591051059f);
    p = fmaf(y, p, 5.100324961653245f);
    p = fmaf(y, p, -10.335425536121228f);
    p = fmaf(y, p, -1.7484556e-7f);                          // 2 pi - (float)(2 pi)
    o.s = fmaf(gp, 6.2831854820251465f, gp * p);            // (float)(2 pi)
    float c = fmaf(y, 0.46285910429932814f, -2.670116930113852f);
    c = fmaf(y, c, 8.117415808996121f);
    c = fmaf(y, c, -9.869604346828243f);
    o.c = fmaf(y, c, 2.0f);
    return o;
}
// 2 cos(2 pi f) from the folded sine: relatively accurate in (2 -/+ result) at both ends
__device__ __forceinline__ float two_cos_from(const Folded &o)
{
    const float c0 = fmaf(-o.s, o.s, 2.0f);
    return o.fold ? -c0 : c0;
}
// 2 sin(2 pi f)
__device__ __forceinline__ float two_sin_from(const Folded &o, const float f) { return copysignf(o.s, f) * o.c; }
// 4 sin^2(pi f) = 2 - 2 cos(2 pi f), relatively accurate for small f (Reinsch's beta)
__device__ __forceinline__ float four_sin2_from(const Folded &o) { return o.fold ? fmaf(-o.s, o.s, 4.0f) : o.s * o.s; }

// 2 cos(2 pi r (w + w_lo)) and 2 sin(2 pi r (w + w_lo)) with hi + lo frequencies
__device__ __forceinline__ float two_cos_turns(float r, float w, float w_lo) { return two_cos_from(sincos_fold(reduce_turns(r, w, w_lo))); }
__device__ __forceinline__ float two_sin_turns_accurate(float r, float w, float w_lo)
{
    const float f = reduce_turns(r, w, w_lo);
    return two_sin_from(sincos_fold(f), f);
}

// accurate sin(q r)/r for one term (slow path): Taylor for |x| < 0.6 (north_star (e)), libdevice sinf otherwise
__device__ __forceinline__ float term_accurate(float qk, float r)
{
    float x = qk * r;
    if (fabsf(x) < 0.6f) {     // remainder x^12/13! < 4e-13
        float x2 = x * x;
        float p = fmaf(x2, -1.0f / 39916800.0f, 1.0f / 362880.0f);
        p = fmaf(x2, p, -1.0f / 5040.0f);
        p = fmaf(x2, p, 1.0f / 120.0f);
        p = fmaf(x2, p, -1.0f / 6.0f);
        p = fmaf(x2, p, 1.0f);
        return qk * p;
    }
    return sinf(x) / r;
}

// ---- mbarrier / bulk copy ------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(u64 *bar, int count) { asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count)); }
__device__ __forceinline__ void mbar_expect_tx(u64 *bar, uint32_t bytes) { asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory"); }
__device__ __forceinline__ void mbar_wait(u64 *bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, uint32_t bytes, u64 *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

// where chain / grid index idx lives: q-chunk and local slot.  Recurrence chunks are residue classes mod S = 8 n_chunks
// (so every chunk starts at the bottom of the grid); the direct variants use contiguous ranges.
// Recurrence index convention (pairs kernel and final kernel must agree):
//   zero-start modes (grid q_k = (k + koff) dq, koff in {0, 1}, at most 2 chunks): idx = k + koff - 1, i.e. the chains
//     start at the first multiple of dq that is not zero (q = 0 is answered by the epilogue: idx = -1 is never stored);
//   general mode: idx = k.
__host__ __device__ inline void slot_of(int variant, int K, int n_chunks, int idx, int &ch, int &l)
{
    if (variant == V_RECUR) {
        int S = 8 * n_chunks;
        ch = (idx % S) / 8;
        l = 8 * (idx / S) + (idx % 8);
    } else {
        ch = idx / K;
        l = idx % K;
    }
}
// accumulators a recurrence launch needs for n_idx chain indices in n_chunks chunks: chunk 0 holds the most; K is kept a
// multiple of 4 (two packed chains) and at least 8
__host__ __device__ inline int recur_slots(int n_idx, int n_chunks)
{
    if (n_idx < 1) return 8;
    const int S = 8 * n_chunks, last = n_idx - 1;
    const int r = last % S;
    const int lmax = 8 * (last / S) + (r < 8 ? r : 7);
    const int K = (lmax + 1 + 3) / 4 * 4;
    return K < 8 ? 8 : K;
}

template <int K, int VAR>
struct PairAcc {
    // FP32 variants: K/2 packed accumulators; F64: K doubles
    typedef typename std::conditional<VAR == V_F64, double, u64>::type elem_t;
    static constexpr int NE = (VAR == V_F64) ? K : K / 2;
    elem_t v[NE];
};

// ---- recurrence variant: per-pair start values, packed hot loop, software-pipelined tile loop ------------------
// All recurrence accumulators hold TWICE sin(q r)/r (the doubled trigonometry above saves five multiplies per
// pair); the final kernel halves the sum.
struct RecurConst {
    float w1, w1_lo;         // dq / 2 pi, hi + lo: theta / 2 pi = r * (w1 + w1_lo)
    float wS, wS_lo;         // S dq / 2 pi (chain stride S = 8 n_chunks)
    float smult;             // (float)S: wS = S w1 exactly (S is a power of two)
    float w4, w4_lo;         // 4 dq / 2 pi (general start: bootstrap stride)
    float cut2;              // r^2 at or below which the pair takes the slow path
    int n_chunks;
};

enum RecurMode : int { RM_P1 = 0, RM_P2A = 1, RM_P2B = 2, RM_G = 3 };
// RM_P1   product form, grid q_k' = k' dq, one chunk  (S = 8):  seeds k0 = 1..8, outputs k' = 8 j + k0
// RM_P2A  product form, two chunks (S = 16), chunk 0: seeds k0 = 1..8, outputs k' = 16 j + k0
// RM_P2B  same, chunk 1: seeds k0 = 9..16
// RM_G    chain form, any uniform grid / any number of chunks: 8 accurate sines at k' = 8 ch - S + (0..7), stride-4 bootstrap
__host__ __device__ constexpr bool recur_is_product(int mode) { return mode != RM_G; }

// The start-up of one pair is split into two stages so that the tile loop can run them one and two groups ahead of the
// packed loop (three-stage software pipeline).
// Stage A (geometry): distance, 1/r, slow-path flag (chain form only) and the two reduced angles (turns, in [-1/2, 1/2]).
struct RecurGeom { float r, rinv, f1, fS; bool slow; };
template <int MODE, bool W>
__device__ __forceinline__ void recur_geom(const float4 pj, const float4 pi, const bool ok, const RecurConst &rc, RecurGeom &g)
{
    const float dx = pj.x - pi.x, dy = pj.y - pi.y, dz = pj.z - pi.z;
    // + 1e-30 keeps rsqrt finite for coincident atoms and changes no other distance; folding it into the FMA chain saves the
    // clamp.  Product form: r = 1e-15 then gives b_k0 = 2 sin(k0 theta)/r its limit 2 k0 dq and W_j = 2 (every step of the
    // start-up keeps RELATIVE accuracy for small theta).  Chain form: such pairs take the slow path.
    const float r2c = fmaf(dx, dx, fmaf(dy, dy, fmaf(dz, dz, 1e-30f)));
    const float rinv = rsqrt_mufu(r2c);
    g.r = r2c * rinv;
    bool small = false;
    if constexpr (!recur_is_product(MODE)) small = !(r2c > rc.cut2);
    // zero for masked / slow-path pairs: every start value becomes exactly 0.  Weighted instantiations (W): pj.w is the j
    // atom's weight; the i atom's weight is applied when the accumulators are flushed
    if constexpr (W) g.rinv = (ok && !small) ? rinv * pj.w : 0.0f;
    else g.rinv = (ok && !small) ? rinv : 0.0f;
    g.slow = small && ok;
    reduce_turns_pair(g.r, rc.w1, rc.w1_lo, rc.smult, g.f1, g.fS);     // f1 is dead code in the general-start mode
}

// ---- product form (RM_P1 / RM_P2A / RM_P2B) ----------------------------------------------------------------------
// Stage B: U = the chunk's 8 seeds b_k0 = 2 sin(k0 theta)/r as 4 pairs; Wt[j] = 2 cos(j S theta) for j = 1 .. J-1.
// Seeds: folded sine / cosine of theta/2 by polynomial, then double-angle / three-term steps, each a single rounding, so
// relative accuracy survives small theta.  T_n = 2 sin(n theta), c_n = 2 cos(n theta).
// Weights: 2 cos(S theta) by its own polynomial on the reduced angle of S theta (not by doubling 2 cos(theta): the
// correlated roundings of that route leave a coherent phase bias); then two interleaved Chebyshev
// chains of stride 2 (W_j = W_2 W_{j-2} - W_{j-4}, W_0 = 2, W_{-1} = W_1), which halves the dependency depth.  An error
// d of 2 cos(S theta) changes W_j by at most j^2 d (6e-8 x 256 = 1.5e-5 of the term at j = 16, pseudo-random over pairs).
template <int MODE, int J>
__device__ __forceinline__ void prod_vals(const RecurGeom &g, const RecurConst &rc, u64 (&U)[4], float (&Wt)[J])
{
    (void)rc;
    const float rinv = g.rinv;
    const Folded h = sincos_fold(g.f1);                // g.f1 = theta / 2 pi reduced: pi f1 = theta / 2
    const float T1 = two_sin_from(h, g.f1);
    const float c1 = two_cos_from(h);
    const float c2 = fmaf(-T1, T1, 2.0f);
    const float c4 = fmaf(c2, c2, -2.0f);     // used for ONE (two for chunk 1 of 2) bootstrap step only: its absolute error of
                                              // one rounding costs 1e-7 relative in u5..u16, no relative accuracy needed
    float u[17];
    u[1] = T1 * rinv; u[2] = c1 * u[1]; u[3] = fmaf(c1, u[2], -u[1]); u[4] = c2 * u[2];
    u[5] = fmaf(c4, u[1], u[3]); u[6] = fmaf(c4, u[2], u[2]); u[7] = fmaf(c4, u[3], u[1]); u[8] = c4 * u[4];
    if constexpr (MODE == RM_P2B) {
#pragma unroll
        for (int n = 9; n <= 16; ++n) u[n] = fmaf(c4, u[n - 4], -u[n - 8]);
        U[0] = pk2(u[9], u[10]); U[1] = pk2(u[11], u[12]); U[2] = pk2(u[13], u[14]); U[3] = pk2(u[15], u[16]);
    } else {
        U[0] = pk2(u[1], u[2]); U[1] = pk2(u[3], u[4]); U[2] = pk2(u[5], u[6]); U[3] = pk2(u[7], u[8]);
    }
    const float cS = two_cos_from(sincos_fold(g.fS));
    if constexpr (J > 1) Wt[1] = cS;
    if constexpr (J > 2) Wt[2] = fmaf(cS, cS, -2.0f);
    if constexpr (J > 3) Wt[3] = fmaf(Wt[2], cS, -cS);
    if constexpr (J > 4) Wt[4] = fmaf(Wt[2], Wt[2], -2.0f);
#pragma unroll
    for (int j = 5; j < J; ++j) Wt[j] = fmaf(Wt[2], Wt[j - 2], -Wt[j - 4]);
    Wt[0] = 1.0f;
}
// Stage C: the outer product.  acc[4 j + a] (slots 8 j + 2 a, 8 j + 2 a + 1) += W_j * U[a]; level 0 has W_0 = 1.
// All K/2 packed operations are independent of one another.
template <int K>
__device__ __forceinline__ void prod_hot(u64 (&acc)[K / 2], const u64 (&U)[4], const float (&Wt)[(K + 7) / 8])
{
    // the compiler orders the K/2 independent packed operations; fixed orders (seed pair or weight outermost, so that one
    // operand stays in the reuse cache) and scalar FFMA were measured on B200 and are slower (profiles/r02_product_form.md)
#pragma unroll
    for (int a = 0; a < 4; ++a)
        if (2 * a < K) acc[a] = add2(acc[a], U[a]);
#pragma unroll
    for (int j = 1; j < (K + 7) / 8; ++j) {
        const u64 wj = pk2(Wt[j], Wt[j]);               // SASS: the scalar-broadcast operand form of FFMA2, no copy
#pragma unroll
        for (int a = 0; a < 4; ++a)
            if (8 * j + 2 * a < K) acc[4 * j + a] = fma2(wj, U[a], acc[4 * j + a]);     // K % 8 == 4: the last level has 4 slots
    }
}

// One shared-memory tile of j atoms against this thread's i atom, product form, NP pairs per iteration.  Stage A of group
// jj + 2 NP and stage B of group jj + NP sit in the same basic block as the outer products of group jj, so the scheduler
// hides their dependency chains (distance, rsqrt, range reduction, polynomials, seed and weight chains: ~70 dependent
// FP32 instructions) under the independent packed instructions.
#define DEBYE_PRAGMA_(x) _Pragma(#x)
#define DEBYE_PRAGMA(x) DEBYE_PRAGMA_(x)
#ifdef DEBYE_PROD_UNROLL
#define DEBYE_PROD_UNROLL_PRAGMA DEBYE_PRAGMA(unroll DEBYE_PROD_UNROLL)
#else
#define DEBYE_PROD_UNROLL_PRAGMA
#endif
// pairs per iteration: two or three (amortises the loop overhead and gives the scheduler independent start-up chains).  Measured
// on B200: two against one +4 % cfg2, +9 % cfg3, +4 % cfg4, +6 % cfg5; three against two on a 10 000-atom structure, T pair.q/s by
// K: 24 6.79/6.83, 32 8.61/8.18, 40 9.45/9.59, 48 10.32/10.42, 56 11.63/11.52, 64 12.67/12.05, 72 12.96/12.72, 80 14.13/13.90,
// 88 14.66/14.54, 96 14.31/14.62, 100 13.54/15.18, 104 13.49/15.09 (2.4 KB of spills at 168 registers), 112 15.55/14.70,
// 120 16.00/15.82, 128 16.84/16.02; cfg4 (K = 64) 0.710 -> 0.757, cfg5 (K = 128) 1.014 -> 1.076 of the 2-lane-op roofline
#ifdef DEBYE_NPP
__host__ __device__ constexpr int prod_np(int K) { return DEBYE_NPP; }
#else
__host__ __device__ constexpr int prod_np(int K) { return ((K >= 56 && K <= 88) || K >= 112 || K == 32) ? 3 : 2; }
#endif
template <int K, int MODE, bool W>
__device__ __forceinline__ void prod_tile(u64 (&acc)[K / 2], const float4 *__restrict__ tile, const int jj0, const int cnt, const float4 pi,
                                          const bool ivalid, const bool diag, const int i_local, const int jl0, const RecurConst &rc,
                                          const int jfree /* warp-uniform: every lane may pair with every tile index >= jfree */)
{
    constexpr int NP = prod_np(K), J = (K + 7) / 8;
    if (jj0 >= cnt) return;
    // first tile index this thread may pair with: masks i >= j on the diagonal and threads without an i atom
    const int jmin = ivalid ? (diag ? max(0, i_local + 1 - jl0) : 0) : 0x7fffffff;
    // masked pairs (before jmin, behind the last atom of the tile: the pipeline reads two groups ahead) get 1/r = 0 and with
    // it seeds that are exactly 0; their coordinates are read from a VALID entry of this tile (index clamp), so that a
    // stale non-finite entry behind the tile can never reach the accumulators (0 * NaN)
    auto geom_masked = [&](const int jbase, RecurGeom (&g)[NP]) {
#pragma unroll
        for (int p = 0; p < NP; ++p) {
            const int j = jbase + p;
            recur_geom<MODE, W>(tile[min(j, cnt - 1)], pi, j >= jmin && j < cnt, rc, g[p]);
        }
    };
    auto geom_free = [&](const int jbase, RecurGeom (&g)[NP]) {
#pragma unroll
        for (int p = 0; p < NP; ++p) recur_geom<MODE, W>(tile[jbase + p], pi, true, rc, g[p]);
    };
    u64 U[NP][4];
    float Wt[NP][J];
    RecurGeom gn[NP];
    geom_masked(jj0, gn);
#pragma unroll
    for (int p = 0; p < NP; ++p) prod_vals<MODE, J>(gn[p], rc, U[p], Wt[p]);
    geom_masked(jj0 + NP, gn);
    // one iteration: stage B of group jj + NP, stage A of group jj + 2 NP, outer products of group jj
#define DEBYE_PROD_ITER(GEOM)                                                                        \
    {                                                                                                \
        u64 Un[NP][4];                                                                               \
        float Wn[NP][J];                                                                             \
        _Pragma("unroll") for (int p = 0; p < NP; ++p) prod_vals<MODE, J>(gn[p], rc, Un[p], Wn[p]);  \
        GEOM(jj + 2 * NP, gn);                                                                       \
        _Pragma("unroll") for (int p = 0; p < NP; ++p) prod_hot<K>(acc, U[p], Wt[p]);                \
        _Pragma("unroll") for (int p = 0; p < NP; ++p) {                                             \
            _Pragma("unroll") for (int a = 0; a < 4; ++a) U[p][a] = Un[p][a];                        \
            _Pragma("unroll") for (int j = 0; j < J; ++j) Wt[p][j] = Wn[p][j];                       \
        }                                                                                            \
    }
    // The interior of a tile needs no mask: all lanes have an i atom below every j of the group whose geometry the iteration
    // computes (jj + 2 NP .. jj + 3 NP - 1 in [jfree, cnt)).  The bounds are warp-uniform; the masked copy of the loop runs the
    // head (diagonal) and the tail of the tile, and whole tiles of warps with a lane that has no i atom (jfree = INT_MAX).
    int jj = jj0;
#pragma unroll 1
    for (int phase = 0; phase < 2; ++phase) {
        const int stop = (phase == 0) ? ((jfree > cnt) ? cnt : min(cnt, max(jj0, jfree - 2 * NP))) : cnt;
#pragma unroll 1
        for (; jj < stop; jj += NP) DEBYE_PROD_ITER(geom_masked)
        if (phase == 0) {
            DEBYE_PROD_UNROLL_PRAGMA
            for (; jj + 3 * NP <= cnt; jj += NP) DEBYE_PROD_ITER(geom_free)
        }
    }
#undef DEBYE_PROD_ITER
}

// ---- centred product form (V_CENT): any uniform piece q = q_s + m dq, 1 lane-operation per term, no telescoping -----------
// With phi = q_c r the angle of a seed and delta a multiple of theta = r dq,
//     2 cos(delta) * 2 sin(phi)/r = 2 [sin(phi + delta) + sin(phi - delta)]/r        =: P
//     2 sin(delta) * 2 cos(phi)/r = 2 [sin(phi + delta) - sin(phi - delta)]/r        =: Q
// so two packed FMA lanes (one into P, one into Q) serve TWO terms, the ones at q_c + delta/r and q_c - delta/r:
//     sum_pairs 4 sin((q_c +/- delta/r) r)/r = P +/- Q            (taken in FP64 by the epilogue).
// Per pair: 8 sine and 8 cosine seeds at phi_k0 = (q_c + k0 dq) r, k0 = 0..7 (q_c in the middle of the piece), and L weight
// pairs 2cos(delta_j), 2sin(delta_j).  K = 16 L + 8: delta_j = 8 j theta and the seeds themselves are level 0 (slots 0..7 hold
// 2 sin(phi_k0)/r); K = 16 L: delta_j = (8 j - 4) theta, no level 0.  Local index m of the piece (q = q_s + m dq):
//     K = 16 L + 8:  seed k0 <-> m = 8 L + k0;      (k0, +j) <-> m = 8 L + k0 + 8 j;      (k0, -j) <-> m = 8 L + k0 - 8 j
//     K = 16 L:                                     (k0, +j) <-> m = 8 L + k0 + 8 (j - 1); (k0, -j) <-> m = 8 L + k0 - 8 j
// Slots: [level 0: 8] then per level j = 1..L: P_j[k0] (8 slots), Q_j[k0] (8 slots).  Unlike the telescoped form nothing is
// chained across q, the start q_s is arbitrary (general-start grids, the pieces of a piecewise-uniform grid), and every
// step of the start-up keeps relative accuracy for small angles (coincident atoms: r = 1e-15 gives the limits 2 q).
struct CentConst {
    float wc, wc_lo;         // q of seed k0 = 0, / 2 pi, hi + lo
    float w1, w1_lo;         // dq / 2 pi
    float smult;             // 8 (K % 16 == 8) or 4 (K % 16 == 0): fS = smult * theta
};
struct CentGeom { float rinv, fc, f1, fS; };
template <bool W>
__device__ __forceinline__ void cent_geom(const float4 pj, const float4 pi, const bool ok, const CentConst &cc, CentGeom &g)
{
    const float dx = pj.x - pi.x, dy = pj.y - pi.y, dz = pj.z - pi.z;
    const float r2c = fmaf(dx, dx, fmaf(dy, dy, fmaf(dz, dz, 1e-30f)));       // as recur_geom
    const float rinv = rsqrt_mufu(r2c);
    const float r = r2c * rinv;
    if constexpr (W) g.rinv = ok ? rinv * pj.w : 0.0f;
    else g.rinv = ok ? rinv : 0.0f;
    g.fc = reduce_turns(r, cc.wc, cc.wc_lo);
    reduce_turns_pair(r, cc.w1, cc.w1_lo, cc.smult, g.f1, g.fS);
}
// Stage B.  Us / Uc: the 8 seeds 2 sin(phi_k0)/r and 2 cos(phi_k0)/r as 4 pairs each; Cw[j], Sw[j] = 2 cos(delta_j), 2 sin(delta_j).
// Seeds: sine and cosine of phi_0 and of theta by the folded polynomials, one exact rotation to phi_1, then the three-term
// recurrence x_{n+1} = 2cos(theta) x_n - x_{n-1} (six steps: rounding errors grow by at most n^2/2 and are unbiased).  Weights:
// the same recurrence in steps of 8 theta from the polynomial values at 8 theta (or 4 theta and one doubling).
template <int K>
__device__ __forceinline__ void cent_vals(const CentGeom &g, u64 (&Us)[4], u64 (&Uc)[4], float (&Cw)[K / 16 + 1], float (&Sw)[K / 16 + 1])
{
    constexpr bool HAS0 = (K % 16) == 8;
    constexpr int L = K / 16;
    const Folded hc = sincos_fold(g.fc);
    float s[8], c[8];
    s[0] = two_sin_from(hc, g.fc) * g.rinv;
    c[0] = two_cos_from(hc) * g.rinv;
    const Folded h1 = sincos_fold(g.f1);
    const float S1 = two_sin_from(h1, g.f1), C1 = two_cos_from(h1);
    const float hs = 0.5f * S1, hk = 0.5f * C1;
    s[1] = fmaf(c[0], hs, s[0] * hk);
    c[1] = fmaf(-s[0], hs, c[0] * hk);
#pragma unroll
    for (int n = 2; n < 8; ++n) { s[n] = fmaf(C1, s[n - 1], -s[n - 2]); c[n] = fmaf(C1, c[n - 1], -c[n - 2]); }
#pragma unroll
    for (int a = 0; a < 4; ++a) { Us[a] = pk2(s[2 * a], s[2 * a + 1]); Uc[a] = pk2(c[2 * a], c[2 * a + 1]); }
    if constexpr (L >= 1) {
        const Folded hS = sincos_fold(g.fS);
        const float SS = two_sin_from(hS, g.fS), CS = two_cos_from(hS);
        Cw[0] = 0.f; Sw[0] = 0.f;
        Cw[1] = CS; Sw[1] = SS;
        if constexpr (HAS0) {            // delta_j = 8 j theta: T_0 = (2, 0)
            if constexpr (L >= 2) { Cw[2] = fmaf(CS, CS, -2.0f); Sw[2] = CS * SS; }
#pragma unroll
            for (int j = 3; j <= L; ++j) { Cw[j] = fmaf(CS, Cw[j - 1], -Cw[j - 2]); Sw[j] = fmaf(CS, Sw[j - 1], -Sw[j - 2]); }
        } else {                         // delta_j = (8 j - 4) theta: step 8 theta, T_0 = (2cos(4 theta), -2 sin(4 theta))
            const float C8 = fmaf(CS, CS, -2.0f);
            if constexpr (L >= 2) { Cw[2] = fmaf(C8, CS, -CS); Sw[2] = fmaf(C8, SS, SS); }
#pragma unroll
            for (int j = 3; j <= L; ++j) { Cw[j] = fmaf(C8, Cw[j - 1], -Cw[j - 2]); Sw[j] = fmaf(C8, Sw[j - 1], -Sw[j - 2]); }
        }
    } else { Cw[0] = 0.f; Sw[0] = 0.f; }
}
// Stage C: K/2 independent packed operations.
template <int K>
__device__ __forceinline__ void cent_hot(u64 (&acc)[K / 2], const u64 (&Us)[4], const u64 (&Uc)[4], const float (&Cw)[K / 16 + 1], const float (&Sw)[K / 16 + 1])
{
    constexpr bool HAS0 = (K % 16) == 8;
    constexpr int L = K / 16, B0 = HAS0 ? 4 : 0;
    if constexpr (HAS0) {
#pragma unroll
        for (int a = 0; a < 4; ++a) acc[a] = add2(acc[a], Us[a]);
    }
#pragma unroll
    for (int j = 1; j <= L; ++j) {
        const u64 wc = pk2(Cw[j], Cw[j]), ws = pk2(Sw[j], Sw[j]);
#pragma unroll
        for (int a = 0; a < 4; ++a) acc[B0 + 8 * (j - 1) + a] = fma2(wc, Us[a], acc[B0 + 8 * (j - 1) + a]);
#pragma unroll
        for (int a = 0; a < 4; ++a) acc[B0 + 8 * (j - 1) + 4 + a] = fma2(ws, Uc[a], acc[B0 + 8 * (j - 1) + 4 + a]);
    }
}
// where local index m of a piece lives: slot of P (or of the level-0 seed), slot of Q (-1: none), sign of Q, and the factor
// that turns the slot sum(s) into sum_pairs sin(q r)/r.  Used by the epilogue.
__host__ __device__ inline void cent_slot_of(int K, int m, int &lp, int &lq, double &sgn, double &scale)
{
    const bool has0 = (K % 16) == 8;
    const int L = K / 16, b0 = has0 ? 8 : 0;
    if (has0 && m >= 8 * L && m < 8 * L + 8) { lp = m - 8 * L; lq = -1; sgn = 0.0; scale = 0.5; return; }
    int j, k0;
    if (m >= 8 * L) { const int d = m - 8 * L - (has0 ? 8 : 0); j = d / 8 + 1; k0 = d % 8; sgn = 1.0; }
    else { const int d = 8 * L - 1 - m; j = d / 8 + 1; k0 = 7 - d % 8; sgn = -1.0; }
    lp = b0 + 16 * (j - 1) + k0; lq = lp + 8; scale = 0.25;
}
// pairs per iteration and occupancy thresholds, measured on B200 (10 000 atoms; T pair.q/s, one pair per iteration -> two):
// K = 104: 10.8 -> 11.6, 2 x K = 56: 7.75 -> 8.45, K = 128: 12.0 -> 13.1; K = 40 at 4 CTAs/SM 6.83, at 3 CTAs/SM 7.00;
// K = 104 at 3 CTAs/SM (168 registers) 9.9 against 11.6 at 2
#ifndef DEBYE_CENT_NP
#define DEBYE_CENT_NP 2
#endif
#ifndef DEBYE_CK4
#define DEBYE_CK4 24
#endif
#ifndef DEBYE_CK3
#define DEBYE_CK3 88
#endif
__host__ __device__ constexpr int cent_min_ctas(int K) { return K <= DEBYE_CK4 ? 4 : (K <= DEBYE_CK3 ? 3 : 2); }
// One tile, the same three-stage pipeline and masking as prod_tile.
template <int K, bool W>
__device__ __forceinline__ void cent_tile(u64 (&acc)[K / 2], const float4 *__restrict__ tile, const int jj0, const int cnt, const float4 pi,
                                          const bool ivalid, const bool diag, const int i_local, const int jl0, const CentConst &cc, const int jfree)
{
    constexpr int NP = DEBYE_CENT_NP, LW = K / 16 + 1;
    if (jj0 >= cnt) return;
    const int jmin = ivalid ? (diag ? max(0, i_local + 1 - jl0) : 0) : 0x7fffffff;
    auto geom_masked = [&](const int jbase, CentGeom (&g)[NP]) {
#pragma unroll
        for (int p = 0; p < NP; ++p) {
            const int j = jbase + p;
            cent_geom<W>(tile[min(j, cnt - 1)], pi, j >= jmin && j < cnt, cc, g[p]);
        }
    };
    auto geom_free = [&](const int jbase, CentGeom (&g)[NP]) {
#pragma unroll
        for (int p = 0; p < NP; ++p) cent_geom<W>(tile[jbase + p], pi, true, cc, g[p]);
    };
    u64 Us[NP][4], Uc[NP][4];
    float Cw[NP][LW], Sw[NP][LW];
    CentGeom gn[NP];
    geom_masked(jj0, gn);
#pragma unroll
    for (int p = 0; p < NP; ++p) cent_vals<K>(gn[p], Us[p], Uc[p], Cw[p], Sw[p]);
    geom_masked(jj0 + NP, gn);
#define DEBYE_CENT_ITER(GEOM)                                                                                   \
    {                                                                                                           \
        u64 Usn[NP][4], Ucn[NP][4];                                                                             \
        float Cwn[NP][LW], Swn[NP][LW];                                                                         \
        _Pragma("unroll") for (int p = 0; p < NP; ++p) cent_vals<K>(gn[p], Usn[p], Ucn[p], Cwn[p], Swn[p]);     \
        GEOM(jj + 2 * NP, gn);                                                                                  \
        _Pragma("unroll") for (int p = 0; p < NP; ++p) cent_hot<K>(acc, Us[p], Uc[p], Cw[p], Sw[p]);            \
        _Pragma("unroll") for (int p = 0; p < NP; ++p) {                                                        \
            _Pragma("unroll") for (int a = 0; a < 4; ++a) { Us[p][a] = Usn[p][a]; Uc[p][a] = Ucn[p][a]; }       \
            _Pragma("unroll") for (int j = 0; j < LW; ++j) { Cw[p][j] = Cwn[p][j]; Sw[p][j] = Swn[p][j]; }      \
        }                                                                                                       \
    }
    int jj = jj0;
#pragma unroll 1
    for (int phase = 0; phase < 2; ++phase) {
        const int stop = (phase == 0) ? ((jfree > cnt) ? cnt : min(cnt, max(jj0, jfree - 2 * NP))) : cnt;
#pragma unroll 1
        for (; jj < stop; jj += NP) DEBYE_CENT_ITER(geom_masked)
        if (phase == 0) {
            for (; jj + 3 * NP <= cnt; jj += NP) DEBYE_CENT_ITER(geom_free)
        }
    }
#undef DEBYE_CENT_ITER
}

// ---- chain form (RM_G) ----------------------------------------------------------------------------------------------
// Stage B (values): Bv = w_0 (the 8 residues), A = w_{-1}, cS = 2 cos(S theta).
// General start (q_0 not a small multiple of dq, or more than 2 chunks): 8 accurate sines at k' = base .. base+7
// (base = -S + 8 ch), then the stride-4 recurrence v_{n+4} = 2cos(4 theta) v_n - v_{n-4} walks up to k' = 8 ch .. 8 ch + 7
__device__ __forceinline__ void recur_vals(const RecurGeom &g, const RecurConst &rc, const float *wtab, u64 (&A)[4], u64 (&Bv)[4], float &cS)
{
    const float r = g.r, rinv = g.rinv;
    // the chain coefficient 2 cos(S theta) is NOT derived from 2 cos(theta) by repeated doubling: the correlated roundings
    // of that route leave a +7e-8 rad coherent phase bias after 16 steps (fp32 emulation)
    cS = two_cos_from(sincos_fold(g.fS));
    float g0[4], g1[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        g0[j] = two_sin_turns_accurate(r, wtab[j], wtab[8 + j]) * rinv;
        g1[j] = two_sin_turns_accurate(r, wtab[4 + j], wtab[12 + j]) * rinv;
    }
    const float c4 = two_cos_turns(r, rc.w4, rc.w4_lo);
    float a0[4], a1[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) { a0[j] = g0[j]; a1[j] = g1[j]; }
    for (int st = 0; st < 2 * rc.n_chunks; ++st) {
#pragma unroll
        for (int j = 0; j < 4; ++j) { float nx = fmaf(c4, g1[j], -g0[j]); g0[j] = g1[j]; g1[j] = nx; }
    }
    Bv[0] = pk2(g0[0], g0[1]); Bv[1] = pk2(g0[2], g0[3]); Bv[2] = pk2(g1[0], g1[1]); Bv[3] = pk2(g1[2], g1[3]);
    A[0] = pk2(-a0[0], -a0[1]); A[1] = pk2(-a0[2], -a0[3]); A[2] = pk2(-a1[0], -a1[1]); A[3] = pk2(-a1[2], -a1[3]);
}

// Packed hot loop of one pair: w_m = sigma_m v_m with sigma = (+,+,-,-): w_{m+1} = (+/-) cS w_m + w_{m-1}; 4 packed chains
// (8 residues), K/8 steps: per term one FFMA2 lane and one FADD2 lane.  A and Bv are consumed.
template <int K>
__device__ __forceinline__ void recur_hot(u64 (&acc)[K / 2], u64 (&A)[4], u64 (&Bv)[4], const float cS)
{
    const u64 cP = pk2(cS, cS), cN = pk2(-cS, -cS);
#pragma unroll
    for (int m = 0; m < (K + 7) / 8; ++m) {
#pragma unroll
        for (int a = 0; a < 4; ++a) {
            if (8 * m + 2 * a < K) {                       // K % 8 == 4: the last step runs chains 0 and 1 only
                if (m & 2) acc[4 * m + a] = sub2(acc[4 * m + a], Bv[a]);
                else acc[4 * m + a] = add2(acc[4 * m + a], Bv[a]);
                if (8 * (m + 1) + 2 * a < K) {
                    u64 nx = fma2((m & 1) ? cN : cP, Bv[a], A[a]);
                    A[a] = Bv[a];
                    Bv[a] = nx;
                }
            }
        }
    }
}

// Slow path of one pair (theta = r dq at or below theta_min, or coincident atoms), chain form.  The three-term chain loses
// the pair's frequency when 2cos(S theta) rounds next to 2 (relative error of theta^2 is 6e-8 / (S theta)^2), so these pairs
// run Reinsch's form of the same chain, which carries beta = 4 sin^2(S theta / 2) = 2 - 2cos(S theta) with full relative
// accuracy:   d_{m+1} = d_m - beta s_m,   s_{m+1} = s_m + d_{m+1},   s_0 = v(k'_j),  d_0 = v(k'_j) - v(k'_j - S).
// Start values are those of the fast path evaluated with the true 1/r (for r = 0 the clamp r^2 >= 1e-30 makes
// 2 sin(n theta)/r come out as its limit 2 n dq).  Three packed lane-operations per term; rare, so cost is irrelevant.
template <int K, bool W>
__device__ __forceinline__ void recur_slow_pair(u64 (&acc)[K / 2], const float4 pj, const float4 pi, const RecurConst &rc, const float *wtab)
{
    RecurConst rs = rc;
    rs.cut2 = -1.0f;                       // never "small": stage A keeps the true 1/r
    RecurGeom g;
    recur_geom<RM_G, W>(pj, pi, true, rs, g);
    u64 A[4], Bv[4];
    float cS;
    recur_vals(g, rc, wtab, A, Bv, cS);
    (void)cS;
    // beta from the polynomial directly (2 - cS would cancel)
    const float nbeta = -four_sin2_from(sincos_fold(g.fS));
    const u64 nb2 = pk2(nbeta, nbeta);
    // stage B returns A = w_{-1} = -v_{-1} (sign convention of the fast loop): d_0 = v_0 - v_{-1} = Bv + A
    u64 s[4], d[4];
#pragma unroll
    for (int a = 0; a < 4; ++a) { s[a] = Bv[a]; d[a] = add2(Bv[a], A[a]); }
#pragma unroll
    for (int m = 0; m < (K + 7) / 8; ++m) {
#pragma unroll
        for (int a = 0; a < 4; ++a) {
            if (8 * m + 2 * a < K) {
                acc[4 * m + a] = add2(acc[4 * m + a], s[a]);
                if (8 * (m + 1) + 2 * a < K) {
                    d[a] = fma2(nb2, s[a], d[a]);
                    s[a] = add2(s[a], d[a]);
                }
            }
        }
    }
}

// Occupancy policy: the K accumulators dominate the register budget.  Product form: K + ~60 registers.
#ifndef DEBYE_K4
#define DEBYE_K4 64
#endif
#ifndef DEBYE_K3
#define DEBYE_K3 104
#endif
__host__ __device__ constexpr int recur_min_ctas(int K) { return K <= DEBYE_K4 ? 4 : (K <= DEBYE_K3 ? 3 : 2); }

// One shared-memory tile of j atoms against this thread's i atom, chain form, one pair per iteration, the same three-stage
// pipeline as prod_tile.
template <int K, bool W>
__device__ __forceinline__ void recur_tile(u64 (&acc)[K / 2], const float4 *__restrict__ tile, const int jj0, const int cnt, const float4 pi,
                                           const bool ivalid, const bool diag, const int i_local, const int jl0, const RecurConst &rc,
                                           const float *wtab)
{
    if (jj0 >= cnt) return;
    const int jmin = ivalid ? (diag ? max(0, i_local + 1 - jl0) : 0) : 0x7fffffff;
    bool had_slow = false;                // some pair of this thread in this tile needs the slow path (handled after the loop)
    auto geom = [&](const int j, RecurGeom &g) {
        recur_geom<RM_G, W>(tile[min(j, cnt - 1)], pi, j >= jmin && j < cnt, rc, g);
        had_slow = had_slow || g.slow;
    };
    u64 A[4], Bv[4];
    float cS;
    RecurGeom gn;
    geom(jj0, gn);
    recur_vals(gn, rc, wtab, A, Bv, cS);
    geom(jj0 + 1, gn);
    for (int jj = jj0; jj < cnt; ++jj) {
        u64 An[4], Bn[4];
        float cSn;
        recur_vals(gn, rc, wtab, An, Bn, cSn);
        geom(jj + 2, gn);
        recur_hot<K>(acc, A, Bv, cS);
#pragma unroll
        for (int a = 0; a < 4; ++a) { A[a] = An[a]; Bv[a] = Bn[a]; }
        cS = cSn;
    }
    // slow-path pairs (theta at or below theta_min, coincident atoms) contributed exactly zero above; they are rare, so
    // the tile is rescanned for them only if some lane of the warp met one
    if (__any_sync(0xffffffffu, had_slow)) {
        if (had_slow) {
            for (int j = max(jj0, jmin); j < cnt; ++j) {
                const float4 pj = tile[j];
                const float dx = pj.x - pi.x, dy = pj.y - pi.y, dz = pj.z - pi.z;
                const float r2c = fmaf(dx, dx, fmaf(dy, dy, fmaf(dz, dz, 1e-30f)));       // as in recur_geom
                if (!(r2c > rc.cut2)) recur_slow_pair<K, W>(acc, pj, pi, rc, wtab);
            }
        }
    }
}

// ---- MUFU variant (any grid): one tile, software pipelined ---------------------------------------------------------------
// One MUFU.SIN per term.  The XU pipe takes one per 8 cycles and scheduler, so the loop is bound by it as long as a MUFU.SIN is
// always ready to issue: the geometry of pair jj + 1 (tile load, distance, MUFU.RSQ) is computed in the same basic block as the
// K terms of pair jj, and pairs below the accuracy cut (theta small: MUFU's absolute error matters; coincident atoms) contribute
// exactly zero here (1/r := 0) and are redone term by term in a rescan of the tile that runs only if some lane met one -- a vote
// and a branch per pair would end the basic block at every pair.
template <int K, bool W>
__device__ __forceinline__ void mufu_tile(u64 (&acc)[K / 2], const float4 *__restrict__ tile, const float *__restrict__ qs, const int jj0, const int cnt,
                                          const float4 pi, const bool ivalid, const bool diag, const int i_local, const int jl0, const float cut2)
{
    if (jj0 >= cnt) return;
    const int jmin = ivalid ? (diag ? max(0, i_local + 1 - jl0) : 0) : 0x7fffffff;
    bool had_slow = false;
    auto geom = [&](const int j, float &rt, float &rinv) {
        const float4 pj = tile[min(j, cnt - 1)];
        const float dx = pj.x - pi.x, dy = pj.y - pi.y, dz = pj.z - pi.z;
        const float r2 = fmaf(dx, dx, fmaf(dy, dy, dz * dz));
        const bool small = !(r2 > cut2), ok = j >= jmin && j < cnt;
        const float r2c = fmaxf(r2, 1e-30f);
        const float ri = rsqrt_mufu(r2c);
        rt = (r2c * ri) * 0.15915494309189535f;                 // r / 2 pi: turns = q_k * rt
        rinv = (ok && !small) ? (W ? ri * pj.w : ri) : 0.0f;
        had_slow = had_slow || (small && ok);
    };
    float rt, rinv;
    geom(jj0, rt, rinv);
    for (int jj = jj0; jj < cnt; ++jj) {
        float rtn, rinvn;
        geom(jj + 1, rtn, rinvn);
        const u64 rinv2 = pk2(rinv, rinv);
#pragma unroll
        for (int l = 0; l < K; l += 4) {
            const float4 q4 = *reinterpret_cast<const float4 *>(&qs[l]);
            acc[l / 2] = fma2(pk2(sin_turns_fma(rt, q4.x), sin_turns_fma(rt, q4.y)), rinv2, acc[l / 2]);
            acc[l / 2 + 1] = fma2(pk2(sin_turns_fma(rt, q4.z), sin_turns_fma(rt, q4.w)), rinv2, acc[l / 2 + 1]);
        }
        rt = rtn; rinv = rinvn;
    }
    if (__any_sync(0xffffffffu, had_slow)) {
        if (had_slow) {
            for (int j = max(jj0, jmin); j < cnt; ++j) {
                const float4 pj = tile[j];
                const float dx = pj.x - pi.x, dy = pj.y - pi.y, dz = pj.z - pi.z;
                const float r2 = fmaf(dx, dx, fmaf(dy, dy, dz * dz));
                if (!(r2 > cut2)) {
                    const float rs = sqrtf(r2);
#pragma unroll
                    for (int l = 0; l < K; ++l) {
                        const float qk = qs[l];
                        float tv = (rs == 0.0f) ? qk : term_accurate(qk, rs);
                        if constexpr (W) tv *= pj.w;
                        float lo_, hi_;
                        upk2(acc[l / 2], lo_, hi_);
                        if (l & 1) hi_ += tv; else lo_ += tv;
                        acc[l / 2] = pk2(lo_, hi_);
                    }
                }
            }
        }
    }
}

// direct variants (MUFU, accurate): CTAs per SM by accumulator count.  The pipelined MUFU loop needs K + ~75 registers: with
// more CTAs per SM than these it spills inside the loop (K = 104 at 3 CTAs/SM, 168 registers: 1.3 KB of spills, 1.36 T
// pair.q/s on cfg2 against 3.22 T at 2 CTAs/SM)
#ifndef DEBYE_MK4
#define DEBYE_MK4 48
#endif
#ifndef DEBYE_MK3
#define DEBYE_MK3 72
#endif
#ifndef DEBYE_FLUSH_J
#define DEBYE_FLUSH_J 512
#endif

#ifdef DEBYE_TRACE
__device__ unsigned long long debye_trace[3 * 4096];
#endif
template <int K, int VAR, bool W, bool SH = false>
__global__ void __launch_bounds__(DEBYE_IB, (VAR == V_F64) ? 1 : (VAR == V_RECUR ? recur_min_ctas(K) : (VAR == V_CENT ? cent_min_ctas(K) : (K <= DEBYE_MK4 ? 4 : (K <= DEBYE_MK3 ? 3 : 2))))) debye_pairs_kernel(const DevPlan *__restrict__ plan, const float4 *__restrict__ sorted, const float *__restrict__ qv,
                                                               double *__restrict__ records, int n_chunks, int is_auto, float theta_min, int alt_gate)
{
    pdl_wait();      // programmatic dependent launch: everything before us in the call has completed (debye_plan.cuh)
    // ---- variant gate (decided on the device so the host never reads q) ---------------------------------------
    if (is_auto) {
        if (plan->variant_auto != VAR) return;
    } else if (VAR == V_RECUR && !plan->uniform) {
        return;   // the final kernel writes NaN in this case
    }
    // recurrence: two accumulator counts may be launched (grid starting at q = 0 needs one chain index fewer, and the
    // host cannot know); alt_gate = 1 runs only if the device chose the smaller one, 0 only if not, -1 always
    if (VAR == V_RECUR && alt_gate >= 0 && plan->recur_alt != alt_gate) return;
    constexpr bool F64 = (VAR == V_F64);
    constexpr int NW = DEBYE_IB / 32;
    __shared__ __align__(128) float4 tile[2][DEBYE_JT + DEBYE_TILE_PAD];
    __shared__ __align__(8) u64 mbar[2];
    __shared__ float tbuf[F64 ? 1 : NW][F64 ? 1 : 32][F64 ? 1 : 33];
    __shared__ double wsum[NW][K];
    __shared__ __align__(16) float qs[(VAR == V_RECUR || VAR == V_CENT) ? 4 : K];
    __shared__ float wtab[16];                        // recurrence, general start: start frequencies (hi[8], lo[8])    // direct variants: q of each local slot (0 for padding)

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int G = gridDim.x, c = blockIdx.x;
    const int N = plan->N, n_tp = plan->n_tp, Bn = plan->B, M = plan->M;
    const int64_t U1 = plan->U1;
    const int64_t Uc = U1 * n_chunks;            // units per conformer
    const int64_t U = Uc * Bn;
    if (U == 0) return;
    const int64_t u0 = debye_range_begin(U, c, G);
    const int64_t u1 = (c + 1 == G) ? U : debye_range_begin(U, c + 1, G);
    if (u0 >= u1) return;
    // tile split of one structure over GPUs (cyclic, which keeps the triangular load balanced): the records of
    // the CTAs that belong to other ranks were zeroed by the host-side memset of debye_partials_shard.  A template parameter,
    // so that the single-GPU instantiations stay instruction for instruction what they were (their register allocation
    // decides +- 4 %: the same test as a run-time branch cost cfg2 0.614 -> 0.587).
    if constexpr (SH) { if (c % plan->shard_world != plan->shard_rank) return; }

#ifdef DEBYE_TRACE      // working builds only: per-CTA start / end time and SM id
    if (tid == 0) { unsigned long long t; unsigned sm; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t)); asm volatile("mov.u32 %0, %%smid;" : "=r"(sm)); debye_trace[3 * c] = t; debye_trace[3 * c + 2] = sm; }
#endif
    // every entry finite from the start: the recurrence pipeline reads up to DEBYE_TILE_PAD entries past the atoms of a tile
    for (int x = tid; x < 2 * (DEBYE_JT + DEBYE_TILE_PAD); x += DEBYE_IB) (&tile[0][0])[x] = make_float4(0.f, 0.f, 0.f, 0.f);
    if (tid == 0) { mbar_init(&mbar[0], 1); mbar_init(&mbar[1], 1); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    __syncthreads();
    uint32_t phase0 = 0, phase1 = 0;

    PairAcc<K, VAR> acc;
#pragma unroll
    for (int i = 0; i < PairAcc<K, VAR>::NE; ++i) acc.v[i] = 0;
    double run = 0.0;                 // thread k < K owns the FP64 running sum of local slot k
    int64_t curX = -1;
    int pending = 0;

    // recurrence constants (rebuilt when the q-chunk changes)
    const double dq_d = plan->dq, q0_d = plan->q0;
    const int koff = plan->zero_start;           // >= 0: grid is (k + koff) dq with koff small; -1: general
    RecurConst rc;
    rc.w1 = rc.w1_lo = rc.wS = rc.wS_lo = rc.w4 = rc.w4_lo = rc.cut2 = 0.f;
    rc.smult = 8.0f;
    rc.n_chunks = n_chunks;
    float cut2 = 0.f;
    int mode = RM_G, ch_cur = 0;
    (void)mode; (void)dq_d; (void)q0_d; (void)koff; (void)cut2;
    CentConst cc;
    cc.wc = cc.wc_lo = cc.w1 = cc.w1_lo = 0.f; cc.smult = 8.0f;
    (void)cc;

    float wi = 1.0f;                  // weighted instantiations: weight of this thread's i atom (accumulators are flushed per row)
    (void)wi;
    auto flush = [&]() {
        // FP32 -> FP64, fixed order.  Each warp transposes 32 slots x 32 lanes through tbuf; lane l sums slot
        // 32 s + l over the 32 lanes in lane order; then threads k < K add the 4 warp sums in warp order.
        if constexpr (!F64) {
#pragma unroll
            for (int s = 0; s < (K + 31) / 32; ++s) {
#pragma unroll
                for (int t = 0; t < 32; t += 2) {
                    int l = 32 * s + t;
                    if (l < K) {
                        float lo, hi;
                        upk2(acc.v[l / 2], lo, hi);
                        if constexpr (W) { lo *= wi; hi *= wi; }
                        tbuf[warp][t][lane] = lo;
                        tbuf[warp][t + 1][lane] = hi;
                        acc.v[l / 2] = 0;
                    }
                }
                __syncwarp();
                if (32 * s + lane < K) {
                    double sum = 0.0;
#pragma unroll
                    for (int j = 0; j < 32; ++j) sum += (double)tbuf[warp][lane][j];
                    wsum[warp][32 * s + lane] = sum;
                }
                __syncwarp();
            }
        } else {
#pragma unroll
            for (int l = 0; l < K; ++l) {
                double v = acc.v[l];
                if constexpr (W) v *= (double)wi;
                acc.v[l] = 0;
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);   // xor tree: same order every run
                if (lane == 0) wsum[warp][l] = v;
            }
        }
        __syncthreads();
        if (tid < K) {
            double s = 0.0;
#pragma unroll
            for (int w = 0; w < NW; ++w) s += wsum[w][tid];
            run += s;
        }
        __syncthreads();
    };
    auto write_record = [&](int64_t X) {
        if (tid < K) { records[((int64_t)c + X) * K + tid] = run; run = 0.0; }
    };

    int64_t u = u0;
    while (u < u1) {
        // ---- decode unit u -> (conformer, type pair, chunk, row, first j) -------------------------------------
        const int b = (int)(u / Uc);
        const int64_t w = u % Uc;
        int lo = 0, hi = n_tp;                    // largest tp with tp_prefix[tp]*n_chunks <= w
        while (hi - lo > 1) { int mid = (lo + hi) >> 1; if (plan->tp_prefix[mid] * n_chunks <= w) lo = mid; else hi = mid; }
        const int tp = lo;
        const int64_t tp_units = plan->tp_prefix[tp + 1] - plan->tp_prefix[tp];
        const int64_t w2 = w - plan->tp_prefix[tp] * n_chunks;
        const int ch = (int)(w2 / tp_units);
        const int64_t v = w2 % tp_units;
        const int ti = plan->tp_ti[tp], tj = plan->tp_tj[tp];
        const bool diag = (ti == tj);
        const int n_i = plan->n_a[ti], n_j = plan->n_a[tj];
        int row; int64_t jo, row_units;
        if (!diag) { row = (int)(v / n_j); jo = v % n_j; row_units = n_j; }
        else {
            int rl = 0, rh = debye_diag_rows(n_i);
            while (rh - rl > 1) { int mid = (rl + rh) >> 1; if (debye_diag_row_prefix(n_i, mid) <= v) rl = mid; else rh = mid; }
            row = rl; jo = v - debye_diag_row_prefix(n_i, row); row_units = (int64_t)n_i - 1 - (int64_t)row * DEBYE_IB;
        }
        const int len = (int)min((int64_t)(u1 - u), row_units - jo);
        const int64_t X = ((int64_t)b * n_tp + tp) * n_chunks + ch;

        if (X != curX) {
            if (curX >= 0) { if (pending) flush(); pending = 0; write_record(curX); }
            curX = X;
            if (ch != ch_cur || u == u0) {
                ch_cur = ch;
                if constexpr (VAR == V_RECUR) {
                    const int S = 8 * n_chunks;
                    // zero-start modes: grid (k + koff) dq with koff in {0, 1} and at most 2 chunks; else general start,
                    // which takes the grid as q0 + k dq whatever q0 is
                    const bool zs = (koff >= 0 && n_chunks <= 2);
                    mode = zs ? (n_chunks == 1 ? RM_P1 : (ch == 0 ? RM_P2A : RM_P2B)) : RM_G;
                    const double qb = q0_d;                               // general start: q of chain index 0
                    const int base = -S + 8 * ch;                         // k' of the first start value
                    __syncthreads();
                    if (tid < 8) {   // turns per Angstrom of the 8 general-start values, hi and lo parts
                        const double wd = (qb + (double)(base + tid) * dq_d) * 0.15915494309189535;
                        const float wh = (float)wd;
                        wtab[tid] = wh; wtab[8 + tid] = (float)(wd - (double)wh);
                    }
                    __syncthreads();
                    const double w1_d = dq_d * 0.15915494309189535;
                    rc.w1 = (float)w1_d; rc.w1_lo = (float)(w1_d - (double)rc.w1);
                    const double wS_d = (double)S * dq_d * 0.15915494309189535, w4_d = 4.0 * dq_d * 0.15915494309189535;
                    rc.wS = (float)wS_d; rc.wS_lo = (float)(wS_d - (double)rc.wS);
                    rc.smult = (float)S;
                    rc.w4 = (float)w4_d; rc.w4_lo = (float)(w4_d - (double)rc.w4);
                    const float rcut = theta_min / fabsf((float)dq_d);
                    rc.cut2 = rcut * rcut;
                } else if constexpr (VAR == V_CENT) {
                    // piece ch of the grid: q = q0 + m dq; seed k0 = 0 sits at local index mc (cent_slot_of)
                    constexpr int mc = (K % 16 == 8) ? 8 * (K / 16) : 8 * (K / 16) - 4;
                    const double pdq = plan->pieces.dq[ch];
                    const double wc_d = fma((double)mc, pdq, plan->pieces.q0[ch]) * 0.15915494309189535, w1_d = pdq * 0.15915494309189535;
                    cc.wc = (float)wc_d; cc.wc_lo = (float)(wc_d - (double)cc.wc);
                    cc.w1 = (float)w1_d; cc.w1_lo = (float)(w1_d - (double)cc.w1);
                    cc.smult = (K % 16 == 8) ? 8.0f : 4.0f;
                } else {
                    __syncthreads();
                    if (tid < K) { int k = ch * K + tid; qs[tid] = (k < M) ? qv[k] : 0.0f; }
                    __syncthreads();
                    const float rcut = theta_min / fmaxf(plan->q_small, 1e-30f);
                    cut2 = (plan->q_small > 0.f) ? rcut * rcut : 0.f;
                }
            }
        }

        // ---- this thread's i atom --------------------------------------------------------------------------------
        const int i_local = row * DEBYE_IB + tid;
        const bool ivalid = i_local < n_i;
        const float4 *conf = sorted + (int64_t)b * N;
        float4 pi = conf[plan->seg_off[ti] + (ivalid ? i_local : 0)];
        if constexpr (W) wi = pi.w;
        const int j_first = diag ? (row * DEBYE_IB + 1 + (int)jo) : (int)jo;   // index within the j type segment
        const float4 *src = conf + plan->seg_off[tj] + j_first;
        const int ntile = (len + DEBYE_JT - 1) / DEBYE_JT;

        if (tid == 0) {
            uint32_t bytes = (uint32_t)min(len, DEBYE_JT) * 16u;
            mbar_expect_tx(&mbar[0], bytes);
            bulk_g2s(&tile[0][0], src, bytes, &mbar[0]);
        }
        for (int t = 0; t < ntile; ++t) {
            const int buf = t & 1;
            if (tid == 0 && t + 1 < ntile) {
                uint32_t bytes = (uint32_t)min(len - (t + 1) * DEBYE_JT, DEBYE_JT) * 16u;
                mbar_expect_tx(&mbar[buf ^ 1], bytes);
                bulk_g2s(&tile[buf ^ 1][0], src + (t + 1) * DEBYE_JT, bytes, &mbar[buf ^ 1]);
            }
            if (buf == 0) { mbar_wait(&mbar[0], phase0); phase0 ^= 1; } else { mbar_wait(&mbar[1], phase1); phase1 ^= 1; }
            const int cnt = min(len - t * DEBYE_JT, DEBYE_JT);
            const int jl0 = j_first + t * DEBYE_JT;
            // on the diagonal, a warp whose every i is >= j has nothing to do for that j: start later
            int jj0 = 0;
            if (diag) { int first_i = row * DEBYE_IB + warp * 32; jj0 = max(0, first_i + 1 - jl0); }
            if constexpr (VAR == V_CENT) {
                const int w_last_i = row * DEBYE_IB + warp * 32 + 31;
                const int jfree = (w_last_i >= n_i) ? 0x7fffffff : (diag ? max(0, w_last_i + 1 - jl0) : 0);
                if (row * DEBYE_IB + warp * 32 < n_i) cent_tile<K, W>(acc.v, tile[buf], jj0, cnt, pi, ivalid, diag, i_local, jl0, cc, jfree);
            } else if constexpr (VAR == V_RECUR) {
                // first tile index from which every lane of this warp pairs with every j: 0 off the diagonal, behind the
                // warp's last i atom on it; never if some lane has no i atom (ragged last row)
                const int w_last_i = row * DEBYE_IB + warp * 32 + 31;
                const int jfree = (w_last_i >= n_i) ? 0x7fffffff : (diag ? max(0, w_last_i + 1 - jl0) : 0);
                // a warp none of whose lanes has an i atom (ragged last row of a small type segment) only keeps the barriers
                if (row * DEBYE_IB + warp * 32 < n_i)
                switch (mode) {      // warp-uniform; one copy of the pipelined loop per mode
                    case RM_P1: prod_tile<K, RM_P1, W>(acc.v, tile[buf], jj0, cnt, pi, ivalid, diag, i_local, jl0, rc, jfree); break;
                    case RM_P2A: prod_tile<K, RM_P2A, W>(acc.v, tile[buf], jj0, cnt, pi, ivalid, diag, i_local, jl0, rc, jfree); break;
                    case RM_P2B: prod_tile<K, RM_P2B, W>(acc.v, tile[buf], jj0, cnt, pi, ivalid, diag, i_local, jl0, rc, jfree); break;
                    default: recur_tile<K, W>(acc.v, tile[buf], jj0, cnt, pi, ivalid, diag, i_local, jl0, rc, wtab); break;
                }
            } else if constexpr (VAR == V_MUFU) {
                if (row * DEBYE_IB + warp * 32 < n_i) mufu_tile<K, W>(acc.v, tile[buf], qs, jj0, cnt, pi, ivalid, diag, i_local, jl0, cut2);
            } else {
            for (int jj = jj0; jj < cnt; ++jj) {
                const float4 pj = tile[buf][jj];
                const bool ok = ivalid && (!diag || (jl0 + jj > i_local));
                if constexpr (F64) {
                    double dx = (double)pj.x - (double)pi.x, dy = (double)pj.y - (double)pi.y, dz = (double)pj.z - (double)pi.z;
                    double r = sqrt(dx * dx + dy * dy + dz * dz);
                    if (ok) {
#pragma unroll
                        for (int l = 0; l < K; ++l) {
                            double qk = (double)qs[l];
                            double x = qk * r;
                            const double tv = (x == 0.0) ? qk : sin(x) / r;
                            acc.v[l] += W ? (double)pj.w * tv : tv;
                        }
                    }
                } else {
                    const float dx = pj.x - pi.x, dy = pj.y - pi.y, dz = pj.z - pi.z;
                    const float r2 = fmaf(dx, dx, fmaf(dy, dy, dz * dz));
                    const bool small = !(r2 > cut2);
                    const float r2c = fmaxf(r2, 1e-30f);
                    float rinv = rsqrt_mufu(r2c);
                    const float r = r2c * rinv;
                    rinv = (ok && !small) ? (W ? rinv * pj.w : rinv) : 0.0f;
                    if (__any_sync(0xffffffffu, small && ok)) {
                        if (small && ok) {
                            const float rs = sqrtf(r2);
#pragma unroll
                            for (int l = 0; l < K; ++l) {
                                const float qk = qs[l];
                                float lo_, hi_;
                                upk2(acc.v[l / 2], lo_, hi_);
                                float tv = (rs == 0.0f) ? qk : term_accurate(qk, rs);
                                if constexpr (W) tv *= pj.w;
                                if (l & 1) hi_ += tv; else lo_ += tv;
                                acc.v[l / 2] = pk2(lo_, hi_);
                            }
                        }
                    }
                    if constexpr (VAR == V_MUFU) {
                        const float rt = r * 0.15915494309189535f;            // r / 2 pi: turns = q_k * rt
                        // The XU pipe takes one MUFU.SIN per 8 cycles and scheduler (16 lanes per clock and SM), so the loop must
                        // issue fewer than 8 instructions per term to be bound by it: four q per LDS.128 (was one LDS per
                        // term) and the scaling by 1/r folded into the accumulation (one packed FMA per two terms instead of
                        // two FMUL and a packed add)
                        const u64 rinv2 = pk2(rinv, rinv);
#pragma unroll
                        for (int l = 0; l < K; l += 4) {
                            const float4 q4 = *reinterpret_cast<const float4 *>(&qs[l]);
                            acc.v[l / 2] = fma2(pk2(sin_turns_fma(rt, q4.x), sin_turns_fma(rt, q4.y)), rinv2, acc.v[l / 2]);
                            acc.v[l / 2 + 1] = fma2(pk2(sin_turns_fma(rt, q4.z), sin_turns_fma(rt, q4.w)), rinv2, acc.v[l / 2 + 1]);
                        }
                    } else {   // V_ACCURATE
#pragma unroll
                        for (int l = 0; l < K; l += 2) {
                            float s0 = sinf(qs[l] * r) * rinv, s1 = sinf(qs[l + 1] * r) * rinv;
                            acc.v[l / 2] = add2(acc.v[l / 2], pk2(s0, s1));
                        }
                    }
                }
            }
            }
            __syncthreads();
            // FP32 -> FP64 at least every DEBYE_FLUSH_J terms per accumulator, also inside a long row segment
            pending += cnt;
            if (pending >= DEBYE_FLUSH_J) { flush(); pending = 0; }
        }
        // weighted calls: the i atom (and with it wi) changes with every row segment, so flush before it does
        if (W && pending) { flush(); pending = 0; }
        u += len;
    }
    if (curX >= 0) { if (pending) flush(); write_record(curX); }
#ifdef DEBYE_TRACE
    if (tid == 0) { unsigned long long t; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t)); debye_trace[3 * c + 1] = t; }
#endif
}

}  // namespace debye
