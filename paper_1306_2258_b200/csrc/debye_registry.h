// debye_registry.h -- lookup of the pairs-kernel instantiations (one per variant and accumulator count K).
#pragma once
#include <cstdint>
#include "debye_plan.cuh"

typedef void (*debye_pairs_fn)(const DevPlan *, const float4 *, const float *, double *, int, int, float, int);

#define DEBYE_KMAX_F32 128
#define DEBYE_KMAX_F64 32

// K must be a multiple of 8 in [8, KMAX] (recurrence: a multiple of 4); returns nullptr otherwise
// sharded: the instantiation whose CTAs skip the tiles of other ranks (debye_partials_shard; unweighted only)
debye_pairs_fn debye_get_pairs_kernel(int variant, int K, bool weighted, bool sharded = false);

// one launch for one small structure (debye_small.cuh): K a multiple of 8 in [8, 128]; nullptr otherwise
typedef void (*debye_small_fn)(const float *, const int32_t *, int, int, const float *, const float *, int, int, double *, double *, int, int32_t *);
debye_small_fn debye_get_small_kernel(int K);

// per-atom form factors on a uniform grid (debye_peratom_recur.cuh): K a multiple of 8 in [8, 128]; nullptr otherwise
namespace debye { struct PeratomPlan; }
typedef void (*debye_peratom_recur_fn)(const float4 *, const float *, const float *, const debye::PeratomPlan *, int, int, int, float, double *, int);
debye_peratom_recur_fn debye_get_peratom_recur_kernel(int K, bool batch);     // batch: several conformers on the unit line

// per-atom form factors, one launch for one small structure (debye_peratom_small.cuh): K a multiple of 8 in [8, 128]; nullptr otherwise
typedef void (*debye_peratom_small_fn)(const float *, const float *, const float *, int, int, int, double *, double *);
debye_peratom_small_fn debye_get_peratom_small_kernel(int K);
