// pairs_recur_s2.cu -- explicit instantiations of debye_pairs_kernel<K, V_RECUR, unweighted, sharded: debye_partials_shard> (split for parallel builds)
#include "debye_pairs.cuh"
#include "debye_registry.h"
debye_pairs_fn debye_get_recur_s2(int K) {
    switch (K) {
        case 12: return debye::debye_pairs_kernel<12, V_RECUR, false, true>;
        case 20: return debye::debye_pairs_kernel<20, V_RECUR, false, true>;
        case 28: return debye::debye_pairs_kernel<28, V_RECUR, false, true>;
        case 36: return debye::debye_pairs_kernel<36, V_RECUR, false, true>;
        case 44: return debye::debye_pairs_kernel<44, V_RECUR, false, true>;
        case 52: return debye::debye_pairs_kernel<52, V_RECUR, false, true>;
        case 60: return debye::debye_pairs_kernel<60, V_RECUR, false, true>;
        default: return nullptr;
    }
}
