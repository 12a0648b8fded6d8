// pairs_recur_s1.cu -- explicit instantiations of debye_pairs_kernel<K, V_RECUR, unweighted, sharded: debye_partials_shard> (split for parallel builds)
#include "debye_pairs.cuh"
#include "debye_registry.h"
debye_pairs_fn debye_get_recur_s1(int K) {
    switch (K) {
        case 72: return debye::debye_pairs_kernel<72, V_RECUR, false, true>;
        case 80: return debye::debye_pairs_kernel<80, V_RECUR, false, true>;
        case 88: return debye::debye_pairs_kernel<88, V_RECUR, false, true>;
        case 96: return debye::debye_pairs_kernel<96, V_RECUR, false, true>;
        case 104: return debye::debye_pairs_kernel<104, V_RECUR, false, true>;
        case 112: return debye::debye_pairs_kernel<112, V_RECUR, false, true>;
        case 120: return debye::debye_pairs_kernel<120, V_RECUR, false, true>;
        case 128: return debye::debye_pairs_kernel<128, V_RECUR, false, true>;
        default: return nullptr;
    }
}
