// pairs_recur_s3.cu -- explicit instantiations of debye_pairs_kernel<K, V_RECUR, unweighted, sharded: debye_partials_shard> (split for parallel builds)
#include "debye_pairs.cuh"
#include "debye_registry.h"
debye_pairs_fn debye_get_recur_s3(int K) {
    switch (K) {
        case 68: return debye::debye_pairs_kernel<68, V_RECUR, false, true>;
        case 76: return debye::debye_pairs_kernel<76, V_RECUR, false, true>;
        case 84: return debye::debye_pairs_kernel<84, V_RECUR, false, true>;
        case 92: return debye::debye_pairs_kernel<92, V_RECUR, false, true>;
        case 100: return debye::debye_pairs_kernel<100, V_RECUR, false, true>;
        case 108: return debye::debye_pairs_kernel<108, V_RECUR, false, true>;
        case 116: return debye::debye_pairs_kernel<116, V_RECUR, false, true>;
        case 124: return debye::debye_pairs_kernel<124, V_RECUR, false, true>;
        default: return nullptr;
    }
}
