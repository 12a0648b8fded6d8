// pairs_mufu_s1.cu -- explicit instantiations of debye_pairs_kernel<K, V_MUFU, unweighted, sharded: debye_partials_shard> (split for parallel builds)
#include "debye_pairs.cuh"
#include "debye_registry.h"
debye_pairs_fn debye_get_mufu_s1(int K) {
    switch (K) {
        case 72: return debye::debye_pairs_kernel<72, V_MUFU, false, true>;
        case 80: return debye::debye_pairs_kernel<80, V_MUFU, false, true>;
        case 88: return debye::debye_pairs_kernel<88, V_MUFU, false, true>;
        case 96: return debye::debye_pairs_kernel<96, V_MUFU, false, true>;
        case 104: return debye::debye_pairs_kernel<104, V_MUFU, false, true>;
        case 112: return debye::debye_pairs_kernel<112, V_MUFU, false, true>;
        case 120: return debye::debye_pairs_kernel<120, V_MUFU, false, true>;
        case 128: return debye::debye_pairs_kernel<128, V_MUFU, false, true>;
        default: return nullptr;
    }
}
