// pairs_cent_s2.cu -- explicit instantiations of debye_pairs_kernel<K, V_CENT, unweighted, sharded> (tile split over GPUs; split for parallel builds)
#include "debye_pairs.cuh"
#include "debye_registry.h"
debye_pairs_fn debye_get_cent_s2(int K) {
    switch (K) {
        case 72: return debye::debye_pairs_kernel<72, V_CENT, false, true>;
        case 80: return debye::debye_pairs_kernel<80, V_CENT, false, true>;
        case 88: return debye::debye_pairs_kernel<88, V_CENT, false, true>;
        case 96: return debye::debye_pairs_kernel<96, V_CENT, false, true>;
        default: return nullptr;
    }
}
