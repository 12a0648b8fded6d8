// pairs_cent_s1.cu -- explicit instantiations of debye_pairs_kernel<K, V_CENT, unweighted, sharded> (tile split over GPUs; split for parallel builds)
#include "debye_pairs.cuh"
#include "debye_registry.h"
debye_pairs_fn debye_get_cent_s1(int K) {
    switch (K) {
        case 40: return debye::debye_pairs_kernel<40, V_CENT, false, true>;
        case 48: return debye::debye_pairs_kernel<48, V_CENT, false, true>;
        case 56: return debye::debye_pairs_kernel<56, V_CENT, false, true>;
        case 64: return debye::debye_pairs_kernel<64, V_CENT, false, true>;
        default: return nullptr;
    }
}
