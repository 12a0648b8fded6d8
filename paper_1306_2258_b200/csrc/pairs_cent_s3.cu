// pairs_cent_s3.cu -- explicit instantiations of debye_pairs_kernel<K, V_CENT, unweighted, sharded> (tile split over GPUs; split for parallel builds)
#include "debye_pairs.cuh"
#include "debye_registry.h"
debye_pairs_fn debye_get_cent_s3(int K) {
    switch (K) {
        case 104: return debye::debye_pairs_kernel<104, V_CENT, false, true>;
        case 112: return debye::debye_pairs_kernel<112, V_CENT, false, true>;
        case 120: return debye::debye_pairs_kernel<120, V_CENT, false, true>;
        case 128: return debye::debye_pairs_kernel<128, V_CENT, false, true>;
        default: return nullptr;
    }
}
