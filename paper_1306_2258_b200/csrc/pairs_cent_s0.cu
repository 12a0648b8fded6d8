// pairs_cent_s0.cu -- explicit instantiations of debye_pairs_kernel<K, V_CENT, unweighted, sharded> (tile split over GPUs; split for parallel builds)
#include "debye_pairs.cuh"
#include "debye_registry.h"
debye_pairs_fn debye_get_cent_s0(int K) {
    switch (K) {
        case 8: return debye::debye_pairs_kernel<8, V_CENT, false, true>;
        case 16: return debye::debye_pairs_kernel<16, V_CENT, false, true>;
        case 24: return debye::debye_pairs_kernel<24, V_CENT, false, true>;
        case 32: return debye::debye_pairs_kernel<32, V_CENT, false, true>;
        default: return nullptr;
    }
}
