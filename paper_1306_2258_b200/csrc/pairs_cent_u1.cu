// pairs_cent_u1.cu -- explicit instantiations of debye_pairs_kernel<K, V_CENT, unweighted> (centred product form; split for parallel builds)
#include "debye_pairs.cuh"
#include "debye_registry.h"
debye_pairs_fn debye_get_cent_u1(int K) {
    switch (K) {
        case 40: return debye::debye_pairs_kernel<40, V_CENT, false>;
        case 48: return debye::debye_pairs_kernel<48, V_CENT, false>;
        case 56: return debye::debye_pairs_kernel<56, V_CENT, false>;
        case 64: return debye::debye_pairs_kernel<64, V_CENT, false>;
        default: return nullptr;
    }
}
