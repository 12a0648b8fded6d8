// pairs_cent_u0.cu -- explicit instantiations of debye_pairs_kernel<K, V_CENT, unweighted> (centred product form; split for parallel builds)
#include "debye_pairs.cuh"
#include "debye_registry.h"
debye_pairs_fn debye_get_cent_u0(int K) {
    switch (K) {
        case 8: return debye::debye_pairs_kernel<8, V_CENT, false>;
        case 16: return debye::debye_pairs_kernel<16, V_CENT, false>;
        case 24: return debye::debye_pairs_kernel<24, V_CENT, false>;
        case 32: return debye::debye_pairs_kernel<32, V_CENT, false>;
        default: return nullptr;
    }
}
