// pairs_cent_w0.cu -- explicit instantiations of debye_pairs_kernel<K, V_CENT, weighted> (centred product form; split for parallel builds)
#include "debye_pairs.cuh"
#include "debye_registry.h"
debye_pairs_fn debye_get_cent_w0(int K) {
    switch (K) {
        case 8: return debye::debye_pairs_kernel<8, V_CENT, true>;
        case 16: return debye::debye_pairs_kernel<16, V_CENT, true>;
        case 24: return debye::debye_pairs_kernel<24, V_CENT, true>;
        case 32: return debye::debye_pairs_kernel<32, V_CENT, true>;
        default: return nullptr;
    }
}
