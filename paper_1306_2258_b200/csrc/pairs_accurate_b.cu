// pairs_accurate_b.cu -- explicit instantiations of debye_pairs_kernel<K, V_ACCURATE> (split for parallel builds)
#include "debye_pairs.cuh"
#include "debye_registry.h"
debye_pairs_fn debye_get_accurate_b(int K) {
    switch (K) {
        case 72: return debye::debye_pairs_kernel<72, V_ACCURATE>;
        case 80: return debye::debye_pairs_kernel<80, V_ACCURATE>;
        case 88: return debye::debye_pairs_kernel<88, V_ACCURATE>;
        case 96: return debye::debye_pairs_kernel<96, V_ACCURATE>;
        case 104: return debye::debye_pairs_kernel<104, V_ACCURATE>;
        case 112: return debye::debye_pairs_kernel<112, V_ACCURATE>;
        case 120: return debye::debye_pairs_kernel<120, V_ACCURATE>;
        case 128: return debye::debye_pairs_kernel<128, V_ACCURATE>;
        default: return nullptr;
    }
}
