// pairs_recur_c.cu -- explicit instantiations of debye_pairs_kernel<K, V_RECUR> (split for parallel builds)
#include "debye_pairs.cuh"
#include "debye_registry.h"
debye_pairs_fn debye_get_recur_c(int K) {
    switch (K) {
        case 12: return debye::debye_pairs_kernel<12, V_RECUR>;
        case 20: return debye::debye_pairs_kernel<20, V_RECUR>;
        case 28: return debye::debye_pairs_kernel<28, V_RECUR>;
        case 36: return debye::debye_pairs_kernel<36, V_RECUR>;
        case 44: return debye::debye_pairs_kernel<44, V_RECUR>;
        case 52: return debye::debye_pairs_kernel<52, V_RECUR>;
        case 60: return debye::debye_pairs_kernel<60, V_RECUR>;
        default: return nullptr;
    }
}
