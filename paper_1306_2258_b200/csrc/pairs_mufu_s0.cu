// pairs_mufu_s0.cu -- explicit instantiations of debye_pairs_kernel<K, V_MUFU, unweighted, sharded: debye_partials_shard> (split for parallel builds)
#include "debye_pairs.cuh"
#include "debye_registry.h"
debye_pairs_fn debye_get_mufu_s0(int K) {
    switch (K) {
        case 8: return debye::debye_pairs_kernel<8, V_MUFU, false, true>;
        case 16: return debye::debye_pairs_kernel<16, V_MUFU, false, true>;
        case 24: return debye::debye_pairs_kernel<24, V_MUFU, false, true>;
        case 32: return debye::debye_pairs_kernel<32, V_MUFU, false, true>;
        case 40: return debye::debye_pairs_kernel<40, V_MUFU, false, true>;
        case 48: return debye::debye_pairs_kernel<48, V_MUFU, false, true>;
        case 56: return debye::debye_pairs_kernel<56, V_MUFU, false, true>;
        case 64: return debye::debye_pairs_kernel<64, V_MUFU, false, true>;
        default: return nullptr;
    }
}
