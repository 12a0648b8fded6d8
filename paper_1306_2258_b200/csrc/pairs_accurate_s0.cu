// pairs_accurate_s0.cu -- explicit instantiations of debye_pairs_kernel<K, V_ACCURATE, unweighted, sharded: debye_partials_shard> (split for parallel builds)
#include "debye_pairs.cuh"
#include "debye_registry.h"
debye_pairs_fn debye_get_accurate_s0(int K) {
    switch (K) {
        case 8: return debye::debye_pairs_kernel<8, V_ACCURATE, false, true>;
        case 16: return debye::debye_pairs_kernel<16, V_ACCURATE, false, true>;
        case 24: return debye::debye_pairs_kernel<24, V_ACCURATE, false, true>;
        case 32: return debye::debye_pairs_kernel<32, V_ACCURATE, false, true>;
        case 40: return debye::debye_pairs_kernel<40, V_ACCURATE, false, true>;
        case 48: return debye::debye_pairs_kernel<48, V_ACCURATE, false, true>;
        case 56: return debye::debye_pairs_kernel<56, V_ACCURATE, false, true>;
        case 64: return debye::debye_pairs_kernel<64, V_ACCURATE, false, true>;
        case 72: return debye::debye_pairs_kernel<72, V_ACCURATE, false, true>;
        case 80: return debye::debye_pairs_kernel<80, V_ACCURATE, false, true>;
        case 88: return debye::debye_pairs_kernel<88, V_ACCURATE, false, true>;
        case 96: return debye::debye_pairs_kernel<96, V_ACCURATE, false, true>;
        case 104: return debye::debye_pairs_kernel<104, V_ACCURATE, false, true>;
        case 112: return debye::debye_pairs_kernel<112, V_ACCURATE, false, true>;
        case 120: return debye::debye_pairs_kernel<120, V_ACCURATE, false, true>;
        case 128: return debye::debye_pairs_kernel<128, V_ACCURATE, false, true>;
        default: return nullptr;
    }
}
