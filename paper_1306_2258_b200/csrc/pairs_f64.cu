// pairs_f64.cu -- explicit instantiations of debye_pairs_kernel<K, V_F64> and the variant/K lookup
#include "debye_pairs.cuh"
#include "debye_registry.h"
debye_pairs_fn debye_get_recur_a(int K); debye_pairs_fn debye_get_recur_b(int K);
debye_pairs_fn debye_get_recur_c(int K); debye_pairs_fn debye_get_recur_d(int K);
debye_pairs_fn debye_get_mufu_a(int K); debye_pairs_fn debye_get_mufu_b(int K);
debye_pairs_fn debye_get_accurate_a(int K); debye_pairs_fn debye_get_accurate_b(int K);
debye_pairs_fn debye_get_f64(int K)
{
    switch (K) {
        case 8: return debye::debye_pairs_kernel<8, V_F64>;
        case 16: return debye::debye_pairs_kernel<16, V_F64>;
        case 24: return debye::debye_pairs_kernel<24, V_F64>;
        case 32: return debye::debye_pairs_kernel<32, V_F64>;
        default: return nullptr;
    }
}
debye_pairs_fn debye_get_pairs_kernel(int variant, int K)
{
    switch (variant) {
        case V_F64: return debye_get_f64(K);
        case V_RECUR: return (K % 8 == 0) ? (K <= 64 ? debye_get_recur_a(K) : debye_get_recur_b(K)) : (K <= 64 ? debye_get_recur_c(K) : debye_get_recur_d(K));
        case V_MUFU: return K <= 64 ? debye_get_mufu_a(K) : debye_get_mufu_b(K);
        case V_ACCURATE: return K <= 64 ? debye_get_accurate_a(K) : debye_get_accurate_b(K);
        default: return nullptr;
    }
}
