// peratom_recur_batch_kernels.cu -- instantiations of debye_peratom_recur_kernel<K, batch of conformers> (debye_peratom_recur.cuh)
#include "debye_peratom_recur.cuh"
#include "debye_registry.h"
debye_peratom_recur_fn debye_get_peratom_recur_batch(int K)
{
    switch (K) {
        case 8: return debye::debye_peratom_recur_kernel<8, true>;
        case 16: return debye::debye_peratom_recur_kernel<16, true>;
        case 24: return debye::debye_peratom_recur_kernel<24, true>;
        case 32: return debye::debye_peratom_recur_kernel<32, true>;
        case 40: return debye::debye_peratom_recur_kernel<40, true>;
        case 48: return debye::debye_peratom_recur_kernel<48, true>;
        case 56: return debye::debye_peratom_recur_kernel<56, true>;
        case 64: return debye::debye_peratom_recur_kernel<64, true>;
        case 72: return debye::debye_peratom_recur_kernel<72, true>;
        case 80: return debye::debye_peratom_recur_kernel<80, true>;
        case 88: return debye::debye_peratom_recur_kernel<88, true>;
        case 96: return debye::debye_peratom_recur_kernel<96, true>;
        case 104: return debye::debye_peratom_recur_kernel<104, true>;
        case 112: return debye::debye_peratom_recur_kernel<112, true>;
        case 120: return debye::debye_peratom_recur_kernel<120, true>;
        case 128: return debye::debye_peratom_recur_kernel<128, true>;
        default: return nullptr;
    }
}
debye_peratom_recur_fn debye_get_peratom_recur_single(int K);
debye_peratom_recur_fn debye_get_peratom_recur_kernel(int K, bool batch) { return batch ? debye_get_peratom_recur_batch(K) : debye_get_peratom_recur_single(K); }
