// peratom_recur_kernels.cu -- instantiations of debye_peratom_recur_kernel<K, single structure> (debye_peratom_recur.cuh)
#include "debye_peratom_recur.cuh"
#include "debye_registry.h"
debye_peratom_recur_fn debye_get_peratom_recur_single(int K)
{
    switch (K) {
        case 8: return debye::debye_peratom_recur_kernel<8, false>;
        case 16: return debye::debye_peratom_recur_kernel<16, false>;
        case 24: return debye::debye_peratom_recur_kernel<24, false>;
        case 32: return debye::debye_peratom_recur_kernel<32, false>;
        case 40: return debye::debye_peratom_recur_kernel<40, false>;
        case 48: return debye::debye_peratom_recur_kernel<48, false>;
        case 56: return debye::debye_peratom_recur_kernel<56, false>;
        case 64: return debye::debye_peratom_recur_kernel<64, false>;
        case 72: return debye::debye_peratom_recur_kernel<72, false>;
        case 80: return debye::debye_peratom_recur_kernel<80, false>;
        case 88: return debye::debye_peratom_recur_kernel<88, false>;
        case 96: return debye::debye_peratom_recur_kernel<96, false>;
        case 104: return debye::debye_peratom_recur_kernel<104, false>;
        case 112: return debye::debye_peratom_recur_kernel<112, false>;
        case 120: return debye::debye_peratom_recur_kernel<120, false>;
        case 128: return debye::debye_peratom_recur_kernel<128, false>;
        default: return nullptr;
    }
}
