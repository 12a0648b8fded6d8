// peratom_small_kernels.cu -- instantiations of debye_peratom_small_kernel<K> (one launch for one small structure, per-atom form factors)
#include "debye_peratom_small.cuh"
#include "debye_registry.h"
debye_peratom_small_fn debye_get_peratom_small_kernel(int K)
{
    switch (K) {
        case 8: return debye::debye_peratom_small_kernel<8>;
        case 16: return debye::debye_peratom_small_kernel<16>;
        case 24: return debye::debye_peratom_small_kernel<24>;
        case 32: return debye::debye_peratom_small_kernel<32>;
        case 40: return debye::debye_peratom_small_kernel<40>;
        case 48: return debye::debye_peratom_small_kernel<48>;
        case 56: return debye::debye_peratom_small_kernel<56>;
        case 64: return debye::debye_peratom_small_kernel<64>;
        case 72: return debye::debye_peratom_small_kernel<72>;
        case 80: return debye::debye_peratom_small_kernel<80>;
        case 88: return debye::debye_peratom_small_kernel<88>;
        case 96: return debye::debye_peratom_small_kernel<96>;
        case 104: return debye::debye_peratom_small_kernel<104>;
        case 112: return debye::debye_peratom_small_kernel<112>;
        case 120: return debye::debye_peratom_small_kernel<120>;
        case 128: return debye::debye_peratom_small_kernel<128>;
        default: return nullptr;
    }
}
