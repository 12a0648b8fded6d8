// pairs_lookup.cu -- variant / K / weighted -> kernel instantiation
#include "debye_registry.h"
debye_pairs_fn debye_get_recur_u0(int K);
debye_pairs_fn debye_get_recur_u1(int K);
debye_pairs_fn debye_get_recur_u2(int K);
debye_pairs_fn debye_get_recur_u3(int K);
debye_pairs_fn debye_get_recur_w0(int K);
debye_pairs_fn debye_get_recur_w1(int K);
debye_pairs_fn debye_get_recur_w2(int K);
debye_pairs_fn debye_get_recur_w3(int K);
debye_pairs_fn debye_get_mufu_u0(int K);
debye_pairs_fn debye_get_mufu_u1(int K);
debye_pairs_fn debye_get_mufu_w0(int K);
debye_pairs_fn debye_get_mufu_w1(int K);
debye_pairs_fn debye_get_accurate_u0(int K);
debye_pairs_fn debye_get_f64_u0(int K);
debye_pairs_fn debye_get_f64_w0(int K);
debye_pairs_fn debye_get_recur_s0(int K);
debye_pairs_fn debye_get_recur_s1(int K);
debye_pairs_fn debye_get_recur_s2(int K);
debye_pairs_fn debye_get_recur_s3(int K);
debye_pairs_fn debye_get_mufu_s0(int K);
debye_pairs_fn debye_get_mufu_s1(int K);
debye_pairs_fn debye_get_f64_s0(int K);
debye_pairs_fn debye_get_cent_u0(int K);
debye_pairs_fn debye_get_cent_u1(int K);
debye_pairs_fn debye_get_cent_u2(int K);
debye_pairs_fn debye_get_cent_u3(int K);
debye_pairs_fn debye_get_cent_w0(int K);
debye_pairs_fn debye_get_cent_w1(int K);
debye_pairs_fn debye_get_cent_w2(int K);
debye_pairs_fn debye_get_cent_w3(int K);
debye_pairs_fn debye_get_cent_s0(int K);
debye_pairs_fn debye_get_cent_s1(int K);
debye_pairs_fn debye_get_cent_s2(int K);
debye_pairs_fn debye_get_cent_s3(int K);
static debye_pairs_fn first_of(debye_pairs_fn (*const *fns)(int), int n, int K)
{
    for (int i = 0; i < n; ++i) { debye_pairs_fn f = fns[i](K); if (f) return f; }
    return nullptr;
}
debye_pairs_fn debye_get_pairs_kernel(int variant, int K, bool weighted, bool sharded)
{
    if (sharded) {      // tile split over GPUs (debye_partials_shard): unweighted only
        if (weighted) return nullptr;
        if (variant == V_RECUR) { static debye_pairs_fn (*const f[])(int) = {debye_get_recur_s0, debye_get_recur_s1, debye_get_recur_s2, debye_get_recur_s3}; return first_of(f, 4, K); }
        if (variant == V_MUFU) { static debye_pairs_fn (*const f[])(int) = {debye_get_mufu_s0, debye_get_mufu_s1}; return first_of(f, 2, K); }
        if (variant == V_ACCURATE) return nullptr;      // the libdevice-sinf reference variant exists for the plain calls only
        if (variant == V_CENT) { static debye_pairs_fn (*const f[])(int) = {debye_get_cent_s0, debye_get_cent_s1, debye_get_cent_s2, debye_get_cent_s3}; return first_of(f, 4, K); }
        if (variant == V_F64) { static debye_pairs_fn (*const f[])(int) = {debye_get_f64_s0}; return first_of(f, 1, K); }
        return nullptr;
    }
    if (variant == V_RECUR && weighted == false) { static debye_pairs_fn (*const f[])(int) = {debye_get_recur_u0, debye_get_recur_u1, debye_get_recur_u2, debye_get_recur_u3}; return first_of(f, 4, K); }
    if (variant == V_RECUR && weighted == true) { static debye_pairs_fn (*const f[])(int) = {debye_get_recur_w0, debye_get_recur_w1, debye_get_recur_w2, debye_get_recur_w3}; return first_of(f, 4, K); }
    if (variant == V_MUFU && weighted == false) { static debye_pairs_fn (*const f[])(int) = {debye_get_mufu_u0, debye_get_mufu_u1}; return first_of(f, 2, K); }
    if (variant == V_MUFU && weighted == true) { static debye_pairs_fn (*const f[])(int) = {debye_get_mufu_w0, debye_get_mufu_w1}; return first_of(f, 2, K); }
    if (variant == V_CENT && weighted == false) { static debye_pairs_fn (*const f[])(int) = {debye_get_cent_u0, debye_get_cent_u1, debye_get_cent_u2, debye_get_cent_u3}; return first_of(f, 4, K); }
    if (variant == V_CENT && weighted == true) { static debye_pairs_fn (*const f[])(int) = {debye_get_cent_w0, debye_get_cent_w1, debye_get_cent_w2, debye_get_cent_w3}; return first_of(f, 4, K); }
    if (variant == V_ACCURATE && weighted == false) { static debye_pairs_fn (*const f[])(int) = {debye_get_accurate_u0}; return first_of(f, 1, K); }
    if (variant == V_ACCURATE && weighted == true) return nullptr;      // reference variant: unweighted, unsharded only
    if (variant == V_F64 && weighted == false) { static debye_pairs_fn (*const f[])(int) = {debye_get_f64_u0}; return first_of(f, 1, K); }
    if (variant == V_F64 && weighted == true) { static debye_pairs_fn (*const f[])(int) = {debye_get_f64_w0}; return first_of(f, 1, K); }
    return nullptr;
}
