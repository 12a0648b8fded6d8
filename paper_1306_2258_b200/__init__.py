"""libdebye for B200 (sm_100a): Debye all-pairs sinc summation (arxiv 1306.2258, Eq. 2).

The public calls live in `paper_1306_2258_b200.binding` (thin ctypes marshalling over the C ABI declared in
include/debye.h); they are re-exported lazily so that importing `workloads` never touches CUDA.  There is
no CPU fallback: a missing libdebye.so raises."""

_API = ("debye_profile", "debye_profile_batch", "debye_profile_host", "debye_profile_batch_host",
        "debye_profile_weighted", "debye_profile_weighted_host", "debye_partials", "debye_partials_shard", "debye_profile_peratom", "debye_profile_peratom_host", "debye_profile_peratom_batch", "debye_profile_from_partials", "debye_profile_static", "static_limits", "q_hint", "q_hint_pieces", "pieces_of", "Plan", "lib", "LibdebyeError", "FLAGS")


def __getattr__(name):
    if name in _API:
        from . import binding
        return getattr(binding, name)
    raise AttributeError(name)
