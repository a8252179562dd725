// trace_kernel<S, NLL, NSRC> instantiations (split path)
#include "tl_dispatch.h"

template <int S_T>
static trace_fn pick_trace(int nll, int nsrc)
{
    if (nll == 0) return nsrc == 1 ? tl::trace_kernel<S_T, 0, 1> : tl::trace_kernel<S_T, 0, 2>;
    return nsrc == 1 ? tl::trace_kernel<S_T, 1, 1> : tl::trace_kernel<S_T, 1, 2>;
}
trace_fn tl_trace_for(int S, int nll, int nsrc)
{
    switch (S) {
    case 1: return pick_trace<1>(nll, nsrc);
    case 2: return pick_trace<2>(nll, nsrc);
    case 4: return pick_trace<4>(nll, nsrc);
    case 8: return pick_trace<8>(nll, nsrc);
    default: return pick_trace<0>(nll, nsrc);
    }
}


// trace_pairs_kernel<S, NLL, NSRC>: the one-pair-per-lane ray-trace of calls with few rows (SIE, even S)
template <int S_T>
static trace_fn pick_trace_pairs(int nll, int nsrc)
{
    if (nll == 0) return nsrc == 1 ? tl::trace_pairs_kernel<S_T, 0, 1> : tl::trace_pairs_kernel<S_T, 0, 2>;
    return nsrc == 1 ? tl::trace_pairs_kernel<S_T, 1, 1> : tl::trace_pairs_kernel<S_T, 1, 2>;
}
trace_fn tl_trace_pairs_for(int S, int nll, int nsrc)
{
    switch (S) {
    case 2: return pick_trace_pairs<2>(nll, nsrc);
    case 4: return pick_trace_pairs<4>(nll, nsrc);
    case 8: return pick_trace_pairs<8>(nll, nsrc);
    default: return nullptr;
    }
}
