// linear-amplitude mode: trace_lin_kernel / fused_lin_kernel instantiations
#include "tl_dispatch.h"

template <int S_T>
static trace_fn pick_trace_lin(int nll, int nsrc)
{
    if (nll == 0) return nsrc == 1 ? tl::trace_lin_kernel<S_T, 0, 1> : tl::trace_lin_kernel<S_T, 0, 2>;
    return nsrc == 1 ? tl::trace_lin_kernel<S_T, 1, 1> : tl::trace_lin_kernel<S_T, 1, 2>;
}
template <int S_T>
static fused_fn pick_fused_lin(int nll, int nsrc)
{
    if (nll == 0) return nsrc == 1 ? tl::fused_lin_kernel<S_T, 0, 1> : tl::fused_lin_kernel<S_T, 0, 2>;
    return nsrc == 1 ? tl::fused_lin_kernel<S_T, 1, 1> : tl::fused_lin_kernel<S_T, 1, 2>;
}
fused_fn tl_fused_lin_for(int S, int nll, int nsrc)
{
    // compile time: only the paper's 4 x 4 supersampling gets the unrolled loop in linear mode
    return S == 4 ? pick_fused_lin<4>(nll, nsrc) : pick_fused_lin<0>(nll, nsrc);
}
trace_fn tl_trace_lin_for(int S, int nll, int nsrc)
{
    return S == 4 ? pick_trace_lin<4>(nll, nsrc) : pick_trace_lin<0>(nll, nsrc);
}

