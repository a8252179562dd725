// elliptical power-law mass model, linear-amplitude mode: trace_lin_kernel / fused_lin_kernel
#include "tl_dispatch.h"

template <int S_T>
static trace_fn pick_trace_lin_epl(int nll, int nsrc)
{
    if (nll == 0) return nsrc == 1 ? tl::trace_lin_kernel<S_T, 0, 1, tl::MASS_EPL> : tl::trace_lin_kernel<S_T, 0, 2, tl::MASS_EPL>;
    return nsrc == 1 ? tl::trace_lin_kernel<S_T, 1, 1, tl::MASS_EPL> : tl::trace_lin_kernel<S_T, 1, 2, tl::MASS_EPL>;
}
template <int S_T>
static fused_fn pick_fused_lin_epl(int nll, int nsrc)
{
    if (nll == 0) return nsrc == 1 ? tl::fused_lin_kernel<S_T, 0, 1, tl::MASS_EPL> : tl::fused_lin_kernel<S_T, 0, 2, tl::MASS_EPL>;
    return nsrc == 1 ? tl::fused_lin_kernel<S_T, 1, 1, tl::MASS_EPL> : tl::fused_lin_kernel<S_T, 1, 2, tl::MASS_EPL>;
}
fused_fn tl_fused_lin_epl_for(int S, int nll, int nsrc)
{
    return S == 4 ? pick_fused_lin_epl<4>(nll, nsrc) : pick_fused_lin_epl<0>(nll, nsrc);
}
trace_fn tl_trace_lin_epl_for(int S, int nll, int nsrc)
{
    return S == 4 ? pick_trace_lin_epl<4>(nll, nsrc) : pick_trace_lin_epl<0>(nll, nsrc);
}
