// elliptical power-law mass model: fused_kernel / trace_kernel instantiations with MASS = MASS_EPL
#include "tl_dispatch.h"

template <int S_T>
static fused_fn pick_fused_epl(int nll, int nsrc)
{
    if (nll == 0) return nsrc == 1 ? tl::fused_kernel<S_T, 0, 1, tl::MASS_EPL> : tl::fused_kernel<S_T, 0, 2, tl::MASS_EPL>;
    return nsrc == 1 ? tl::fused_kernel<S_T, 1, 1, tl::MASS_EPL> : tl::fused_kernel<S_T, 1, 2, tl::MASS_EPL>;
}
template <int S_T>
static trace_fn pick_trace_epl(int nll, int nsrc)
{
    if (nll == 0) return nsrc == 1 ? tl::trace_kernel<S_T, 0, 1, tl::MASS_EPL> : tl::trace_kernel<S_T, 0, 2, tl::MASS_EPL>;
    return nsrc == 1 ? tl::trace_kernel<S_T, 1, 1, tl::MASS_EPL> : tl::trace_kernel<S_T, 1, 2, tl::MASS_EPL>;
}
fused_fn tl_fused_epl_for(int S, int nll, int nsrc)
{
    return S == 4 ? pick_fused_epl<4>(nll, nsrc) : pick_fused_epl<0>(nll, nsrc);
}
trace_fn tl_trace_epl_for(int S, int nll, int nsrc)
{
    return S == 4 ? pick_trace_epl<4>(nll, nsrc) : pick_trace_epl<0>(nll, nsrc);
}
