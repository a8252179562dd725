// fused_kernel<S, NLL, NSRC> instantiations
#include "tl_dispatch.h"

template <int S_T>
static fused_fn pick_fused(int nll, int nsrc)
{
    if (nll == 0) return nsrc == 1 ? tl::fused_kernel<S_T, 0, 1> : tl::fused_kernel<S_T, 0, 2>;
    return nsrc == 1 ? tl::fused_kernel<S_T, 1, 1> : tl::fused_kernel<S_T, 1, 2>;
}
fused_fn tl_fused_for(int S, int nll, int nsrc)
{
    switch (S) {
    case 1: return pick_fused<1>(nll, nsrc);
    case 2: return pick_fused<2>(nll, nsrc);
    case 4: return pick_fused<4>(nll, nsrc);
    case 8: return pick_fused<8>(nll, nsrc);
    default: return pick_fused<0>(nll, nsrc);
    }
}

// the three-CTAs-per-SM variant (256 threads, PSF up to 21 x 21): S = 2 only, where the pair loop holds one
// pair per sub-row and fits in 85 registers
fused_fn tl_fused_small_for(int S, int nll, int nsrc)
{
    if (S != 2) return nullptr;
    if (nll == 0) return nsrc == 1 ? tl::fused_kernel<2, 0, 1, tl::MASS_SIE, 1> : tl::fused_kernel<2, 0, 2, tl::MASS_SIE, 1>;
    return nsrc == 1 ? tl::fused_kernel<2, 1, 1, tl::MASS_SIE, 1> : tl::fused_kernel<2, 1, 2, tl::MASS_SIE, 1>;
}
