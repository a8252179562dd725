// serve_kernel<S, NLL, NSRC> instantiations (the persistent kernel of tl_serve_start, tl_serve.cuh)
#include "tl_dispatch.h"
#include "tl_serve.cuh"

template <int S_T>
static serve_fn pick_serve(int nll, int nsrc)
{
    if (nll == 0) return nsrc == 1 ? tl::serve_kernel<S_T, 0, 1> : tl::serve_kernel<S_T, 0, 2>;
    return nsrc == 1 ? tl::serve_kernel<S_T, 1, 1> : tl::serve_kernel<S_T, 1, 2>;
}
serve_fn tl_serve_for(int S, int nll, int nsrc)
{
    switch (S) {
    case 2: return pick_serve<2>(nll, nsrc);
    case 4: return pick_serve<4>(nll, nsrc);
    case 8: return pick_serve<8>(nll, nsrc);
    default: return nullptr;                 // the one-pair-per-lane ray-trace needs an even S
    }
}
