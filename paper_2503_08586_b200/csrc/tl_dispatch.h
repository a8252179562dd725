// tl_dispatch.h -- kernel tables.  The template kernels are instantiated in translation units of
// their own (tl_inst_fused.cu, tl_inst_split.cu, tl_inst_lin.cu; tl_inst_epl.cu, tl_inst_epl_lin.cu) so that nvcc can compile
// them in parallel; tinylens.cu only asks for the function pointer that matches a context.
#pragma once
#include "tl_kernels.cuh"
namespace tl { struct ServeCtl; struct ServeDev; }

typedef void (*fused_fn)(const tl::KArgs);
typedef void (*trace_fn)(const tl::KArgs, int);
typedef void (*serve_fn)(const tl::KArgs, const tl::PrologueArgs, tl::ServeCtl *, tl::ServeDev *, float *, unsigned long long, unsigned long long);

fused_fn tl_fused_for(int S, int n_lens_light, int n_source);          // fused_kernel<S, NLL, NSRC>
fused_fn tl_fused_small_for(int S, int n_lens_light, int n_source);    // fused_kernel<S, NLL, NSRC, SIE, 1> (256 threads, K <= 21), or null
trace_fn tl_trace_for(int S, int n_lens_light, int n_source);          // trace_kernel<S, NLL, NSRC>
serve_fn tl_serve_for(int S, int n_lens_light, int n_source);          // serve_kernel<S, NLL, NSRC> (persistent), or null (odd S)
trace_fn tl_trace_pairs_for(int S, int n_lens_light, int n_source);    // trace_pairs_kernel<S, NLL, NSRC>, or null (odd S)
fused_fn tl_fused_lin_for(int S, int n_lens_light, int n_source);      // fused_lin_kernel<...>
trace_fn tl_trace_lin_for(int S, int n_lens_light, int n_source);      // trace_lin_kernel<...>
// mass_model = MASS_EPL (compile time: S = 4 unrolled, any other S through the generic loop)
fused_fn tl_fused_epl_for(int S, int n_lens_light, int n_source);
trace_fn tl_trace_epl_for(int S, int n_lens_light, int n_source);
fused_fn tl_fused_lin_epl_for(int S, int n_lens_light, int n_source);
trace_fn tl_trace_lin_epl_for(int S, int n_lens_light, int n_source);
