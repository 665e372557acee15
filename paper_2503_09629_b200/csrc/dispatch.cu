// dispatch.cu — picks the kernel set: the tuned sm_100a kernels (default) or the straightforward
// reference kernels (environment SC_KERNELS=ref; A/B checks and debugging only). Both are CUDA.
#include "kernels.h"

namespace sc {

void launch_rhs_stage_ref(const RhsArgs& a, cudaStream_t st);
void launch_ghost_fill_ref(const GhostArgs& a, cudaStream_t st);
void launch_periodic_fill_ref(const BoxView& b, int V, double* y, cudaStream_t st);
void launch_restrict_ref(const BoxView& ch, const BoxView& pa, int V, const double* yc, double* yp, cudaStream_t st);

void launch_ghost_fill_opt(const GhostArgs& a, cudaStream_t st);
void launch_restrict_opt(const BoxView& ch, const BoxView& pa, int V, const double* yc, double* yp, cudaStream_t st);

static int g_mode = 1;
void select_kernels(int mode) { g_mode = mode; }

void launch_rhs_stage(const RhsArgs& a, cudaStream_t st) { launch_rhs_stage_ref(a, st); }
void launch_ghost_fill(const GhostArgs& a, cudaStream_t st) {
  if (g_mode == 0) launch_ghost_fill_ref(a, st);
  else launch_ghost_fill_opt(a, st);
}
void launch_periodic_fill(const BoxView& b, int V, double* y, cudaStream_t st) { launch_periodic_fill_ref(b, V, y, st); }
void launch_restrict(const BoxView& ch, const BoxView& pa, int V, const double* yc, double* yp, cudaStream_t st) {
  if (g_mode == 0) launch_restrict_ref(ch, pa, V, yc, yp, st);
  else launch_restrict_opt(ch, pa, V, yc, yp, st);
}

}  // namespace sc
