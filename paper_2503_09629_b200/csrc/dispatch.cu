// dispatch.cu — picks the kernel set: the tuned sm_100a kernels (default) or the straightforward
// direct-load kernels of kernels_basic.cu (environment SC_KERNELS=ref; A/B checks and debugging only).
// Both are CUDA; there is no CPU path.
#include "kernels.h"

namespace sc {

void launch_stage_direct(const StageArgs& a, cudaStream_t st);
void launch_ghost_fill_direct(const GhostArgs& a, cudaStream_t st);
void launch_restrict_ref(const BoxView& ch, const BoxView& pa, int V, const double* yc, double* yp, cudaStream_t st);

void launch_restrict_opt(const BoxView& ch, const BoxView& pa, int V, const double* yc, double* yp, cudaStream_t st);

static int g_mode = 1;
void select_kernels(int mode) { g_mode = mode; }
int selected_kernels() { return g_mode; }

void launch_stage(const StageArgs& a, cudaStream_t st) { launch_stage_direct(a, st); }
void launch_ghost_fill(const GhostArgs& a, cudaStream_t st) { launch_ghost_fill_direct(a, st); }
void launch_restrict(const BoxView& ch, const BoxView& pa, int V, const double* yc, double* yp, cudaStream_t st) {
  if (g_mode == 0) launch_restrict_ref(ch, pa, V, yc, yp, st);
  else launch_restrict_opt(ch, pa, V, yc, yp, st);
}
bool make_box_tensor_map(const BoxView&, int, void*, void*) { return false; }
void build_ghost_tiles(const BoxView&, std::vector<GhostTile>& tiles) { tiles.clear(); }

}  // namespace sc
