// dispatch.cu — picks the kernel set: the tuned sm_100a kernels (default: stage_tma.cu, ghost_tma.cu,
// restrict_zmarch.cu) or the straightforward direct-load kernels of kernels_basic.cu (environment
// SC_KERNELS=ref; A/B checks and debugging only). Both are CUDA; there is no CPU path.
#include <atomic>
#include <cstdlib>

#include "kernels.h"

namespace sc {

void launch_stage_direct(const StageArgs& a, cudaStream_t st);
void launch_stage_fd8(const StageArgs& a, cudaStream_t st);
int launch_stage_tma(const StageArgs& a, cudaStream_t st);
bool make_box_tensor_map_tma(const BoxView& b, int narrays, void* base, const unsigned box[4], int l2_promotion,
                             bool swizzle64, void* out_map128);
void stage_box_dims(int variant, unsigned box[4]);
void restrict_box_dims(unsigned box[4]);
void launch_ghost_fill_direct(const GhostArgs& a, cudaStream_t st);
void launch_ghost_fill_tma(const GhostArgs& a, cudaStream_t st);
void launch_ghost_fill_tiled(const GhostArgs& a, cudaStream_t st);
bool ghost_tma_takes(const GhostArgs& a);
void ghost_box_dims(int axis, unsigned box[4]);
void launch_restrict_ref(const RestrictArgs& a, cudaStream_t st);
void launch_restrict_opt(const RestrictArgs& a, cudaStream_t st);
void launch_restrict_tiled(const RestrictArgs& a, cudaStream_t st);
void launch_stage_ko_direct(const StageKOArgs& a, cudaStream_t st);
void launch_stage_ko_tma(const StageKOArgs& a, cudaStream_t st);
bool stage_ko_tma_takes(const StageKOArgs& a);
void stageko_box_dims(int variant, unsigned box[4]);
void launch_stage_gen_tma(const StageKOArgs& a, cudaStream_t st);
bool stage_gen_tma_takes(const StageKOArgs& a);
void stagegen_box_dims(int H, unsigned box[4]);

// process-wide (it mirrors the environment variable SC_KERNELS, read when a hierarchy is created); atomic: hierarchies
// may be created from several host threads
static std::atomic<int> g_mode{1};
void select_kernels(int mode) { g_mode.store(mode, std::memory_order_relaxed); }
int selected_kernels() { return g_mode.load(std::memory_order_relaxed); }

int launch_stage(const StageArgs& a, cudaStream_t st) {
  if (g_mode == 0) { launch_stage_direct(a, st); return 1; }
  if (a.fd_order == 8) { launch_stage_fd8(a, st); return 1; }  // the TMA z-march is radius 2 only
  return launch_stage_tma(a, st);
}
void launch_stage_ko(const StageKOArgs& a, cudaStream_t st) {
  if (g_mode != 0 && stage_gen_tma_takes(a)) launch_stage_gen_tma(a, st);      // 8th-order differences
  else if (g_mode != 0 && stage_ko_tma_takes(a)) launch_stage_ko_tma(a, st);   // 4th-order
  else { launch_stage_ko_direct(a, st); return; }
  if (a.rad_nb > 0) {  // radiative level 0 (S29): the boundary points again, with the radiative operator
    StageKOArgs z = a;
    z.zone_only = 1;
    launch_stage_ko_direct(z, st);
  }
}
void launch_ghost_fill(const GhostArgs& a, cudaStream_t st) {
  const bool s3 = a.np == 5 && a.pmin == -2;  // the tuned kernel has the quartic cell-centred operator built in
  if (g_mode == 0) launch_ghost_fill_direct(a, st);                          // SC_KERNELS=ref: the np^3-point gather
  else if (!s3 || !ghost_tma_takes(a)) launch_ghost_fill_tiled(a, st);       // any width / stencil / shape, separable
  else launch_ghost_fill_tma(a, st);
}
void launch_restrict(const RestrictArgs& a, cudaStream_t st) {
  if (g_mode == 0) launch_restrict_ref(a, st);
  else if (a.nr == 1) launch_restrict_ref(a, st);  // injection: one load per parent cell
  else if (a.nr != 6 || !a.tmap) launch_restrict_tiled(a, st);
  else launch_restrict_opt(a, st);
}
bool make_box_tensor_map(const BoxView& b, int narrays, void* base, int kind, void* out_map128) {
  unsigned box[4];
  if (kind == 0 || kind == 8) stage_box_dims(kind == 8, box);  // the stage kernels' halo tile: 32 x 16 or 64 x 7 cells
  else if (kind == 1) restrict_box_dims(box);
  else if (kind <= 4) ghost_box_dims(kind - 2, box);
  else if (kind == 5 || kind == 9) stageko_box_dims(kind == 9, box);  // the dissipative stage kernel's halo-3 tile, 32 x 16 / 64 x 7
  else if (kind != 8) stagegen_box_dims(kind == 7 ? 5 : 4, box);  // kinds 6, 7: the general path's halo-4 / halo-5 tiles
  // streaming tiles (stage, restriction) promote misses to 256-byte fetches; the ghost fill's footprint rows are
  // 64-160 bytes and isolated: promotion there only multiplies the DRAM traffic. The x-slab footprint (kind 2,
  // 64-byte rows) is swizzled so that one-thread-per-row reads are bank-conflict free (ghost_tma.cu).
  return make_box_tensor_map_tma(b, narrays, base, box, (kind <= 1 || kind >= 5) ? 256 : 0, kind == 2, out_map128);
}

}  // namespace sc
