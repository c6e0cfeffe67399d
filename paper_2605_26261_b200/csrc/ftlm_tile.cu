// TILE kernels (B200 design) - placeholder until the first GPU parity run
// of the ROW path; the plan is absent so the dispatcher uses the ROW kernels.
#include "ftlm_common.cuh"

int ftlm_tile_plan_create(ftlm_ctx* c) { c->tile = nullptr; return FTLM_OK; }
void ftlm_tile_plan_destroy(ftlm_ctx* c) { c->tile = nullptr; }
int ftlm_launch_hv_tile(ftlm_ctx*, const void*, const void*, void*, int, cudaStream_t) {
  ftlm_set_error("TILE kernel not built"); return FTLM_EUNSUPPORTED;
}
int ftlm_launch_neighbors_tile(ftlm_ctx*, int64_t, int64_t, int64_t*, cudaStream_t) {
  ftlm_set_error("TILE kernel not built"); return FTLM_EUNSUPPORTED;
}
