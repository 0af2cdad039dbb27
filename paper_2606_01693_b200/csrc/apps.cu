// apps.cu — application drivers of PAPER.md §V-B (L365-366): BFS and the tile-based tracer.
#include "gq.h"
extern "C" int bfs_run(int, const uint64_t*, const uint32_t*, uint32_t, uint32_t, int32_t*, gq_bfs_stats*, void*) { return GQ_E_INVAL; }
extern "C" int rt_render(int, const gq_rt_scene*, float*, gq_rt_stats*, void*) { return GQ_E_INVAL; }
