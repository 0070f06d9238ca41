// a6-a8, Blackwell kernel: TMA-gathered K/V pages, tcgen05.mma with TMEM accumulators.
#include "attn_schedule.cuh"
#include "common.cuh"

namespace omnimem {

bool attn_tcgen05_supported(const AttnArgs&) { return false; }
size_t attn_tcgen05_workspace_bytes(int32_t, int32_t, int32_t, int32_t) { return 0; }
int32_t launch_attn_tcgen05(const AttnArgs&) { return fail(OMNIMEM_EUNSUPPORTED, "tcgen05 attention kernel not built"); }

}  // namespace omnimem
