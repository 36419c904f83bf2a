// Fused shot-tile path (S0-S5 in one kernel). Placeholder: not attempted yet, the general
// kernels run.
#pragma once
#include "tpx3_common.cuh"

namespace tpx3 {

inline int enqueue_fused(int num_sms, uint64_t* launches, Ctrl* ctrl, unsigned long long* tiles, cudaStream_t st,
                         const Params& prm, const uint16_t* x, const uint16_t* y, const uint64_t* toa,
                         const uint16_t* tot, uint32_t* perm, uint32_t* label, uint64_t max_clusters,
                         const tpx3_clusters_t& out, uint32_t* n_clusters) {
  (void)num_sms; (void)launches; (void)ctrl; (void)tiles; (void)st; (void)prm; (void)x; (void)y; (void)toa; (void)tot;
  (void)perm; (void)label; (void)max_clusters; (void)out; (void)n_clusters;
  return TPX3_OK;
}

}  // namespace tpx3
