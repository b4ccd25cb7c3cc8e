// tdse_taylor_blocked.cuh -- temporally blocked Taylor step (all orders of one step in a single pass over HBM).
#pragma once
#include "tdse_device.cuh"

namespace tdse {

struct BlockedCfg {
    int supported = 0;
};

inline int blocked_configure(BlockedCfg *cfg, const tdse_grid &) { cfg->supported = 0; return TDSE_OK; }
inline bool blocked_supported(const BlockedCfg &cfg, int) { return cfg.supported != 0; }
inline int launch_taylor_blocked(const BlockedCfg &, const GridDev &, const double2 *, double2 *, const double *,
                                 const double *, int, cudaStream_t) {
    return TDSE_ERR_UNSUPPORTED;
}

}  // namespace tdse
