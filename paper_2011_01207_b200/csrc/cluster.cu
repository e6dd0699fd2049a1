// cluster.cu -- CLUSTER list mode (filtered 8-atom-cluster -> atom lists).  Not built yet:
// the context falls back to TILES (see api.cu), so these entry points are never reached.
#include "common.cuh"

namespace tkhp {

size_t cluster_workspace_bytes(const tkhp_params *, int) { return 0; }
int cluster_build(Ctx *c, cudaStream_t) { c->list_mode_in_use = TKHP_LIST_TILES; return TKHP_OK; }
int cluster_tmatvec(Ctx *c, cudaStream_t) { return set_err(c, TKHP_EINVAL, "cluster lists not available%s"); }
int cluster_field(Ctx *c, cudaStream_t) { return set_err(c, TKHP_EINVAL, "cluster lists not available%s"); }
long long cluster_slots(Ctx *) { return 0; }

}  // namespace tkhp
