// a3 + a4 on the 5th-generation tensor cores (tcgen05 / TMEM / TMA).  Placeholder until the kernels land:
// reports "not available" so that DHP_MLP_AUTO uses the SIMT path.
#include "dhp_internal.cuh"

namespace dhp {
bool mlp_tc_available(Ctx*) { return false; }
int mlp_tc_alloc(Ctx*) { return DHP_OK; }
void mlp_tc_free(Ctx*) {}
int mlp_tc_weights(Ctx*, Weights*) { return DHP_OK; }
void mlp_tc_weights_free(Ctx*, Weights*) {}
int mlp_tc(Ctx*, const Weights*) { return DHP_E_NOTIMPL; }
}  // namespace dhp
