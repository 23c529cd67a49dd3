// gda_dense.cu -- S2 + S4 for dense QUBO (tcgen05 GEMM gradient).  Placeholder until the kernel lands.
#include "gda_internal.cuh"

static gda_status nyi() { gda_set_error("dense path: not built yet"); return GDA_ERR_UNSUPPORTED; }
gda_status dense_prepare(gda_problem*, const float*, const float*) { return nyi(); }
gda_status dense_make_operand(gda_problem*, int32_t, const float*, __nv_bfloat16*, int, cudaStream_t, int64_t*) { return nyi(); }
gda_status dense_step(gda_problem*, int32_t, float*, float*, const __nv_bfloat16*, __nv_bfloat16*, const UpdParams&,
                      const RunState*, uint32_t, cudaStream_t, int64_t*) { return nyi(); }
gda_status dense_grad(gda_problem*, int32_t, const float*, float*, cudaStream_t) { return nyi(); }
gda_status dense_score_partials(gda_problem*, int32_t, const float*, void*, int32_t*, cudaStream_t, int64_t*) { return nyi(); }
int32_t dense_num_partials(const gda_problem*, int32_t) { return 1; }
void dense_release(gda_problem*) {}
