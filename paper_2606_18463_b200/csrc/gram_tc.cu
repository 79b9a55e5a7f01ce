// gram_tc.cu -- placeholder until the tcgen05 kernel lands (next commit).
#include <cstdio>
#include "common.cuh"
namespace casgd {
struct GramTcPlan { int unused; };
GramTcPlan *gram_tc_plan_create(const uint16_t *, int32_t, int32_t, int32_t, const uint16_t *, char *err, int errlen)
{
    snprintf(err, errlen, "tcgen05 Gram kernel not built yet; set CASGD_OPT_GRAM_IMPL = 1");
    return nullptr;
}
void gram_tc_plan_destroy(GramTcPlan *p) { delete p; }
int launch_gram_tc(cudaStream_t, GramTcPlan *, int32_t, int32_t, float *, int32_t, float *, int, char *, int) { return -1; }
}  // namespace casgd
