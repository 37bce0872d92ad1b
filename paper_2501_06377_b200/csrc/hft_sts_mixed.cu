// hft_sts_mixed.cu -- k_sts_upipe with fp32 storage and fp64 arithmetic (hft_options.f32_arith = 0), a translation unit
// of its own: its coefficient table (fp64) has its own constant bank, and the units build in parallel.
#define HFT_STS_MIXED_TU
#include "hft_sts_upipe.cuh"

namespace hft {
#define HFT_INST(K)                                                                                                              \
    template int sts_upipe_launch<float, double, K>(const StsBlockedPlan<float>&, const UPipePlan&, Tables<float>&, const Geom&, \
                                                    int, const float*, const float*, float*, float*, bool, int64_t*);
HFT_INST(2) HFT_INST(4) HFT_INST(6) HFT_INST(8)
#undef HFT_INST
}  // namespace hft
