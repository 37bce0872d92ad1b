// hft_sts_f32.cu -- the temporally blocked STS step in float: every k_sts_pipe / k_sts_capseq / k_sts_blocked instantiation
// of this precision lives in this translation unit (explicit instantiation; hft_api.cu declares it extern).
#include "hft_sts_pipe.cuh"

template int hft::sts_blocked_step<float>(hft::StsBlockedPlan<float>&, hft::Tables<float>&, const hft::Geom&, int, int64_t*);
