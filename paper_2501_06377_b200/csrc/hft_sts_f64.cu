// hft_sts_f64.cu -- the temporally blocked STS step in double: every k_sts_pipe / k_sts_upipe / k_sts_capseq instantiation
// of this precision lives in this translation unit (explicit instantiation; hft_api.cu declares it extern).
#include "hft_sts_step.cuh"

template int hft::sts_blocked_step<double>(hft::StsBlockedPlan<double>&, hft::Tables<double>&, const hft::Geom&, int64_t*);
