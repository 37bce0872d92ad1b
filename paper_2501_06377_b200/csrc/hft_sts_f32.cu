// hft_sts_f32.cu -- the temporally blocked STS step in float (see hft_sts_f64.cu); the fp32-storage / fp64-arithmetic
// instantiations of k_sts_upipe are compiled in hft_sts_mixed.cu.
#include "hft_sts_step.cuh"

template int hft::sts_blocked_step<float>(hft::StsBlockedPlan<float>&, hft::Tables<float>&, const hft::Geom&, int64_t*);
