// host_lhcs_avx512.cpp -- worker systems of Algorithm 2, 8 worker(s) per step.
// See host_lhcs_lanes.inc.  Build flags: -mavx512f -mavx512dq and -ffp-contract=off.
#define VCRYPT_LANES 8
#define VCRYPT_FN derive_workers_avx512
#include "host_lhcs_lanes.inc"
