// host_lhcs_avx2.cpp -- worker systems of Algorithm 2, 4 worker(s) per step.
// See host_lhcs_lanes.inc.  Build flags: -mavx2 and -ffp-contract=off.
#define VCRYPT_LANES 4
#define VCRYPT_FN derive_workers_avx2
#include "host_lhcs_lanes.inc"
