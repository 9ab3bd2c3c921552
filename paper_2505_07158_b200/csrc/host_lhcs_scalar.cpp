// host_lhcs_scalar.cpp -- worker systems of Algorithm 2, 1 worker(s) per step.
// See host_lhcs_lanes.inc.  Build flags: (baseline x86-64) and -ffp-contract=off.
#define VCRYPT_LANES 1
#define VCRYPT_FN derive_workers_scalar
#include "host_lhcs_lanes.inc"
