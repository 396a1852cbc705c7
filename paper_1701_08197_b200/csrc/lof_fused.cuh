// lof_fused.cuh — shape-specialised fused kernels (filled in below the generic path).
#pragma once
#include "lof_common.cuh"
