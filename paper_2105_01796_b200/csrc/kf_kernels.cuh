// kf_kernels.cuh -- every kernel template of the thread-per-track and lanes-per-track variants.
#pragma once

#include "kf_common.cuh"
#include "kf_forward.cuh"
#include "kf_rts.cuh"
