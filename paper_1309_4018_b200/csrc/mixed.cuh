// mixed.cuh -- PYGBE_PRECISION_MIXED: P2P / M2P arithmetic in fp32, fp64 accumulation (a6, a7 at
// BASELINE.json config 4's precision).  Placeholder until the fp32 kernels land.
#pragma once
#include "common.cuh"

static int mixed_build_region(pygbe_handle *h, Region &R)
{
    (void)h; (void)R;
    pygbe_set_error("PYGBE_PRECISION_MIXED is not implemented yet");
    return PYGBE_EINVAL;
}
static int mixed_region_sum(pygbe_handle *h, Region &R, const int *skip)
{
    (void)h; (void)R; (void)skip;
    pygbe_set_error("PYGBE_PRECISION_MIXED is not implemented yet");
    return PYGBE_EINVAL;
}
