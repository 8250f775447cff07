// gram_i8tc.cuh -- tensor-core engine of the all-pairs kernel (tcgen05 kind::i8).  Placeholder until the
// kernel lands: reports "unsupported" so AUTO falls back to the FFMA engine.
#pragma once
#include "common.cuh"

namespace clusco {

static inline bool i8tc_supported(int32_t) { return false; }

static inline int i8tc_prepare(const float*, int64_t, int32_t, const Workspace&, char*, ModelStat*, cudaStream_t)
{
    return CLUSCO_ERR_INVALID_ARG;
}

static inline int i8tc_compute(int64_t, int32_t, int64_t, int64_t, float*, const Workspace&, char*, ModelStat*, int,
                               cudaStream_t)
{
    return CLUSCO_ERR_INVALID_ARG;
}

}  // namespace clusco
