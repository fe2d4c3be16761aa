#include "etp_internal.h"
extern "C" etp_status etp_shard_linear(etp_ctx* ctx, etp_linear_mode mode, etp_dtype dtype, const void* x, int64_t tokens,
                                       int64_t in_features, int64_t out_features, const etp_tensor* w,
                                       const etp_shard* layout, int32_t n_shards, int64_t features_per_unit, void* y,
                                       void* stream) {
    ETP_FAIL(ETP_ERR_UNSUPPORTED, "etp_shard_linear: not built yet");
}
