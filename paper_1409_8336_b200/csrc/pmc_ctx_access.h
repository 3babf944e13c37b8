// pmc_ctx_access.h — the few facts about a pmc_ctx (defined in pmc_api.cu) that another translation unit of libpmc
// needs: which device and stream it was created on, its SM count, and how to leave an error message in it.
#pragma once
#include <cuda_runtime.h>

#include "../../include/pmc.h"

namespace pmc {
int ctx_device(const pmc_ctx *c);
cudaStream_t ctx_stream(const pmc_ctx *c);
int ctx_sm_count(const pmc_ctx *c);
int ctx_fail(pmc_ctx *c, int code, const char *msg);      // stores msg (if c is not null) and returns code
}  // namespace pmc
