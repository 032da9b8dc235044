// peek_api.cu — status strings, thread-local error detail, workspace sizing (include/peek.h).
#include <stdarg.h>
#include <string.h>

#include "peek_common.cuh"

namespace peek {

static thread_local char g_err[512] = "";

void set_error(const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
}

peek_status cuda_fail(cudaError_t e, const char* what) {
    set_error("%s: %s", what, cudaGetErrorString(e));
    return PEEK_ERR_CUDA;
}

int sm_count() {
    int dev = 0, n = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return 148;
    if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) return 148;
    return n;
}

i64 block_hash_ws_bytes(i64 N);
i64 lpm_ws_bytes(i64 N);
i64 pending_tree_ws_bytes(i64 N);
i64 demand_rank_ws_bytes(i64 N, i64 S);

}  // namespace peek

extern "C" const char* peek_status_string(peek_status s) {
    switch (s) {
        case PEEK_OK: return "PEEK_OK";
        case PEEK_ERR_INVALID_ARG: return "PEEK_ERR_INVALID_ARG";
        case PEEK_ERR_CAPACITY: return "PEEK_ERR_CAPACITY";
        case PEEK_ERR_WORKSPACE: return "PEEK_ERR_WORKSPACE";
        case PEEK_ERR_CUDA: return "PEEK_ERR_CUDA";
        case PEEK_ERR_UNSUPPORTED: return "PEEK_ERR_UNSUPPORTED";
        case PEEK_ERR_UNIMPLEMENTED: return "PEEK_ERR_UNIMPLEMENTED";
        default: return "PEEK_ERR_UNKNOWN";
    }
}

extern "C" const char* peek_last_error(void) { return peek::g_err; }

extern "C" int32_t peek_version(void) { return 100; }

extern "C" peek_status peek_workspace_bytes(int32_t call_id, int64_t N, int64_t T, int64_t NB,
                                            int64_t S, int64_t V, int64_t* out_bytes) {
    (void)T; (void)NB; (void)V;
    if (!out_bytes || N < 0 || S < 0) {
        peek::set_error("peek_workspace_bytes: bad argument");
        return PEEK_ERR_INVALID_ARG;
    }
    switch (call_id) {
        case PEEK_CALL_BLOCK_HASH: *out_bytes = peek::block_hash_ws_bytes(N); break;
        case PEEK_CALL_LPM: *out_bytes = peek::lpm_ws_bytes(N); break;
        case PEEK_CALL_PENDING_TREE: *out_bytes = peek::pending_tree_ws_bytes(N); break;
        case PEEK_CALL_DEMAND_RANK: *out_bytes = peek::demand_rank_ws_bytes(N, S); break;
        default:
            peek::set_error("peek_workspace_bytes: unknown call_id %d", call_id);
            return PEEK_ERR_INVALID_ARG;
    }
    if (*out_bytes < 256) *out_bytes = 256;
    return PEEK_OK;
}
