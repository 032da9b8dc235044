// peek_api.cu — status strings, thread-local error detail, workspace sizing (include/peek.h).
#include <stdarg.h>
#include <string.h>

#include <mutex>
#include <vector>

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

static int g_grid_limit = 0;  // PEEK_OPT_GRID_LIMIT
bool grid_limited() { return g_grid_limit > 0; }  // the test hook is set: small-queue shortcuts stand aside
int persistent_ctas() {       // CTAs of a persistent cooperative kernel: one per SM unless capped
    int n = sm_count();
    return (g_grid_limit > 0 && g_grid_limit < n) ? g_grid_limit : n;
}

cudaError_t func_smem_optin(const void* func, int bytes) {
    struct Done { int dev; const void* func; int bytes; };
    static std::mutex mu;
    static std::vector<Done> done;
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    std::lock_guard<std::mutex> lock(mu);
    for (const Done& d : done)
        if (d.dev == dev && d.func == func && d.bytes >= bytes) return cudaSuccess;
    e = cudaFuncSetAttribute(func, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    if (e == cudaSuccess) done.push_back(Done{dev, func, bytes});
    return e;
}

static std::mutex g_side_mu;
bool side_fork(cudaStream_t st, SideStream* ss) {
    struct PerDev { int dev; SideStream s; };
    static std::vector<PerDev> made;
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(st, &cs) != cudaSuccess || cs != cudaStreamCaptureStatusNone) {
        cudaGetLastError();
        return false;
    }
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return false;
    g_side_mu.lock();
    const SideStream* found = nullptr;
    for (const PerDev& d : made)
        if (d.dev == dev) found = &d.s;
    if (!found) {
        SideStream n{};
        if (cudaStreamCreateWithFlags(&n.side, cudaStreamNonBlocking) != cudaSuccess ||
            cudaEventCreateWithFlags(&n.fork, cudaEventDisableTiming) != cudaSuccess ||
            cudaEventCreateWithFlags(&n.join, cudaEventDisableTiming) != cudaSuccess) {
            cudaGetLastError();
            g_side_mu.unlock();
            return false;
        }
        made.push_back(PerDev{dev, n});
        found = &made.back().s;
    }
    *ss = *found;
    if (cudaEventRecord(ss->fork, st) != cudaSuccess || cudaStreamWaitEvent(ss->side, ss->fork, 0) != cudaSuccess) {
        cudaGetLastError();
        g_side_mu.unlock();
        return false;
    }
    return true;  // side_join unlocks
}
cudaError_t side_join(cudaStream_t st, const SideStream& ss) {
    cudaError_t e = cudaEventRecord(ss.join, ss.side);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(st, ss.join, 0);
    g_side_mu.unlock();
    return e;
}

int sm_count() {
    int dev = 0, n = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return 148;
    if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) return 148;
    return n;
}

// ---- tracing ---------------------------------------------------------------------------
static const char* const g_prof_names[PROF_NSLOTS] = {
    "hash.nb_scan", "hash.content", "hash.chain", "tree.persistent", "lpm.radix_walk", "lpm.hash_probe",
    "lpm.resolve_scan", "lpm.dual_walk", "demand.count", "rank.clpm_sort", "signals.clpm", "rank.full_key", "offline.phase1"};
static constexpr int PROF_RING = 512;
struct ProfSlotState {
    cudaEvent_t ev[PROF_RING][2];
    int created, used;
};
static ProfSlotState g_prof[PROF_NSLOTS];
static bool g_prof_on = false;
static long long g_launches = 0;

void prof_begin(int slot, cudaStream_t st) {
    if (!g_prof_on) return;
    ProfSlotState& p = g_prof[slot];
    if (p.used >= PROF_RING) return;
    if (p.used >= p.created) {
        if (cudaEventCreate(&p.ev[p.created][0]) != cudaSuccess) return;
        if (cudaEventCreate(&p.ev[p.created][1]) != cudaSuccess) return;
        p.created++;
    }
    cudaEventRecord(p.ev[p.used][0], st);
}

void prof_end(int slot, cudaStream_t st, int launches) {
    g_launches += launches;
    if (!g_prof_on) return;
    ProfSlotState& p = g_prof[slot];
    if (p.used >= PROF_RING || p.used >= p.created) return;
    cudaEventRecord(p.ev[p.used][1], st);
    p.used++;
}

i64 block_hash_ws_bytes(i64 N);
i64 lpm_ws_bytes(i64 N, i64 V);
i64 pending_tree_ws_bytes(i64 N);
i64 demand_rank_ws_bytes(i64 N, i64 S);
i64 clpm_signals_ws_bytes(i64 N, i64 S);
i64 clpm_order_full_ws_bytes(i64 N);
i64 group_major_ws_bytes(i64 N);
i64 offline_phase1_ws_bytes(i64 N);
i64 pending_tree_update_ws_bytes(i64 N_old, i64 N_new, i64 M);
void lpm_set_option(int key, i64 v);
void tree_set_option(int key, i64 v);

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
    if (!out_bytes || N < 0 || S < 0) {
        peek::set_error("peek_workspace_bytes: bad argument");
        return PEEK_ERR_INVALID_ARG;
    }
    switch (call_id) {
        case PEEK_CALL_BLOCK_HASH: *out_bytes = peek::block_hash_ws_bytes(N); break;
        case PEEK_CALL_LPM: *out_bytes = peek::lpm_ws_bytes(N, V > 0 ? V : 0); break;
        case PEEK_CALL_PENDING_TREE: *out_bytes = peek::pending_tree_ws_bytes(N); break;
        case PEEK_CALL_DEMAND_RANK: *out_bytes = peek::demand_rank_ws_bytes(N, S); break;
        case PEEK_CALL_CLPM_SIGNALS: *out_bytes = peek::clpm_signals_ws_bytes(N, S); break;
        case PEEK_CALL_CLPM_ORDER_FULL: *out_bytes = peek::clpm_order_full_ws_bytes(N); break;
        case PEEK_CALL_CLPM_GROUP_MAJOR: *out_bytes = peek::group_major_ws_bytes(N); break;
        case PEEK_CALL_OFFLINE_PHASE1: *out_bytes = peek::offline_phase1_ws_bytes(N); break;
        case PEEK_CALL_PENDING_TREE_UPDATE:  // N = N_new, T = N_old, NB = M
            if (T < 0 || NB < 0) { peek::set_error("peek_workspace_bytes: bad sizes"); return PEEK_ERR_INVALID_ARG; }
            *out_bytes = peek::pending_tree_update_ws_bytes(T, N, NB);
            break;
        default:
            peek::set_error("peek_workspace_bytes: unknown call_id %d", call_id);
            return PEEK_ERR_INVALID_ARG;
    }
    if (*out_bytes < 256) *out_bytes = 256;
    return PEEK_OK;
}

extern "C" peek_status peek_set_option(int32_t key, int64_t value) {
    if ((key == PEEK_OPT_LPM_STRATEGY && value >= 0 && value <= 2) ||
        (key == PEEK_OPT_LPM_WINDOW && value >= 0 && value <= (1 << 20))) {
        peek::lpm_set_option(key, value);
        return PEEK_OK;
    }
    if (key == PEEK_OPT_TREE_LOCAL_CAP && value >= 0 && value <= (1 << 20)) {
        peek::tree_set_option(key, value);
        return PEEK_OK;
    }
    if (key == PEEK_OPT_GRID_LIMIT && value >= 0 && value <= 65536) {
        peek::g_grid_limit = (int)value;
        return PEEK_OK;
    }
    peek::set_error("peek_set_option: unknown key %d or bad value %lld", key, (long long)value);
    return PEEK_ERR_INVALID_ARG;
}

extern "C" void peek_profile_enable(int32_t on) { peek::g_prof_on = on != 0; }
extern "C" int32_t peek_profile_slots(void) { return peek::PROF_NSLOTS; }
extern "C" const char* peek_profile_name(int32_t slot) {
    return (slot >= 0 && slot < peek::PROF_NSLOTS) ? peek::g_prof_names[slot] : "";
}
extern "C" peek_status peek_profile_read(int32_t slot, double* total_ms, int64_t* groups, int32_t reset) {
    if (slot < 0 || slot >= peek::PROF_NSLOTS || !total_ms || !groups) {
        peek::set_error("peek_profile_read: bad argument");
        return PEEK_ERR_INVALID_ARG;
    }
    peek::ProfSlotState& p = peek::g_prof[slot];
    double tot = 0;
    for (int i = 0; i < p.used; ++i) {
        PEEK_CUDA(cudaEventSynchronize(p.ev[i][1]));
        float ms = 0;
        PEEK_CUDA(cudaEventElapsedTime(&ms, p.ev[i][0], p.ev[i][1]));
        tot += ms;
    }
    *total_ms = tot;
    *groups = p.used;
    if (reset) p.used = 0;
    return PEEK_OK;
}
extern "C" int64_t peek_launch_count(void) { return peek::g_launches; }
