/* peek.h — C ABI of libpeek.so: the data-parallel hot path behind PEEK
 * (arxiv/paper_2607_02525, "Predictive Queue-Informed KV Cache Management for LLM
 * Serving"), as hand-written sm_100a CUDA kernels.
 *
 * Four calls (BASELINE.json north_star):
 *   peek_block_hash    chained per-block hashes of CSR int32 token sequences
 *                      ("k_i = hash(k_{i-1}, tuple(s[iB:(i+1)B]))", B = 16)
 *   peek_pending_tree  the pending radix tree as a batch build: lexicographic order of the
 *                      requests' hash chains, adjacent LCP, groups and clusters
 *                      (PAPER.md:94 section 3.1, :287 section A.1.3, :125 has_sharing)
 *   peek_lpm           per-request hit length against the engine's prefix cache: a radix cache
 *                      (Alg. 1) and/or a flat block-hash table
 *                      ("per-request find_longest_cache_hit")
 *   peek_demand_rank   per-cached-block pending demand for the eviction hook (PAPER.md:115-119
 *                      Eq. 2 pending_count; :281 inverted index block_hash -> demand) and the cLPM
 *                      admission order, sub-key (-h, -|cluster|, arrival) of Eq. 1
 * and the next rows of SURVEY.md 8(f), declared further down: peek_clpm_signals (sections, ancestor
 * score, Eq. 2 eviction score), peek_radix_demand, peek_clpm_order_full (the five-part key of Eq. 1),
 * peek_clpm_group_major, peek_clpm_lane_b, peek_dynamic_lane, peek_stride_interleave (Alg. 2 of
 * PAPER.md:325 end to end), peek_pending_tree_update (incremental maintenance) and
 * peek_offline_phase1 (PEEK-offline's reordering and guards).
 *
 * Conventions (the paper is silent on all of them):
 *   Pointers   every array pointer is caller-owned DEVICE memory unless marked [host]; it must
 *              stay valid until the work enqueued on `stream` has completed.  The library keeps
 *              no state between calls, allocates no device memory and frees none.
 *   Workspace  `ws` is caller-allocated device scratch of at least peek_workspace_bytes(...)
 *              bytes, 256-byte aligned; contents undefined before and after.  Too small ->
 *              PEEK_ERR_WORKSPACE, nothing enqueued.
 *   Stream     `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).
 *              Calls only enqueue work: no device synchronisation, no device->host copy.
 *   Errors     return code only (0 = PEEK_OK, < 0 = error); peek_last_error() gives a
 *              thread-local detail string.  Argument errors are detected on the host before
 *              anything is enqueued.  Contents of device arrays are trusted (monotone offsets,
 *              valid child indices, >= 1 EMPTY table slot) and not validated.
 *   Sizes      N = 0 is PEEK_OK and touches nothing.  N < 2^31 - 1.  block_size must be 16
 *              (every config) else PEEK_ERR_UNSUPPORTED.  The element counts of
 *              `tokens` and `hashes` live on the device (tok_off[N], blk_off[N]), so the host
 *              checks cannot see them: an array that a requested output needs must be non-NULL
 *              even when it holds no element (a queue without a full block has NB = 0); it is
 *              then never read.
 *   Aliasing   inputs and outputs never alias each other or `ws`.
 *   Determinism outputs are a pure function of the inputs (no dependence on atomics order).
 *   There is no CPU fallback anywhere in this library.
 */
#ifndef PEEK_H_
#define PEEK_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef int32_t peek_status;
enum {
    PEEK_OK = 0,
    PEEK_ERR_INVALID_ARG = -1,   /* NULL where required, negative size, S not a power of two, ... */
    PEEK_ERR_CAPACITY = -2,      /* an output capacity the host can check is too small */
    PEEK_ERR_WORKSPACE = -3,     /* ws NULL / misaligned / smaller than peek_workspace_bytes */
    PEEK_ERR_CUDA = -4,          /* a CUDA runtime call failed; see peek_last_error() */
    PEEK_ERR_UNSUPPORTED = -5,   /* block_size != 16 */
    PEEK_ERR_UNIMPLEMENTED = -6
};

/* Table EMPTY sentinel: no chained hash ever equals it (peek_block_hash remaps). */
#define PEEK_EMPTY_KEY 0xFFFFFFFFFFFFFFFFull

/* Static strings, never freed.  peek_last_error is thread-local, "" if none. */
const char* peek_status_string(peek_status s);
const char* peek_last_error(void);
int32_t peek_version(void); /* major*10000 + minor*100 + patch */

/* ---- workspace -------------------------------------------------------------------------- */
enum {
    PEEK_CALL_BLOCK_HASH = 0,
    PEEK_CALL_LPM = 1,
    PEEK_CALL_PENDING_TREE = 2,
    PEEK_CALL_DEMAND_RANK = 3,
    PEEK_CALL_CLPM_SIGNALS = 4,
    PEEK_CALL_CLPM_ORDER_FULL = 5,
    PEEK_CALL_CLPM_GROUP_MAJOR = 6,
    PEEK_CALL_OFFLINE_PHASE1 = 7,
    PEEK_CALL_PENDING_TREE_UPDATE = 8 /* pass N = N_new, T = N_old, NB = M */
};
/* Bytes of device scratch `call_id` needs for the given sizes [host out].  N requests, T tokens,
 * NB hashed blocks, S table slots, V radix nodes; pass 0 for sizes a call does not use. */
peek_status peek_workspace_bytes(int32_t call_id, int64_t N, int64_t T, int64_t NB, int64_t S,
                                 int64_t V, int64_t* out_bytes);

/* ---- a1: chained block hash ----------------------------------------- */
/* tokens  int32[T]  CSR token pool, request r = tokens[tok_off[r] .. tok_off[r+1]); the pointer must
 *                    be 16-byte aligned (the kernel stages tokens with 16-byte bulk copies)
 * tok_off int64[N+1] monotone, tok_off[0] >= 0
 * seed    k_{-1} of every chain
 * blk_off int64[N+1] OUT exclusive prefix sum of nb_r = floor(len_r / block_size)
 * hashes  uint64[NB] OUT k^r_i at hashes[blk_off[r] + i]; the trailing partial block of a request
 *                    is not hashed.  hashes_capacity = number of uint64 the buffer holds; the
 *                    caller computes NB = sum floor(len_r/B) on the host (it owns tok_off);
 *                    kernels never write at or beyond hashes_capacity.
 * Hash function (the paper names none; R1): tokens as uint32 bit patterns,
 *   S_i = sum_j (tok[iB+j] + 1) * M_j,  M_j = mix64(j+1)|1,  c_i = mix64(S_i),
 *   k_i = mix64(k_{i-1} ^ c_i), remapped to 0xFF..FE if it equals PEEK_EMPTY_KEY (remapped value
 *   is stored and carried); mix64 = the splitmix64 finaliser. */
peek_status peek_block_hash(const int32_t* tokens, const int64_t* tok_off, int64_t N,
                            int32_t block_size, uint64_t seed, int64_t* blk_off, uint64_t* hashes,
                            int64_t hashes_capacity, void* ws, int64_t ws_bytes, void* stream);

/* The same operation for callers that cannot allocate device memory (code under CUDA-graph capture,
 * serving loops and harnesses that forbid cudaMalloc): no `ws` - the scratch is a 32 KB file-scope
 * `static __device__` array inside the library, which every GPU that loads the library holds until
 * the process exits.  Arguments, layouts, outputs and error behaviour are those of peek_block_hash;
 * in addition N > PEEK_BLOCK_HASH_STATIC_MAX_N is rejected with PEEK_ERR_CAPACITY (nothing is
 * touched).  The call makes no cudaMalloc / cudaFree and no allocating library call.  ALL calls on
 * a device share the one array: two calls that overlap on the GPU (different streams, or two host
 * threads on different streams) race and corrupt each other - serialise them on one stream or use
 * peek_block_hash with separate workspaces.  The array keeps the last call's contents; the kernels
 * rewrite everything they read from it, so nothing has to be cleared between calls. */
#define PEEK_BLOCK_HASH_STATIC_MAX_N 4194304
peek_status peek_block_hash_static(const int32_t* tokens, const int64_t* tok_off, int64_t N,
                                   int32_t block_size, uint64_t seed, int64_t* blk_off,
                                   uint64_t* hashes, int64_t hashes_capacity, void* stream);

/* ---- the engine's prefix cache, read-only --------------------------------- */
/* Radix cache flattened to arrays.  Node 0 is the root (empty label).  Node u's label is
 * c_tokens[n_tok_off[u] .. + n_tok_len[u]).  The children of node v are edges
 * n_child_off[v] .. n_child_off[v+1]; within a node edges are sorted ascending by e_first_tok
 * (signed int32), first tokens are distinct, and e_first_tok[e] == first label token of
 * e_child[e] ("children keyed by the first edge token"). */
typedef struct {
    const int32_t* c_tokens;    /* int32[CT] */
    int64_t CT;
    const int64_t* n_tok_off;   /* int64[V] */
    const int32_t* n_tok_len;   /* int32[V] */
    const int32_t* n_child_off; /* int32[V+1] */
    int32_t V;
    const int32_t* e_first_tok; /* int32[E] */
    const int32_t* e_child;     /* int32[E] */
    int32_t E;
} peek_radix;

/* Flat block-hash cache: open addressing, linear probing, home = key & (S-1), S a power of two,
 * empty slots hold PEEK_EMPTY_KEY, each key at most once, no tombstones, >= 1 empty slot. */
typedef struct {
    const uint64_t* t_keys; /* uint64[S] */
    int64_t S;
} peek_table;

/* Optional accelerator for peek_lpm: outputs of peek_pending_tree over the SAME hashes/blk_off.
 * order/lcp are by sorted position.  With it, peek_lpm co-descends: a request whose sorted
 * predecessor's hit ends inside their common prefix copies that hit without touching the cache;
 * otherwise it resumes at the common depth (Alg. 1 "one cache walk per pending edge",
 * PAPER.md:73-82, :96).  Results are identical with and without it. */
typedef struct {
    const int32_t* order; /* int32[N] */
    const int32_t* lcp;   /* int32[N] */
} peek_tree_view;

/* ---- a5/a6: longest prefix match (Alg. 1; hash mode PAPER.md:87-89) -- */
/* hit_radix int32[N] OUT (NULL to skip; needs radix, tokens, tok_off): tokens of request r matched
 *           from the root; a partial edge match ends the walk; token-granular; not capped at len-1.
 * hit_hash  int32[N] OUT (NULL to skip; needs table, hashes, blk_off): block_size * number of
 *           leading blocks whose chained hash is in the table, scanning to the FIRST miss.
 * tree      optional (NULL = naive per-request walk; needs hashes/blk_off as given to
 *           peek_pending_tree).
 * Streams   With a tree view and BOTH modes requested (queues above 2048 requests) the two walks are
 *           independent kernels: the hash probes run on a side stream that the library creates once
 *           per device (one non-blocking stream and two events, kept until the process exits; no
 *           device memory), forked from and joined back into `stream`, so for the caller the call is
 *           still ordered on `stream` alone.  If `stream` is being captured into a CUDA graph, or the
 *           side stream cannot be made, both kernels stay on `stream`.  Calls from several host
 *           threads share the side stream: they stay correct and serialise on it. */
peek_status peek_lpm(const int32_t* tokens, const int64_t* tok_off, const uint64_t* hashes,
                     const int64_t* blk_off, int64_t N, int32_t block_size,
                     const peek_radix* radix /*host struct*/, const peek_table* table /*host struct*/,
                     const peek_tree_view* tree /*host struct*/, int32_t* hit_radix,
                     int32_t* hit_hash, void* ws, int64_t ws_bytes, void* stream);

/* ---- a2-a4: pending radix tree at block granularity ------------ */
/* order         int32[N] OUT sorted position -> request; chains compared word by word as unsigned
 *               64-bit, a proper prefix first, identical chains by ascending request index
 * lcp           int32[N] OUT lcp[0] = 0; lcp[j] = leading equal hash words of order[j-1], order[j]
 * group_id      int32[N] OUT by request: dense id (in sorted order) of the root-child subtree;
 *               a new group starts at sorted position j iff lcp[j] == 0
 * group_size    int32[N] OUT by request: members of its group   (has_sharing <=> max >= 2)
 * cluster_depth int32[N] OUT by request: depth in blocks of the deepest node on its path with
 *               pending_count >= 2 (0 = none: singleton)
 * cluster_size  int32[N] OUT by request: that node's pending_count (1 for singletons)
 * cluster_id    int64[N] OUT by request: (first sorted position under the node << 32) | depth;
 *               (sorted position << 32) for singletons
 * n_groups      int32[1] OUT device scalar
 * Any of group_id .. n_groups may be NULL (skipped); order and lcp are required.
 * Relies on the chain property "k_i equal => k_j equal for all j < i" (true unless two distinct
 * blocks collide in 64 bits; R15). */
peek_status peek_pending_tree(const uint64_t* hashes, const int64_t* blk_off, int64_t N,
                              int32_t* order, int32_t* lcp, int32_t* group_id, int32_t* group_size,
                              int32_t* cluster_depth, int32_t* cluster_size, int64_t* cluster_id,
                              int32_t* n_groups, void* ws, int64_t ws_bytes, void* stream);

/* ---- a7/a8: eviction demand and cLPM order (Eq. 1) */
/* demand     int32[S] OUT (NULL to skip; needs hashes, blk_off, order, lcp, table): for an occupied
 *            slot the number of (request, block) pairs whose chained hash equals its key, 0 for
 *            empty slots.  Independent of hit lengths.
 * clpm_order int32[N] OUT (NULL to skip; needs hit, cluster_size): request indices sorted ascending
 *            by (-hit[r], -cluster_size[r], arrival[r], r); arrival NULL => arrival[r] = r. */
peek_status peek_demand_rank(const uint64_t* hashes, const int64_t* blk_off, int64_t N,
                             const int32_t* order, const int32_t* lcp,
                             const peek_table* table /*host struct*/, const int32_t* hit,
                             const int32_t* cluster_size, const int32_t* arrival, int32_t* demand,
                             int32_t* clpm_order, void* ws, int64_t ws_bytes, void* stream);

/* ---- a9/a10: the remaining signals of Eq. 1 and Eq. 2 ------------------ */
/* Read off the pending tree (order, lcp of peek_pending_tree) - DESIGN.md R20-R23.
 * section     int32[N] OUT by request (NULL to skip; needs hit): 0 warm if hit[r] > tau; else
 *             1 pioneer if r has the smallest (arrival, index) among the cold requests that share its
 *             first theta = 32 tokens (= two blocks; one block for a one-block prompt; a request with
 *             no full block is always a pioneer), else 2 sibling.  Equivalent to the sequential
 *             `seen` loop of Alg. 2 in arrival order.  arrival NULL => the index.
 * score       int64[N] OUT by request (NULL to skip): ancestor score of PAPER.md:102,
 *             16 * sum over the blocks i of r of pending_count(block i of r), pending_count = number
 *             of pending (request, block) pairs with that chained hash.
 * evict_score int64[S] OUT (NULL to skip; needs hashes, table): Eq. 2 per table
 *             slot - for a slot whose key is block i of some pending chain, the maximum over
 *             j <= i of pending_count(block j) * 16 * (j + 1); 0 for empty slots and for slots on no
 *             pending chain (zero-demand victims).  Lowest evicts first.
 * All pointers device; hit, arrival, hashes may be NULL when the outputs that need them are. */
peek_status peek_clpm_signals(const uint64_t* hashes, const int64_t* blk_off, int64_t N,
                              const int32_t* order, const int32_t* lcp, const int32_t* hit, int32_t tau,
                              const int32_t* arrival, const peek_table* table /*host struct*/,
                              int32_t* section, int64_t* score, int64_t* evict_score,
                              void* ws, int64_t ws_bytes, void* stream);

/* clpm_order int32[N] OUT request indices sorted ascending by the full key of Eq. 1
 *            (section[r], -hit[r], -score[r], -cluster_size[r], arrival[r], r); arrival NULL => r.
 * All inputs device arrays by request; all but arrival required. */
peek_status peek_clpm_order_full(const int32_t* section, const int32_t* hit, const int64_t* score,
                                 const int32_t* cluster_size, const int32_t* arrival, int64_t N,
                                 int32_t* clpm_order, void* ws, int64_t ws_bytes, void* stream);

/* a9b: per-radix-node pending demand (R26), the radix-cache
 * counterpart of `demand`: node_demand[v] int32[V] OUT = pending requests whose longest-prefix match
 * enters node v (matches >= 1 token of its label); node_demand[0] (root) = N.
 * hit_radix int32[N] must be peek_lpm's radix-mode result for the same queue and cache. */
peek_status peek_radix_demand(const int32_t* tokens, const int64_t* tok_off, int64_t N,
                              const peek_radix* radix /*host struct*/, const int32_t* hit_radix,
                              int32_t* node_demand, void* stream);

/* a11 (first part): group-major admission (worked example
 * PAPER.md:55; R24).
 * lane_order int32[N] a permutation of the requests (the cache-locality lane: peek_clpm_order_full)
 * cluster_id int64[N] by request (peek_pending_tree)
 * gm_order   int32[N] OUT requests ordered by (lane position of the first member of their cluster,
 *            own lane position): every cluster comes out contiguous, right behind its first member. */
peek_status peek_clpm_group_major(const int32_t* lane_order, const int64_t* cluster_id, int64_t N,
                                  int32_t* gm_order, void* ws, int64_t ws_bytes, void* stream);

/* a11b: the fairness lane of Alg. 2 line 18: request indices sorted ascending by
 * (section[r], arrival[r], -hit[r], r); arrival NULL => r.  Workspace: PEEK_CALL_CLPM_ORDER_FULL. */
peek_status peek_clpm_lane_b(const int32_t* section, const int32_t* hit, const int32_t* arrival, int64_t N,
                             int32_t* lane_b_order, void* ws, int64_t ws_bytes, void* stream);

/* a11c: the dynamic-lane controller of PAPER.md:111-113 (Alg. 2 line 20; R27):
 * out[0] = 0.3 * clamp(0.15 + 0.5 * singleton_frac + 0.3 * age_pressure, 0.10, 0.60)
 *          + 0.7 * prev_fair_share     (the new fairness share 1 - alpha, double, every product and
 *          sum rounded once), out[1] = singleton_frac = fraction of requests with cluster_size == 1.
 * out double[2] device; age_pressure = min(1, oldest singleton wait / 2 s) is the engine's to supply.
 * Workspace: >= 256 bytes. */
peek_status peek_dynamic_lane(const int32_t* cluster_size, int64_t N, double age_pressure,
                              double prev_fair_share, double* out, void* ws, int64_t ws_bytes, void* stream);

/* a13: incremental maintenance of the pending tree (PAPER.md:21, :94, :287:
 * the paper inserts and removes requests instead of rebuilding).  The new queue has N_new requests:
 * the survivors of the old queue, renumbered by `remap`, and M arrivals at indices
 * N_new - M .. N_new - 1; hashes / blk_off describe the NEW queue (survivors' chains unchanged).
 * old_order, old_lcp int32[N_old]  the previous result of peek_pending_tree / _update
 * remap     int32[N_old]           old request index -> new index, -1 = removed; increasing on the
 *                                  survivors (so that identical chains stay ordered by index)
 * Outputs as peek_pending_tree, and equal to what it returns on the new queue, without sorting the
 * survivors again: compaction + the arrivals' own sort + a bisection merge.  Pays off when M << N. */
peek_status peek_pending_tree_update(const uint64_t* hashes, const int64_t* blk_off, int64_t N_new, int64_t M,
                                     const int32_t* old_order, const int32_t* old_lcp, int64_t N_old,
                                     const int32_t* remap, int32_t* order, int32_t* lcp, int32_t* group_id,
                                     int32_t* group_size, int32_t* cluster_depth, int32_t* cluster_size,
                                     int64_t* cluster_id, int32_t* n_groups, void* ws, int64_t ws_bytes,
                                     void* stream);

/* a11d: the stride interleave of Alg. 2 line 22, which the paper names but does
 * not define; R28: admission slot k = 0, 1, .. belongs to Lane A iff
 * floor((k+1) * alpha) > floor(k * alpha) (double products rounded once), else to Lane B, and the lane
 * admits its first request not admitted yet.
 * lane_a, lane_b int32[N] permutations of the requests (peek_clpm_order_full / _group_major, _lane_b)
 * alpha in [0, 1]: the share of Lane A (1 - out[0] of peek_dynamic_lane; default 0.7)
 * out    int32[N] the admission order.  Workspace: (N + 31) / 32 * 4 bytes when that exceeds 160 KB
 * (N > 1.3 M), none otherwise.  Sequential across slots: one CTA, 1024 slots per step. */
peek_status peek_stride_interleave(const int32_t* lane_a, const int32_t* lane_b, int64_t N, double alpha,
                                   int32_t* out, void* ws, int64_t ws_bytes, void* stream);

/* a12: PEEK-offline phase 1 (R25).
 * depth_blocks the trie covers the first depth_blocks blocks of every chain (the paper's D = 128
 *              tokens = 8), 1..16
 * order        int32[N] OUT the permutation of the depth-first traversal that emits a node's
 *              terminators first (ascending request index) and visits children in descending
 *              subtree request count (ties: smallest request index below)
 * guards       double[4] OUT (device): duplication (fraction of requests whose whole chain equals an
 *              earlier request's), coverage (fraction sharing >= 2 blocks = 32 tokens with another),
 *              mean sharing depth in tokens over the first depth_blocks blocks, and 1.0 if any
 *              guard fires (duplication > 0.5, coverage < 0.1, depth < 64), else 0.0 */
peek_status peek_offline_phase1(const uint64_t* hashes, const int64_t* blk_off, int64_t N, int32_t depth_blocks,
                                int32_t* order, double* guards, void* ws, int64_t ws_bytes, void* stream);

/* ---- options: tuning and test hooks ------------------------------------------------------- */
/* Process-wide, not thread-safe against concurrent calls; results never depend on them.
 * PEEK_OPT_LPM_STRATEGY  how peek_lpm co-descends when a tree view is given:
 *     PEEK_LPM_AUTO (default)  dual-walk; queues of at most 2048 requests take one launch of
 *                              per-request walks (both modes)
 *     PEEK_LPM_DUAL_WALK       a warp walks a run of sorted positions in order, carrying the
 *                              predecessor's hit and cache path (Alg. 1's co-descent)
 *     PEEK_LPM_SPECULATIVE     every position walks in parallel from its shared depth, a scan
 *                              resolves which walks were needed
 * PEEK_OPT_LPM_WINDOW    sorted positions per dual-walk window (0 = automatic)
 * PEEK_OPT_GRID_LIMIT    cap on the CTAs of the persistent (cooperative) kernels of
 *                        peek_pending_tree and peek_demand_rank; 0 = one per SM (default).  A test
 *                        hook: a small cap makes every CTA loop over several tiles at small N.
 * PEEK_OPT_TREE_LOCAL_CAP  peek_pending_tree: the largest unresolved segment (in sorted positions) that
 *                        one CTA finishes out of shared memory; larger ones go through another
 *                        grid-wide refinement round first.  0 = the built-in capacity (default);
 *                        values 128 .. capacity lower it (a test hook: the grid-wide rounds and the
 *                        work-item queues then run at small N).
 * Unknown key or bad value -> PEEK_ERR_INVALID_ARG. */
enum { PEEK_OPT_LPM_STRATEGY = 1, PEEK_OPT_LPM_WINDOW = 2, PEEK_OPT_GRID_LIMIT = 3, PEEK_OPT_TREE_LOCAL_CAP = 4 };
enum { PEEK_LPM_AUTO = 0, PEEK_LPM_DUAL_WALK = 1, PEEK_LPM_SPECULATIVE = 2 };
peek_status peek_set_option(int32_t key, int64_t value);

/* ---- work counters of peek_lpm (the amortisation claim) ---- */
/* counters: NULL (default: off) or uint64[4] [device, caller-owned, zeroed by the caller], valid
 * until switched off again.  While set, every peek_lpm call ADDS, per mode it runs:
 * [0] walks started at the root of the cache (one per request without a tree view; one per run of
 * sorted positions in the dual walk - every other position copies its predecessor's hit or resumes
 * below their shared prefix), [1] child lookups (radix mode; a resumed walk costs lookups, no
 * re-descent), [2] tokens compared against edge labels (matched tokens plus the mismatching one),
 * [3] table slots' first probes (hash mode).  [2] and [3] are the work the dual walk amortises
 * (PAPER.md:293 O(C x D) against O(N x D)).  Process-wide like the options; results never depend on it. */
peek_status peek_lpm_counters(uint64_t* counters);

/* ---- tracing (CUDA events per kernel group) --------------------------- */
/* Off by default.  When on, every kernel group a call enqueues is bracketed by a pair of CUDA
 * events on the caller's stream (up to 512 pairs per slot between reads; later ones are dropped).
 * peek_profile_read synchronises on the recorded events of `slot`, returns their summed elapsed
 * milliseconds and the number of bracketed groups [host out], and optionally resets the slot.
 * peek_launch_count: kernels this library has launched in this process (always counted). */
void peek_profile_enable(int32_t on);
int32_t peek_profile_slots(void);
const char* peek_profile_name(int32_t slot);
peek_status peek_profile_read(int32_t slot, double* total_ms, int64_t* groups, int32_t reset);
int64_t peek_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif /* PEEK_H_ */
