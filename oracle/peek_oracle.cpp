// peek_oracle.cpp — TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, obviously-correct CPU implementation of what the PEEK hot path
// computes (arxiv/paper_2607_02525).  Only tests/, __graft_entry__.smoke() and
// bench.py's cpu_baseline / --impl reference legs may build, load or call this
// file.  It shares no code, header, table or constant generator with the CUDA
// path under paper_2607_02525_b200/csrc/, and neither includes the other.
//
// Every function is the plain definition written out (the paper's dual-walk,
// Alg. 1, reaches the per-request longest prefix match exactly,
// PAPER.md:73-82 "H[r] <- max(H[r], h)", "a partial match
// terminates the branch"), so there is no blocking, fusion or reordering here.
// Readings of silent / garbled passages are DESIGN.md "Readings" R1..R14
// (= SURVEY.md section 8(c) O1-O5, S1-S26).
//
// Pins (tests/test_oracle_*.py, run with -m "not gpu"):
//   orc_block_hash    splitmix64 known-answer stream + survey-computed vectors
//                     (tests/golden/hash_vectors.txt), python big-int restatement
//   orc_lpm_radix     brute force max-LCP over all cached sequences; std::mismatch
//                     reduction for a one-sequence cache; planted structure
//   orc_lpm_hash      python set of chained keys; mirror identity hit_hash =
//                     B*floor(hit_radix/B)
//   orc_pending_tree  python sorted() of tuples, O(N^2 nb) cluster definition,
//                     paper worked example PAPER.md:55 (sizes 3/3/2), Fig. 6(a)
//   orc_demand        nested-loop count; root-block demand = N
//   orc_clpm_order    python sorted() of tuples; worked-example order
//   orc_score / orc_evict_score / orc_sections / orc_clpm_order_full (NEXT-1 rows)
//                     token-level brute force on tiny queues (path counts by tuple
//                     prefixes, Alg. 2's sequential `seen` loop), closed forms on
//                     planted queues, the worked example's pioneers and siblings
// No function here is "parity unpinned".
//
// Threading: the per-request loops (hash, radix walk, hash probes) carry an
// OpenMP "parallel for"; results do not depend on the thread count.  The sorts
// and the demand map are single-threaded.

#include <algorithm>
#include <cstdint>
#include <cstring>
#include <numeric>
#include <unordered_map>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef uint64_t u64;
typedef int64_t i64;
typedef int32_t i32;

static const u64 ORC_EMPTY = 0xFFFFFFFFFFFFFFFFull;  // table EMPTY sentinel (R5)

// ---------------------------------------------------------------------------
// O1. Chained block hash.  PAPER.md:596  k_i = hash(k_{i-1}, tuple(s[iB:(i+1)B])),
// B = 16; "hashes each block by token content and prefix position via
// chained hashing".  The paper names no hash function (R1): this is the
// splitmix64 finaliser over an order-sensitive multiply-add of the block.
// ---------------------------------------------------------------------------
static inline u64 orc_mix64(u64 x) {
    x ^= x >> 30;
    x *= 0xBF58476D1CE4E5B9ull;
    x ^= x >> 27;
    x *= 0x94D049BB133111EBull;
    x ^= x >> 31;
    return x;
}

extern "C" u64 orc_mix64_export(u64 x) { return orc_mix64(x); }

// M_j = mix64(j+1) | 1   (odd per-position multiplier)
extern "C" u64 orc_position_multiplier(i32 j) { return orc_mix64((u64)j + 1) | 1ull; }

extern "C" int orc_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

extern "C" void orc_set_num_threads(int n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

// blk_off[r] = sum_{q<r} floor(len_q / B); trailing partial block not hashed (R3).
// hashes must have room for blk_off[N] words.  Returns NB.
extern "C" i64 orc_block_hash(const i32* tokens, const i64* tok_off, i64 N, i32 B, u64 seed,
                              i64* blk_off, u64* hashes) {
    blk_off[0] = 0;
    for (i64 r = 0; r < N; ++r) blk_off[r + 1] = blk_off[r] + (tok_off[r + 1] - tok_off[r]) / B;
    if (!hashes) return blk_off[N];
    std::vector<u64> M(B);
    for (i32 j = 0; j < B; ++j) M[j] = orc_position_multiplier(j);
#pragma omp parallel for schedule(dynamic, 64)
    for (i64 r = 0; r < N; ++r) {
        const i32* s = tokens + tok_off[r];
        i64 nb = blk_off[r + 1] - blk_off[r];
        u64 k = seed;  // k_{-1} = seed (R2)
        for (i64 i = 0; i < nb; ++i) {
            u64 S = 0;
            for (i32 j = 0; j < B; ++j) {
                u64 t = (u64)(uint32_t)s[i * B + j];  // bit pattern as u32, widened (R6)
                S += (t + 1) * M[j];
            }
            u64 c = orc_mix64(S);
            k = orc_mix64(k ^ c);
            if (k == ORC_EMPTY) k = 0xFFFFFFFFFFFFFFFEull;  // remapped value stored AND carried (R5)
            hashes[blk_off[r] + i] = k;
        }
    }
    return blk_off[N];
}

// ---------------------------------------------------------------------------
// O2a. LPM against the radix cache (the result of Alg. 1): for
// each request independently walk from the root; a partial edge match ends the
// walk.  Token-granular, not rounded to B, not capped at len-1
// (R9, R10).  Children of node v are edges n_child_off[v] .. n_child_off[v+1];
// the child is found by linear scan on e_first_tok (R11).
// ---------------------------------------------------------------------------
extern "C" void orc_lpm_radix(const i32* tokens, const i64* tok_off, i64 N,
                              const i32* c_tokens, const i64* n_tok_off, const i32* n_tok_len,
                              const i32* n_child_off, const i32* e_first_tok, const i32* e_child,
                              i32* hit_radix) {
#pragma omp parallel for schedule(dynamic, 64)
    for (i64 r = 0; r < N; ++r) {
        const i32* s = tokens + tok_off[r];
        i64 len = tok_off[r + 1] - tok_off[r];
        i32 v = 0;
        i64 d = 0;
        for (;;) {
            if (d == len) break;
            i32 u = -1;
            for (i32 e = n_child_off[v]; e < n_child_off[v + 1]; ++e)
                if (e_first_tok[e] == s[d]) { u = e_child[e]; break; }
            if (u < 0) break;
            const i32* lab = c_tokens + n_tok_off[u];
            i64 L = n_tok_len[u];
            i64 m = 0;
            while (m < L && d + m < len && lab[m] == s[d + m]) ++m;
            d += m;
            if (m < L) break;
            v = u;
        }
        hit_radix[r] = (i32)d;
    }
}

// ---------------------------------------------------------------------------
// O2b. LPM against the flat block-hash table ("per-request
// find_longest_cache_hit", O(N x b)).  Scan to the FIRST miss (R12).  Table:
// open addressing, linear probing, home = key & (S-1), EMPTY = all ones (R13).
// ---------------------------------------------------------------------------
static inline bool orc_lookup(const u64* t_keys, i64 S, u64 key) {
    i64 p = (i64)(key & (u64)(S - 1));
    while (t_keys[p] != ORC_EMPTY) {
        if (t_keys[p] == key) return true;
        p = (p + 1) & (S - 1);
    }
    return false;
}

extern "C" void orc_lpm_hash(const u64* hashes, const i64* blk_off, i64 N, i32 B,
                             const u64* t_keys, i64 S, i32* hit_hash) {
#pragma omp parallel for schedule(dynamic, 64)
    for (i64 r = 0; r < N; ++r) {
        const u64* k = hashes + blk_off[r];
        i64 nb = blk_off[r + 1] - blk_off[r];
        i64 i = 0;
        while (i < nb && orc_lookup(t_keys, S, k[i])) ++i;
        hit_hash[r] = (i32)(B * i);
    }
}

// ---------------------------------------------------------------------------
// O3. Pending radix tree at block granularity (R7): the
// sorted order of the hash chains is the DFS order of the compressed trie,
// adjacent LCPs are its branching depths.
// ---------------------------------------------------------------------------
struct OrcChainLess {
    const u64* hashes;
    const i64* blk_off;
    // word-by-word unsigned compare; a proper prefix sorts first; equal chains
    // are "not less" either way so stable_sort keeps ascending request index.
    bool operator()(i32 a, i32 b) const {
        const u64* ka = hashes + blk_off[a];
        const u64* kb = hashes + blk_off[b];
        i64 na = blk_off[a + 1] - blk_off[a], nb = blk_off[b + 1] - blk_off[b];
        i64 m = na < nb ? na : nb;
        for (i64 i = 0; i < m; ++i) {
            if (ka[i] != kb[i]) return ka[i] < kb[i];
        }
        return na < nb;
    }
};

extern "C" void orc_pending_tree(const u64* hashes, const i64* blk_off, i64 N,
                                 i32* order, i32* lcp, i32* group_id, i32* group_size,
                                 i32* cluster_depth, i32* cluster_size, i64* cluster_id,
                                 i32* n_groups) {
    // O3.1 order
    for (i64 r = 0; r < N; ++r) order[r] = (i32)r;
    OrcChainLess less{hashes, blk_off};
    std::stable_sort(order, order + N, less);
    // O3.2 adjacent LCP in blocks, lcp[0] = 0; sentinel lcp[N] = 0 kept locally
    std::vector<i32> L(N + 1, 0);
    for (i64 j = 1; j < N; ++j) {
        i32 a = order[j - 1], b = order[j];
        const u64* ka = hashes + blk_off[a];
        const u64* kb = hashes + blk_off[b];
        i64 na = blk_off[a + 1] - blk_off[a], nb = blk_off[b + 1] - blk_off[b];
        i64 m = na < nb ? na : nb, i = 0;
        while (i < m && ka[i] == kb[i]) ++i;
        L[j] = (i32)i;
    }
    for (i64 j = 0; j < N; ++j) lcp[j] = L[j];
    // O3.3 flat groups: a new group starts at j iff lcp[j] == 0 (root-child
    // subtrees, the ones has_sharing looks at)
    i32 g = -1;
    std::vector<i32> gsize;
    for (i64 j = 0; j < N; ++j) {
        if (L[j] == 0) { ++g; gsize.push_back(0); }
        group_id[order[j]] = g;
        gsize[g] += 1;
    }
    for (i64 j = 0; j < N; ++j) group_size[order[j]] = gsize[group_id[order[j]]];
    *n_groups = g + 1;
    // O3.4 cluster = deepest node on the request's path with pending_count >= 2
    // (PAPER.md:94, :287); pending_count includes requests ending at the node (R8).
    for (i64 j = 0; j < N; ++j) {
        i32 r = order[j];
        i32 cd = L[j] > L[j + 1] ? L[j] : L[j + 1];
        if (cd == 0) {
            cluster_depth[r] = 0;
            cluster_size[r] = 1;
            cluster_id[r] = (i64)((u64)j << 32);
            continue;
        }
        i64 a = j;
        while (!(L[a] < cd)) --a;  // largest p <= j with lcp[p] < cd (lcp[0] = 0 < cd)
        i64 b = j;
        while (!(L[b + 1] < cd)) ++b;  // smallest q >= j with lcp[q+1] < cd (lcp[N] = 0)
        cluster_depth[r] = cd;
        cluster_size[r] = (i32)(b - a + 1);
        cluster_id[r] = (i64)(((u64)a << 32) | (u64)(uint32_t)cd);
    }
}

// ---------------------------------------------------------------------------
// O4. Per-table-slot pending demand (PAPER.md:281 inverted index
// block_hash -> demand; pending_count in Eq. 2).  Independent of
// hit lengths.  demand[p] = 0 for EMPTY slots.
// ---------------------------------------------------------------------------
extern "C" void orc_demand(const u64* hashes, const i64* blk_off, i64 N,
                           const u64* t_keys, i64 S, i32* demand) {
    std::unordered_map<u64, i64> slot_of;
    slot_of.reserve((size_t)S);
    for (i64 p = 0; p < S; ++p) {
        demand[p] = 0;
        if (t_keys[p] != ORC_EMPTY) slot_of.emplace(t_keys[p], p);
    }
    i64 NB = blk_off[N];
    for (i64 x = 0; x < NB; ++x) {
        auto it = slot_of.find(hashes[x]);
        if (it != slot_of.end()) demand[it->second] += 1;
    }
}

// ---------------------------------------------------------------------------
// O5. cLPM order: the (-h, -|cluster|, arrival) sub-key of Eq. 1
// with the request index as the last tie-break (R14).  arrival == NULL => index.
// ---------------------------------------------------------------------------
extern "C" void orc_clpm_order(const i32* hit, const i32* cluster_size, const i32* arrival,
                               i64 N, i32* clpm_order) {
    for (i64 r = 0; r < N; ++r) clpm_order[r] = (i32)r;
    std::sort(clpm_order, clpm_order + N, [&](i32 a, i32 b) {
        if (hit[a] != hit[b]) return hit[a] > hit[b];
        if (cluster_size[a] != cluster_size[b]) return cluster_size[a] > cluster_size[b];
        i32 aa = arrival ? arrival[a] : a, ab = arrival ? arrival[b] : b;
        if (aa != ab) return aa < ab;
        return a < b;
    });
}

// has_sharing guard: true iff some root child has pending_count >= 2.
extern "C" i32 orc_has_sharing(const i32* group_size, i64 N) {
    for (i64 r = 0; r < N; ++r)
        if (group_size[r] >= 2) return 1;
    return 0;
}

// ===========================================================================
// Next rows: the full Eq. 1 key and Eq. 2 score.
// Readings R20-R23 in DESIGN.md.  Trie nodes exist at block granularity (R7), so
// an edge is one block of B tokens and pending_count of the node reached by
// block i of request r is the number of pending (request, block) pairs whose
// chained hash equals k^r_i - the same count orc_demand takes per table slot.
// ===========================================================================
static void orc_pending_counts(const u64* hashes, i64 NB, std::unordered_map<u64, i64>& pc) {
    pc.reserve((size_t)NB);
    for (i64 x = 0; x < NB; ++x) pc[hashes[x]] += 1;
}

// O6. Ancestor score: score(r) = sum over the nodes v on r's path of
// pending_count(v) * |edge(v)|, |edge| = B tokens per block (R20).
extern "C" void orc_score(const u64* hashes, const i64* blk_off, i64 N, i32 block_size, i64* score) {
    std::unordered_map<u64, i64> pc;
    orc_pending_counts(hashes, blk_off[N], pc);
    for (i64 r = 0; r < N; ++r) {
        i64 s = 0;
        for (i64 x = blk_off[r]; x < blk_off[r + 1]; ++x) s += pc[hashes[x]] * block_size;
        score[r] = s;
    }
}

// O7. Eviction score (Eq. 2): for the cached block b,
// max over the ancestors v of b (b's own node included) of pending_count(v) * depth(v),
// depth in tokens (R23).  Per table slot; a slot whose key is on no pending chain has no
// pending ancestor that can be named through the keys-only table and scores 0 (R23).
extern "C" void orc_evict_score(const u64* hashes, const i64* blk_off, i64 N, i32 block_size,
                                const u64* t_keys, i64 S, i64* evict) {
    std::unordered_map<u64, i64> pc;
    orc_pending_counts(hashes, blk_off[N], pc);
    std::unordered_map<u64, i64> slot_of;
    slot_of.reserve((size_t)S);
    for (i64 p = 0; p < S; ++p) {
        evict[p] = 0;
        if (t_keys[p] != ORC_EMPTY) slot_of.emplace(t_keys[p], p);
    }
    for (i64 r = 0; r < N; ++r) {
        i64 best = 0;  // max over blocks 0..i of r's path
        for (i64 x = blk_off[r]; x < blk_off[r + 1]; ++x) {
            i64 depth_tokens = (x - blk_off[r] + 1) * block_size;
            i64 v = pc[hashes[x]] * depth_tokens;
            if (v > best) best = v;
            auto it = slot_of.find(hashes[x]);
            if (it != slot_of.end()) evict[it->second] = best;
        }
    }
}

// O8. Sections (Alg. 2 lines 3-13): in arrival order (ties by
// request index), warm (0) if h > tau; else pioneer (1) if the prompt's first theta = 32 tokens
// have not been seen this cycle, else sibling (2).  At block granularity (R22) the first
// theta tokens are the first two blocks: the prefix key is k_1 for nb >= 2, k_0 for nb == 1
// (a shorter prompt is a different prefix than any longer one), and a request with no full
// block is never "seen".
extern "C" void orc_sections(const u64* hashes, const i64* blk_off, i64 N, const i32* hit, i32 tau,
                             const i32* arrival, i32* section) {
    std::vector<i64> by_arrival((size_t)N);
    for (i64 r = 0; r < N; ++r) by_arrival[(size_t)r] = r;
    std::stable_sort(by_arrival.begin(), by_arrival.end(), [&](i64 a, i64 b) {
        i32 aa = arrival ? arrival[a] : (i32)a, ab = arrival ? arrival[b] : (i32)b;
        return aa < ab;
    });
    std::unordered_map<u64, int> seen2, seen1;  // by k_1 (nb >= 2) and by k_0 (nb == 1)
    for (i64 q = 0; q < N; ++q) {
        i64 r = by_arrival[(size_t)q];
        if (hit[r] > tau) { section[r] = 0; continue; }
        i64 nb = blk_off[r + 1] - blk_off[r];
        if (nb == 0) { section[r] = 1; continue; }
        std::unordered_map<u64, int>& seen = nb >= 2 ? seen2 : seen1;
        u64 p = nb >= 2 ? hashes[blk_off[r] + 1] : hashes[blk_off[r]];
        if (seen.count(p)) section[r] = 2;
        else { section[r] = 1; seen[p] = 1; }
    }
}

// O9. The full cLPM key of Eq. 1: (section, -h, -score, -|cluster|, arrival),
// request index last (R14).
extern "C" void orc_clpm_order_full(const i32* section, const i32* hit, const i64* score,
                                    const i32* cluster_size, const i32* arrival, i64 N, i32* out) {
    for (i64 r = 0; r < N; ++r) out[r] = (i32)r;
    std::sort(out, out + N, [&](i32 a, i32 b) {
        if (section[a] != section[b]) return section[a] < section[b];
        if (hit[a] != hit[b]) return hit[a] > hit[b];
        if (score[a] != score[b]) return score[a] > score[b];
        if (cluster_size[a] != cluster_size[b]) return cluster_size[a] > cluster_size[b];
        i32 aa = arrival ? arrival[a] : a, ab = arrival ? arrival[b] : b;
        if (aa != ab) return aa < ab;
        return a < b;
    });
}

// O10. Group-major admission ("emits all members of one cluster contiguously";
// worked example PAPER.md:55).  Reading R24: walking the cache-locality lane (Eq. 1 order), the
// first member of a cluster pulls the rest of its cluster right behind it, in lane order; i.e.
// requests are ordered by (lane position of their cluster's first member, own lane position).
// A singleton is its own cluster (its cluster_id is unique).
extern "C" void orc_group_major(const i32* lane_order, const i64* cluster_id, i64 N, i32* out) {
    std::vector<i64> pos((size_t)N);
    for (i64 p = 0; p < N; ++p) pos[(size_t)lane_order[p]] = p;
    std::unordered_map<i64, i64> first;
    for (i64 p = 0; p < N; ++p) {
        i64 c = cluster_id[lane_order[p]];
        if (!first.count(c)) first[c] = p;
    }
    for (i64 r = 0; r < N; ++r) out[r] = (i32)r;
    std::sort(out, out + N, [&](i32 a, i32 b) {
        i64 fa = first[cluster_id[a]], fb = first[cluster_id[b]];
        if (fa != fb) return fa < fb;
        return pos[(size_t)a] < pos[(size_t)b];
    });
}

// O11. PEEK-offline phase 1: a prefix trie over the first D = 128 tokens of
// every prompt (= the first 8 blocks, R7); each node records the requests terminating there and
// its subtree request count; a depth-first traversal that visits children in DESCENDING
// subtree-count order emits the permutation.  Reading R25: a node first emits its terminators in
// ascending request index; children with equal counts go by the smallest request index below them.
// Guards: duplication = fraction of requests whose whole chain equals that of an
// earlier request; coverage = fraction of requests sharing >= 32 tokens (2 blocks) with another;
// depth = mean over the requests of 16 * (leading blocks, of the first `depth_blocks`, shared
// with another request).  guards[3] = 1 if duplication > 0.5 or coverage < 0.1 or depth < 64.
namespace {
struct OffNode {
    std::unordered_map<u64, int> child;
    std::vector<i32> term;
    i64 count = 0;
    i32 minidx = 0x7fffffff;
};
}  // namespace
extern "C" void orc_offline_phase1(const u64* hashes, const i64* blk_off, i64 N, i32 depth_blocks,
                                   i32* order, double* guards) {
    std::vector<OffNode> nodes(1);
    std::vector<std::vector<int>> path((size_t)N);
    for (i64 r = 0; r < N; ++r) {
        int v = 0;
        nodes[0].count += 1;
        if ((i32)r < nodes[0].minidx) nodes[0].minidx = (i32)r;
        i64 L = blk_off[r + 1] - blk_off[r];
        if (L > depth_blocks) L = depth_blocks;
        for (i64 i = 0; i < L; ++i) {
            u64 k = hashes[blk_off[r] + i];
            auto it = nodes[(size_t)v].child.find(k);
            int c;
            if (it == nodes[(size_t)v].child.end()) {
                c = (int)nodes.size();
                nodes[(size_t)v].child.emplace(k, c);
                nodes.emplace_back();
            } else c = it->second;
            v = c;
            nodes[(size_t)v].count += 1;
            if ((i32)r < nodes[(size_t)v].minidx) nodes[(size_t)v].minidx = (i32)r;
            path[(size_t)r].push_back(v);
        }
        nodes[(size_t)v].term.push_back((i32)r);
    }
    i64 out = 0;
    std::vector<int> stack{0};
    while (!stack.empty()) {  // explicit stack: children pushed in reverse visiting order
        int v = stack.back();
        stack.pop_back();
        for (i32 r : nodes[(size_t)v].term) order[out++] = r;  // inserted in ascending index
        std::vector<int> ch;
        for (auto& kv : nodes[(size_t)v].child) ch.push_back(kv.second);
        std::sort(ch.begin(), ch.end(), [&](int a, int b) {
            if (nodes[(size_t)a].count != nodes[(size_t)b].count) return nodes[(size_t)a].count > nodes[(size_t)b].count;
            return nodes[(size_t)a].minidx < nodes[(size_t)b].minidx;
        });
        for (auto it = ch.rbegin(); it != ch.rend(); ++it) stack.push_back(*it);
    }
    // guards
    std::unordered_map<u64, std::vector<i64>> by_last;  // (last hash) -> requests, to find equal chains
    i64 dup = 0, cov = 0;
    double depth_sum = 0;
    std::unordered_map<u64, int> seen_chain;
    for (i64 r = 0; r < N; ++r) {
        i64 nb = blk_off[r + 1] - blk_off[r];
        // whole-chain identity: same length and same words
        bool is_dup = false;
        u64 tag = nb ? hashes[blk_off[r + 1] - 1] : 0x1234567ull;
        for (i64 q : by_last[tag]) {
            i64 nq = blk_off[q + 1] - blk_off[q];
            if (nq == nb && std::equal(hashes + blk_off[r], hashes + blk_off[r + 1], hashes + blk_off[q])) { is_dup = true; break; }
        }
        by_last[tag].push_back(r);
        if (is_dup) ++dup;
        const std::vector<int>& p = path[(size_t)r];
        if (p.size() >= 2 && nodes[(size_t)p[1]].count >= 2) ++cov;
        i64 d = 0;
        while (d < (i64)p.size() && nodes[(size_t)p[(size_t)d]].count >= 2) ++d;
        depth_sum += 16.0 * (double)d;
    }
    guards[0] = N ? (double)dup / (double)N : 0.0;
    guards[1] = N ? (double)cov / (double)N : 0.0;
    guards[2] = N ? depth_sum / (double)N : 0.0;
    guards[3] = (guards[0] > 0.5 || guards[1] < 0.1 || guards[2] < 64.0) ? 1.0 : 0.0;
}

// O12. Per-radix-node pending demand (the SGLang-side counterpart of the
// block_hash -> demand index, "PeekDemandStrategy scores candidate nodes").
// Reading R26: node_demand[v] = number of pending requests whose longest-prefix match enters v
// (matches at least one token of v's label); the root, whose label is empty, is entered by every
// request, so node_demand[root] = N.  Same walk as orc_lpm_radix.
extern "C" void orc_radix_demand(const i32* tokens, const i64* tok_off, i64 N, const i32* c_tokens,
                                 const i64* n_tok_off, const i32* n_tok_len, const i32* n_child_off,
                                 const i32* e_first_tok, const i32* e_child, i32 V, i32* node_demand) {
    for (i32 v = 0; v < V; ++v) node_demand[v] = 0;
    for (i64 r = 0; r < N; ++r) {
        const i32* s = tokens + tok_off[r];
        i64 len = tok_off[r + 1] - tok_off[r];
        i32 v = 0;
        i64 d = 0;
        node_demand[0] += 1;
        for (;;) {
            if (d == len) break;
            i32 u = -1;
            for (i32 e = n_child_off[v]; e < n_child_off[v + 1]; ++e)
                if (e_first_tok[e] == s[d]) { u = e_child[e]; break; }
            if (u < 0) break;
            node_demand[u] += 1;  // the first token of the edge matched: u is entered
            const i32* lab = c_tokens + n_tok_off[u];
            i64 L = n_tok_len[u], m = 0;
            while (m < L && d + m < len && lab[m] == s[d + m]) ++m;
            d += m;
            if (m < L) break;
            v = u;
        }
    }
}

// O13. Fairness lane (Alg. 2 line 18): R_B = sort by
// (section, arrival, -h), request index last (R14).
extern "C" void orc_lane_b(const i32* section, const i32* hit, const i32* arrival, i64 N, i32* out) {
    for (i64 r = 0; r < N; ++r) out[r] = (i32)r;
    std::sort(out, out + N, [&](i32 a, i32 b) {
        if (section[a] != section[b]) return section[a] < section[b];
        i32 aa = arrival ? arrival[a] : a, ab = arrival ? arrival[b] : b;
        if (aa != ab) return aa < ab;
        if (hit[a] != hit[b]) return hit[a] > hit[b];
        return a < b;
    });
}

// O14. Dynamic-lane controller (Alg. 2 line 20):
// 1 - alpha <- EMA_{beta=0.3}(clamp(0.15 + 0.5*singleton_frac + 0.3*age_pressure, 0.10, 0.60)),
// singleton_frac = fraction of requests in no cluster (cluster_size == 1).  Reading R27: the EMA is
// new = beta * x + (1 - beta) * previous, in double precision, each product and sum rounded once.
extern "C" void orc_dynamic_lane(const i32* cluster_size, i64 N, double age_pressure, double prev,
                                 double* out) {
    i64 single = 0;
    for (i64 r = 0; r < N; ++r) single += cluster_size[r] == 1;
    volatile double sf = N ? (double)single / (double)N : 0.0;
    volatile double a = 0.5 * sf, b = 0.3 * age_pressure;
    volatile double x = 0.15 + a;
    x = x + b;
    if (x < 0.10) x = 0.10;
    if (x > 0.60) x = 0.60;
    volatile double p = 0.3 * x, q = 0.7 * prev;
    out[0] = p + q;  // the new fairness share 1 - alpha
    out[1] = sf;
}

// O15. Stride interleave of the two lanes (Alg. 2 line 22; "a fraction
// alpha of admissions come from Lane A, 1 - alpha from Lane B").  The paper names the routine but
// does not define it.  Reading R28: admission slot k = 0, 1, ... belongs to Lane A iff
// floor((k+1)*alpha) > floor(k*alpha) - after any k slots Lane A has had floor(k*alpha) of them and
// Lane B's slots are never more than ceil(1/(1-alpha)) apart - else to Lane B; the lane admits its
// first request not admitted yet.  Both lanes list every request, so neither runs dry early.
extern "C" void orc_stride_interleave(const i32* lane_a, const i32* lane_b, i64 N, double alpha, i32* out) {
    std::vector<char> done((size_t)N, 0);
    i64 ia = 0, ib = 0;
    for (i64 k = 0; k < N; ++k) {
        volatile double x0 = (double)k * alpha, x1 = (double)(k + 1) * alpha;
        bool from_a = (i64)x1 > (i64)x0;  // alpha in [0, 1]: the products are >= 0, truncation = floor
        if (from_a) {
            while (done[(size_t)lane_a[ia]]) ++ia;
            out[k] = lane_a[ia];
        } else {
            while (done[(size_t)lane_b[ib]]) ++ib;
            out[k] = lane_b[ib];
        }
        done[(size_t)out[k]] = 1;
    }
}
