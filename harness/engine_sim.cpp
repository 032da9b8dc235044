// engine_sim.cpp — host-side stand-in for the serving engine's prefix cache.
//
// PEEK matches pending requests against a cache it does not own: SGLang's radix
// tree or vLLM's flat chained-block-hash table.  Neither engine is
// available here, so the seeded workload generators (workloads.py) use this file
// to BUILD those read-only inputs: a compressed token trie flattened to the
// arrays of include/peek.h `peek_radix`, and an open-addressed key table
// (`peek_table`).  It holds none of the method's arithmetic: no hash function,
// no longest-prefix walk over a finished cache, no probe of a finished table.
// It is linked into neither libpeek.so nor the oracle.
#include <algorithm>
#include <cstdint>
#include <cstring>
#include <deque>
#include <map>
#include <vector>

typedef int32_t i32;
typedef int64_t i64;
typedef uint64_t u64;

namespace {
struct Node {
    const i32* lab;  // label tokens (points into an owned copy of the sequence pool)
    i64 len;
    i64 sd;  // depth at which the label starts
    std::map<i32, i32> kids;  // first token -> node id (ordered = signed ascending)
};
struct Builder {
    std::vector<Node> nodes;
    std::deque<std::vector<i32>> pool;  // owned copies of accepted sequences
    i32 B;
    i64 max_blocks;
    i64 blocks;
    bool full;
};
}  // namespace

extern "C" void* esim_radix_new(i32 B, i64 max_blocks) {
    Builder* b = new Builder();
    b->B = B;
    b->max_blocks = max_blocks;
    b->blocks = 0;
    b->full = false;
    b->nodes.push_back(Node{nullptr, 0, 0, {}});
    return b;
}

extern "C" void esim_radix_free(void* h) { delete (Builder*)h; }

// Insert sequences in order until `max_blocks` distinct full blocks are held
// (a full block = a block-aligned prefix of some inserted sequence); the
// sequence that would overshoot is truncated at a block boundary.  Writes the
// accepted length of each sequence (0 if dropped) and returns how many were
// accepted (length > 0 or empty input).
extern "C" i64 esim_radix_insert(void* h, const i32* tokens, const i64* off, i64 n_seq,
                                 i64* accepted_len) {
    Builder* b = (Builder*)h;
    const i32 B = b->B;
    i64 n_acc = 0;
    for (i64 s = 0; s < n_seq; ++s) {
        accepted_len[s] = 0;
        if (b->full) continue;
        const i32* t = tokens + off[s];
        i64 len = off[s + 1] - off[s];
        // divergence depth with the current trie
        i32 v = 0;
        i64 d = 0;
        i32 split_node = -1;
        i64 split_m = 0;
        while (d < len) {
            auto it = b->nodes[v].kids.find(t[d]);
            if (it == b->nodes[v].kids.end()) break;
            i32 u = it->second;
            const Node& nu = b->nodes[u];
            i64 m = 0;
            while (m < nu.len && d + m < len && nu.lab[m] == t[d + m]) ++m;
            d += m;
            if (m < nu.len) { split_node = u; split_m = m; break; }
            v = u;
        }
        i64 new_blocks = len / B - d / B;
        if (b->max_blocks > 0 && b->blocks + new_blocks >= b->max_blocks) {
            i64 room = b->max_blocks - b->blocks;
            len = (d / B + room) * (i64)B;  // truncate at a block boundary
            new_blocks = room;
            b->full = true;
        }
        accepted_len[s] = len;
        ++n_acc;
        if (len <= d) continue;  // nothing new below the divergence point
        b->blocks += new_blocks;
        b->pool.emplace_back(t, t + len);
        const i32* own = b->pool.back().data();
        if (split_node >= 0) {
            // split edge (parent v) -> split_node at split_m
            Node& old = b->nodes[split_node];
            Node mid{old.lab, split_m, old.sd, {}};
            i32 mid_id = (i32)b->nodes.size();
            i32 first = old.lab[0];
            old.lab += split_m;
            old.len -= split_m;
            old.sd += split_m;
            mid.kids[old.lab[0]] = split_node;
            b->nodes.push_back(mid);
            b->nodes[v].kids[first] = mid_id;
            v = mid_id;
        }
        Node leaf{own + d, len - d, d, {}};
        i32 leaf_id = (i32)b->nodes.size();
        b->nodes.push_back(leaf);
        b->nodes[v].kids[own[d]] = leaf_id;
    }
    return n_acc;
}

extern "C" void esim_radix_sizes(void* h, i64* V, i64* E, i64* CT, i64* blocks, i32* full) {
    Builder* b = (Builder*)h;
    i64 ct = 0, e = 0;
    for (const Node& n : b->nodes) { ct += n.len; e += (i64)n.kids.size(); }
    *V = (i64)b->nodes.size();
    *E = e;
    *CT = ct;
    *blocks = b->blocks;
    *full = b->full ? 1 : 0;
}

// Flatten: BFS node numbering from the root (node 0, empty label); children of
// a node occupy consecutive edges sorted ascending by first token (signed).
extern "C" void esim_radix_export(void* h, i32* c_tokens, i64* n_tok_off, i32* n_tok_len,
                                  i32* n_child_off, i32* e_first_tok, i32* e_child) {
    Builder* b = (Builder*)h;
    i64 V = (i64)b->nodes.size();
    std::vector<i32> bfs;  // new id -> old id
    bfs.reserve(V);
    std::vector<i32> newid(V, -1);
    bfs.push_back(0);
    newid[0] = 0;
    for (size_t q = 0; q < bfs.size(); ++q) {
        for (auto& kv : b->nodes[bfs[q]].kids) {
            newid[kv.second] = (i32)bfs.size();
            bfs.push_back(kv.second);
        }
    }
    i64 ct = 0;
    i32 e = 0;
    for (i64 nv = 0; nv < V; ++nv) {
        const Node& n = b->nodes[bfs[nv]];
        n_tok_off[nv] = ct;
        n_tok_len[nv] = (i32)n.len;
        if (n.len) memcpy(c_tokens + ct, n.lab, sizeof(i32) * n.len);
        ct += n.len;
        n_child_off[nv] = e;
        for (auto& kv : n.kids) {
            e_first_tok[e] = kv.first;
            e_child[e] = newid[kv.second];
            ++e;
        }
    }
    n_child_off[V] = e;
}

// Open addressing, linear probing, home = key & (S-1), EMPTY = all ones; keys
// only.  Inserts keys in the given order, skipping duplicates, until `max_keys`
// keys are held (<= 0: no cap).  Caller initialises t_keys to EMPTY.  Returns
// the number of keys held after the call given `held` before it.
extern "C" i64 esim_table_insert(u64* t_keys, i64 S, const u64* keys, i64 n, i64 held,
                                 i64 max_keys) {
    const u64 EMPTY = ~0ull;
    for (i64 i = 0; i < n; ++i) {
        if (max_keys > 0 && held >= max_keys) break;
        if (held >= S - 1) break;  // always keep one EMPTY slot
        u64 k = keys[i];
        i64 p = (i64)(k & (u64)(S - 1));
        bool dup = false;
        while (t_keys[p] != EMPTY) {
            if (t_keys[p] == k) { dup = true; break; }
            p = (p + 1) & (S - 1);
        }
        if (dup) continue;
        t_keys[p] = k;
        ++held;
    }
    return held;
}
