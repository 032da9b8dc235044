"""Definitions written out in pure Python, independently of oracle/ and of the CUDA path.

Used only by tests to pin the oracle on tiny inputs:
every function is the *definition* of the quantity, not an algorithm for it.
"""
MASK = (1 << 64) - 1
EMPTY = MASK


def mix64(x):
    x &= MASK
    x ^= x >> 30
    x = (x * 0xBF58476D1CE4E5B9) & MASK
    x ^= x >> 27
    x = (x * 0x94D049BB133111EB) & MASK
    x ^= x >> 31
    return x


def chain(tokens, B=16, seed=0):
    """PAPER.md:596 k_i = hash(k_{i-1}, block_i) with the DESIGN.md R1 function."""
    M = [mix64(j + 1) | 1 for j in range(B)]
    k = seed
    out = []
    for i in range(len(tokens) // B):
        S = 0
        for j in range(B):
            S = (S + ((tokens[i * B + j] & 0xFFFFFFFF) + 1) * M[j]) & MASK
        k = mix64(k ^ mix64(S))
        if k == EMPTY:
            k = EMPTY - 1
        out.append(k)
    return out


def lcp(a, b):
    n = 0
    for x, y in zip(a, b):
        if x != y:
            break
        n += 1
    return n


def hit_radix(req, cached_seqs):
    """max over cached sequences of LCP(request, sequence) (north_star)."""
    return max([lcp(req, s) for s in cached_seqs], default=0)


def hit_hash(chain_r, keyset, B=16):
    i = 0
    while i < len(chain_r) and chain_r[i] in keyset:
        i += 1
    return B * i


def pending_tree(chains):
    """order / lcp / groups / clusters from the definitions."""
    N = len(chains)
    order = sorted(range(N), key=lambda r: (tuple(chains[r]), r))  # prefix sorts first
    L = [0] * N
    for j in range(1, N):
        L[j] = lcp(chains[order[j - 1]], chains[order[j]])
    # groups: requests sharing the first block (root-child subtrees); nb=0 alone
    group_id = [0] * N
    g = -1
    for j in range(N):
        if L[j] == 0:
            g += 1
        group_id[order[j]] = g
    gsz = [0] * (g + 1)
    for r in range(N):
        gsz[group_id[r]] += 1
    group_size = [gsz[group_id[r]] for r in range(N)]
    # cluster: largest d >= 1 such that >= 2 requests share r's first d blocks; count them
    cdepth, csize = [0] * N, [1] * N
    for r in range(N):
        best_d, best_c = 0, 1
        for d in range(len(chains[r]), 0, -1):
            pre = chains[r][:d]
            c = sum(1 for q in range(N) if chains[q][:d] == pre)
            if c >= 2:
                best_d, best_c = d, c
                break
        cdepth[r], csize[r] = best_d, best_c
    return order, L, group_id, group_size, cdepth, csize, g + 1


def demand(chains, t_keys):
    out = [0] * len(t_keys)
    for p, key in enumerate(t_keys):
        if key == EMPTY:
            continue
        for ch in chains:
            for k in ch:
                if k == key:
                    out[p] += 1
    return out


def clpm_order(hit, csize, arrival):
    N = len(hit)
    arr = arrival if arrival is not None else list(range(N))
    return sorted(range(N), key=lambda r: (-hit[r], -csize[r], arr[r], r))


def table_from_keys(keys, S):
    t = [EMPTY] * S
    for k in keys:
        p = k & (S - 1)
        while t[p] != EMPTY and t[p] != k:
            p = (p + 1) & (S - 1)
        t[p] = k
    return t
