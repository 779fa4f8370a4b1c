"""Seeded synthetic diagram sets shaped like the paper's 1-5 loop workloads (BASELINE.json configs[0..4]).

This module is the input generator shared by tests/, bench.py and smoke(): it holds none of the method's
arithmetic (no sampler, no integrand) and imports neither oracle/ nor the CUDA path. A "graph" is the tuple
(loops, ext_pos, chords) both sides accept. The paper's workload is "all 5-loop graphs without lepton loops"
(PAPER.md:86-91), a purely combinatorial object; configs 3 and 4 are seeded subsets of it (A12).
"""

M0, M1, W0, W1 = 0xD2511F53, 0xCD9E8D57, 0x9E3779B9, 0xBB67AE85


def philox4x32_10(ctr, key):
    """public Philox4x32-10 (PAPER.md:94 names the generator); used here only to draw graph subsets"""
    c0, c1, c2, c3 = ctr
    k0, k1 = key
    for _ in range(10):
        p0, p1 = M0 * c0, M1 * c2
        c0, c1, c2, c3 = ((p1 >> 32) ^ c1 ^ k0) & 0xFFFFFFFF, p1 & 0xFFFFFFFF, ((p0 >> 32) ^ c3 ^ k1) & 0xFFFFFFFF, p0 & 0xFFFFFFFF
        k0, k1 = (k0 + W0) & 0xFFFFFFFF, (k1 + W1) & 0xFFFFFFFF
    return c0, c1, c2, c3


def _matchings(free):
    if not free:
        yield []
        return
    first = free[0]
    for j in range(1, len(free)):
        rest = free[1:j] + free[j + 1:]
        for tail in _matchings(rest):
            yield [(first, free[j])] + tail


def is_valid(loops, ext_pos, chords):
    """1PI vertex graph: every electron line t (joining positions t, t+1) is spanned by a chord"""
    return all(any(a <= t < b for a, b in chords) for t in range(2 * loops))


_CACHE = {}


def all_graphs(loops):
    """canonical order: ascending external position, then lexicographic sorted chord list (A19)"""
    if loops not in _CACHE:
        out = []
        for e in range(2 * loops + 1):
            free = [p for p in range(2 * loops + 1) if p != e]
            for ch in _matchings(free):
                if is_valid(loops, e, ch):
                    out.append((loops, e, tuple(ch)))
        _CACHE[loops] = out
    return _CACHE[loops]


def graph_class(graph):
    """(k, m, n) of PAPER.md:104"""
    _, e, chords = graph
    k = sum(1 for a, b in chords if a < e < b)
    left = sum(1 for a, b in chords if b < e)
    right = sum(1 for a, b in chords if a > e)
    return (k, max(left, right), min(left, right))


def _shuffle(items, seed, stream):
    """Fisher-Yates driven by Philox(key=seed, ctr=(i, 0, stream, 0xD1A6))"""
    items = list(items)
    for i in range(len(items) - 1, 0, -1):
        r = philox4x32_10((i, 0, stream, 0xD1A6), (seed & 0xFFFFFFFF, seed >> 32))[0]
        j = r % (i + 1)
        items[i], items[j] = items[j], items[i]
    return items


def config_graphs(config):
    """list of (canonical_index, graph) of BASELINE.json configs[config]"""
    if config in (0, 1, 2):
        gs = all_graphs(config + 1)
        return list(enumerate(gs))
    if config == 3:
        gs = all_graphs(4)
        pick = sorted(_shuffle(range(len(gs)), 4, 0)[:128])
        return [(i, gs[i]) for i in pick]
    if config == 4:
        gs = all_graphs(5)
        by_class = {}
        for i, g in enumerate(gs):
            by_class.setdefault(graph_class(g), []).append(i)
        classes = sorted(by_class)
        total, want = len(gs), 256
        quota = {c: max(1, (want * len(by_class[c])) // total) for c in classes}
        rem = sorted(classes, key=lambda c: -((want * len(by_class[c])) % total))
        k = 0
        while sum(quota.values()) < want:
            quota[rem[k % len(rem)]] += 1
            k += 1
        while sum(quota.values()) > want:
            big = max(classes, key=lambda c: quota[c])
            quota[big] -= 1
        pick = []
        for ci, c in enumerate(classes):
            pick += _shuffle(by_class[c], 5, ci + 1)[:quota[c]]
        return [(i, gs[i]) for i in sorted(pick)]
    raise ValueError("config must be 0..4")


CONFIG_SEED = {0: 1, 1: 2, 2: 3, 3: 4, 4: 5}
CONFIG_POINTS_TOTAL = {0: 10 ** 7, 1: 6 * 10 ** 8, 2: 10 ** 9, 3: 10 ** 10, 4: 10 ** 11}
