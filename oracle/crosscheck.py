"""oracle.crosscheck — TEST INFRASTRUCTURE.  Second, independent clustering implementation used
only to cross-check ``po_cluster`` (SURVEY.md 8(c) "implementation (ii)"): union-find over kept
digis, neighbours found through a dict keyed (row, col); label = minimum index per set, computed
in a final pass.  Pure Python: small inputs only."""
from __future__ import annotations

import numpy as np

INVALID = 0xFFFFFFFF


def cluster_union_find(module, row, col, kept):
    D = len(module)
    parent = list(range(D))

    def find(a):
        while parent[a] != a:
            parent[a] = parent[parent[a]]
            a = parent[a]
        return a

    def union(a, b):
        ra, rb = find(a), find(b)
        if ra != rb:
            parent[rb] = ra          # arbitrary direction: the minimum is taken afterwards

    cells = {}                       # (module,row,col) -> list of digi indices (duplicates, A6)
    for d in range(D):
        if kept[d]:
            cells.setdefault((int(module[d]), int(row[d]), int(col[d])), []).append(d)
    for (m, r, c), ds in cells.items():
        for d in ds[1:]:
            union(ds[0], d)          # equal coordinates are adjacent (A6)
        for dr in (-1, 0, 1):
            for dc in (-1, 0, 1):
                if (dr or dc) and (m, r + dr, c + dc) in cells:
                    union(ds[0], cells[(m, r + dr, c + dc)][0])
    label = np.full(D, INVALID, np.uint32)
    minimum = {}
    for d in range(D):
        if kept[d]:
            r = find(d)
            minimum[r] = min(minimum.get(r, d), d)
    for d in range(D):
        if kept[d]:
            label[d] = minimum[find(d)]
    return label
