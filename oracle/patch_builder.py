"""CPU oracle of the Ramses GPU patch builder (the only procedure the paper lists,
PAPER.md:55-57, §3 "Hence, for the GPU a specific procedure has been designed", Figure 1 at :41):

  1. "at a given level of refinement, AMR cells are ordered according to a space filling curve based layout"
  2. "cells are grouped in compact (i.e. with no holes) cubic patches of maximum possible size"
  3. "neighbouring patches are grouped in large chunks collecting all the data necessary" (gather)

TEST INFRASTRUCTURE: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
may import this module; it shares no code with the CUDA path (paper_1412_0934_b200/csrc/patch_builder.cu).

Plain numpy / Python, written to be checked against the text by eye.  Readings where the paper is silent
(DESIGN.md §11): the space-filling curve is the Morton (Z-order) curve, x the least significant bit of each
triple; a "cubic patch" is an octree-aligned cube of side 2^k cells, k <= kmax; "compact" = every one of its
8^k cells is a leaf cell of the level; "maximum possible size" = each cell belongs to the largest such cube
that contains it (these cubes are disjoint and cover all cells); patches are listed in curve order.

Pins (tests/test_oracle_patch_builder.py): the textbook bit interleave on hand-computed keys; brute force over
every aligned cube of tiny random cell sets; disjoint cover / fullness / maximality on random sets; a full
grid gives (N / 2^kmax)^3 patches; the worked example of tests/golden/patch_builder_example.txt.
"""
from __future__ import annotations

import numpy as np


def morton_key(x, y, z, bits: int) -> np.ndarray:
    """Step 1: Morton key, bit b of x -> bit 3b, of y -> 3b+1, of z -> 3b+2 (one loop per bit)."""
    x = np.asarray(x, dtype=np.uint64)
    y = np.asarray(y, dtype=np.uint64)
    z = np.asarray(z, dtype=np.uint64)
    key = np.zeros(x.shape, dtype=np.uint64)
    one = np.uint64(1)
    for b in range(bits):
        sb = np.uint64(b)
        key |= ((x >> sb) & one) << np.uint64(3 * b)
        key |= ((y >> sb) & one) << np.uint64(3 * b + 1)
        key |= ((z >> sb) & one) << np.uint64(3 * b + 2)
    return key


def morton_decode(key, bits: int):
    key = np.asarray(key, dtype=np.uint64)
    x = np.zeros(key.shape, dtype=np.int64)
    y = np.zeros(key.shape, dtype=np.int64)
    z = np.zeros(key.shape, dtype=np.int64)
    one = np.uint64(1)
    for b in range(bits):
        x |= (((key >> np.uint64(3 * b)) & one) << np.uint64(b)).astype(np.int64)
        y |= (((key >> np.uint64(3 * b + 1)) & one) << np.uint64(b)).astype(np.int64)
        z |= (((key >> np.uint64(3 * b + 2)) & one) << np.uint64(b)).astype(np.int64)
    return x, y, z


def curve_order(xyz: np.ndarray, bits: int):
    """Step 1.  xyz: int [3, ncell] (unique cells).  Returns (perm, keys_sorted): perm[i] = input index of
    the i-th cell along the curve (a stable sort of the keys; keys are unique, so the order is unique)."""
    key = morton_key(xyz[0], xyz[1], xyz[2], bits)
    perm = np.argsort(key, kind="stable")
    return perm.astype(np.int64), key[perm]


def build_patches(keys_sorted: np.ndarray, kmax: int):
    """Step 2, written as the definition itself: the cells are a SET of coordinates; an
    octree-aligned cube of side 2^k is compact iff every one of its 8^k coordinates is in the set; every cell
    belongs to the largest compact cube (k <= kmax) that contains it.  The cells are visited in curve order;
    a cell no earlier patch covers starts a patch: the largest k whose aligned cube around it is compact, by
    direct membership tests (each aligned cube is tested once and the answer remembered).  Aligned cubes are
    nested or disjoint, so the cubes found are disjoint, cover the cells, and the visited cell is the cube's
    first cell along the curve.  No property of sorted keys is used.
    Returns (first, level): first[p] = position in curve order of the first cell of patch p, level[p] = k."""
    keys = np.asarray(keys_sorted, dtype=np.uint64)
    n = keys.shape[0]
    bits = max(1, (int(keys.max()).bit_length() + 2) // 3) if n else 1
    x, y, z = morton_decode(keys, bits)
    coords = list(zip(x.tolist(), y.tolist(), z.tolist()))
    cells = set(coords)
    assert len(cells) == n, "cells are unique"
    compact = {}                                   # (k, ox, oy, oz) -> every coordinate of the cube is a cell

    def is_compact(k, ox, oy, oz):
        key = (k, ox, oy, oz)
        if key not in compact:
            s = 1 << k
            compact[key] = all((ox + a, oy + b, oz + c) in cells
                               for c in range(s) for b in range(s) for a in range(s))
        return compact[key]

    covered = set()
    first, level = [], []
    for i, (cx, cy, cz) in enumerate(coords):
        if (cx, cy, cz) in covered:
            continue
        k_found = 0
        for k in range(kmax, 0, -1):
            s = 1 << k
            if is_compact(k, cx // s * s, cy // s * s, cz // s * s):
                k_found = k
                break
        s = 1 << k_found
        ox, oy, oz = cx // s * s, cy // s * s, cz // s * s
        covered.update((ox + a, oy + b, oz + c) for c in range(s) for b in range(s) for a in range(s))
        first.append(i)
        level.append(k_found)
    return np.asarray(first, dtype=np.int64), np.asarray(level, dtype=np.int32)


def patch_origins(keys_sorted, first, bits: int):
    x, y, z = morton_decode(np.asarray(keys_sorted)[first], bits)
    return np.stack([x, y, z], axis=1).astype(np.int32)


def gather_level(fields: np.ndarray, perm, keys_sorted, first, level, k: int, bits: int):
    """Step 3 for the patches of side n = 2^k: out[f, p, lz, ly, lx] = field f of the cell at
    origin_p + (lx, ly, lz), patches in curve order.  fields: [nf, ncell] in INPUT order.
    Returns (out [nf, np_k, n, n, n], origin [np_k, 3])."""
    n = 1 << k
    sel = np.nonzero(np.asarray(level) == k)[0]
    out = np.zeros((fields.shape[0], len(sel), n, n, n), dtype=fields.dtype)
    org = patch_origins(keys_sorted, np.asarray(first)[sel], bits)
    lx, ly, lz = morton_decode(np.arange(8 ** k, dtype=np.uint64), k)   # Morton offset inside the cube -> (lx, ly, lz)
    for s, p in enumerate(sel):
        f0 = int(first[p])
        out[:, s, lz, ly, lx] = fields[:, perm[f0:f0 + 8 ** k]]
    return out, org
