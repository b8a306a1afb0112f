"""Pins of the patch-builder oracle (oracle/patch_builder.py): the textbook
bit interleave on hand-computed keys, the hand-worked example of tests/golden/patch_builder_example.txt,
brute force over aligned cubes on tiny random cell sets (no Morton arithmetic on that side), and the
invariants that define the result (disjoint cover, compactness, maximality, curve order)."""
import os

import numpy as np
import pytest

from oracle import patch_builder as pb

GOLD = os.path.join(os.path.dirname(__file__), "golden", "patch_builder_example.txt")


def _interleave_int(x, y, z, bits):
    """Independent key: plain Python integers, one bit at a time."""
    k = 0
    for b in range(bits):
        k |= ((x >> b) & 1) << (3 * b) | ((y >> b) & 1) << (3 * b + 1) | ((z >> b) & 1) << (3 * b + 2)
    return k


def test_morton_key_hand_values():
    # (3,5,6): x=011 y=101 z=110 -> bit triples (z y x) per level b: b0: x1 y1 z0 -> 011 = 3; b1: x1 y0 z1 -> 101 = 5;
    # b2: x0 y1 z1 -> 110 = 6  => key = 3 + 5*8 + 6*64 = 427
    assert int(pb.morton_key(3, 5, 6, 3)) == 427
    assert [int(pb.morton_key(*c, 2)) for c in ((1, 0, 0), (0, 1, 0), (0, 0, 1), (2, 0, 0), (0, 2, 0), (0, 0, 2))] == [1, 2, 4, 8, 16, 32]
    rng = np.random.default_rng(5)
    xyz = rng.integers(0, 1 << 7, size=(3, 200))
    keys = pb.morton_key(xyz[0], xyz[1], xyz[2], 7)
    assert [int(k) for k in keys] == [_interleave_int(int(a), int(b), int(c), 7) for a, b, c in xyz.T]
    x, y, z = pb.morton_decode(keys, 7)
    assert np.array_equal(np.stack([x, y, z]), xyz)


def _read_gold():
    sec, out = None, {"cells": [], "order": [], "patches": []}
    for ln in open(GOLD):
        ln = ln.strip()
        if not ln or ln.startswith("#"):
            continue
        if ln in out:
            sec = ln
            continue
        out[sec].append([int(v) for v in ln.split()])
    return out


def test_worked_example():
    g = _read_gold()
    xyz = np.array(g["cells"]).T
    perm, keys = pb.curve_order(xyz, 2)
    assert perm.tolist() == g["order"][0]
    first, level = pb.build_patches(keys, 2)
    org = pb.patch_origins(keys, first, 2)
    got = [list(map(int, o)) + [1 << int(k)] for o, k in zip(org, level)]
    assert got == g["patches"]


def _brute_force_patches(cells: set, bits: int, kmax: int):
    """For every cell the largest aligned compact cube containing it, by direct membership tests."""
    found = set()
    for (x, y, z) in cells:
        best = (x, y, z, 1)
        for k in range(1, kmax + 1):
            s = 1 << k
            ox, oy, oz = x // s * s, y // s * s, z // s * s
            if all((ox + i, oy + j, oz + l) in cells for i in range(s) for j in range(s) for l in range(s)):
                best = (ox, oy, oz, s)
        found.add(best)
    return found


@pytest.mark.parametrize("seed", range(6))
def test_brute_force_tiny(seed):
    rng = np.random.default_rng([11, seed])
    bits, kmax = 3, (2 if seed % 2 else 3)
    N = 1 << bits
    # a union of a few aligned cubes of mixed sizes plus random single cells: patches of every size occur
    occ = np.zeros((N, N, N), bool)
    for _ in range(3):
        s = 1 << int(rng.integers(1, 3))
        o = rng.integers(0, N // s, 3) * s
        occ[o[0]:o[0] + s, o[1]:o[1] + s, o[2]:o[2] + s] = True
    occ |= rng.random((N, N, N)) < (0.9 if seed == 5 else 0.15)
    if seed == 4:
        occ[:] = True
    xyz = np.array(np.nonzero(occ))
    xyz = xyz[:, rng.permutation(xyz.shape[1])]
    perm, keys = pb.curve_order(xyz, bits)
    first, level = pb.build_patches(keys, kmax)
    org = pb.patch_origins(keys, first, bits)
    got = {(int(o[0]), int(o[1]), int(o[2]), 1 << int(k)) for o, k in zip(org, level)}
    cells = {tuple(int(v) for v in c) for c in xyz.T}
    assert got == _brute_force_patches(cells, bits, kmax)
    # curve order of the patch list: increasing key of the origin, keys computed independently
    ok = [_interleave_int(int(o[0]), int(o[1]), int(o[2]), bits) for o in org]
    assert ok == sorted(ok)
    # disjoint cover
    assert int((8 ** level.astype(np.int64)).sum()) == xyz.shape[1]
    if seed == 4:
        assert len(first) == (N >> kmax) ** 3 and (level == kmax).all()


def test_gather_places_cells():
    rng = np.random.default_rng(3)
    bits, kmax = 4, 2
    N = 1 << bits
    occ = np.zeros((N, N, N), bool)
    occ[4:12, 0:8, 8:16] = True
    occ[0:2, 0:2, 0:2] = True
    occ[13, 13, 13] = True
    xyz = np.array(np.nonzero(occ))
    xyz = xyz[:, rng.permutation(xyz.shape[1])]
    # field 0 = x + 100 y + 10000 z of the cell, field 1 = its input index
    F = np.stack([xyz[0] + 100.0 * xyz[1] + 10000.0 * xyz[2], np.arange(xyz.shape[1], dtype=np.float64)])
    perm, keys = pb.curve_order(xyz, bits)
    first, level = pb.build_patches(keys, kmax)
    for k in (1, 2):
        out, org = pb.gather_level(F, perm, keys, first, level, k, bits)
        n = 1 << k
        assert out.shape[1] == (8 if k == 2 else 1)        # the 8^3 box = eight 4^3 patches; one 2^3 patch
        lz, ly, lx = np.meshgrid(np.arange(n), np.arange(n), np.arange(n), indexing="ij")
        for s in range(out.shape[1]):
            exp = (org[s, 0] + lx) + 100.0 * (org[s, 1] + ly) + 10000.0 * (org[s, 2] + lz)
            assert np.array_equal(out[0, s], exp)
            idx = out[1, s].astype(int)
            assert np.array_equal(xyz[0][idx], org[s, 0] + lx) and np.array_equal(xyz[2][idx], org[s, 2] + lz)
