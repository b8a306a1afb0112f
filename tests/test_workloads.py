"""The seeded input generators (workloads/): shapes, seeds, stated statistics."""
import numpy as np

import workloads as wk


def test_config1_shape_and_state():
    wl = wk.config1_sod()
    lev = wl.levels[0]
    assert lev.U.shape == (5, 1, 32, 32, 32) and lev.bc == (1,) * 6 and wl.gamma == 1.4
    assert np.all(lev.U[0, 0, :, :, :16] == 1.0) and np.all(lev.U[0, 0, :, :, 16:] == 0.125)
    assert np.allclose(lev.U[4, 0, 0, 0, [0, 31]], [2.5, 0.25])


def test_config2_statistics_and_determinism():
    a = wk.config2_random_patches(npatch=4)
    b = wk.config2_random_patches(npatch=4)
    assert np.array_equal(a.levels[0].U, b.levels[0].U)
    U = a.levels[0].U
    assert np.allclose(U[0].mean(axis=(1, 2, 3)), 1.0, atol=1e-14)
    assert abs(np.log(U[0]).std() - 0.5) < 0.02
    v = U[1:4] / U[0]
    mach = np.sqrt((v ** 2).sum(axis=0).mean()) / np.sqrt(5.0 / 3.0)
    assert abs(mach - 1.0) < 0.03
    assert not np.array_equal(U[:, 0], U[:, 1])


def test_morton_order_and_patch_split_roundtrip():
    o = wk.morton_patch_origins(4, 4, 4, 16)
    assert o[:8].tolist() == [[0, 0, 0], [16, 0, 0], [0, 16, 0], [16, 16, 0], [0, 0, 16], [16, 0, 16],
                              [0, 16, 16], [16, 16, 16]]
    assert len({tuple(r) for r in o.tolist()}) == 64
    G = np.arange(2 * 64 ** 3, dtype=np.float64).reshape(2, 64, 64, 64)
    U = wk.split_into_patches(G, 16, o)
    assert np.array_equal(wk.configs.join_patches(U, o, (64, 64, 64)), G)


def test_config3_orszag_tang_state():
    wl = wk.config3_orszag_tang(N=32)
    lev = wl.levels[0]
    assert lev.U.shape == (9, 8, 16, 16, 16) and lev.domain_cells == (32, 32, 32)
    assert np.allclose(lev.U[0], 25 / (36 * np.pi)) and np.all(lev.U[8] == 0) and np.all(lev.U[7] == 0)
    G = wk.configs.join_patches(lev.U, lev.origin, (32, 32, 32))
    # central-difference div B vanishes identically (B_x depends on y only, B_y on x only)
    div = (np.roll(G[5], -1, 2) - np.roll(G[5], 1, 2)) + (np.roll(G[6], -1, 1) - np.roll(G[6], 1, 1))
    assert np.abs(div).max() < 1e-15


def test_config5_statistics_small():
    wl = wk.config5_turbulence(N=64, n=32)
    lev = wl.levels[0]
    U = lev.U
    assert U.shape == (9, 8, 32, 32, 32) and np.all(U[0] == 1.0)
    v2 = (U[1:4] ** 2).sum(axis=0).mean()
    assert abs(np.sqrt(v2) - 3 * np.sqrt(5 / 3)) < 1e-12
    assert abs((U[5:8] ** 2).sum(axis=0).mean() - 0.02) < 1e-14
    G = wk.configs.join_patches(U, lev.origin, (64, 64, 64))
    assert abs(G[5].mean()) < 1e-15
    # spectrally solenoidal: k . B^ = 0
    Bh = [np.fft.fftn(G[5 + c]) for c in range(3)]
    k = np.fft.fftfreq(64) * 64
    KZ, KY, KX = np.meshgrid(k, k, k, indexing="ij")
    keep = (np.abs(KX) < 32) & (np.abs(KY) < 32) & (np.abs(KZ) < 32)
    div = (KX * Bh[0] + KY * Bh[1] + KZ * Bh[2])[keep]
    assert np.abs(div).max() < 1e-8 * np.abs(Bh[0]).max()


def test_config4_geometry_small():
    wl = wk.config4_two_level(True, nfine=64, threshold=3.0)
    lc, lf = wl.levels
    assert lc.U.shape == (9, 8, 16, 16, 16) and lf.U.shape[1] == 16
    assert np.all(lf.origin % 16 == 0) and lf.dx == lc.dx / 2
    # root = 2x2x2 mean of the fine data under every fine patch
    Gc = wk.configs.join_patches(lc.U, lc.origin, (32, 32, 32))
    p = 3
    ox, oy, oz = lf.origin[p] // 2
    blk = lf.U[:, p].reshape(9, 8, 2, 8, 2, 8, 2).mean(axis=(2, 4, 6))
    assert np.allclose(Gc[:, oz:oz + 8, oy:oy + 8, ox:ox + 8], blk, rtol=1e-13, atol=1e-16)
    assert abs(Gc[7].mean() - 1e-3) < 1e-12
