"""-m gpu parity at BASELINE.json's full sizes, in the launch configuration bench.py times: sampled outputs
the oracle computes one by one (tests/gpu_harness.sampled_patch_parity), plus properties that hold at any
size (conservation on the periodic domain, finite state, event counters).  Inputs are the seeded synthetic
workloads of bench.py."""
import numpy as np
import pytest

import workloads as wk

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def H():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("-m gpu tests need a CUDA device (there is no CPU fallback)")
    import gpu_harness
    return gpu_harness


def test_config5_full_size_sampled_fp32(oracle, H):
    """Config 5 as bench.py runs it and as BASELINE.json states it: 512^3 = 4096 patches of 32^3, MHD fp32,
    MC + HLLD + GLM, 10 steps.  EVERY step is checked on 64 seeded sample patches
    against the fp64 oracle restarted from the GPU's own input state of that step (A17: the fp32 bound is per
    step); conserved totals over all 10 steps."""
    import torch
    import paper_1412_0934_b200 as amr
    dev = torch.device("cuda:0")
    U, origin = wk.turbulence_patches_torch(512, 32, dev)
    U0 = U.cpu().numpy()
    del U
    torch.cuda.empty_cache()
    wlp = dict(gamma=5.0 / 3.0, cfl=0.3, limiter=wk.configs.LIM_MC, riemann=wk.configs.RS_HLLD, alpha=0.4)
    nf, npatch = U0.shape[:2]
    b = amr.PatchBatch(npatch, 32, nf, amr.AMR_F32, 1.0 / 512, origin=origin, domain_cells=(512,) * 3, bc=(0,) * 6, nghost=3)
    b.upload(U0)
    tot0 = b.conserved_totals()
    rng = np.random.default_rng([wk.SEED, 5, 512])
    before = U0
    worst = []
    for step in range(10):
        dt, sm = b.cfl_dt(wlp["gamma"], wlp["cfl"])
        b.mhd_step(dt, wlp["gamma"], wlp["limiter"], wlp["riemann"], sm, wlp["alpha"])
        after = b.download()
        ids = rng.choice(npatch, size=64, replace=False)
        errs = H.sampled_patch_parity(oracle, before, after, origin, 32, (512,) * 3, 1.0 / 512, wlp, dt, sm, ids, np.float32)
        worst.append(max(e.max() for e in errs))
        assert worst[-1] <= 1e-5, (step, worst)
        before = after
    tot = b.conserved_totals()
    absn = np.abs(U0.astype(np.float64)).sum(axis=(1, 2, 3, 4))
    grp = np.array([absn[0], absn[1:4].max(), absn[1:4].max(), absn[1:4].max(), absn[4], absn[5:8].max(), absn[5:8].max(), absn[5:8].max()])
    assert (np.abs(tot - tot0)[:8] / grp).max() <= 3e-6       # fp32 round-off of 10 x 1.3e8 cell updates, summed in fp64
    c = b.step_counters()
    assert c["nonpositive_rho_after"] == 0 and np.isfinite(tot).all()


@pytest.mark.parametrize("np_dtype", [np.float64, np.float32])
def test_config3_full_size_sampled(oracle, H, np_dtype):
    """Config 3 as stated: 256^3 Orszag-Tang = 4096 patches of 16^3, MHD, 5 steps; the last step is checked on
    16 seeded sample patches (fp64: 1e-12 per step; fp32: 1e-5), conservation over the 5 steps."""
    import paper_1412_0934_b200 as amr
    w = wk.config3_orszag_tang(N=256)
    lev = w.levels[0]
    U0 = lev.U.astype(np_dtype)
    wlp = dict(gamma=w.gamma, cfl=w.cfl, limiter=w.limiter, riemann=w.riemann, alpha=w.alpha)
    dtype = amr.AMR_F64 if np_dtype == np.float64 else amr.AMR_F32
    b = amr.PatchBatch(lev.npatch, 16, 9, dtype, lev.dx, origin=lev.origin, domain_cells=lev.domain_cells, bc=(0,) * 6, nghost=3)
    b.upload(U0)
    tot0 = b.conserved_totals()
    for step in range(5):
        if step == 4:
            before = b.download()
        dt, sm = b.cfl_dt(wlp["gamma"], wlp["cfl"])
        b.mhd_step(dt, wlp["gamma"], wlp["limiter"], wlp["riemann"], sm, wlp["alpha"])
    after = b.download()
    rng = np.random.default_rng([wk.SEED, 3, 256])
    ids = rng.choice(lev.npatch, size=16, replace=False)
    errs = H.sampled_patch_parity(oracle, before, after, lev.origin, 16, lev.domain_cells, lev.dx, wlp, dt, sm, ids, np_dtype)
    tol = 1e-12 if np_dtype == np.float64 else 1e-5
    assert max(e.max() for e in errs) <= tol, errs
    tot = b.conserved_totals()
    absn = np.abs(U0.astype(np.float64)).sum(axis=(1, 2, 3, 4))
    grp = np.array([absn[0], absn[1:4].max(), absn[1:4].max(), absn[1:4].max(), absn[4], absn[5:8].max(), absn[5:8].max(), absn[5:8].max()])
    assert (np.abs(tot - tot0)[:8] / grp).max() <= (1e-13 if np_dtype == np.float64 else 1e-6)


@pytest.mark.parametrize("mhd", [False, True])
def test_config4_full_size_fp32(oracle, H, mhd):
    """Config 4 as stated: 128^3 root = 512 patches of 16^3 + level-1 patches on the flagged blocks (A15), fp32,
    one coarse step with two fine substeps (O9), element by element against the fp64 oracle started from the
    fp32-rounded data (fp32 degeneracy thresholds), composite conservation to fp32 round-off."""
    wl = wk.config4_two_level(mhd)
    lc, lf = wl.levels
    assert lc.npatch == 512 and 80 <= lf.npatch <= 125          # "about 20 % extra cells"
    lc.U = lc.U.astype(np.float32).astype(np.float64)
    lf.U = lf.U.astype(np.float32).astype(np.float64)
    ref = oracle.two_level_step(wl, eps=oracle.default_eps(np.float32))
    got = H.gpu_two_level_step(wl, np_dtype=np.float32)
    assert abs(got["dt0"] - ref["dt0"]) <= 4e-6 * ref["dt0"]
    ps = ref["smax"] * max(np.abs(ref["Uc"][5:8]).max(), 1e-300) if mhd else None
    ec = H.rel_err(got["Uc"], ref["Uc"], psi_scale=ps)
    ef = H.rel_err(got["Uf"], ref["Uf"], psi_scale=ps)
    assert ec.max() <= 2e-5 and ef.max() <= 2e-5, (ec, ef)      # two fine substeps + restriction + reflux: 2 x 1e-5
    tot = oracle.composite_totals(oracle.ghosted(got["Uc"].astype(np.float64), lc.g), lc,
                                  oracle.ghosted(got["Uf"].astype(np.float64), lf.g), lf)
    nfc = 8 if mhd else 5
    absn = np.array([np.abs(lc.U[f]).sum() * lc.dx ** 3 for f in range(lc.nfields)])
    assert (np.abs(tot - ref["totals_before"])[:nfc] / absn[:nfc]).max() <= 2e-6
