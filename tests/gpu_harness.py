"""Sequencing helpers for the -m gpu parity tests: drive the CUDA path through the Python binding
exactly as oracle.api.advance / two_level_step sequence the oracle (same order of calls), and the
error norm of reading A18.  No arithmetic of the method lives here."""
import numpy as np

import paper_1412_0934_b200 as amr


def gpu_dtype(np_dtype):
    return amr.AMR_F64 if np.dtype(np_dtype) == np.float64 else amr.AMR_F32


def gpu_step(b, wl, dt, ch, limiter=None, riemann=None):
    lim = wl.limiter if limiter is None else limiter
    rs = wl.riemann if riemann is None else riemann
    if wl.mhd:
        b.mhd_step(dt, wl.gamma, lim, rs, ch, wl.alpha)
    else:
        b.hydro_step(dt, wl.gamma, lim, rs)


def gpu_advance(level, wl, nsteps, np_dtype=np.float64, dt_fixed=None, limiter=None, riemann=None):
    """Every step: amr_cfl_dt (O7; fused value after the first step) -> dt = cfl dx / smax, c_h = smax
    -> amr_*_step (O0..O6).  Returns dict(U, dts, smaxs, counters, batch)."""
    b = amr.PatchBatch.from_level(level, gpu_dtype(np_dtype))
    dts, smaxs = [], []
    for _ in range(nsteps):
        dt, sm = b.cfl_dt(wl.gamma, wl.cfl)
        if dt_fixed is not None:
            dt = dt_fixed
        gpu_step(b, wl, dt, sm, limiter, riemann)
        dts.append(dt)
        smaxs.append(sm)
    return dict(U=b.download(), dts=dts, smaxs=smaxs, counters=b.step_counters(), batch=b)


def gpu_ppm_advance(level, wl, nsteps, np_dtype=np.float64, dt_fixed=None, riemann=None):
    """PPM in the order of oracle.api.ppm_advance: amr_cfl_dt -> dt, then amr_hydro_step_ppm with the sweep order
    x-y-z on even steps, z-y-x on odd steps (the halo is gathered inside every sweep)."""
    b = amr.PatchBatch.from_level(level, gpu_dtype(np_dtype))
    rs = wl.riemann if riemann is None else riemann
    dts, smaxs = [], []
    for step_no in range(nsteps):
        dt, sm = b.cfl_dt(wl.gamma, wl.cfl)
        if dt_fixed is not None:
            dt = dt_fixed
        b.hydro_step_ppm(dt, wl.gamma, rs, step_no % 2)
        dts.append(dt)
        smaxs.append(sm)
    return dict(U=b.download(), dts=dts, smaxs=smaxs, counters=b.step_counters(), batch=b)


def gpu_two_level_step(wl, np_dtype=np.float64, do_reflux=True):
    """O9 in the order of oracle.api.two_level_step."""
    lc, lf = wl.levels
    dt_ = gpu_dtype(np_dtype)
    bc = amr.PatchBatch.from_level(lc, dt_)
    bf = amr.PatchBatch.from_level(lf, dt_)
    link = amr.LevelLink(bc, bf)
    _, s0 = bc.cfl_dt(wl.gamma, wl.cfl)
    _, s1 = bf.cfl_dt(wl.gamma, wl.cfl)
    sm = max(s0, s1)
    dt0 = wl.cfl * lc.dx / sm
    link.flux_clear()
    gpu_step(bc, wl, dt0, sm)
    for theta in (0.0, 0.5):
        link.prolong_ghosts(theta)
        gpu_step(bf, wl, 0.5 * dt0, sm)
    link.restrict()
    if do_reflux:
        link.reflux(dt0)
    out = dict(Uc=bc.download(), Uf=bf.download(), dt0=dt0, smax=sm, coarse=bc, fine=bf, link=link)
    return out


def gpu_hierarchy_step(wl, np_dtype=np.float64, do_reflux=True, nsteps=1):
    """f3 through amr_hierarchy_cfl_dt / amr_hierarchy_step (the recursion runs inside the library, in the
    order of oracle.api.hierarchy_step)."""
    h = amr.Hierarchy.from_workload(wl, gpu_dtype(np_dtype))
    dts = []
    for _ in range(nsteps):
        dt0, sm = h.cfl_dt(wl.gamma, wl.cfl)
        h.step(dt0, wl.gamma, wl.limiter, wl.riemann, sm, wl.alpha, do_reflux)
        dts.append(dt0)
    return dict(U=[b.download() for b in h.levels], dt0=dts[-1], dts=dts, smax=sm, hierarchy=h)


def field_groups(nf):
    """A18: momentum and B are normalised by the max over their three components."""
    g = [[0], [1, 2, 3], [4]]
    if nf == 9:
        g += [[5, 6, 7], [8]]
    return g


def rel_err(got, ref, psi_scale=None):
    """Per field group: max|got-ref| / max|ref| (psi: / psi_scale when given, since it starts at 0)."""
    got = np.asarray(got, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    errs = []
    for grp in field_groups(ref.shape[0]):
        num = np.abs(got[grp] - ref[grp]).max()
        den = np.abs(ref[grp]).max()
        if grp == [8] and psi_scale is not None:
            den = max(den, psi_scale)
        errs.append(num / max(den, 1e-300))
    return np.array(errs)


def per_step_parity(oracle, level, wl, nsteps, np_dtype, psi_floor=None):
    """Per-step parity inside a multi-step GPU run (reading A17): at every step the fp64
    oracle is restarted from the GPU's own state of that step (rounded values, promoted to fp64) and
    takes one step with the GPU's dt and c_h; its result is compared with the GPU's next state.
    Returns (list of per-step rel_err arrays, final GPU state, batch)."""
    b = amr.PatchBatch.from_level(level, gpu_dtype(np_dtype))
    g = level.g
    errs = []
    U = b.download()
    for _ in range(nsteps):
        dt, sm = b.cfl_dt(wl.gamma, wl.cfl)
        gpu_step(b, wl, dt, sm)
        Unew = b.download()
        Ug = oracle.ghosted(U.astype(np.float64), g)
        oracle.fill_ghosts(Ug, g, level.origin, level.domain_cells, level.bc, level.self_periodic)
        r = oracle.step(Ug, g, dt, level.dx, wl.gamma, wl.limiter, wl.riemann, ch=sm, alpha=wl.alpha,
                        eps=oracle.default_eps(np_dtype))
        ref = oracle.interior(r["U"], g)
        ps = sm * np.abs(ref[5:8]).max() if wl.mhd else None
        errs.append(rel_err(Unew, ref, psi_scale=ps))
        U = Unew
    return errs, U, b


def sampled_patch_parity(oracle, U0, U1, origin, n, domain, dx, wl, dt, ch, sample_ids, np_dtype):
    """Full-size parity on sampled outputs: for each sampled patch the oracle takes the same step on a
    3x3x3-patch mini-level cut out of the GPU's input state U0 (the patch and its 26 periodic neighbours:
    everything the radius-2 stencil of the centre patch can reach), with the GPU's dt and c_h, and its centre
    patch is compared element by element with the GPU's output U1.  Returns the per-patch rel_err arrays."""
    where = {tuple(int(v) for v in o): i for i, o in enumerate(np.asarray(origin))}
    dom = np.asarray(domain)
    mini_origin = np.array([[i * n, j * n, k * n] for k in range(3) for j in range(3) for i in range(3)], np.int32)
    import workloads as wk
    errs = []
    for s in sample_ids:
        o = np.asarray(origin[s])
        ids = [where[tuple(int(v) for v in (o + (mo - n)) % dom)] for mo in mini_origin]
        Um = np.ascontiguousarray(U0[:, ids]).astype(np.float64)
        lev = wk.Level(n=n, g=3, level=0, dx=dx, origin=mini_origin, domain_cells=(3 * n,) * 3, bc=(0,) * 6,
                       self_periodic=False, U=Um)
        Ug = oracle.ghosted(Um, 3)
        oracle.fill_ghosts(Ug, 3, lev.origin, lev.domain_cells, lev.bc, False)
        # O1..O6 act patch by patch on the ghosted arrays: only the centre patch (index 13) is stepped
        Uc = np.ascontiguousarray(Ug[:, 13:14])
        r = oracle.step(Uc, 3, dt, dx, wl["gamma"], wl["limiter"], wl["riemann"], ch=ch, alpha=wl["alpha"],
                        eps=oracle.default_eps(np_dtype))
        ref = oracle.interior(r["U"], 3)[:, 0]
        got = np.asarray(U1[:, s], dtype=np.float64)
        ps = ch * np.abs(ref[5:8]).max() if ref.shape[0] == 9 else None
        errs.append(rel_err(got[:, None], ref[:, None], psi_scale=ps))
    return errs


_ROT = {0: [0, 1, 2, 3, 4, 5, 6, 7, 8], 1: [0, 2, 3, 1, 4, 6, 7, 5, 8], 2: [0, 3, 1, 2, 4, 7, 5, 6, 8]}


def cells_next_to_a_marginal_decision(oracle, level, wl, dt, ch, limiter, riemann, eps, cells, rel=1e-4):
    """Readings A7 / A19: the HLL fallback (p_T* <= 0) and the skipped rotational waves (B_n^2 < eps p_T*) are the
    discontinuous decisions of the MHD solver; the kernel takes them in the batch dtype, the oracle in fp64, so a face
    whose criterion lies within fp32 round-off of its threshold may be decided differently and then changes its two
    cells by O(1e-3).  For each cell (p, k, j, i) this returns whether one of its six faces is such a face ACCORDING
    TO THE ORACLE: |p_T*| <= rel * max(p_TL, p_TR) or |B_n^2 - eps p_T*| <= rel * eps p_T* (oracle.hlld_states on the
    oracle's own face states).  Everything else must meet the plain bound."""
    g = level.g
    Ug = oracle.ghosted(level.U, g)
    oracle.fill_ghosts(Ug, g, level.origin, level.domain_cells, level.bc, level.self_periodic)
    FS = oracle.step(Ug, g, dt, level.dx, wl.gamma, limiter, riemann, ch=ch, alpha=wl.alpha, eps=eps,
                     want_face_states=True)["FS"]          # [d][0: W^-_d, 1: W^+_d][field][patch][M^3]
    out = []
    for (p, k, j, i) in cells:
        c = [k + g, j + g, i + g]
        marginal = False
        for d in range(3):
            e = [0, 0, 0]
            e[2 - d] = 1
            for upper in (0, 1):
                lo = c if upper else [c[a] - e[a] for a in range(3)]
                hi = [c[a] + e[a] for a in range(3)] if upper else c
                WL = FS[d, 1, :, p, lo[0], lo[1], lo[2]][_ROT[d]]
                WR = FS[d, 0, :, p, hi[0], hi[1], hi[2]][_ROT[d]]
                st = oracle.hlld_states(WL, WR, wl.gamma, ch, eps)
                if st["S"][0] >= 0 or st["S"][4] <= 0:
                    continue                                # supersonic face: no star state is formed
                pts, bn2 = st["ptstar"], st["Bn"] ** 2
                ptk = max(WL[4] + 0.5 * (WL[5:8] ** 2).sum(), WR[4] + 0.5 * (WR[5:8] ** 2).sum())
                if abs(pts) <= rel * ptk or abs(bn2 - eps * pts) <= rel * eps * abs(pts):
                    marginal = True
        out.append(marginal)
    return out
