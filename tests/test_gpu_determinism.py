"""-m gpu: the CUDA path gives the same BITS when the same work is run again (a tripwire for shared-memory races in
the step kernels - whose phases hand data between warps with two barriers per plane, a warp-level fence and
unsynchronised private scratch, DESIGN.md section 6.1 - and for order-dependent accumulation in the AMR operators:
the reflux list is appended through an atomic counter, the flux registers are summed with result-less atomics).
compute-sanitizer is not available on the GPU boxes of this pool; a race would show here as differing bits between
repeated runs on data whose neighbouring values differ everywhere."""
import numpy as np
import pytest

import workloads as wk

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def H():
    import gpu_harness
    return gpu_harness


def _hydro_of(wl):
    lev = wl.levels[0]
    U = lev.U.copy()
    U[4] -= 0.5 * (U[5] ** 2 + U[6] ** 2 + U[7] ** 2)
    lev.U = np.ascontiguousarray(U[:5])
    return wk.Workload(wl.name + "_hydro", [lev], wl.gamma, False, wl.limiter, wk.configs.RS_HLLC, wl.cfl, 1, 0.0)


@pytest.mark.parametrize("np_dtype", [np.float32, np.float64])
@pytest.mark.parametrize("mhd", [False, True])
@pytest.mark.parametrize("n", [16, 32])
def test_three_steps_twice_give_the_same_bits(H, np_dtype, mhd, n):
    """config-5 turbulence at 64^3 (every tile has neighbours in all directions; Mach 3, so limiter and solver take
    every branch), three steps, run five times from the same state: states, dt and signal speeds bitwise equal."""
    wl = wk.config5_turbulence(N=64, n=n)
    if not mhd:
        wl = _hydro_of(wl)
    lev = wl.levels[0]
    first = H.gpu_advance(lev, wl, 3, np_dtype=np_dtype)
    assert np.isfinite(first["U"]).all()
    for _ in range(4):
        again = H.gpu_advance(lev, wl, 3, np_dtype=np_dtype)
        assert again["dts"] == first["dts"] and again["smaxs"] == first["smaxs"]
        assert np.array_equal(again["U"], first["U"])


@pytest.mark.parametrize("np_dtype", [np.float32, np.float64])
def test_hierarchy_root_steps_twice_give_the_same_bits(H, np_dtype):
    """Three-level MHD hierarchy, two root steps (prolongation, restriction, reflux from a device-built list, flux
    registers accumulated by atomics, levels overlapped on streams), run three times: every level bitwise equal."""
    wl = wk.config_hierarchy(True, 3, 256, n=16)
    first = H.gpu_hierarchy_step(wl, np_dtype=np_dtype, nsteps=2)
    for _ in range(2):
        again = H.gpu_hierarchy_step(wl, np_dtype=np_dtype, nsteps=2)
        assert again["dts"] == first["dts"]
        for a, b in zip(again["U"], first["U"]):
            assert np.array_equal(a, b)


def test_ppm_steps_twice_give_the_same_bits(H):
    """The config-5 gas without the field at Mach 1 (PPM has no pressure floor either), 64^3 on 16^3 patches."""
    G = wk.configs.turbulence_state(64, mach=1.0)
    G[4] -= 0.5 * (G[5] ** 2 + G[6] ** 2 + G[7] ** 2)
    wl = wk.configs.uniform_grid_workload("turbulence_hydro_mach1", np.ascontiguousarray(G[:5]), 16, 5.0 / 3.0, False,
                                          wk.configs.LIM_MC, wk.configs.RS_HLLC, 0.3, 2)
    lev = wl.levels[0]
    first = H.gpu_ppm_advance(lev, wl, 2, np_dtype=np.float32)
    for _ in range(3):
        again = H.gpu_ppm_advance(lev, wl, 2, np_dtype=np.float32)
        assert np.array_equal(again["U"], first["U"])
