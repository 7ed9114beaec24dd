"""Full-size checks in the launch configuration bench.py times (pytest -m gpu).

The oracle runs the full-size configs for as many steps as it finishes in about a minute on the
GPU box's host cores (element-wise parity on every cell); beyond that the checks are properties
that hold at any size: mass conservation, the spreading moment identity sum_X G = sum_k Delta u_k
(pin K6) and bitwise run-to-run determinism."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL = 2e-6


def _stream():
    import torch
    return torch.cuda.Stream()


@pytest.fixture(scope="module")
def api():
    from paper_1904_02108_b200 import api as _api
    return _api


def _parity(api, wl, steps):
    import oracle
    sim = api.from_workload(wl, stream=_stream())
    ref = oracle.from_workload(wl)
    sim.step(steps, wl.mdf_iters)
    ref.step(steps, wl.mdf_iters)
    sim.sync()
    rho, u, f = sim.read_fields()
    r_rho, r_u, r_f = ref.read_fields()
    e_u, e_r = np.abs(u - r_u).max(), np.abs(rho - r_rho).max()
    assert e_u <= TOL and e_r <= TOL, (e_u, e_r)
    if wl.n_markers:
        assert np.abs(f - r_f).max() <= 1e-5 * np.abs(r_f).max()
        mk, rm = sim.read_markers(), ref.read_markers()
        assert np.abs(mk["force"] - rm["du"]).max() <= 1e-5 * np.abs(rm["du"]).max()
        perm_ref = oracle.reference_sort(mk["cell"].astype(np.int64))
        assert np.array_equal(mk["perm"].astype(np.int64), perm_ref)
    sim.close()
    ref.close()
    return e_u, e_r


def test_w2_full_256_parity_at_step_100(api):
    """configs[1] at full size, parity at step 100 (BJ:north_star) + the plane-mean profile is held."""
    from paper_1904_02108_b200 import workloads
    wl = workloads.get("W2")
    e = _parity(api, wl, 100)
    print("W2 full errors (u, rho):", e)


def test_w2_full_poiseuille_profile_is_held_1000_steps(api):
    """configs[1]: after 1000 steps the x-y plane means of u_x stay within 1e-5 of the analytic
    discrete Poiseuille profile (pin K9's closed form, typed here)."""
    from paper_1904_02108_b200 import workloads
    wl = workloads.get("W2")
    sim = api.from_workload(wl, stream=_stream())
    sim.step(1000, 0)
    rho, u, _ = sim.read_fields(force=False)
    tau, g, H = wl.tau, wl.g[0], wl.nz
    nu = (tau - 0.5) / 3.0
    z = np.arange(H, dtype=np.float64)
    exact = g / (2 * nu) * (z + 0.5) * (H - 0.5 - z) + g * (16 * tau * tau - 20 * tau + 3) / (4 * (2 * tau - 1))
    prof = u[0].astype(np.float64).mean(axis=(1, 2))
    assert np.abs(prof - exact).max() < 1e-5
    assert abs(rho.astype(np.float64).mean() - 1.0) < 1e-6
    sim.close()


def test_w4_full_256_parity_at_step_100(api):
    """configs[3] at full size (1,179,648 markers), every cell and marker against the oracle."""
    from paper_1904_02108_b200 import workloads
    e = _parity(api, workloads.get("W4"), 100)
    print("W4 full errors (u, rho):", e)


def _properties(api, wl, steps):
    outs = []
    for rep in range(2):
        sim = api.from_workload(wl, stream=_stream())
        rho0, _, _ = sim.read_fields(u=False, force=False)
        m0 = rho0.astype(np.float64).sum()
        sim.step(steps, wl.mdf_iters)
        sim.sync()
        rho, u, G = sim.read_fields()
        mk = sim.read_markers(pos=False, perm=False, cell=False)
        sim.close()
        # mass: fp32 read-out summed in fp64
        assert abs(rho.astype(np.float64).sum() - m0) <= 2e-7 * m0
        # K6: zeroth moment of the spread force equals the sum of the marker forces
        tot_g = G.astype(np.float64).reshape(3, -1).sum(axis=1)
        tot_m = mk["force"].astype(np.float64).sum(axis=0)
        scale = np.abs(mk["force"]).astype(np.float64).sum()
        assert np.abs(tot_g - tot_m).max() <= 1e-6 * scale
        assert np.isfinite(u).all() and np.abs(u).max() < 0.3
        outs.append((rho, u, G, mk["force"]))
    for a, b in zip(*outs):
        assert np.array_equal(a, b)          # bitwise determinism at full size


def test_w4_full_properties_100_steps(api):
    from paper_1904_02108_b200 import workloads
    _properties(api, workloads.get("W4"), 100)


def test_w5_full_512_parity_20_steps_and_properties(api):
    """configs[4] at full size (134 M cells, 11.8 M markers): 20 steps against the oracle on every cell and
    marker (the fp64 oracle needs ~50 GB and ~10 s per step on the GPU box's host cores: step 100 at full size would
    take the whole test budget; it is checked on the 128^3 reduction of the recipe, test_w5_recipe_128_100_steps),
    then properties and bitwise determinism over 20 steps."""
    from paper_1904_02108_b200 import workloads
    wl = workloads.get("W5")
    e = _parity(api, wl, 20)
    print("W5 full errors (u, rho):", e)
    _properties(api, wl, 20)


def test_paper_shaped_case_p6_parity_and_p18_properties(api):
    """the paper's 160 x 160 x 320 box with 6 propellers of 3936 points
    (spacing 1, s = 1): 20 steps against the oracle on every cell and marker; 18 propellers (the
    paper's extreme case, 70,848 points): properties over 50 steps.  nx = 160 is a multiple of 32,
    ny = 160, nz = 320 of 4: the two-candidate collect path; s = 1 makes the MDF iteration matrix
    the stiffest of all workloads."""
    from paper_1904_02108_b200 import workloads
    e = _parity(api, workloads.get("P6"), 20)
    print("P6 errors (u, rho):", e)
    _properties(api, workloads.get("P18"), 50)
