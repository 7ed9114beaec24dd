"""Randomised differential test (pytest -m gpu): seeded random lattices, walls, marker sets and option sets, the CUDA
path against the fp64 oracle at north_star's tolerances.

A run of 7,000 such cases found the one bug the workload tests could not see (two markers far apart in one chunk,
`test_two_markers_far_apart_in_one_chunk_activate_the_cells_between_them`); this file keeps 80 of them in the suite.
The marker sets are deliberately unlike a propeller: uniform clouds, clusters that put hundreds of markers into a few
cells, sheets, markers exactly on cell faces, static sets with a prescribed velocity next to rotating ones."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL_U, TOL_RHO, TOL_F = 2e-6, 2e-6, 1e-5


def _marker_set(rng, n, dims, wall):
    mode = rng.integers(0, 3)
    if mode == 0:                                    # a uniform cloud
        pos = rng.uniform(0, 1, (n, 3)) * dims
    elif mode == 1:                                  # clusters: a few cells hold everything
        c = rng.uniform(0, 1, (int(rng.integers(1, 5)), 3)) * dims
        pos = c[rng.integers(0, len(c), n)] + rng.normal(scale=rng.uniform(0.2, 1.5), size=(n, 3))
    else:                                            # a sheet
        pos = rng.uniform(0, 1, (n, 3)) * dims
        pos[:, int(rng.integers(0, 3))] = rng.uniform(2, 4) + rng.normal(scale=0.05, size=n)
    for a in range(3):
        # R17: next to a wall the stencil floor(x)-1 .. floor(x)+2 has to stay inside the box
        pos[:, a] = np.clip(pos[:, a], 1.0, dims[a] - 2.001) if wall[a] else np.mod(pos[:, a], dims[a])
    if rng.random() < 0.2:                           # some markers exactly on cell faces / corners
        k = min(n, 5)
        pos[:k] = np.floor(pos[:k])
        for a in range(3):
            if wall[a]:
                pos[:k, a] = np.clip(pos[:k, a], 1.0, dims[a] - 3.0)
    pos = pos.astype(np.float32)
    for a in range(3):
        if not wall[a]:
            pos[:, a] = np.where(pos[:, a] >= np.float32(dims[a]), np.float32(0), pos[:, a])
    vel = rng.normal(scale=0.01, size=(n, 3)).astype(np.float32)
    area = rng.uniform(0.02, 0.3, n).astype(np.float32) / max(1.0, n / 300)
    return pos, vel, area


def _run_case(api, orc, seed):
    import torch
    rng = np.random.default_rng(seed)
    nx, ny, nz = int(rng.integers(8, 44)), int(rng.integers(4, 26)), int(rng.integers(4, 26))
    wall = tuple(int(rng.random() < 0.3) for _ in range(3)) if rng.random() < 0.4 else (0, 0, 0)
    tau = float(rng.uniform(0.55, 1.2))
    g = tuple(float(x) for x in rng.normal(scale=2e-6, size=3))
    sim = api.LbmIbm(nx, ny, nz, tau, wall=wall, g=g, stream=torch.cuda.Stream())
    ref = orc.Oracle(nx, ny, nz, tau, wall=wall, g=g)
    dims = np.array([nx, ny, nz], float)
    for _ in range(int(rng.integers(1, 4))):
        m = _marker_set(rng, int(rng.choice([1, 7, 40, 300, 1500, 4000])), dims, wall)
        sim.set_markers(*m)
        ref.set_markers(*m)
        if sum(wall) == 0 and rng.random() < 0.7:    # a rotating body (no wall: nothing for the swept sphere to cross)
            axis = rng.normal(size=3)
            axis /= np.linalg.norm(axis)
            centre = rng.uniform(0, 1, 3) * dims
            omega = float(rng.uniform(-0.02, 0.02)) if rng.random() < 0.8 else 0.0
            sim.set_kinematics(omega, axis, centre)
            ref.set_kinematics(omega, axis, centre)
    opts = {}
    if rng.random() < 0.7: opts["tile_rows"] = int(rng.choice([0, 1, 2, 4]))
    if rng.random() < 0.7: opts["persistent"] = int(rng.choice([0, 1, 2]))
    if rng.random() < 0.7: opts["overlap"] = int(rng.choice([0, 1, 2, 3]))
    if rng.random() < 0.5: opts["pipeline"] = int(rng.choice([0, 1, 2]))
    if rng.random() < 0.2: opts["tile_warps"] = 2
    for k, v in opts.items():
        sim.set_option(getattr(api, "OPT_" + k.upper()), v)
    mdf, steps = int(rng.integers(1, 7)), int(rng.integers(2, 14))
    sim.step(steps, mdf)
    ref.step(steps, mdf)
    if rng.random() < 0.3:                           # pure steps in between
        sim.step(2, 0); ref.step(2, 0)
        sim.step(2, mdf); ref.step(2, mdf)
    sim.sync()
    rho, u, _ = sim.read_fields()
    r_rho, r_u, _ = ref.read_fields()
    mk, rm = sim.read_markers(), ref.read_markers()
    sim.close()
    what = f"seed {seed}: {nx}x{ny}x{nz} wall {wall} tau {tau:.2f} mdf {mdf} steps {steps} {opts}"
    if not np.isfinite(r_u).all() or np.abs(r_u).max() > 0.15 or np.abs(r_rho - 1).max() > 0.2:
        return False                                 # the random set-up diverges (also in fp64): nothing to compare
    assert np.abs(u - r_u).max() <= TOL_U, what
    assert np.abs(rho - r_rho).max() <= TOL_RHO, what
    assert np.abs(mk["force"] - rm["du"]).max() <= TOL_F * max(np.abs(rm["du"]).max(), 1e-30), what
    # positions: within a few fp32 ulp, modulo the box on periodic axes (23.9999988 in fp64 is 0 in fp32, R20)
    d = np.abs(mk["pos"] - rm["x"])
    for a in range(3):
        if not wall[a]:
            d[:, a] = np.minimum(d[:, a], dims[a] - d[:, a])
    assert d.max() <= 16 * np.spacing(np.float32(max(nx, ny, nz))), what
    assert np.array_equal(mk["perm"].astype(np.int64), orc.reference_sort(mk["cell"].astype(np.int64))), what
    return True


def test_eighty_random_cases_match_the_oracle():
    import torch
    assert torch.cuda.is_available()
    from paper_1904_02108_b200 import api
    import oracle as orc
    # 41861: the case (of 1,500) that fails on the library before the active-cell capacity fix
    compared = sum(_run_case(api, orc, seed) for seed in list(range(41000, 41080)) + [41861])
    assert compared >= 60            # a few random set-ups are unstable and skipped, most must be compared
