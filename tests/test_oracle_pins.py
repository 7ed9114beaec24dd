"""Pins K1..K13: the fp64 oracle against what the paper and the
mathematics fix -- closed forms, invariants, brute force over the whole lattice, textbook limits.
None of these re-uses the oracle's own formulae: every expected value below is either a literal
closed form typed here from the mathematics, a conservation law, or a brute-force evaluation of
the paper's definition (sums over ALL lattice cells, P:78 / P:98) written independently in numpy.
"""
import math

import numpy as np
import pytest

import oracle
from oracle import Oracle


# ----------------------------------------------------------------------------------------------
# K1: the delta kernel w(r) (reading R6)
def test_K1_delta_closed_values():
    golden = {}
    with open(__file__.rsplit("/", 1)[0] + "/golden/peskin4_values.txt") as fh:
        for line in fh:
            if line.startswith("#") or not line.strip():
                continue
            r, v = line.split()[:2]
            golden[float(r)] = float(v)
    assert len(golden) >= 7
    for r, v in golden.items():
        assert oracle.delta_w(r) == pytest.approx(v, abs=1e-15)
        assert oracle.delta_w(-r) == pytest.approx(v, abs=1e-15)


def test_K1_delta_moment_identities():
    rng = np.random.default_rng(1)
    for r in list(rng.uniform(-1.0, 1.0, size=200)) + [0.0, 0.5, 1.0, -1.0, 0.25]:
        js = np.arange(-4, 5)
        w = np.array([oracle.delta_w(r - j) for j in js])
        assert w.sum() == pytest.approx(1.0, abs=1e-14)                 # partition of unity
        assert ((r - js) * w).sum() == pytest.approx(0.0, abs=1e-14)    # first moment
        assert (w * w).sum() == pytest.approx(3.0 / 8.0, abs=1e-14)     # sum of squares
        assert w[js % 2 == 0].sum() == pytest.approx(0.5, abs=1e-14)    # even / odd balance
        assert (w >= 0).all()
    assert oracle.delta_w(2.0) == 0.0 and oracle.delta_w(2.5) == 0.0 and oracle.delta_w(-3.0) == 0.0


def test_K1_printed_second_branch_is_garbled():
    """R6: the second branch as printed ('sqrt(1 - 7 + 12|r| - 4r^2)') breaks partition of
    unity by several per cent; the standard Peskin form does not."""
    def printed(r):
        a = abs(r)
        if a <= 1:
            return (3 - 2 * a + math.sqrt(1 + 4 * a - 4 * a * a)) / 8
        if a <= 2:
            return (5 - 2 * a - math.sqrt(max(0.0, 1 - 7 + 12 * a - 4 * a * a))) / 8
        return 0.0
    r = 0.3
    s_printed = sum(printed(r - j) for j in range(-3, 4))
    assert abs(s_printed - 1.0) > 0.03


# ----------------------------------------------------------------------------------------------
def _brute_weights(o: Oracle, x):
    """W(X,Y,Z) over ALL lattice cells for one point (periodic minimum-image distance)."""
    def w1d(xa, n, periodic):
        X = np.arange(n, dtype=np.float64)
        d = xa - X
        if periodic:
            d = d - n * np.round(d / n)
        a = np.abs(d)
        out = np.zeros(n)
        m1 = a <= 1
        m2 = (a > 1) & (a < 2)
        out[m1] = (3 - 2 * a[m1] + np.sqrt(1 + 4 * a[m1] - 4 * a[m1] ** 2)) / 8
        out[m2] = (5 - 2 * a[m2] - np.sqrt(-7 + 12 * a[m2] - 4 * a[m2] ** 2)) / 8
        return out
    wx = w1d(x[0], o.nx, True)
    wy = w1d(x[1], o.ny, True)
    wz = w1d(x[2], o.nz, True)
    return wz[:, None, None] * wy[None, :, None] * wx[None, None, :]


def _random_markers(rng, n, box):
    pos = rng.uniform(0.0, 1.0, size=(n, 3)) * np.array(box)
    return pos.astype(np.float32), rng.uniform(0.1, 0.5, size=n).astype(np.float32)


def test_K2_constant_and_linear_fields_reproduced():
    rng = np.random.default_rng(2)
    o = Oracle(12, 10, 9, 0.8)
    # keep markers away from the periodic seam so that the linear field is linear in the stencil
    pos = (rng.uniform(2.5, 6.0, size=(40, 3))).astype(np.float32)
    o.set_markers(pos, None, np.ones(40, dtype=np.float32))
    o.markers_at_rest()
    Z, Y, X = np.meshgrid(np.arange(9.0), np.arange(10.0), np.arange(12.0), indexing="ij")
    U = np.stack([0.3 + 0 * X, 0.1 * X - 0.2 * Y + 0.05 * Z + 1.0, -0.7 * Z + 0.01 * X])
    u = o.interpolate(U)
    p = pos.astype(np.float64)
    assert np.allclose(u[:, 0], 0.3, atol=1e-14)
    assert np.allclose(u[:, 1], 0.1 * p[:, 0] - 0.2 * p[:, 1] + 0.05 * p[:, 2] + 1.0, atol=1e-13)
    assert np.allclose(u[:, 2], -0.7 * p[:, 2] + 0.01 * p[:, 0], atol=1e-13)


def test_K3_bruteforce_all_cells_interpolation_and_spreading():
    rng = np.random.default_rng(3)
    o = Oracle(8, 7, 6, 0.8)   # periodic, includes markers whose stencil wraps
    pos, area = _random_markers(rng, 10, (8, 7, 6))
    o.set_markers(pos, None, area)
    o.markers_at_rest()
    U = rng.normal(size=(3, 6, 7, 8))
    u = o.interpolate(U)
    v = rng.normal(size=(10, 3))
    F = o.spread(v)
    F_ref = np.zeros_like(F)
    for k in range(10):
        W = _brute_weights(o, pos[k].astype(np.float64))
        assert W.sum() == pytest.approx(1.0, abs=1e-13)
        for a in range(3):
            assert u[k, a] == pytest.approx((U[a] * W).sum(), abs=1e-13)
            F_ref[a] += v[k, a] * W
    assert np.allclose(F, F_ref, atol=1e-13)


def test_K4_adjointness():
    rng = np.random.default_rng(4)
    o = Oracle(9, 8, 10, 0.8)
    pos, area = _random_markers(rng, 50, (9, 8, 10))
    o.set_markers(pos, None, area)
    o.markers_at_rest()
    U = rng.normal(size=(3, 10, 8, 9))
    Fk = rng.normal(size=(50, 3))
    s = area.astype(np.float64)
    lhs = (o.spread(Fk * s[:, None]) * U).sum()
    rhs = (s[:, None] * Fk * o.interpolate(U)).sum()
    assert lhs == pytest.approx(rhs, rel=1e-13)


def test_K5_single_marker_uniform_flow_geometric_series():
    """One marker in uniform flow U0: g_m = (u_k - U0) (1 - s (3/8)^3)^m, Delta u = s sum_m g_m."""
    U0 = np.array([0.03, -0.02, 0.01])
    uk = np.array([0.05, 0.01, -0.04])
    s = 0.7
    o = Oracle(10, 10, 10, 0.8)
    o.set_markers(np.array([[4.3, 5.6, 4.9]], dtype=np.float32), uk[None].astype(np.float32),
                  np.array([s], dtype=np.float32))
    o.markers_at_rest()
    s = float(np.float32(s))
    uk = uk.astype(np.float32).astype(np.float64)
    U = np.broadcast_to(U0[:, None, None, None], (3, 10, 10, 10)).copy()
    q = 1.0 - s * 0.052734375        # (3/8)^3 typed as a literal
    for N in (1, 2, 5):
        o.set_U(U)
        o.mdf(N)
        m = o.read_markers()
        g_last = (uk - U0) * q ** (N - 1)
        du = s * (uk - U0) * sum(q ** i for i in range(N))
        assert np.allclose(m["g"][0], g_last, atol=1e-15)
        assert np.allclose(m["du"][0], du, atol=1e-15)


def test_K6_force_moments_and_K7_bookkeeping():
    rng = np.random.default_rng(6)
    o = Oracle(16, 14, 12, 0.8)
    pos = rng.uniform(3.0, 9.0, size=(60, 3)).astype(np.float32)     # stencils inside the box
    area = rng.uniform(0.1, 0.3, size=60).astype(np.float32)
    vel = rng.normal(scale=0.02, size=(60, 3)).astype(np.float32)
    o.set_markers(pos, vel, area)
    o.markers_at_rest()
    U = rng.normal(scale=0.01, size=(3, 12, 14, 16))
    o.set_U(U)
    o.mdf(4, also_last_u=True)
    m = o.read_markers()
    # G is only reachable through read_fields (which recomputes moments from f, not touching G)
    _, _, G = o.read_fields()
    du = m["du"]
    # zeroth moment
    assert np.allclose(G.reshape(3, -1).sum(axis=1), du.sum(axis=0), atol=1e-14)
    # first moment: sum_X X x G(X) = sum_k x_k x du_k
    Z, Y, X = np.meshgrid(np.arange(12.0), np.arange(14.0), np.arange(16.0), indexing="ij")
    R = np.stack([X, Y, Z]).reshape(3, -1)
    torque_grid = np.cross(R.T, G.reshape(3, -1).T).sum(axis=0)
    torque_mark = np.cross(pos.astype(np.float64), du).sum(axis=0)
    assert np.allclose(torque_grid, torque_mark, atol=1e-12)
    # K7: if the last iteration also updates U then U^N = U^0 + G cell by cell (reading R8)
    assert np.allclose(o.get_Um(), U + G, atol=1e-15)


def test_K13_reductions():
    """mdf_iters = 0 or zero markers == pure LBM; one iteration with s = 1 == classical single
    direct forcing: G = spread(u_k - interp(U))."""
    rng = np.random.default_rng(13)
    u0 = rng.normal(scale=0.01, size=(3, 8, 8, 8))
    a = Oracle(8, 8, 8, 0.7)
    b = Oracle(8, 8, 8, 0.7)
    c = Oracle(8, 8, 8, 0.7)
    for o in (a, b, c):
        o.set_fields(None, u0)
    pos = rng.uniform(0, 8, size=(5, 3)).astype(np.float32)
    b.set_markers(pos, None, np.ones(5, dtype=np.float32))
    c.set_markers(pos, None, np.ones(5, dtype=np.float32))
    a.step(3, 5)          # no markers
    b.step(3, 0)          # markers but zero iterations
    c.step(3, 1)
    fa, fb, fc = a.populations().copy(), b.populations().copy(), c.populations().copy()
    assert np.array_equal(fa, fb)
    assert not np.array_equal(fa, fc)
    # single direct forcing
    d = Oracle(8, 8, 8, 0.7)
    d.set_markers(pos, None, np.ones(5, dtype=np.float32))
    d.markers_at_rest()
    U = rng.normal(scale=0.01, size=(3, 8, 8, 8))
    d.set_U(U)
    d.mdf(1)
    _, _, G = d.read_fields()
    assert np.allclose(G, d.spread(0.0 - d.interpolate(U)), atol=1e-16)


# ----------------------------------------------------------------------------------------------
# K8: collide / stream invariants
def test_K8_rest_state_is_invariant():
    """rho = 1, u = 0, no force is a fixed point.  In plain fp64 sum_i t_i rounds to 1 - O(1e-16),
    so the pin is: no drift beyond a few ulp however many steps are taken (the CUDA path, which
    stores f_i - t_i, is checked bit-for-bit in the gpu tests)."""
    o = Oracle(6, 5, 4, 0.8, wall=(0, 1, 0))
    f0 = o.populations().copy()
    o.step(7, 0)
    assert np.abs(o.populations() - f0).max() < 5e-16
    o.step(200, 0)
    assert np.abs(o.populations() - f0).max() < 5e-16
    rho, u, G = o.read_fields()
    assert np.array_equal(rho, np.ones_like(rho)) or np.allclose(rho, 1.0, atol=2e-16)
    assert np.abs(u).max() < 1e-16


def test_K8_mass_conserved_and_momentum_balance():
    rng = np.random.default_rng(8)
    for forcing in ("guo", "shift"):
        g = (1e-4, -2e-4, 5e-5)
        o = Oracle(10, 9, 8, 0.75, g=g, forcing=forcing)
        u0 = rng.normal(scale=0.02, size=(3, 8, 9, 10))
        rho0 = 1.0 + rng.normal(scale=0.01, size=(8, 9, 10))
        o.set_fields(rho0, u0)
        pos = rng.uniform(0, 8, size=(30, 3)).astype(np.float32)
        vel = rng.normal(scale=0.02, size=(30, 3)).astype(np.float32)
        o.set_markers(pos, vel, np.full(30, 0.25, dtype=np.float32))
        E = np.array([[0, 0, 0], [1, 0, 0], [-1, 0, 0], [0, 1, 0], [0, -1, 0], [0, 0, 1], [0, 0, -1],
                      [1, 1, 0], [-1, -1, 0], [1, -1, 0], [-1, 1, 0], [1, 0, 1], [-1, 0, -1], [1, 0, -1],
                      [-1, 0, 1], [0, 1, 1], [0, -1, -1], [0, 1, -1], [0, -1, 1]], dtype=np.float64)
        mass0 = o.populations().sum()
        for _ in range(5):
            f = o.populations()
            mom_before = np.einsum("ia,izyx->a", E, f)
            rho, _, _ = o.read_fields()
            o.step(1, 3)
            _, _, G = o.read_fields()
            mom_after = np.einsum("ia,izyx->a", E, o.populations())
            a = G + np.array(g)[:, None, None, None]
            expect = (rho[None] * a).reshape(3, -1).sum(axis=1)
            assert np.allclose(mom_after - mom_before, expect, rtol=0, atol=1e-12)
        assert o.populations().sum() == pytest.approx(mass0, rel=1e-13)


def test_K8_mass_with_walls():
    rng = np.random.default_rng(81)
    o = Oracle(6, 7, 8, 0.6, wall=(1, 0, 1), g=(1e-5, 0, 0))
    o.set_fields(1.0 + rng.normal(scale=0.01, size=(8, 7, 6)), rng.normal(scale=0.02, size=(3, 8, 7, 6)))
    m0 = o.populations().sum()
    o.step(50, 0)
    assert o.populations().sum() == pytest.approx(m0, rel=1e-13)


# ----------------------------------------------------------------------------------------------
# K9: exact discrete Poiseuille solution (collide + stream + half-way bounce-back + force)
@pytest.mark.parametrize("forcing", ["guo", "shift"])
@pytest.mark.parametrize("tau", [0.6, 0.8, 0.933, 1.0])
def test_K9_poiseuille_exact_discrete_profile(tau, forcing):
    H, g = 16, 1e-5
    nu = (tau - 0.5) / 3.0
    o = Oracle(2, 2, H, tau, wall=(0, 0, 1), g=(g, 0.0, 0.0), forcing=forcing)
    z = np.arange(H, dtype=np.float64)
    slip = g * (16 * tau * tau - 20 * tau + 3) / (4 * (2 * tau - 1))
    exact = g / (2 * nu) * (z + 0.5) * (H - 0.5 - z) + slip
    o.set_fields(None, np.stack([np.broadcast_to(exact[:, None, None], (H, 2, 2)),
                                 np.zeros((H, 2, 2)), np.zeros((H, 2, 2))]))
    nsteps = int(12 * H * H / nu)
    o.step(nsteps, 0)
    rho, u, _ = o.read_fields()
    prof = u[0].mean(axis=(1, 2))
    assert np.abs(prof - exact).max() < 1e-8 * g            # 1e-13 absolute
    assert np.abs(u[1]).max() < 1e-12 and np.abs(u[2]).max() < 1e-12
    assert np.allclose(rho, 1.0, atol=1e-12)


def test_K9_poiseuille_from_rest_converges_to_the_exact_profile():
    """K9 started from rest (u0 = 0) instead of from the answer: the profile must be REACHED, not merely held.
    tau = 1 makes the diffusive time short (nu = 1/6): H^2 / nu = 384 steps for H = 8; 40 diffusive times."""
    H, g, tau = 8, 1e-5, 1.0
    nu = (tau - 0.5) / 3.0
    for forcing in ("guo", "shift"):
        o = Oracle(2, 2, H, tau, wall=(0, 0, 1), g=(g, 0.0, 0.0), forcing=forcing)
        z = np.arange(H, dtype=np.float64)
        slip = g * (16 * tau * tau - 20 * tau + 3) / (4 * (2 * tau - 1))
        exact = g / (2 * nu) * (z + 0.5) * (H - 0.5 - z) + slip
        o.step(int(40 * H * H / nu), 0)
        rho, u, _ = o.read_fields()
        prof = u[0].mean(axis=(1, 2))
        assert prof.max() > 0.9 * exact.max()                  # it did move away from rest
        assert np.abs(prof - exact).max() < 1e-8 * g


# ----------------------------------------------------------------------------------------------
# K14: second moment of the forced collision (the part of the Guo source term K8 / K9 do not see)
_E = np.array([[0, 0, 0], [1, 0, 0], [-1, 0, 0], [0, 1, 0], [0, -1, 0], [0, 0, 1], [0, 0, -1],
               [1, 1, 0], [-1, -1, 0], [1, -1, 0], [-1, 1, 0], [1, 0, 1], [-1, 0, -1], [1, 0, -1],
               [-1, 0, 1], [0, 1, 1], [0, -1, -1], [0, 1, -1], [0, -1, 1]], dtype=np.float64)


def test_K14_guo_source_second_moment_closed_form():
    """Uniform periodic box, rho = 1, uniform u0 and uniform acceleration a: streaming maps a uniform state onto
    itself, so a step is the collision alone and every moment follows a closed recurrence.

    Moments of the D3Q19 equilibrium and of the Guo source S_i = t_i rho [3 (e_i - u*).a + 9 (e_i.u*)(e_i.a)]
    (P:56 force inclusion, reading R3; u* = U + a/2):
        sum_i e e^T Eq_i(rho, u) = rho (I/3 + u u^T),      sum_i e e^T S_i = rho (u* a^T + a u*^T),
        sum_i e Eq_i = rho u,  sum_i e S_i = rho a,  sum_i S_i = 0.
    With f' = f - (f - Eq(rho, u*))/tau + (1 - 1/(2 tau)) S the momentum gains rho a per step (U_{n+1} = U_n + a)
    and the second moment Pi = sum_i e e^T f_i obeys
        Pi_{n+1} = (1 - 1/tau) Pi_n + (1/tau) rho (I/3 + u* u*^T) + (1 - 1/(2 tau)) rho (u* a^T + a u*^T),
    whose solution from Pi_0 = rho (I/3 + u0 u0^T) is
        Pi_n = rho [ I/3 + U_n U_n^T - (1/4) a a^T (1 - (1 - 1/tau)^n) ].
    (Check: insert, use u* = U_n + a/2 and U_{n+1} = U_n + a; the a a^T terms give -1/4 + (1/tau)(1/4) ... = the
    stated factor.)  Dropping the 9 (e.u*)(e.a) term, or writing U for u* in the source, changes Pi at O(|u||a|)
    and O(|a|^2): the mutated recurrences below miss the oracle by many orders of magnitude more than the pin allows."""
    tau = 0.8
    u0 = np.array([0.021, -0.013, 0.008])
    a = np.array([0.011, 0.007, -0.009])
    nx, ny, nz = 3, 4, 5
    o = Oracle(nx, ny, nz, tau, g=tuple(a))
    o.set_fields(None, np.broadcast_to(u0[:, None, None, None], (3, nz, ny, nx)).copy())

    def second_moment():
        f = o.populations()
        assert np.abs(f - f[:, :1, :1, :1]).max() < 1e-15            # stays uniform
        return np.einsum("ia,ib,i->ab", _E, _E, f[:, 0, 0, 0])

    def recurrence(P, U, variant):
        us = U + 0.5 * a
        uv = U if variant == "U_for_ustar" else us
        src = np.outer(uv, a) + np.outer(a, uv)
        if variant == "no_second_order":                              # only 3 (e - u*).a kept: -(u*.a) I
            src = -np.dot(us, a) * np.eye(3)
        return (1 - 1 / tau) * P + (1 / tau) * (np.eye(3) / 3 + np.outer(us, us)) + (1 - 0.5 / tau) * src

    P = {v: np.eye(3) / 3 + np.outer(u0, u0) for v in ("exact", "no_second_order", "U_for_ustar")}
    U = u0.copy()
    assert np.abs(second_moment() - P["exact"]).max() < 1e-15
    worst = {v: 0.0 for v in P}
    for n in range(1, 8):
        o.step(1, 0)
        for v in P:
            P[v] = recurrence(P[v], U, v)
        U = U + a
        got = second_moment()
        closed = np.eye(3) / 3 + np.outer(U, U) - 0.25 * np.outer(a, a) * (1 - (1 - 1 / tau) ** n)
        assert np.abs(got - closed).max() < 1e-14, n
        assert np.abs(got - P["exact"]).max() < 1e-14, n
        for v in P:
            worst[v] = max(worst[v], np.abs(got - P[v]).max())
        rho, u, _ = o.read_fields()
        assert np.abs(u[:, 0, 0, 0] - U).max() < 1e-15 and abs(rho[0, 0, 0] - 1) < 1e-15
    assert worst["no_second_order"] > 1e-5 and worst["U_for_ustar"] > 1e-5      # the pin discriminates


# K10: tau <-> nu through the decay of a periodic shear wave
def test_K10_shear_wave_decay():
    L, tau, A = 32, 0.8, 1e-4
    nu = (tau - 0.5) / 3.0
    o = Oracle(2, 2, L, tau)
    z = np.arange(L)
    u0 = np.zeros((3, L, 2, 2))
    u0[0] = (A * np.sin(2 * np.pi * z / L))[:, None, None]
    o.set_fields(None, u0)
    o.step(200, 0)       # let the non-hydrodynamic transient die
    _, u1, _ = o.read_fields()
    a1 = 2.0 / L * (u1[0, :, 0, 0] * np.sin(2 * np.pi * z / L)).sum()
    T = 400
    o.step(T, 0)
    _, u2, _ = o.read_fields()
    a2 = 2.0 / L * (u2[0, :, 0, 0] * np.sin(2 * np.pi * z / L)).sum()
    k = 2 * np.pi / L
    nu_meas = -math.log(a2 / a1) / (k * k * T)
    assert nu_meas == pytest.approx(nu, rel=k * k)      # O(k^2) discretisation error


# K11: rigid rotation invariants
def test_K11_kinematics():
    rng = np.random.default_rng(11)
    omega = 2 * math.pi / 64
    axis = np.array([0.3, -0.5, 0.8])
    axis /= np.linalg.norm(axis)
    c = np.array([20.0, 21.0, 19.5])
    o = Oracle(40, 40, 40, 0.8, wall=(1, 1, 1))
    pos = (c + rng.uniform(-8, 8, size=(25, 3))).astype(np.float32)
    o.set_markers(pos, None, np.ones(25, dtype=np.float32))
    o.set_kinematics(omega, axis * 3.0, c)        # un-normalised axis must be normalised
    p = pos.astype(np.float64)
    rperp = np.linalg.norm(np.cross(p - c, axis), axis=1)
    for n in range(64):
        o.step(1, 1)
        m = o.read_markers()
        assert np.allclose(np.linalg.norm(m["x"] - c, axis=1), np.linalg.norm(p - c, axis=1), atol=1e-12)
        assert np.allclose(np.linalg.norm(m["uk"], axis=1), 2 * rperp * math.sin(omega / 2), atol=1e-13)
        assert np.allclose((m["x"] - c) @ axis, (p - c) @ axis, atol=1e-12)
    assert np.allclose(m["x"], p, atol=1e-11)       # back at rest after 2 pi / omega steps
    # quarter turn about z, typed by hand: (x,y) -> (-y,x)
    o2 = Oracle(40, 40, 40, 0.8, wall=(1, 1, 1))
    o2.set_markers(np.array([[25.0, 20.0, 20.0]], dtype=np.float32), None, np.ones(1, dtype=np.float32))
    o2.set_kinematics(math.pi / 2, np.array([0.0, 0.0, 1.0]), np.array([20.0, 20.0, 20.0]))
    o2.step(1, 1)
    m2 = o2.read_markers()
    assert np.allclose(m2["x"][0], [20.0, 25.0, 20.0], atol=1e-14)
    assert np.allclose(m2["uk"][0], [-5.0, 5.0, 0.0], atol=1e-14)


def test_K11_periodic_wrap_of_positions():
    o = Oracle(16, 16, 16, 0.8)
    o.set_markers(np.array([[15.5, 0.25, 8.0]], dtype=np.float32), None, np.ones(1, dtype=np.float32))
    o.set_kinematics(math.pi, np.array([0.0, 0.0, 1.0]), np.array([15.0, 0.0, 8.0]))
    o.step(1, 1)
    x = o.read_markers()["x"][0]
    assert np.allclose(x, [14.5, 15.75, 8.0], atol=1e-13)    # (14.5, -0.25) wrapped into [0,16)


# K12: direction tables -- a lattice symmetry applied to the whole set-up permutes the result
def test_K12_lattice_symmetry_axis_permutation_and_mirror():
    rng = np.random.default_rng(12)
    n = 8
    u0 = rng.normal(scale=0.02, size=(3, n, n, n))      # [comp][z][y][x]
    rho0 = 1.0 + rng.normal(scale=0.01, size=(n, n, n))
    pos = rng.uniform(0, n, size=(12, 3))
    vel = rng.normal(scale=0.02, size=(12, 3))
    g = np.array([1e-4, -3e-4, 2e-4])

    def run(perm, sign):
        """relabel axes: new axis a = old axis perm[a], mirrored if sign[a] = -1"""
        # field arrays are indexed [z][y][x] = axes (2,1,0)
        def xf_scalar(A):
            B = np.transpose(A, [2 - perm[2 - d] for d in range(3)])
            for a in range(3):
                if sign[a] < 0:
                    B = np.flip(B, axis=2 - a)
            return B
        r = xf_scalar(rho0)
        v = np.stack([sign[a] * xf_scalar(u0[perm[a]]) for a in range(3)])
        p = np.stack([pos[:, perm[a]] if sign[a] > 0 else (n - 1) - pos[:, perm[a]] for a in range(3)], axis=1)
        p = np.mod(p, n)
        w = np.stack([sign[a] * vel[:, perm[a]] for a in range(3)], axis=1)
        gg = [sign[a] * g[perm[a]] for a in range(3)]
        o = Oracle(n, n, n, 0.7, g=gg)
        o.set_fields(r, v)
        o.set_markers(p.astype(np.float64).astype(np.float32), w.astype(np.float32), np.full(12, 0.25, dtype=np.float32))
        o.step(4, 2)
        rr, uu, GG = o.read_fields()
        return rr, uu, GG, xf_scalar

    # markers must be float32-exact in both frames: use dyadic positions
    pos = np.round(pos * 64) / 64
    vel = np.round(vel * 4096) / 4096
    r0, u_0, G0, _ = run([0, 1, 2], [1, 1, 1])
    for perm, sign in (([1, 2, 0], [1, 1, 1]), ([0, 1, 2], [-1, 1, 1]), ([2, 1, 0], [1, -1, 1])):
        r1, u1, G1, xf = run(perm, sign)
        assert np.allclose(r1, xf(r0), atol=1e-13)
        for a in range(3):
            assert np.allclose(u1[a], sign[a] * xf(u_0[perm[a]]), atol=1e-13)
            assert np.allclose(G1[a], sign[a] * xf(G0[perm[a]]), atol=1e-13)


def test_reference_sort_is_stable():
    rng = np.random.default_rng(5)
    keys = rng.integers(0, 50, size=1000)
    perm = oracle.reference_sort(keys)
    expect = np.argsort(keys, kind="stable")
    assert np.array_equal(perm, expect)
