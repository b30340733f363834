"""Pins for the CPU oracle: what the paper and the mathematics fix (P1..P9).

None of these tests retype the oracle's formulas or re-call its routines to
produce the expected value: expected values are paper-printed numbers
(tests/golden/paper_values.json), closed forms, invariants, textbook special
cases, or an independent dense-matrix / polynomial-fit formulation written
here in numpy in a different style (hard-coded integer matrices from the
literature ordering, np.linalg.inv, np.polyfit).
"""
import math

import numpy as np
import pytest

from oracle.oracle import Oracle, wall_derivative
from paper_2509_01099_b200 import inputs

SQ3 = math.sqrt(3.0)


def make(dim, n, mesh="tanh", stretch=1.3, Ra=1e5, Ma=0.1 * SQ3, threads=1):
    w = inputs.custom_workload("t", dim, n, mesh=mesh, stretch=stretch, Ra=Ra, Ma=Ma)
    return Oracle(w.coords, w.delta, w.Ra, w.Pr, w.Ma, threads=threads), w


# --------------------------------------------------------------------------
# P3  lattice algebra
# --------------------------------------------------------------------------

# Standard second-order polynomial equilibrium in velocity space (textbook):
W9 = np.array([4 / 9] + [1 / 9] * 4 + [1 / 36] * 4)
W19 = np.array([1 / 3] + [1 / 18] * 6 + [1 / 36] * 12)


def feq2(e, wts, rho, u):
    eu = e @ u
    return wts * rho * (1 + 3 * eu + 4.5 * eu**2 - 1.5 * (u @ u))


def guo_force_velocity_space(e, wts, u, F):
    """Guo et al. forcing, velocity space: w_i [3 (e_i - u) + 9 (e_i.u) e_i] . F"""
    return np.array([w * ((3 * (ei - u) + 9 * (ei @ u) * ei) @ F) for ei, w in zip(e, wts)])


@pytest.mark.parametrize("dim", [2, 3])
def test_P3_rows_orthogonal_and_inverse(dim):
    o, _ = make(dim, 6)
    m = o.matrices()
    for A, Ai in ((m["M"], m["Minv"]), (m["N"], m["Ninv"])):
        G = A @ A.T
        assert np.allclose(G - np.diag(np.diag(G)), 0.0, atol=1e-12)
        assert np.allclose(Ai @ A, np.eye(len(A)), atol=1e-14)
        assert np.allclose(Ai, np.linalg.inv(A), atol=1e-14)
    ef, eg = o.velocities()
    # velocity sets: opposite pairs present, isotropy sums
    assert (ef.sum(0) == 0).all() and (eg.sum(0) == 0).all()
    assert len({tuple(v) for v in ef.tolist()}) == o.qf
    assert (ef[: o.qg] == eg).all()


@pytest.mark.parametrize("dim", [2, 3])
def test_P3_meq_is_projection_of_polynomial_equilibrium(dim):
    o, _ = make(dim, 6)
    ef, _ = o.velocities()
    M = o.matrices()["M"]
    wts = W9 if dim == 2 else W19
    rng = np.random.default_rng(1)
    for _ in range(5):
        rho = 1.0 + 0.1 * rng.uniform(-1, 1)
        u = 0.1 * rng.uniform(-1, 1, 3)
        if dim == 2:
            u[2] = 0.0
        assert np.allclose(M @ feq2(ef.astype(float), wts, rho, u), o.meq(rho, u), atol=1e-14)


@pytest.mark.parametrize("dim", [2, 3])
def test_P3_forcing_moments_are_projection_of_guo(dim):
    """Eq. 12 with the corrected last entry (reading A8) and Eq. 13."""
    o, _ = make(dim, 6)
    ef, _ = o.velocities()
    M = o.matrices()["M"]
    wts = W9 if dim == 2 else W19
    rng = np.random.default_rng(2)
    for _ in range(5):
        u = 0.1 * rng.uniform(-1, 1, 3)
        F = 1e-3 * rng.uniform(-1, 1, 3)
        if dim == 2:
            u[2] = F[2] = 0.0
        ref = M @ guo_force_velocity_space(ef.astype(float), wts, u, F)
        got = o.mforce(u, F)
        assert np.allclose(got, ref, atol=1e-17), (got - ref)
    if dim == 2:  # the entry as PRINTED (uFx + vFy) is not the projection
        u, F = np.array([0.05, -0.02, 0.0]), np.array([1e-3, 2e-3, 0.0])
        ref = M @ guo_force_velocity_space(ef.astype(float), wts, u, F)
        assert abs(ref[8] - (u[0] * F[0] + u[1] * F[1])) > 1e-6


@pytest.mark.parametrize("dim", [2, 3])
def test_P3_temperature_equilibrium_weights_match_printed_omega(dim, golden):
    """N^-1 n_eq(u=0) = (rest weight, omega/2 ...) with omega as printed at PAPER.md:177."""
    o, _ = make(dim, 6)
    p = o.params()
    num, den = golden["omega_bc"]["d2q5" if dim == 2 else "d3q7"]
    omega = (num + p["a_T"]) / den
    assert p["omega_bc"] == pytest.approx(omega, rel=1e-15)
    Ni = o.matrices()["Ninv"]
    geq = Ni @ o.neq(1.0, np.zeros(3))
    assert np.allclose(geq[1:], omega / 2, atol=1e-15)
    assert geq.sum() == pytest.approx(1.0, abs=1e-15)
    # a_T as printed at PAPER.md:124
    c, d = golden["a_T"]["d2q5" if dim == 2 else "d3q7"]
    assert p["a_T"] == pytest.approx(c * SQ3 * p["alpha"] - d, rel=1e-14)
    # q_kappa closed form: alpha = cs_T^2 (1/q_k - 1/2), cs_T^2 = omega (2-D: (4+a_T)/10; 3-D: (6+a_T)/21)
    qk = o.matrices()["Q"][1]
    assert p["alpha"] == pytest.approx(omega * (1 / qk - 0.5), rel=1e-13)


@pytest.mark.parametrize("dim", [2, 3])
def test_P3_collision_invariants(dim):
    o, _ = make(dim, 6)
    ef, _ = o.velocities()
    p = o.params()
    rng = np.random.default_rng(3)
    for _ in range(5):
        f = (1 + 0.05 * rng.uniform(-1, 1, o.qf)) / o.qf
        g = 0.3 * rng.uniform(-1, 1, o.qg)
        fp, gp = o.collide_node(f, g)
        rho, T = f.sum(), g.sum()
        assert fp.sum() == pytest.approx(rho, rel=1e-15)
        assert gp.sum() == pytest.approx(T, abs=1e-15)
        F = np.array([0.0, rho * p["gbeta"] * T, 0.0])
        dj = ef.T @ fp - ef.T @ f
        assert np.allclose(dj, F, atol=1e-16)
    # equilibrium without force is a fixed point of the collision
    o.set_buoyancy_scale(0.0)
    u = np.array([0.03, -0.02, 0.01 if dim == 3 else 0.0])
    feq = o.matrices()["Minv"] @ o.meq(1.02, u)
    geq = o.matrices()["Ninv"] @ o.neq(0.2, u)
    fp, gp = o.collide_node(feq, geq)
    assert np.allclose(fp, feq, atol=1e-16) and np.allclose(gp, geq, atol=1e-16)


def test_P3_relaxation_rates():
    o, _ = make(2, 6)
    p, m = o.params(), o.matrices()
    tau = p["tau_f"]
    assert p["nu"] == pytest.approx((tau - 0.5) / 3.0, rel=1e-14)  # nu = c_s^2 (tau - 1/2)
    S = m["S"]
    assert S[7] == pytest.approx(1 / tau) and S[8] == pytest.approx(1 / tau)
    assert S[0] == 0 and S[3] == 0 and S[5] == 0
    assert m["Q"][1] == pytest.approx(3 - SQ3) and m["Q"][2] == pytest.approx(3 - SQ3)
    o3, _ = make(3, 6)
    S3 = o3.matrices()["S"]
    t3 = o3.params()["tau_f"]
    for k in (9, 11, 13, 14, 15):
        assert S3[k] == pytest.approx(1 / t3)
    for k in (0, 3, 5, 7):
        assert S3[k] == 0


# --------------------------------------------------------------------------
# P1  quadratic interpolation is exact on quadratics (stretched mesh)
# --------------------------------------------------------------------------

@pytest.mark.parametrize("dim", [2, 3])
def test_P1_weights_reproduce_quadratics(dim):
    o, w = make(dim, 17, stretch=1.8)
    for axis in range(dim):
        x = w.coords[axis]
        for c in (-1, 1):
            base, wt = o.weights(axis, c)
            for j in range(len(x)):
                if (j == 0 and c == 1) or (j == len(x) - 1 and c == -1):
                    continue  # departure point beyond the wall: bounce-back, no stencil
                xd = x[j] - c * w.delta
                xs = x[base[j]: base[j] + 3]
                assert xs[0] - 1e-15 <= xd <= xs[2] + 1e-15      # interpolation, never extrapolation
                assert wt[j].sum() == pytest.approx(1.0, abs=1e-13)
                for poly in (lambda t: 1 + 0 * t, lambda t: t, lambda t: 3 * t * t - t + 0.5):
                    assert wt[j] @ poly(xs) == pytest.approx(float(poly(xd)), abs=1e-13)
                # independent construction: the parabola through the three nodes
                ys = np.array([0.3, -1.1, 0.7])
                coef = np.polyfit(xs - x[j], ys, 2)
                assert wt[j] @ ys == pytest.approx(np.polyval(coef, -c * w.delta), abs=1e-11)


@pytest.mark.parametrize("dim", [2, 3])
def test_P1_stream_is_exact_on_separable_quadratics(dim):
    """f+ = p(x)p(y)p(z), deg <= 2 per axis  =>  streamed value = p at the departure point."""
    o, w = make(dim, 9, stretch=1.5)
    ef, eg = o.velocities()
    x = w.coords[0]
    nz = o.shape[0]

    def P(t, k):
        return 1.0 + (0.5 + 0.1 * k) * t - (0.7 - 0.05 * k) * t * t

    X = [x, x, x if dim == 3 else np.zeros(1)]
    fp = np.empty((o.qf,) + o.shape)
    gp = np.empty((o.qg,) + o.shape)
    for i in range(o.qf):
        fp[i] = P(X[2], i)[:, None, None] * P(X[1], i + 1)[None, :, None] * P(X[0], i + 2)[None, None, :] if dim == 3 else (
            np.ones(1)[:, None, None] * P(X[1], i + 1)[None, :, None] * P(X[0], i + 2)[None, None, :])
    for i in range(o.qg):
        gp[i] = fp[i] * 0.5
    o.set_post_collision(fp, gp)
    o.stream()
    f, g = o.get_populations()
    n = len(x)
    checked = 0
    for i in range(o.qf):
        e = ef[i]
        for iz in range(nz):
            for iy in range(n):
                for ix in range(n):
                    idx = (ix, iy, iz)
                    if any((e[a] == 1 and idx[a] == 0) or (e[a] == -1 and idx[a] == n - 1) for a in range(dim)):
                        continue
                    xd = x[ix] - e[0] * w.delta
                    yd = x[iy] - e[1] * w.delta
                    val = P(np.float64(yd), i + 1) * P(np.float64(xd), i + 2)
                    if dim == 3:
                        val *= P(np.float64(x[iz] - e[2] * w.delta), i)
                    assert f[i, iz, iy, ix] == pytest.approx(val, abs=2e-13)
                    if i < o.qg:
                        assert g[i, iz, iy, ix] == pytest.approx(0.5 * val, abs=2e-13)
                    checked += 1
    assert checked > 0


# --------------------------------------------------------------------------
# P2  uniform mesh: ISLBM streaming == textbook pull streaming + half-way BB
# --------------------------------------------------------------------------

def textbook_stream(fp, e, opp, wall_rule):
    """Pull streaming on a unit lattice with half-way bounce-back, by index shifts."""
    q, nz, ny, nx = fp.shape
    out = np.empty_like(fp)
    dims = (nx, ny, nz)
    for i in range(q):
        for iz in range(nz):
            for iy in range(ny):
                for ix in range(nx):
                    src = (ix - e[i][0], iy - e[i][1], iz - e[i][2])
                    hit = [a for a in range(3) if not (0 <= src[a] < dims[a])]
                    if hit:
                        out[i, iz, iy, ix] = wall_rule(i, hit[0], (ix, iy, iz), fp[opp[i], iz, iy, ix])
                    else:
                        out[i, iz, iy, ix] = fp[i, src[2], src[1], src[0]]
    return out


@pytest.mark.parametrize("dim,n", [(2, 16), (3, 8)])
def test_P2_uniform_mesh_reduces_to_textbook_streaming_bitwise(dim, n):
    o, w = make(dim, n, mesh="uniform")
    ef, eg = o.velocities()
    opp_f = [int(np.where((ef == -ef[i]).all(1))[0][0]) for i in range(o.qf)]
    opp_g = [int(np.where((eg == -eg[i]).all(1))[0][0]) for i in range(o.qg)]
    fp, gp = inputs.random_state(o.shape, o.qf, o.qg, seed=5)
    o.set_post_collision(fp, gp)
    o.stream()
    f, g = o.get_populations()
    omega = o.params()["omega_bc"]
    ref_f = textbook_stream(fp, ef, opp_f, lambda i, a, idx, v: v)                      # Eq. 21

    def thermal(i, a, idx, v):
        if a == 0:                                                                     # Eq. 22
            return -v + omega * (0.5 if idx[0] == 0 else -0.5)
        return v                                                                       # Eq. 23

    ref_g = textbook_stream(gp, eg, opp_g, thermal)
    assert np.array_equal(f, ref_f)
    assert np.array_equal(g, ref_g)


# --------------------------------------------------------------------------
# P4  mass
# --------------------------------------------------------------------------

def test_P4_mass_conserved_on_uniform_mesh():
    o, _ = make(2, 32, mesh="uniform", Ra=1e5)
    o.init(0, 1e-3)
    m0 = o.mass()["plain"]
    o.step(1000)
    m1 = o.mass()["plain"]
    assert abs(m1 - m0) / m0 < 1e-13
    # the flow actually started (buoyancy acts): Re > 0
    assert o.nusselt()["Re"] > 1e-3


def test_P4_rest_state_keeps_mass_on_stretched_mesh():
    """Interpolated streaming is not conservative in general (reading A18), but a
    uniform rest state (T = 0, so no force) must stay exactly at rest."""
    o, _ = make(2, 24, stretch=1.6)
    o.init(0, 0.0)
    f0, g0 = o.get_populations()
    o.set_buoyancy_scale(0.0)
    o.step(50)
    f1, g1 = o.get_populations()
    assert np.abs(f1 - f0).max() < 1e-15


# --------------------------------------------------------------------------
# P5  conduction fixed point with buoyancy off (reading A19)
# --------------------------------------------------------------------------

def conduction_state(o, w):
    """u = 0, rho = 1, T linear between the walls; g_i = w_i T - (w_i/q_k) e_i.gradT."""
    ef, eg = o.velocities()
    p = o.params()
    qk = 3.0 - SQ3
    x = w.coords[0]
    xw = x[0] - w.delta / 2
    G_lu = -1.0 / (p["L_eff_x"] / w.delta)            # dT/dx per lattice unit
    T = 0.5 + G_lu * (x - xw) / w.delta
    wr = np.full(o.qg, p["omega_bc"] / 2)
    wr[0] = 1.0 - wr[1:].sum()
    wf = W9 if o.dim == 2 else W19
    f = np.empty((o.qf,) + o.shape)
    g = np.empty((o.qg,) + o.shape)
    for i in range(o.qf):
        f[i] = wf[i]
    for i in range(o.qg):
        g[i] = (wr[i] * T - wr[i] / qk * eg[i][0] * G_lu)[None, None, :]
    return f, g, T


@pytest.mark.parametrize("dim,n,steps", [(2, 32, 1000), (3, 12, 200)])
def test_P5_conduction_state_is_fixed_point_on_stretched_mesh(dim, n, steps):
    o, w = make(dim, n, stretch=1.5)
    o.set_buoyancy_scale(0.0)
    f0, g0, T = conduction_state(o, w)
    o.set_populations(f0, g0)
    o.step(steps)
    f1, g1 = o.get_populations()
    assert np.abs(f1 - f0).max() < 1e-13
    assert np.abs(g1 - g0).max() < 1e-13
    nu = o.nusselt()
    assert nu["Nu_hot"] == pytest.approx(1.0, abs=1e-11)
    assert nu["Nu_cold"] == pytest.approx(1.0, abs=1e-11)
    assert nu["Nu_vol"] == pytest.approx(1.0, abs=1e-12)
    assert nu["Re"] == pytest.approx(0.0, abs=1e-9)   # round-off velocity x sqrt(Ra/Pr)/U ~ 4e3
    assert np.allclose(o.fields()["T"][0, 0], T, atol=1e-13)


def test_P5b_thermal_diffusivity_from_decay_of_a_sine_mode():
    """Buoyancy off: T = conduction + A sin(pi (x - x_wall)/H) satisfies both
    Dirichlet walls and decays like exp(-alpha (pi/H)^2 t) — fixes alpha(q_kappa, a_T)."""
    o, w = make(2, 48, mesh="uniform", Ra=2e4)
    o.set_buoyancy_scale(0.0)
    p = o.params()
    f0, g0, T = conduction_state(o, w)
    H = p["H_lu"]
    xs = (w.coords[0] - (w.coords[0][0] - w.delta / 2)) / w.delta
    A = 1e-2
    mode = A * np.sin(math.pi * xs / H)
    wr = np.full(o.qg, p["omega_bc"] / 2)
    wr[0] = 1.0 - wr[1:].sum()
    g = g0 + wr[:, None, None, None] * mode[None, None, None, :]
    o.set_populations(f0, g)
    k2 = (math.pi / H) ** 2
    o.step(200)   # let the non-equilibrium part settle
    a1 = ((o.fields()["T"][0, 5] - T) * np.sin(math.pi * xs / H)).sum()
    nsteps = 1500
    o.step(nsteps)
    a2 = ((o.fields()["T"][0, 5] - T) * np.sin(math.pi * xs / H)).sum()
    alpha_measured = -math.log(a2 / a1) / (nsteps * k2)
    assert alpha_measured == pytest.approx(p["alpha"], rel=5e-3)


def test_P5c_viscosity_from_decay_of_a_shear_wave_away_from_walls():
    """Interior shear wave v(x) = A sin(kx): decays like exp(-nu k^2 t) until wall
    information (speed <= 1 node/step) reaches the probe — fixes nu(tau_f)."""
    n, lam = 96, 24
    o, w = make(2, n, mesh="uniform", Ra=3e4)
    o.set_buoyancy_scale(0.0)
    p, m = o.params(), o.matrices()
    k = 2 * math.pi / lam
    A = 1e-3
    ix = np.arange(n)
    f = np.empty((9, 1, n, n))
    g = np.zeros((5, 1, n, n))
    for i in range(n):
        f[:, 0, :, i] = (m["Minv"] @ o.meq(1.0, np.array([0.0, A * math.sin(k * ix[i]), 0.0])))[:, None]
    o.set_populations(f, g)
    rows = slice(n // 2 - 2, n // 2 + 2)
    cols = slice(n // 2 - lam, n // 2 + lam)           # two full wavelengths in the middle
    sinp = np.sin(k * ix[cols])
    o.step(4)
    a1 = (o.fields()["v"][0, rows, cols] * sinp).sum()
    nsteps = 16
    o.step(nsteps)
    a2 = (o.fields()["v"][0, rows, cols] * sinp).sum()
    nu_measured = -math.log(a2 / a1) / (nsteps * k * k)
    assert nu_measured == pytest.approx(p["nu"], rel=3e-2)


# --------------------------------------------------------------------------
# P6  wall derivative
# --------------------------------------------------------------------------

def test_P6_eq28_reduces_to_eq27_and_is_exact_on_quadratics(golden):
    c = golden["eq27_coeffs"]
    for which, coef in (("wall", (1, 0, 0)), ("first", (0, 1, 0)), ("second", (0, 0, 1))):
        assert wall_derivative(1.0, *coef) == pytest.approx(c[which] / c["denominator"], rel=1e-15)
    for q in (1.0, 1.37, 2.5):
        poly = lambda s: 0.4 - 1.3 * s + 0.8 * s * s        # s = distance from the wall in l.u.
        d = wall_derivative(q, poly(0.0), poly(0.5), poly(0.5 + q))
        assert d == pytest.approx(-1.3, abs=1e-13)


# --------------------------------------------------------------------------
# P7  brute force: one full step by an independent dense formulation
# --------------------------------------------------------------------------

# Literature matrices typed out (Lallemand & Luo D2Q9 in the velocity order
# 0,E,N,W,S,NE,NW,SW,SE; d'Humieres D3Q19 rows evaluated below from the typed
# velocity list) — a second, independent route to M.
M9_TYPED = np.array([
    [1, 1, 1, 1, 1, 1, 1, 1, 1],
    [-4, -1, -1, -1, -1, 2, 2, 2, 2],
    [4, -2, -2, -2, -2, 1, 1, 1, 1],
    [0, 1, 0, -1, 0, 1, -1, -1, 1],
    [0, -2, 0, 2, 0, 1, -1, -1, 1],
    [0, 0, 1, 0, -1, 1, 1, -1, -1],
    [0, 0, -2, 0, 2, 1, 1, -1, -1],
    [0, 1, -1, 1, -1, 0, 0, 0, 0],
    [0, 0, 0, 0, 0, 1, -1, 1, -1]], dtype=float)
N5_TYPED = np.array([
    [1, 1, 1, 1, 1],
    [0, 1, 0, -1, 0],
    [0, 0, 1, 0, -1],
    [-4, 1, 1, 1, 1],
    [0, 1, -1, 1, -1]], dtype=float)
E9 = np.array([(0, 0, 0), (1, 0, 0), (0, 1, 0), (-1, 0, 0), (0, -1, 0), (1, 1, 0), (-1, 1, 0), (-1, -1, 0), (1, -1, 0)])
E19 = np.array([(0, 0, 0), (1, 0, 0), (-1, 0, 0), (0, 1, 0), (0, -1, 0), (0, 0, 1), (0, 0, -1),
                (1, 1, 0), (-1, 1, 0), (1, -1, 0), (-1, -1, 0), (1, 0, 1), (-1, 0, 1), (1, 0, -1), (-1, 0, -1),
                (0, 1, 1), (0, -1, 1), (0, 1, -1), (0, -1, -1)])
N7_TYPED = np.array([
    [1, 1, 1, 1, 1, 1, 1],
    [0, 1, -1, 0, 0, 0, 0],
    [0, 0, 0, 1, -1, 0, 0],
    [0, 0, 0, 0, 0, 1, -1],
    [-6, 1, 1, 1, 1, 1, 1],
    [0, 2, 2, -1, -1, -1, -1],
    [0, 0, 0, 1, 1, -1, -1]], dtype=float)
# d'Humieres et al. (2002) D3Q19 rows for the axis (|c|^2=1) and diagonal (|c|^2=2) shells
M19_SHELL = {"e": (-30, -11, 8), "eps": (12, -4, 1), "q": (0, -4, 1), "pi": (0, -2, 1)}


def M19_typed():
    e = E19.astype(float)
    c2 = (e**2).sum(1)
    shell = c2.astype(int)
    rows = [np.ones(19),
            np.array([M19_SHELL["e"][s] for s in shell], float),
            np.array([M19_SHELL["eps"][s] for s in shell], float)]
    for a in range(3):
        rows.append(e[:, a])
        rows.append(np.array([M19_SHELL["q"][s] for s in shell]) * e[:, a])
    pxx = 3 * e[:, 0] ** 2 - c2
    pww = e[:, 1] ** 2 - e[:, 2] ** 2
    pi = np.array([M19_SHELL["pi"][s] for s in shell], float)
    rows += [pxx, pi * pxx, pww, pi * pww, e[:, 0] * e[:, 1], e[:, 1] * e[:, 2], e[:, 0] * e[:, 2],
             (e[:, 1] ** 2 - e[:, 2] ** 2) * e[:, 0], (e[:, 2] ** 2 - e[:, 0] ** 2) * e[:, 1], (e[:, 0] ** 2 - e[:, 1] ** 2) * e[:, 2]]
    return np.array(rows)


def brute_force_step(dim, coords, delta, Ra, Pr, Ma, f, g):
    """One collide + stream, dense matrices, generic inverse, polyfit interpolation."""
    e = (E9 if dim == 2 else E19).astype(int)
    qf, qg = len(e), (5 if dim == 2 else 7)
    M = M9_TYPED if dim == 2 else M19_typed()
    N = N5_TYPED if dim == 2 else N7_TYPED
    Mi, Ni = np.linalg.inv(M), np.linalg.inv(N)
    x = coords[0]
    n = len(x)
    H = (x[-1] - x[0] + delta) / delta
    U = Ma / SQ3
    nu = U * H * math.sqrt(Pr / Ra)
    alpha = nu / Pr
    gbeta = U * U / H
    tau = 3 * nu + 0.5
    sq = 8 * (2 * tau - 1) / (8 * tau - 1)
    qk, qe = 3 - SQ3, 4 * SQ3 - 6
    if dim == 2:
        aT = 20 * SQ3 * alpha - 4
        omega = (4 + aT) / 10
        S = np.diag([0, 1 / tau, 1 / tau, 0, sq, 0, sq, 1 / tau, 1 / tau])
        Qm = np.diag([0, qk, qk, qe, qe])
    else:
        aT = 42 * SQ3 * alpha - 6
        omega = (6 + aT) / 21
        S = np.diag([0, 1 / tau, 1 / tau, 0, sq, 0, sq, 0, sq] + [1 / tau] * 7 + [sq] * 3)
        Qm = np.diag([0, qk, qk, qk, qe, qe, qe])
    wts = W9 if dim == 2 else W19
    nz = f.shape[1]
    fp, gp = np.empty_like(f), np.empty_like(g)
    I = np.eye(qf)
    for iz in range(nz):
        for iy in range(n):
            for ix in range(n):
                fn, gn = f[:, iz, iy, ix], g[:, iz, iy, ix]
                T, rho = gn.sum(), fn.sum()
                F = np.array([0.0, rho * gbeta * T, 0.0])
                u = (e.T @ fn + F / 2) / rho
                feq = feq2(e.astype(float), wts, rho, u)                    # velocity-space equilibrium
                Fi = guo_force_velocity_space(e.astype(float), wts, u, F)   # velocity-space forcing
                fp[:, iz, iy, ix] = fn - Mi @ S @ M @ (fn - feq) + Mi @ (I - S / 2) @ M @ Fi
                neq = np.zeros(qg)
                neq[0] = T
                neq[1:dim + 1] = u[:dim] * T
                neq[dim + 1] = aT * T
                gp[:, iz, iy, ix] = gn - Ni @ Qm @ (N @ gn - neq)

    def pull(arr, i, ei, idx):
        # tensor-product parabola through the 3 nearest-in-index nodes per moving axis
        sl, pts = [], []
        for a in range(3):
            if a < dim and ei[a] != 0:
                b = min(max(idx[a] - 1, 0), n - 3)
                sl.append(range(b, b + 3))
                pts.append(x[idx[a]] - ei[a] * delta)
            else:
                sl.append([idx[a]])
                pts.append(None)
        vals = np.array([[[arr[i, kz, ky, kx] for kx in sl[0]] for ky in sl[1]] for kz in sl[2]])
        for a, axis_np in ((0, 2), (1, 1), (2, 0)):           # reduce x, then y, then z
            if pts[a] is None:
                vals = vals.take(0, axis=axis_np)
            else:
                xs = x[list(sl[a])]
                vals = np.apply_along_axis(lambda v: np.polyval(np.polyfit(xs - xs[1], v, 2), pts[a] - xs[1]), axis_np, vals)
            vals = np.expand_dims(vals, axis_np)
        return float(vals.reshape(()))

    def opposite(ei):
        return int(np.where((e == -ei).all(1))[0][0])

    fo, go = np.empty_like(f), np.empty_like(g)
    dims = (n, n, nz)
    for iz in range(nz):
        for iy in range(n):
            for ix in range(n):
                idx = (ix, iy, iz)
                for i in range(qf):
                    out = [a for a in range(dim) if (e[i][a] == 1 and idx[a] == 0) or (e[i][a] == -1 and idx[a] == dims[a] - 1)]
                    if out:
                        fo[i, iz, iy, ix] = fp[opposite(e[i]), iz, iy, ix]
                    else:
                        fo[i, iz, iy, ix] = pull(fp, i, e[i], idx)
                    if i < qg:
                        if out:
                            v = gp[opposite(e[i]), iz, iy, ix]
                            go[i, iz, iy, ix] = (-v + omega * (0.5 if ix == 0 else -0.5)) if out[0] == 0 else v
                        else:
                            go[i, iz, iy, ix] = pull(gp, i, e[i], idx)
    return fo, go


@pytest.mark.parametrize("dim,n", [(2, 5), (3, 4)])
def test_P7_brute_force_step_on_tiny_mesh(dim, n):
    o, w = make(dim, n, stretch=1.1, Ra=2e3)
    f, g = inputs.random_state(o.shape, o.qf, o.qg, seed=11, amp=0.05)
    o.set_populations(f, g)
    o.step(1)
    f1, g1 = o.get_populations()
    fb, gb = brute_force_step(dim, w.coords, w.delta, w.Ra, w.Pr, w.Ma, f, g)
    assert np.abs(f1 - fb).max() < 1e-13
    assert np.abs(g1 - gb).max() < 1e-13


def test_P7_typed_matrices_equal_polynomial_rows():
    o2, _ = make(2, 5)
    o3, _ = make(3, 4)
    assert np.array_equal(o2.matrices()["M"], M9_TYPED)
    assert np.array_equal(o2.matrices()["N"], N5_TYPED)
    assert np.array_equal(o3.matrices()["M"], M19_typed())
    assert np.array_equal(o3.matrices()["N"], N7_TYPED)
    assert np.array_equal(o2.velocities()[0], E9) and np.array_equal(o3.velocities()[0], E19)


# --------------------------------------------------------------------------
# P8 / P9  parameter map and paper-mode mesh
# --------------------------------------------------------------------------

def test_P8_unit_map(golden):
    y, d = inputs.erf_mesh(129, 1.5)
    o = Oracle([y, y], d, 1e6, 0.71, 0.1)
    p = o.params()
    # dt*/dx* = (U/H_lu) / (1/H_lu) = U = Ma c_s ~ 0.0577
    assert round(p["dt_star"] * p["H_lu"], 4) == golden["dt_over_dx_ma0p1"]["value"]
    assert p["U"] == pytest.approx(0.1 / SQ3, rel=1e-15)
    # Table 1: characteristic length (1/y1 - 1) l.u., effective height 1 - y1
    assert p["H_lu"] == pytest.approx(1.0 / d - 1.0, rel=1e-12)
    assert p["L_eff_y"] == pytest.approx(1.0 - d, rel=1e-12)
    # Ra and Pr recovered from the lattice-unit transport coefficients (Eq. 8)
    assert p["gbeta"] * p["H_lu"] ** 3 / (p["nu"] * p["alpha"]) == pytest.approx(1e6, rel=1e-12)
    assert p["nu"] / p["alpha"] == pytest.approx(0.71, rel=1e-14)
    # uniform mesh, Eq. 24-25: H = N l.u.
    xu, du = inputs.uniform_mesh(64)
    assert Oracle([xu, xu], du, 1e6, 0.71, 0.1).params()["H_lu"] == pytest.approx(64.0, rel=1e-13)


def test_P9_erf_mesh_quality_as_printed(golden):
    y = inputs.erf_points(513, 1.5)
    d = np.diff(y)
    growth = max((d[1:] / d[:-1]).max(), (d[:-1] / d[1:]).max())
    aspect = d.max() / d.min()
    gq = golden["mesh_quality_513_a1p5"]
    assert round(growth, 4) == gq["max_growth_rate"]
    assert round(aspect, 2) == gq["max_aspect_ratio"]
    assert y[0] == 0.0 and y[-1] == pytest.approx(1.0, abs=1e-15)


def test_bj_config_parameters_match_survey_table():
    """SURVEY.md section 8(a) table (derived there by an independent probe)."""
    expect = {"c1_64sq": (140.00, 0.037304, 0.61191, -2.17991), "c2_512sq": (1698.33, 0.045253, 0.63576, -1.79208),
              "c4_128cu": (416.10, 0.035061, 0.60518, -2.40764)}
    for name, (H, nu, tau, aT) in expect.items():
        w = inputs.workload(name)
        p = Oracle(w.coords, w.delta, w.Ra, w.Pr, w.Ma).params()
        assert p["H_lu"] == pytest.approx(H, abs=6e-3)
        assert p["nu"] == pytest.approx(nu, abs=6e-7)
        assert p["tau_f"] == pytest.approx(tau, abs=6e-6)
        assert p["a_T"] == pytest.approx(aT, abs=6e-6)
        assert p["U"] == pytest.approx(0.1, rel=1e-14)


# --------------------------------------------------------------------------
# init, step_node, threads, input validation
# --------------------------------------------------------------------------

def test_init_noise_follows_splitmix64(golden):
    o, _ = make(2, 8)
    amp = 1e-3
    o.init(0, amp)
    T = o.fields()["T"].ravel()
    for k, hx in enumerate(golden["splitmix64_seed0"]["outputs_hex"]):
        r = (int(hx, 16) >> 11) * 2.0**-53
        assert T[k] == pytest.approx(amp * (2 * r - 1), abs=1e-18)
    assert np.abs(T).max() <= amp and np.abs(T).max() > 0.5 * amp
    fl = o.fields()
    assert np.allclose(fl["rho"], 1.0, atol=1e-15) and np.abs(fl["u"]).max() == 0.0
    # buoyancy sign (reading A9): hot fluid rises -> v > 0 next to the hot wall after a few steps
    o.step(200)
    fl = o.fields()
    assert fl["v"][0, 2:-2, 0].mean() > 0 and fl["v"][0, 2:-2, -1].mean() < 0


@pytest.mark.parametrize("dim,n", [(2, 9), (3, 6)])
def test_step_node_equals_full_step(dim, n):
    o, _ = make(dim, n, stretch=1.4)
    f, g = inputs.random_state(o.shape, o.qf, o.qg, seed=3)
    o.set_populations(f, g)
    samples = [(ix, iy, iz) for ix in (0, 1, n // 2, n - 2, n - 1) for iy in (0, n // 2, n - 1)
               for iz in ((0, n // 2, n - 1) if dim == 3 else (0,))]
    pre = {s: o.step_node(*s) for s in samples}
    o.step(1)
    f1, g1 = o.get_populations()
    for (ix, iy, iz), (nf, ng) in pre.items():
        assert np.array_equal(nf, f1[:, iz, iy, ix]) and np.array_equal(ng, g1[:, iz, iy, ix])


def test_threads_are_bit_identical():
    o1, w = make(2, 40, stretch=1.7)
    o4 = Oracle(w.coords, w.delta, w.Ra, w.Pr, w.Ma, threads=4)
    for o in (o1, o4):
        o.init(7, 1e-3)
        o.step(25)
    a, b = o1.get_populations(), o4.get_populations()
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])


def test_create_rejects_bad_input():
    x, d = inputs.tanh_mesh(16, 1.2)
    with pytest.raises(ValueError):
        Oracle([x, x[::-1].copy()], d, 1e5, 0.71, 0.1)            # not increasing
    with pytest.raises(ValueError):
        Oracle([x, x], 2 * d, 1e5, 0.71, 0.1)                     # spacing < delta
    with pytest.raises(ValueError):
        Oracle([x[:2], x], d, 1e5, 0.71, 0.1)                     # n < 3


# ---------------------------------------------------------------------------
# Nu_middle, Eq. 33 (reading A23)
# ---------------------------------------------------------------------------
def _state_with(o, T_of_x, u0=0.0):
    """rest-weight flow populations carrying a uniform x-velocity u0, temperature populations w_i * T(x)."""
    ef, _ = o.velocities()
    o.init(0, 0.0)
    f0, _ = o.get_populations()
    w = f0[:, 0, 0, 0].copy()
    f = np.empty((o.qf,) + o.shape)
    for i in range(o.qf):
        f[i] = w[i] * (1.0 + 3.0 * ef[i][0] * u0)
    T = T_of_x(np.asarray(o.coords[0]))
    g = np.empty((o.qg,) + o.shape)
    wg = np.full(o.qg, o.params()["omega_bc"] / 2)
    wg[0] = 1 - wg[1:].sum()
    for i in range(o.qg):
        g[i] = (wg[i] * T)[None, None, :]
    return f, g


@pytest.mark.parametrize("dim,n", [(2, 21), (2, 20), (3, 9), (3, 8), (2, 3)])
def test_nu_middle_is_exact_on_quadratic_temperature_and_uniform_advection(dim, n):
    """Eq. 33 on states whose centre-plane flux has a closed form: T quadratic in x (the 3-point derivative and the
    linear interpolation between the bracketing columns are then exact, odd and even n), plus a uniform u0."""
    w = inputs.custom_workload("m", dim, n, stretch=1.3, Ra=2e4)
    o = Oracle(w.coords, w.delta, w.Ra, w.Pr, w.Ma)
    p = o.params()
    x = np.asarray(w.coords[0])
    xw = x[0] - w.delta / 2
    L = (x[-1] - x[0] + w.delta)
    xm = xw + L / 2
    a, b, c = 0.3, -0.8, (0.0 if n == 3 else 0.45)
    s = lambda xx: (xx - xw) / w.delta                       # lattice units from the hot wall
    Tq = lambda xx: a + b * s(xx) / p["H_lu"] + c * (s(xx) / p["H_lu"]) ** 2
    u0 = 0.01 * p["U"]
    f, g = _state_with(o, Tq, u0)
    o.set_populations(f, g)
    dTdxstar = b + 2 * c * s(xm) / p["H_lu"]                 # d T / d x*  with x* = x_lu / H_lu
    if n % 2 == 1:
        T_mid = Tq(xm)
    else:                                                    # linear interpolation of u*T between two columns
        i0 = n // 2 - 1
        a1 = (xm - x[i0]) / (x[i0 + 1] - x[i0])
        T_mid = (1 - a1) * Tq(x[i0]) + a1 * Tq(x[i0 + 1])
    expect = math.sqrt(w.Ra * w.Pr) * 0.01 * T_mid - dTdxstar
    assert o.nusselt_middle() == pytest.approx(expect, rel=1e-11, abs=1e-12)


def test_nu_middle_of_the_conduction_state_is_one():
    w = inputs.custom_workload("m", 2, 24, stretch=1.5, Ra=1e5)
    o = Oracle(w.coords, w.delta, w.Ra, w.Pr, w.Ma)
    p = o.params()
    x = np.asarray(w.coords[0])
    lin = lambda xx: 0.5 - ((xx - (x[0] - w.delta / 2)) / w.delta) / p["H_lu"]
    f, g = _state_with(o, lin)
    o.set_populations(f, g)
    assert o.nusselt_middle() == pytest.approx(1.0, abs=1e-12)


# ---------------------------------------------------------------------------
# A2 alternative: upwind stencil {j-2,j-1,j} / {j,j+1,j+2}
# ---------------------------------------------------------------------------
@pytest.mark.parametrize("dim", [2, 3])
def test_upwind_stencil_weights_bracket_the_departure_point_and_reproduce_quadratics(dim):
    o, w = make(dim, 17, stretch=1.8)
    o.set_stencil(1)
    for axis in range(dim):
        x = w.coords[axis]
        n = len(x)
        for c in (-1, 1):
            base, wt = o.weights(axis, c)
            for j in range(n):
                if (j == 0 and c == 1) or (j == n - 1 and c == -1):
                    continue
                want = min(max(j - 2 if c == 1 else j, 0), n - 3)
                assert base[j] == want
                xd = x[j] - c * w.delta
                xs = x[base[j]: base[j] + 3]
                assert xs[0] - 1e-15 <= xd <= xs[2] + 1e-15
                assert wt[j].sum() == pytest.approx(1.0, abs=1e-13)
                for poly in (lambda t: 1 + 0 * t, lambda t: t, lambda t: 3 * t * t - t + 0.5):
                    assert wt[j] @ poly(xs) == pytest.approx(float(poly(xd)), abs=1e-13)
    o.set_stencil(0)                                           # and back: the central tables are restored
    base, _ = o.weights(0, 1)
    assert list(base[:4]) == [0, 0, 1, 2]


@pytest.mark.parametrize("dim,n", [(2, 16), (3, 8)])
def test_upwind_stencil_on_uniform_mesh_is_textbook_streaming_bitwise(dim, n):
    o, w = make(dim, n, mesh="uniform")
    o.set_stencil(1)
    ef, eg = o.velocities()
    opp_f = [int(np.where((ef == -ef[i]).all(1))[0][0]) for i in range(o.qf)]
    fp, gp = inputs.random_state(o.shape, o.qf, o.qg, seed=6)
    o.set_post_collision(fp, gp)
    o.stream()
    f, _ = o.get_populations()
    assert np.array_equal(f, textbook_stream(fp, ef, opp_f, lambda i, a, idx, v: v))


def test_upwind_and_central_stencils_differ_on_a_stretched_mesh_but_share_the_conduction_fixed_point():
    w = inputs.custom_workload("s", 2, 24, stretch=1.5, Ra=1e5)
    res = []
    for kind in (0, 1):
        o = Oracle(w.coords, w.delta, w.Ra, w.Pr, w.Ma)
        o.set_stencil(kind)
        o.init(0, 1e-3)
        o.step(50)
        res.append(o.fields()["T"].copy())
    assert 1e-9 < np.abs(res[0] - res[1]).max() < 1e-2


# ---------------------------------------------------------------------------
# normalisation of <Re>, <u*^2>_V and <Nu> (Eq. 31, 34)
# ---------------------------------------------------------------------------
@pytest.mark.parametrize("dim,n", [(2, 14), (3, 7)])
def test_volume_diagnostics_closed_forms_for_uniform_velocity(dim, n):
    """Uniform velocity (u0, v0[, w0]), buoyancy off, T = c + (antisymmetric about the cavity centre): the Eq. 29
    weights are symmetric and sum to L_eff, so <Re> = sqrt(Ra/Pr)|u0|/U, <u*^2> = |u0|^2/U^2 and
    <Nu> = 1 + sqrt(Ra Pr) (u0/U) c, whatever the stretching."""
    w = inputs.custom_workload("d", dim, n, stretch=1.6, Ra=3e4)
    o = Oracle(w.coords, w.delta, w.Ra, w.Pr, w.Ma)
    o.set_buoyancy_scale(0.0)
    p = o.params()
    ef, _ = o.velocities()
    o.init(0, 0.0)
    f0, _ = o.get_populations()
    wts = f0[:, 0, 0, 0].copy()
    u0 = np.array([0.013, -0.007, 0.004])[:dim] * p["U"]
    f = np.empty((o.qf,) + o.shape)
    for i in range(o.qf):
        eu = float(ef[i][:dim] @ u0)
        f[i] = wts[i] * (1.0 + 3.0 * eu + 4.5 * eu * eu - 1.5 * float(u0 @ u0))     # second-order equilibrium: sum e f = rho u0
    x = np.asarray(w.coords[0])
    xc = 0.5 * (x[0] + x[-1])
    c = 0.21
    T = c + 0.4 * np.sin(3.0 * (x - xc)) + 0.1 * (x - xc) ** 3                      # c + odd function of (x - centre)
    wg = np.full(o.qg, p["omega_bc"] / 2)
    wg[0] = 1 - wg[1:].sum()
    g = np.empty((o.qg,) + o.shape)
    for i in range(o.qg):
        g[i] = (wg[i] * T)[None, None, :]
    o.set_populations(f, g)
    fl = o.fields()
    assert np.abs(fl["u"] - u0[0]).max() < 1e-15 and np.abs(fl["rho"] - 1).max() < 1e-14
    d = o.nusselt()
    speed = float(np.linalg.norm(u0))
    assert d["Re"] == pytest.approx(math.sqrt(w.Ra / w.Pr) * speed / p["U"], rel=1e-12)
    assert d["u2"] == pytest.approx(speed ** 2 / p["U"] ** 2, rel=1e-12)
    assert d["Nu_vol"] == pytest.approx(1.0 + math.sqrt(w.Ra * w.Pr) * (u0[0] / p["U"]) * c, rel=1e-11)


# ---------------------------------------------------------------------------
# Eq. 28 with q != 1 INSIDE oracle_nusselt (q = second / first mesh spacing > 1)
# ---------------------------------------------------------------------------
def _q_mesh(kind, dim):
    """(coords, delta, Ma): the paper's own mesh (Eq. 26, a = 1.5, 257 points in 2-D / 65 in 3-D, delta = y_1: q = 1.009 /
    1.036) or the hand-made mesh with q = 2.5 at the hot wall and 1.75 at the cold wall."""
    if kind == "erf":
        x, d = inputs.erf_mesh(257 if dim == 2 else 65, 1.5)
        return [x.copy() for _ in range(dim)], d, 0.1
    x, d = inputs.wallgap_mesh(24 if dim == 2 else 14)
    return [x.copy() for _ in range(dim)], d, 0.1 * SQ3


@pytest.mark.parametrize("kind,dim", [("erf", 2), ("wallgap", 2), ("erf", 3), ("wallgap", 3)])
def test_P6b_wall_nusselt_of_the_conduction_state_is_one_for_q_not_one(kind, dim):
    """The conduction profile is linear in x, and Eq. 28 is exact on it for ANY q (it is the wall derivative of the
    parabola through the wall value, node 1 at 0.5 l.u. and node 2 at 0.5 + q l.u.), so Nu_hot = Nu_cold = 1 to
    round-off through oracle_nusselt exactly when q_lo and q_hi are the right spacing ratios at the right walls.
    The meshes have q != 1 (every other Nu test runs on tanh meshes, where q = 1 and Eq. 28 is Eq. 27), and the
    hand-made one has different q at the two walls, so an inverted ratio, a wrong spacing or a swapped pair fails:
    the test also shows by how much."""
    coords, delta, Ma = _q_mesh(kind, dim)
    o = Oracle(coords, delta, 1e5, 0.71, Ma, threads=4)
    o.set_buoyancy_scale(0.0)
    x = coords[0]
    q_lo, q_hi = (x[1] - x[0]) / delta, (x[-1] - x[-2]) / delta
    assert q_lo > 1.005 and q_hi > 1.005
    if kind == "wallgap":
        assert q_lo == pytest.approx(2.5, rel=1e-12) and q_hi == pytest.approx(1.75, rel=1e-12)

    class W:                      # what conduction_state reads
        pass
    w = W()
    w.coords, w.delta = coords, delta
    f0, g0, T = conduction_state(o, w)
    o.set_populations(f0, g0)
    o.step(20)                    # still the fixed point (P5) on these meshes
    f1, g1 = o.get_populations()
    assert np.abs(f1 - f0).max() < 1e-13 and np.abs(g1 - g0).max() < 1e-13
    nu = o.nusselt()
    assert nu["Nu_hot"] == pytest.approx(1.0, abs=1e-11)
    assert nu["Nu_cold"] == pytest.approx(1.0, abs=1e-11)
    assert o.nusselt_middle() == pytest.approx(1.0, abs=1e-11)
    # what a plausible mistake would give on this state (closed form of Eq. 28 on a linear profile: the slope comes
    # out multiplied by (2 q'^2 + 2 q' - q) / (q' (2 q' + 1)) when q' is used instead of the true q)
    wrong = lambda qp, q: (2 * qp * qp + 2 * qp - q) / (qp * (2 * qp + 1))
    for qp, q in ((1.0, q_lo), (1.0 / q_lo, q_lo), (q_hi if kind == "wallgap" else 1.0, q_lo)):
        assert abs(wrong(qp, q) - 1.0) > 1e-3
    assert wrong(q_lo, q_lo) == pytest.approx(1.0, abs=1e-15)


def test_P6c_eq28_inside_nusselt_matches_the_parabola_through_wall_and_two_nodes():
    """A curved profile: T quadratic in x, buoyancy off, on the hand-made mesh.  The expected Nu_hot / Nu_cold are the
    wall derivatives of the quadratic itself (closed form), which Eq. 28 reproduces exactly only with the right q."""
    coords, delta, Ma = _q_mesh("wallgap", 2)
    o = Oracle(coords, delta, 1e5, 0.71, Ma)
    p = o.params()
    x = np.asarray(coords[0])
    s = lambda xx: (xx - (x[0] - delta / 2)) / delta / p["H_lu"]       # x* from the hot wall, in [0, 1]
    a, b, c = 0.5, -1.7, 0.7                                           # T(0) = T_hot = 0.5, T(1) = T_cold = -0.5
    f, g = _state_with(o, lambda xx: a + b * s(xx) + c * s(xx) ** 2)
    o.set_populations(f, g)
    nu = o.nusselt()
    assert nu["Nu_hot"] == pytest.approx(-b, rel=1e-11)                # -dT/dx* at x* = 0
    assert nu["Nu_cold"] == pytest.approx(-(b + 2 * c), rel=1e-11)     # -dT/dx* at x* = 1
