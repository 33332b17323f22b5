"""Pins of the CPU oracle against what the paper and the mathematics fix.

None of these compares the oracle with itself or with the CUDA path: they use
hand-derived shell sums (tests/golden), brute force written in numpy, closed
forms (Laplacian of a quadratic, gradient of a linear field), invariants
(symmetry, momentum conservation), a dense LAPACK solve and the hydrostatic
law rho*g*h.  Pin numbers T1..T12 follow SURVEY.md 8(c).4 / DESIGN.md section 4.
"""
import math
import os

import numpy as np
import pytest

from oracle import mps_oracle as O
from paper_2105_01677_b200 import scenes

GOLD = {}
with open(os.path.join(os.path.dirname(__file__), "golden", "lattice_constants.txt")) as _f:
    for _ln in _f:
        _k, _v = _ln.split("#")[0].split()
        GOLD[_k] = float(_v)

L0 = 0.01


def brute_sets_numpy(x, y, z, valid, re):
    """O(N^2) definition of the neighbour set with reading Q2's rounding."""
    dx = x[None, :] - x[:, None]
    dy = y[None, :] - y[:, None]
    dz = z[None, :] - z[:, None]
    r2 = (dx * dx + dy * dy) + dz * dz
    m = r2 < re * re
    np.fill_diagonal(m, False)
    m &= valid[None, :] & valid[:, None]
    return m


def csr_to_mask(counts, idx, n):
    m = np.zeros((n, n), bool)
    rows = np.repeat(np.arange(n), counts)
    m[rows, idx] = True
    return m


# ---- T1: neighbour sets ----------------------------------------------------
@pytest.mark.parametrize("kind", ["lattice7", "cloud", "tank"])
@pytest.mark.parametrize("cell_div", [1, 2])
def test_T1_neighbour_sets_equal_numpy_brute_force(kind, cell_div):
    if kind == "lattice7":
        s = scenes.fluid_blob(L0, (7, 7, 7))
    elif kind == "cloud":
        s = scenes.random_cloud(2000, 10 * 3.1 * L0, seed=3)
        s.params["l0"] = L0
        s.params["re_n"], s.params["re_lap"] = 2.1 * L0, 3.1 * L0
    else:
        s = scenes.small_tank(shuffle=True)
    o = O.Oracle(s, cell_div=cell_div)
    for re in (s.params["re_n"], s.params["re_lap"]):
        cnt, idx = o.neighbours(re)
        valid = o.get("type") != scenes.GHOST
        ref = brute_sets_numpy(s.x, s.y, s.z, valid, re)
        got = csr_to_mask(cnt, idx, s.n)
        assert (ref == got).all()
        assert cnt.max() <= 300
        # rows ascending
        rows = np.repeat(np.arange(s.n), cnt)
        same_row = rows[1:] == rows[:-1]
        assert (np.diff(idx)[same_row] > 0).all()


def test_T1_grid_equals_oracle_brute_on_config1():
    s = scenes.make_scene(1)
    a = O.Oracle(s)
    b = O.Oracle(s, brute=True)
    sub = None
    for re in (s.params["re_n"], s.params["re_lap"]):
        ca, ia = a.neighbours(re)
        cb, ib = b.neighbours(re)
        assert (ca == cb).all() and (ia == ib).all()


# ---- T2: n0, lambda ---------------------------------------------------------
@pytest.mark.parametrize("dim,tag", [(3, "3d"), (2, "2d")])
@pytest.mark.parametrize("re", [2.1, 3.1])
@pytest.mark.parametrize("l0", [0.01, 0.005, 0.004])
def test_T2_lattice_constants(dim, tag, re, l0):
    n0, lam, cnt = O.lattice_constants(dim, l0, re * l0)
    assert cnt == int(GOLD[f"count_{tag}_{re}"])
    assert n0 == pytest.approx(GOLD[f"n0_{tag}_{re}"], rel=1e-13)
    assert lam / (l0 * l0) == pytest.approx(GOLD[f"lambda_{tag}_{re}"], rel=1e-13)


def test_T2_survey_printed_values():
    # the values SURVEY.md 8(c).4 T2 prints
    assert GOLD["n0_3d_2.1"] == pytest.approx(14.4185754082867, rel=1e-13)
    assert GOLD["n0_3d_3.1"] == pytest.approx(54.3212093818204, rel=1e-13)
    assert GOLD["lambda_3d_3.1"] == pytest.approx(3.24342167603806, rel=1e-13)


# ---- T3: density on an un-jittered block ------------------------------------
def test_T3_block_density_values():
    m = 7
    s = scenes.fluid_blob(L0, (m, m, m))
    o = O.Oracle(s)
    o.density()
    n = o.get("n").reshape(m, m, m)  # z, y, x
    n0 = GOLD["n0_3d_2.1"]
    core = n[2:-2, 2:-2, 2:-2]
    assert np.allclose(core, n0, rtol=1e-13, atol=0)
    assert n[1, 3, 3] == pytest.approx(GOLD["n_depth1_3d_2.1"], rel=1e-13)
    assert n[3, 3, 1] == pytest.approx(GOLD["n_depth1_3d_2.1"], rel=1e-13)
    assert n[0, 3, 3] == pytest.approx(GOLD["n_face_3d_2.1"], rel=1e-13)
    assert n[3, 0, 3] == pytest.approx(GOLD["n_face_3d_2.1"], rel=1e-13)
    assert o.stats()["max_nb"] == 32


# ---- T4: free-surface flags --------------------------------------------------
@pytest.mark.parametrize("m", [5, 8])
def test_T4_free_surface_is_outer_shell(m):
    s = scenes.fluid_blob(L0, (m, m, m))
    o = O.Oracle(s)
    o.density()
    o.ppe_flags()
    bc = o.get("bc").reshape(m, m, m)
    inner = np.zeros((m, m, m), bool)
    inner[1:-1, 1:-1, 1:-1] = True
    assert (bc[inner] == 0).all()
    assert (bc[~inner] == 1).all()
    assert o.stats()["n_surface"] == m ** 3 - (m - 2) ** 3


def test_T4_dummy_and_beta_threshold():
    s = scenes.small_tank(jitter=0.0)
    o = O.Oracle(s)
    o.density()
    o.ppe_flags()
    bc, ty, n = o.get("bc"), o.get("type"), o.get("n")
    assert (bc[ty == scenes.DUMMY] == -1).all()
    nd = ty != scenes.DUMMY
    assert ((bc[nd] == 1) == (n[nd] < 0.97 * GOLD["n0_3d_2.1"])).all()
    # a wall particle under the fluid has a full neighbourhood -> not surface (Q3)
    under = nd & (ty == scenes.WALL) & (s.z < 0) & (s.x > 2 * L0) & (s.x < 4 * L0) \
        & (s.y > 2 * L0) & (s.y < 4 * L0)
    assert under.any() and (bc[under] == 0).all()


# ---- T5: Laplacian of a quadratic --------------------------------------------
def _interior_mask(s, m, margin):
    ix = np.rint(s.x / L0 - 0.5).astype(int)
    iy = np.rint(s.y / L0 - 0.5).astype(int)
    iz = np.rint(s.z / L0 - 0.5).astype(int)
    ok = np.ones(s.n, bool)
    for a in (ix, iy, iz):
        ok &= (a >= margin) & (a < m - margin)
    return ok


def test_T5_laplacian_of_quadratic_and_linear():
    m = 10
    s = scenes.fluid_blob(L0, (m, m, m))
    a = np.array([1.3, -0.7, 2.9])
    b = np.array([0.4, 5.0, -1.1])
    phi = a[0] * s.x ** 2 + a[1] * s.y ** 2 + a[2] * s.z ** 2 + b[0] * s.x + b[1] * s.y + b[2] * s.z + 3.0
    lin = b[0] * s.x + b[1] * s.y + b[2] * s.z + 3.0
    o = O.Oracle(s, nu=(1.0, 1.0), g=(0.0, 0.0, 0.0))
    o.set("u", phi)
    o.set("v", lin)
    o.viscosity()
    core = _interior_mask(s, m, 4)
    assert core.sum() == 8
    lap = o.get("ax")[core]
    assert np.allclose(lap, 2 * a.sum(), rtol=1e-11)
    assert np.abs(o.get("ay")[core]).max() < 1e-9 * np.abs(lin).max() / L0 ** 2 * 1e-3
    # gravity is added as is
    o2 = O.Oracle(s, nu=(0.0, 0.0))
    o2.viscosity()
    assert (o2.get("az") == -9.81).all() and (o2.get("ax") == 0).all()


# ---- T6: gradient of a linear field -------------------------------------------
@pytest.mark.parametrize("variant,expect", [(0, 1.0), (1, 0.0), (2, 1.0)])
def test_T6_gradient_of_linear_field(variant, expect):
    m = 9
    s = scenes.fluid_blob(L0, (m, m, m))
    g = np.array([700.0, -300.0, 9810.0])
    p = g[0] * s.x + g[1] * s.y + g[2] * s.z + 50.0
    o = O.Oracle(s, grad_variant=variant)
    o.set("p", p)
    o.phat()
    o.gradient()
    core = _interior_mask(s, m, 4)  # needs phat_j of neighbours to be interior too
    G = np.stack([o.get("gx"), o.get("gy"), o.get("gz")], 1)[core]
    if variant == 0:
        # (p_j - phat_i): the constant phat_i cancels on a symmetric lattice
        assert np.allclose(G, g[None, :], rtol=1e-11)
    elif variant == 2:
        # (p_i + p_j): the constant p_i cancels on a symmetric lattice
        assert np.allclose(G, g[None, :], rtol=1e-11)
    else:
        # Eq. 14 as printed: hat terms cancel the linear part (Q13)
        assert np.abs(G).max() < 1e-9 * np.abs(g).max()
    # phat is the minimum over the closed r_n ball
    ph = o.get("phat")
    i = int(np.nonzero(core)[0][0])
    d2 = (s.x - s.x[i]) ** 2 + (s.y - s.y[i]) ** 2 + (s.z - s.z[i]) ** 2
    assert ph[i] == p[d2 < (2.1 * L0) ** 2].min()


# ---- T7: equation of state ----------------------------------------------------
def test_T7_equation_of_state():
    n0 = GOLD["n0_3d_2.1"]
    assert O.eos(1000.0, 10.0, 7.0, n0, n0) == 0.0
    assert O.eos(1000.0, 10.0, 7.0, 1.01 * n0, n0) == pytest.approx(GOLD["eos_1.01"], rel=1e-13)
    assert GOLD["eos_1.01"] == pytest.approx(1030.5050301001, rel=1e-12)
    # general-gamma branch agrees with the gamma = 7 product form, and is monotone
    assert O.eos(1000.0, 10.0, 7.0 + 1e-13, 1.01 * n0, n0) == pytest.approx(GOLD["eos_1.01"], rel=1e-11)
    v = [O.eos(800.0, 10.0, 7.0, q * n0, n0) for q in (0.9, 0.99, 1.0, 1.02, 1.1)]
    assert all(b > a for a, b in zip(v, v[1:]))
    s = scenes.small_tank()
    o = O.Oracle(s)
    o.density()
    o.pressure_explicit()
    p, ty = o.get("p"), o.get("type")
    assert (p >= 0).all() and (p[ty == scenes.DUMMY] == 0).all()
    o2 = O.Oracle(s, clamp_negative_p=0)
    o2.density()
    o2.pressure_explicit()
    assert o2.get("p").min() < 0  # free-surface particles have n < n0


# ---- T8: PPE operator invariants ----------------------------------------------
def _moved_tank():
    s = scenes.small_tank(shuffle=True)
    o = O.Oracle(s)
    o.step(2, 0)  # two explicit steps so that the particles are off-lattice
    o.viscosity(); o.predict(); o.density(); o.ppe_flags(); o.ppe_rhs()
    return s, o


def test_T8_operator_symmetric_positive_rowsum():
    s, o = _moved_tank()
    bc = o.get("bc")
    rows = bc == 0
    rng = np.random.default_rng(0)
    x = np.where(rows, rng.standard_normal(s.n), 0.0)
    y = np.where(rows, rng.standard_normal(s.n), 0.0)
    Ax, Ay = o.ppe_apply(x), o.ppe_apply(y)
    assert (Ax[~rows] == 0).all()
    assert x @ Ay == pytest.approx(Ax @ y, rel=1e-11)
    assert x @ Ax > 0 and y @ Ay > 0
    # row sums: A.1 = compress/dt^2 + sum over surface neighbours of c_ij
    one = np.where(rows, 1.0, 0.0)
    A1 = o.ppe_apply(one)
    c = o.constants()
    dt, re = s.params["dt"], s.params["re_lap"]
    X, Y, Z = o.get("x"), o.get("y"), o.get("z")
    valid = o.get("type") != scenes.GHOST
    m = brute_sets_numpy(X, Y, Z, valid, re)
    r = np.sqrt((X[None] - X[:, None]) ** 2 + (Y[None] - Y[:, None]) ** 2 + (Z[None] - Z[:, None]) ** 2)
    with np.errstate(divide="ignore"):
        cij = np.where(m, c["A_lap"] * (re / r - 1.0) / 1000.0, 0.0)
    expect = 1e-7 / dt ** 2 + (cij * (bc[None, :] == 1)).sum(1)
    assert np.allclose(A1[rows], expect[rows], rtol=1e-11)
    # points of the domain far from any surface: pure compress term
    deep = rows & ((cij * (bc[None, :] == 1)).sum(1) == 0)
    assert deep.any()
    assert np.allclose(A1[deep], 1e-7 / dt ** 2, rtol=1e-9)


# ---- T9: CG against a dense solve ---------------------------------------------
def _dense_A(o, s, rho_pair=None):
    """Assemble A per Listing 2: -val off-diagonal, +val and
    +1e-7/dt^2 on the diagonal, dummies skipped, surface columns dropped."""
    c = o.constants()
    bc = o.get("bc")
    X, Y, Z = o.get("x"), o.get("y"), o.get("z")
    re, dt = s.params["re_lap"], s.params["dt"]
    valid = o.get("type") != scenes.GHOST
    m = brute_sets_numpy(X, Y, Z, valid, re)
    r = np.sqrt((X[None] - X[:, None]) ** 2 + (Y[None] - Y[:, None]) ** 2 + (Z[None] - Z[:, None]) ** 2)
    if rho_pair is None:
        rho_pair = 1000.0
    with np.errstate(divide="ignore", invalid="ignore"):
        val = np.where(m & (bc[None, :] != -1), c["A_lap"] * (re / r - 1.0) / rho_pair, 0.0)
    rows = np.nonzero(bc == 0)[0]
    A = -val[np.ix_(rows, rows)]
    A[np.arange(rows.size), np.arange(rows.size)] = val[rows].sum(1) + o.params["compress"] / dt ** 2
    return A, rows


@pytest.mark.parametrize("compress", [1e-7, 0.0])
def test_T9_cg_equals_dense_solve(compress):
    s = scenes.small_tank(shuffle=True)
    o = O.Oracle(s, compress=compress)
    o.step(2, 0)
    o.viscosity(); o.predict(); o.density(); o.ppe_flags(); o.ppe_rhs()
    A, rows = _dense_A(o, s)
    assert 100 < rows.size <= 1200
    assert np.allclose(A, A.T, rtol=1e-12)
    b = o.get("b")[rows]
    xd = np.linalg.solve(A, b)
    it = o.ppe_solve(1e-12, 5000)
    assert it > 0
    xc = o.get("xcg")[rows]
    assert np.linalg.norm(xc - xd) <= 1e-9 * np.linalg.norm(xd)
    # operator == dense matrix
    rng = np.random.default_rng(1)
    v = np.zeros(s.n); v[rows] = rng.standard_normal(rows.size)
    assert np.allclose(o.ppe_apply(v)[rows], A @ v[rows], rtol=1e-10, atol=1e-10 * np.abs(A @ v[rows]).max())
    # default tolerance: relative residual as stated (Q15)
    it2 = o.ppe_solve(1e-8, 5000)
    x8 = o.get("xcg")[rows]
    assert np.linalg.norm(b - A @ x8) <= 1.5e-8 * np.linalg.norm(b)
    assert 0 < it2 <= it


def test_T9_two_phase_operator_matches_dense():
    s = scenes.small_tank(shuffle=True)
    s.phase[(s.z > 0.03)] = 1
    o = O.Oracle(s, n_phases=2, rho=(1000.0, 800.0))
    o.density(); o.ppe_flags(); o.ppe_rhs()
    rho = np.where(s.phase == 1, 800.0, 1000.0)
    A, rows = _dense_A(o, s, rho_pair=0.5 * (rho[None, :] + rho[:, None]))
    v = np.zeros(s.n); v[rows] = np.random.default_rng(2).standard_normal(rows.size)
    assert np.allclose(o.ppe_apply(v)[rows], A @ v[rows], rtol=1e-10, atol=1e-10 * np.abs(A @ v[rows]).max())
    oh = O.Oracle(s, n_phases=2, rho=(1000.0, 800.0), rho_pair_mean=1)
    oh.density(); oh.ppe_flags()
    Ah, _ = _dense_A(oh, s, rho_pair=2 * rho[None, :] * rho[:, None] / (rho[None, :] + rho[:, None]))
    assert np.allclose(oh.ppe_apply(v)[rows], Ah @ v[rows], rtol=1e-10, atol=1e-10 * np.abs(Ah @ v[rows]).max())


# ---- T10: momentum conservation -------------------------------------------------
@pytest.mark.parametrize("variant", [1, 2])
def test_T10_antisymmetric_gradient_conserves_momentum(variant):
    s = scenes.fluid_blob(L0, (6, 5, 7), seed=5, jitter=0.2)
    rng = np.random.default_rng(4)
    o = O.Oracle(s, grad_variant=variant)
    o.set("p", rng.uniform(0, 1000.0, s.n))
    o.phat(); o.gradient()
    G = np.stack([o.get("gx"), o.get("gy"), o.get("gz")], 1)
    assert np.abs(G.sum(0)).max() <= 1e-12 * np.linalg.norm(G, axis=1).sum()
    o0 = O.Oracle(s, grad_variant=0)
    o0.set("p", o.get("p")); o0.phat(); o0.gradient()
    G0 = np.stack([o0.get("gx"), o0.get("gy"), o0.get("gz")], 1)
    assert np.abs(G0.sum(0)).max() > 1e-6 * np.linalg.norm(G0, axis=1).sum()  # variant 0 is not


# ---- T12: stable sort invariants --------------------------------------------------
@pytest.mark.parametrize("cell_div", [1, 2, 3])
def test_T12_sort_invariants(cell_div):
    s = scenes.small_tank(shuffle=True)
    s.x[5] = 10.0  # one particle outside the domain -> GHOST
    o = O.Oracle(s, cell_div=cell_div)
    key, perm, cs = o.bin()
    nx, ny, nz, ncells = o.grid()
    assert sorted(perm.tolist()) == list(range(s.n))
    ks = key[perm]
    assert (np.diff(ks) >= 0).all()
    eq = np.diff(ks) == 0
    assert (np.diff(perm)[eq] > 0).all()
    assert key[5] == ncells and o.get("type")[5] == scenes.GHOST and perm[-1] == 5
    assert cs[0] == 0 and cs[-1] == s.n - 1 and (np.diff(cs) >= 0).all()
    assert (cs == np.searchsorted(ks, np.arange(ncells + 1), side="left")).all()
    # the key itself: independent restatement with numpy floor
    c = o.constants()
    dmin = s.params["domain_min"]
    ci = [np.floor((a - m) * c["inv_h"]).astype(np.int64) for a, m in zip((s.x, s.y, s.z), dmin)]
    k2 = ci[0] + nx * (ci[1] + ny * ci[2])
    ok = np.arange(s.n) != 5
    assert (key[ok] == k2[ok]).all()
    assert c["h"] == max(s.params["re_n"], s.params["re_lap"]) / cell_div
    ext = [hi - lo for lo, hi in zip(dmin, s.params["domain_max"])]
    assert [nx, ny, nz] == [math.ceil(e * c["inv_h"]) for e in ext]


# ---- Smagorinsky: simple shear ------------------------------------------------------
def test_smagorinsky_simple_shear():
    m = 9
    s = scenes.fluid_blob(L0, (m, m, m))
    gdot = 3.5
    o = O.Oracle(s, cs=0.12)
    o.set("u", gdot * s.y)
    o.viscosity()
    core = _interior_mask(s, m, 3)
    nut = o.get("nut")[core]
    assert np.allclose(nut, (0.12 * L0) ** 2 * gdot, rtol=1e-11)
    # rigid rotation has no strain
    o.set("u", -2.0 * s.y); o.set("v", 2.0 * s.x)
    o.viscosity()
    assert np.abs(o.get("nut")[core]).max() < 1e-12 * (0.12 * L0) ** 2 * 2.0 * 1e3


# ---- predictor / corrector arithmetic -------------------------------------------------
def test_predictor_corrector_closed_form():
    s = scenes.small_tank()
    o = O.Oracle(s)
    rng = np.random.default_rng(9)
    fl = s.type == scenes.FLUID
    u0 = np.where(fl, rng.standard_normal(s.n), 0.0)
    ax = rng.standard_normal(s.n)
    o.set("u", u0); o.set("ax", ax)
    dt = s.params["dt"]
    o.predict()
    us = o.get("u")
    assert np.array_equal(us[fl], (u0 + dt * ax)[fl]) and np.array_equal(us[~fl], u0[~fl])
    assert np.array_equal(o.get("x")[fl], (s.x + dt * us)[fl]) and np.array_equal(o.get("x")[~fl], s.x[~fl])
    gx = rng.standard_normal(s.n) * 1e4
    o.set("gx", gx)
    xs = o.get("x")
    o.correct()
    un = o.get("u")
    assert np.allclose(un[fl], (us - dt / 1000.0 * gx)[fl], rtol=1e-14)
    assert np.allclose(o.get("x")[fl], (xs + dt * (un - us))[fl], rtol=1e-15)
    assert np.array_equal(o.get("x")[~fl], s.x[~fl]) and (un[~fl] == 0).all()


# ---- T11: hydrostatic pressure rho*g*h -------------------------------------------------
# Loose physics-sanity pins (north_star: "hydrostatic pressure rho*g*h in a resting
# tank").  On the un-jittered lattice the layer one spacing below the surface starts
# with n = n0 - 0.05 (T3), a negative source that dominates the first steps; the column
# settles by a fraction of l0 and then carries the hydrostatic gradient, with the usual
# MPS pressure noise.  Measured with this oracle: slope/(rho g) = 1.03-1.11 over steps
# 20-200 (PPE), bottom-layer mean ringing around 1.1 rho g H at period ~4H/c0 (EoS).
def _hydro(route, nsteps, avg_from):
    depth = 8
    s = scenes.hydrostatic_tank(L0, foot=(10, 10), depth=depth, height=11)
    o = O.Oracle(s)
    fl = s.type == scenes.FLUID
    H = depth * L0
    slopes, bottoms = [], []
    for k in range(1, nsteps + 1):
        o.step(1, route)
        if k > avg_from:
            p, z = o.get("p"), o.get("z")
            d = H - z
            sel = fl & (d > 2 * L0)
            slopes.append(np.polyfit(d[sel], p[sel], 1)[0])
            bottoms.append(p[fl & (s.z < L0)].mean())
    assert o.stats()["n_ghost"] == 0
    return np.mean(slopes), np.mean(bottoms), H


def test_T11_hydrostatic_ppe():
    slope, bottom, H = _hydro(route=1, nsteps=60, avg_from=30)
    rg = 1000.0 * 9.81
    assert slope == pytest.approx(rg, rel=0.15)
    assert bottom == pytest.approx(rg * (H - L0), rel=0.25)


def test_T11_hydrostatic_explicit():
    slope, bottom, H = _hydro(route=0, nsteps=400, avg_from=200)
    rg = 1000.0 * 9.81
    assert slope == pytest.approx(rg, rel=0.20)
    assert bottom == pytest.approx(rg * H, rel=0.20)


# ---- NEXT-1: higher-order source (HS, Eq. 15), higher-order Laplacian (HL, Eq. 16), ECS ----
def _numpy_dndt(x, y, z, u, v, w, re):
    """Brute force: Dn/Dt_i = d/dt sum_j (re/r_ij - 1) = -sum_j re/r^3 (x_ij . u_ij)."""
    dx = x[None, :] - x[:, None]; dy = y[None, :] - y[:, None]; dz = z[None, :] - z[:, None]
    du = u[None, :] - u[:, None]; dv = v[None, :] - v[:, None]; dw = w[None, :] - w[:, None]
    r2 = (dx * dx + dy * dy) + dz * dz
    m = r2 < re * re
    np.fill_diagonal(m, False)
    r2 = np.where(m, r2, 1.0)
    return -(np.where(m, re / (r2 * np.sqrt(r2)) * (dx * du + dy * dv + dz * dw), 0.0)).sum(axis=1)


def test_HS_dndt_uniform_dilation_closed_form():
    # u = a x on the ideal lattice: x_ij . u_ij = a r^2, so Dn/Dt = -a sum re/r = -a (n0 + 32)
    m = 9
    s = scenes.fluid_blob(L0, (m, m, m))
    a = 0.37
    o = O.Oracle(s)
    o.set("u", a * s.x); o.set("v", a * s.y); o.set("w", a * s.z)
    o.bin(); o.dndt()
    core = _interior_mask(s, m, 3)
    expect = -a * (GOLD["n0_3d_2.1"] + GOLD["count_3d_2.1"])
    assert core.sum() == 27
    assert np.allclose(o.get("dndt")[core], expect, rtol=1e-12)


def test_HS_dndt_equals_brute_force_and_finite_difference_of_density():
    s = scenes.small_tank(shuffle=True)
    rng = np.random.default_rng(4)
    fl = s.type == scenes.FLUID
    for k in "uvw":
        getattr(s, k)[fl] = rng.standard_normal(fl.sum())
    o = O.Oracle(s)
    o.bin(); o.dndt()
    d = o.get("dndt")
    ref = _numpy_dndt(s.x, s.y, s.z, s.u, s.v, s.w, s.params["re_n"])
    assert np.allclose(d, ref, rtol=1e-12, atol=1e-9 * np.abs(ref).max())
    # it is the time derivative of Eq. 5 along the motion: central difference of the oracle's
    # own density at r -/+ eps u (walls do not move), on particles with no pair near r_n
    eps = 1e-9
    dens = []
    for sgn in (-1.0, 1.0):
        o2 = O.Oracle(s)
        for k, vel in zip("xyz", "uvw"):
            o2.set(k, getattr(s, k) + sgn * eps * getattr(s, vel))
        o2.bin(); o2.density()
        dens.append(o2.get("n"))
    fd = (dens[1] - dens[0]) / (2 * eps)
    # exclude particles that have a pair within 1e-6 l0 of r_n (the weight has a kink there)
    dx = s.x[None, :] - s.x[:, None]; dy = s.y[None, :] - s.y[:, None]; dz = s.z[None, :] - s.z[:, None]
    r = np.sqrt(dx * dx + dy * dy + dz * dz)
    near = (np.abs(r - s.params["re_n"]) < 1e-6 * s.params["l0"]).any(axis=1)
    ok = ~near
    assert ok.sum() > 0.9 * s.n
    assert np.allclose(fd[ok], d[ok], rtol=2e-5, atol=2e-5 * np.abs(d).max())


def test_HS_and_ECS_right_hand_side_worked_example():
    # ideal lattice scaled by s (same 32 neighbours for 0.94 < s <= 1) with u = a X:
    #   n^k = (n0 + 32)/s - 32,  (Dn/Dt)^k = -a (n0 + 32)/s   (every r scales by s)
    m, sc, a = 9, 0.98, -0.8
    n0, cnt = GOLD["n0_3d_2.1"], GOLD["count_3d_2.1"]
    s = scenes.fluid_blob(L0, (m, m, m))
    core = _interior_mask(s, m, 3)
    for src in (1, 2):
        o = O.Oracle(s, ppe_source=src, re_n=2.1 * L0, beta=0.0)
        X, Y, Z = sc * s.x, sc * s.y, sc * s.z
        o.set("x", X); o.set("y", Y); o.set("z", Z)
        o.set("u", a * X); o.set("v", a * Y); o.set("w", a * Z)
        o.bin(); o.density(); o.dndt(); o.dndt(keep=True)
        nk = (n0 + cnt) / sc - cnt
        dk = -a * (n0 + cnt) / sc
        assert np.allclose(o.get("n")[core], nk, rtol=1e-12)
        assert np.allclose(o.get("dndt_k")[core], dk, rtol=1e-12)
        o.set("n_k", o.get("n"))
        o.ppe_flags(); o.ppe_rhs()
        dt = s.params["dt"]
        if src == 1:      # Eq. 15 (sign: Q22): b = (Dn/Dt)* / (n0 dt)
            expect = dk / (n0 * dt)
        else:             # Eq. 17-18 by hand with alpha = (n^k - n0)/n0, beta = dt (Dn/Dt)^k / n0
            alpha = (nk - n0) / n0
            beta = dt * dk / n0
            expect = (dk / n0 + abs(alpha) * dk / n0 + abs(beta) * alpha / dt) / dt
        assert expect > 0  # compression (a < 0) must raise the pressure
        assert np.allclose(o.get("b")[core], expect, rtol=1e-12)


def test_HL_operator_closed_form_symmetry_and_dense_solve():
    # Eq. 16 applied to phi = x^2 at an interior lattice particle: (1/n0) sum 2 x_ij^2 re / r^3
    # = (2/3)(1/n0) sum re/r = (2/3)(n0 + 122)/n0 (cubic symmetry); the operator is -(1/rho) lap
    m = 10
    s = scenes.fluid_blob(L0, (m, m, m))
    o = O.Oracle(s, ppe_laplacian=1, compress=0.0, beta=0.0)
    o.bin(); o.density(); o.ppe_flags()
    assert (o.get("bc") == 0).all()
    y = o.ppe_apply(s.x ** 2)
    core = _interior_mask(s, m, 4)
    n0l, cnt = GOLD["n0_3d_3.1"], GOLD["count_3d_3.1"]
    assert np.allclose(y[core], -(2.0 / 3.0) * (n0l + cnt) / n0l / 1000.0, rtol=1e-11)  # rho = 1000
    # symmetric positive definite, and CG = dense solve
    st = scenes.small_tank()
    o = O.Oracle(st, ppe_laplacian=1)
    o.bin(); o.density(); o.ppe_flags(); o.ppe_rhs()
    rows = np.nonzero(o.get("bc") == 0)[0]
    rng = np.random.default_rng(7)
    xv = np.zeros(st.n); yv = np.zeros(st.n)
    xv[rows] = rng.standard_normal(rows.size); yv[rows] = rng.standard_normal(rows.size)
    Ax, Ay = o.ppe_apply(xv), o.ppe_apply(yv)
    assert abs(xv @ Ay - Ax @ yv) <= 1e-12 * abs(xv @ Ay)
    assert xv @ Ax > 0
    A = np.zeros((rows.size, rows.size))
    for k, i in enumerate(rows):
        e = np.zeros(st.n); e[i] = 1.0
        A[:, k] = o.ppe_apply(e)[rows]
    b = o.get("b")[rows]
    it = o.ppe_solve(1e-12, 5000)
    assert it > 0
    xd = np.linalg.solve(A, b)
    assert np.linalg.norm(o.get("xcg")[rows] - xd) <= 1e-9 * np.linalg.norm(xd)


# ---- NEXT-3 (part): two-dimensional mode (P:292 item 1; the paper's timed scenes are 2D) ----
def _lattice_2d(m, l0=L0):
    i = np.arange(m)
    Y, X = np.meshgrid(i, i, indexing="ij")
    x = (X.ravel() + 0.5) * l0; y = (Y.ravel() + 0.5) * l0
    s = scenes.dam_break_2d(l0, (m, m), (m, m), seed=1, jitter=0.0)
    keep = s.type == scenes.FLUID
    for k in ("x", "y", "z", "u", "v", "w", "type", "phase"):
        setattr(s, k, np.ascontiguousarray(getattr(s, k)[keep]))
    pad = 8.0 * l0
    s.params["domain_min"] = (-pad, -pad, -0.5 * l0)
    s.params["domain_max"] = (m * l0 + pad, m * l0 + pad, 0.5 * l0)
    assert np.allclose(np.sort(s.x), np.sort(x)) and np.allclose(np.sort(s.y), np.sort(y))
    return s


def test_2d_density_laplacian_and_gradient_closed_forms():
    m = 12
    s = _lattice_2d(m)
    ix = np.rint(s.x / L0 - 0.5).astype(int); iy = np.rint(s.y / L0 - 0.5).astype(int)
    core = (ix >= 4) & (ix < m - 4) & (iy >= 4) & (iy < m - 4)
    o = O.Oracle(s, nu=(1.0, 1.0), g=(0.0, 0.0, 0.0))
    c = o.constants()
    assert abs(c["n0_n"] - GOLD["n0_2d_2.1"]) <= 1e-12 * GOLD["n0_2d_2.1"]
    assert abs(c["n0_lap"] - GOLD["n0_2d_3.1"]) <= 1e-12 * GOLD["n0_2d_3.1"]
    assert abs(c["lam"] / L0 ** 2 - GOLD["lambda_2d_3.1"]) <= 1e-12 * GOLD["lambda_2d_3.1"]
    o.bin(); o.density()
    assert np.allclose(o.get("n")[core], GOLD["n0_2d_2.1"], rtol=1e-12)
    cnt, _ = o.neighbours(s.params["re_lap"])
    assert (cnt[core] == GOLD["count_2d_3.1"]).all()
    # Eq. 10 with d = 2 on a quadratic: 2 (a_x + a_y)
    a = np.array([1.7, -0.6])
    o.set("u", a[0] * s.x ** 2 + a[1] * s.y ** 2 + 0.3 * s.x - 2.0 * s.y + 1.0)
    o.viscosity()
    assert np.allclose(o.get("ax")[core], 2 * a.sum(), rtol=1e-11)
    # gradient of a linear pressure with d = 2: variants 0 and 2 return the slope
    gvec = np.array([3.0, -2.0])
    p = gvec[0] * s.x + gvec[1] * s.y + 50.0
    for variant in (0, 2):
        o2 = O.Oracle(s, grad_variant=variant)
        o2.bin(); o2.set("p", p); o2.phat(); o2.gradient()
        gx, gy = o2.get("gx")[core], o2.get("gy")[core]
        if variant == 0:   # (p_j - phat_i): the constant phat_i drops out on the symmetric lattice
            assert np.allclose(gx, gvec[0], rtol=1e-10) and np.allclose(gy, gvec[1], rtol=1e-10)
        else:              # (p_i + p_j): same, the 2 p_i part cancels by symmetry
            assert np.allclose(gx, gvec[0], rtol=1e-10) and np.allclose(gy, gvec[1], rtol=1e-10)
        assert np.abs(o2.get("gz")).max() == 0.0


def test_2d_neighbour_sets_equal_numpy_brute_force_and_cg_equals_dense():
    s = scenes.dam_break_2d(L0, (24, 20), (8, 14), seed=5)
    o = O.Oracle(s)
    o.bin()
    valid = np.ones(s.n, bool)
    for re in (s.params["re_n"], s.params["re_lap"]):
        cnt, idx = o.neighbours(re)
        assert np.array_equal(csr_to_mask(cnt, idx, s.n), brute_sets_numpy(s.x, s.y, s.z, valid, re))
    o.density(); o.ppe_flags(); o.ppe_rhs()
    rows = np.nonzero(o.get("bc") == 0)[0]
    assert 50 < rows.size < 600
    A = np.zeros((rows.size, rows.size))
    for k, i in enumerate(rows):
        e = np.zeros(s.n); e[i] = 1.0
        A[:, k] = o.ppe_apply(e)[rows]
    assert np.allclose(A, A.T, rtol=0, atol=1e-12 * np.abs(A).max())
    b = o.get("b")[rows]
    assert o.ppe_solve(1e-12, 5000) > 0
    xd = np.linalg.solve(A, b)
    assert np.linalg.norm(o.get("xcg")[rows] - xd) <= 1e-9 * np.linalg.norm(xd)


# ---- NEXT-3 (part): the (1 - r/re)^3 kernel of Eq. 4 ---------------------------------
@pytest.mark.parametrize("dim,tag", [(3, "3d"), (2, "2d")])
@pytest.mark.parametrize("re", [2.1, 3.1])
def test_eq4_kernel_lattice_constants(dim, tag, re):
    n0, lam, cnt = O.lattice_constants(dim, L0, re * L0, kernel=1)
    assert abs(n0 - GOLD[f"n0_eq4_{tag}_{re}"]) <= 1e-13 * n0
    assert abs(lam / L0 ** 2 - GOLD[f"lambda_eq4_{tag}_{re}"]) <= 1e-13 * lam / L0 ** 2
    assert cnt == GOLD[f"count_{tag}_{re}"]


def test_eq4_kernel_density_laplacian_gradient():
    # density = NumPy brute force of Eq. 5 with Eq. 4 on a jittered tank
    s = scenes.small_tank(shuffle=True)
    o = O.Oracle(s, kernel=1)
    o.bin(); o.density()
    re = s.params["re_n"]
    dx = s.x[None, :] - s.x[:, None]; dy = s.y[None, :] - s.y[:, None]; dz = s.z[None, :] - s.z[:, None]
    r = np.sqrt((dx * dx + dy * dy) + dz * dz)
    m = r < re
    np.fill_diagonal(m, False)
    ref = np.where(m, (1.0 - r / re) ** 3, 0.0).sum(axis=1)
    assert np.allclose(o.get("n"), ref, rtol=1e-12, atol=1e-13)
    # lambda makes Eq. 10 exact on a quadratic for any kernel; the gradient model is exact on a
    # linear field on the symmetric lattice for any kernel
    mm = 10
    b = scenes.fluid_blob(L0, (mm, mm, mm))
    core = _interior_mask(b, mm, 4)
    a = np.array([0.9, 1.4, -2.2])
    o = O.Oracle(b, kernel=1, nu=(1.0, 1.0), g=(0.0, 0.0, 0.0))
    o.set("u", a[0] * b.x ** 2 + a[1] * b.y ** 2 + a[2] * b.z ** 2 - 3.0 * b.x + 7.0)
    o.viscosity()
    assert np.allclose(o.get("ax")[core], 2 * a.sum(), rtol=1e-11)
    gvec = np.array([2.0, -1.0, 0.5])
    o2 = O.Oracle(b, kernel=1, grad_variant=2)
    o2.bin(); o2.set("p", gvec[0] * b.x + gvec[1] * b.y + gvec[2] * b.z + 10.0); o2.phat(); o2.gradient()
    for k, comp in enumerate(("gx", "gy", "gz")):
        assert np.allclose(o2.get(comp)[core], gvec[k], rtol=1e-10)


# ---- NEXT-3 (part): neighbour-list reuse (Q24) -------------------------------------
def test_list_reuse_is_the_stored_set_retested_at_the_current_distance():
    s = scenes.small_tank(shuffle=True)
    o = O.Oracle(s, rebin_every=4)
    o.freeze_lists()                                   # lists of both radii at positions A
    rng = np.random.default_rng(11)
    fl = s.type == scenes.FLUID
    xb, yb, zb = s.x.copy(), s.y.copy(), s.z.copy()
    for arr in (xb, yb, zb):
        arr[fl] += rng.uniform(-0.3, 0.3, fl.sum()) * s.params["l0"]   # positions B: sets change
    o.set("x", xb); o.set("y", yb); o.set("z", zb)
    o.density()
    re = s.params["re_n"]
    valid = np.ones(s.n, bool)
    at_a = brute_sets_numpy(s.x, s.y, s.z, valid, re)
    at_b = brute_sets_numpy(xb, yb, zb, valid, re)
    assert (at_a != at_b).sum() > 100                  # the move does change the exact sets
    dx = xb[None, :] - xb[:, None]; dy = yb[None, :] - yb[:, None]; dz = zb[None, :] - zb[:, None]
    r = np.sqrt((dx * dx + dy * dy) + dz * dz)
    r = np.where(at_a & at_b, r, 1.0)
    ref = np.where(at_a & at_b, re / r - 1.0, 0.0).sum(axis=1)
    assert np.allclose(o.get("n"), ref, rtol=1e-12, atol=1e-12)
    # dropping the lists gives the exact sets at B again
    o.freeze_lists(False)
    o.density()
    r = np.where(at_b, np.sqrt((dx * dx + dy * dy) + dz * dz), 1.0)
    assert np.allclose(o.get("n"), np.where(at_b, re / r - 1.0, 0.0).sum(axis=1), rtol=1e-12, atol=1e-12)


def test_list_reuse_equals_exact_mode_while_no_pair_crosses_a_radius():
    # a fluid at rest in a full tank barely moves in 4 steps: same sets, so the same trajectory
    # up to the order of the sums
    s = scenes.hydrostatic_tank(foot=(8, 8), depth=6, height=9)
    a = O.Oracle(s); b = O.Oracle(s, rebin_every=4)
    a.step(4, 0); b.step(4, 0)
    for k in "xyz":
        assert np.abs(a.get(k) - b.get(k)).max() <= 1e-12 * s.params["l0"]


# ---- NEXT-2: multi-density pressure term of the weakly-compressible model (Eq. 11-12) ----
def test_smoothed_density_closed_form_at_a_flat_interface():
    # lattice block, lower half rho_a, upper half rho_b.  A particle in the layer just below the
    # interface sees, above it, the offsets (0,0,1), 4 x (1,0,1), 4 x (1,1,1), (0,0,2) within 2.1 l0:
    # S1 = 1.1 + 4 (2.1/sqrt2 - 1) + 4 (2.1/sqrt3 - 1) + 0.05; <rho> = (rho_a (n0 - S1) + rho_b S1)/n0
    m = 10
    s = scenes.fluid_blob(L0, (m, m, m))
    iz = np.rint(s.z / L0 - 0.5).astype(int)
    s.phase[iz >= m // 2] = 1
    ra, rb = 1000.0, 800.0
    o = O.Oracle(s, n_phases=2, rho=(ra, rb), grad_variant=3)
    o.bin(); o.smooth_density()
    rs = o.get("rho_s")
    n0 = GOLD["n0_3d_2.1"]
    S1 = 1.1 + 4 * (2.1 / math.sqrt(2) - 1) + 4 * (2.1 / math.sqrt(3) - 1) + 0.05
    S2 = 0.05                                             # two layers below: only (0,0,2) reaches across
    core_xy = _interior_mask(s, m, 3)
    below1 = core_xy & (iz == m // 2 - 1); below2 = core_xy & (iz == m // 2 - 2)
    above1 = core_xy & (iz == m // 2)
    assert below1.sum() > 0 and below2.sum() > 0
    assert np.allclose(rs[below1], (ra * (n0 - S1) + rb * S1) / n0, rtol=1e-13)
    assert np.allclose(rs[below2], (ra * (n0 - S2) + rb * S2) / n0, rtol=1e-13)
    assert np.allclose(rs[above1], (rb * (n0 - S1) + ra * S1) / n0, rtol=1e-13)
    # single phase: <rho> = rho exactly
    o1 = O.Oracle(scenes.small_tank(), grad_variant=3)
    o1.bin(); o1.smooth_density()
    assert np.allclose(o1.get("rho_s"), 1000.0, rtol=1e-14, atol=0)


def test_multiphase_pressure_term_brute_force_and_single_phase_limit():
    s = scenes.small_tank(shuffle=True)
    s.phase[s.z > 0.03] = 1
    rho = np.array([1000.0, 800.0])
    o = O.Oracle(s, n_phases=2, rho=tuple(rho), grad_variant=3)
    o.bin(); o.smooth_density()
    rng = np.random.default_rng(9)
    p = rng.uniform(0.0, 500.0, s.n)
    p[s.type == scenes.DUMMY] = 0.0
    o.set("p", p); o.gradient()
    re = s.params["re_n"]
    dx = s.x[None, :] - s.x[:, None]; dy = s.y[None, :] - s.y[:, None]; dz = s.z[None, :] - s.z[:, None]
    r2 = (dx * dx + dy * dy) + dz * dz
    m = (r2 < re * re) & (s.type != scenes.DUMMY)[None, :]
    np.fill_diagonal(m, False)
    r2s = np.where(m, r2, 1.0)
    w = np.where(m, re / np.sqrt(r2s) - 1.0, 0.0)
    # smoothed density (all neighbours, dummies included)
    mall = r2 < re * re
    np.fill_diagonal(mall, False)
    wall_ = np.where(mall, re / np.sqrt(np.where(mall, r2, 1.0)) - 1.0, 0.0)
    rj = rho[s.phase]
    rs = (wall_ * rj[None, :]).sum(axis=1) / wall_.sum(axis=1)
    assert np.allclose(o.get("rho_s"), rs, rtol=1e-12)
    al = p / rj
    coef = (rs[None, :] / rs[:, None]) * al[None, :] - al[:, None]
    c = coef / r2s * w
    n0 = GOLD["n0_3d_2.1"]
    fluid = s.type == scenes.FLUID
    for comp, d in (("gx", dx), ("gy", dy), ("gz", dz)):
        ref = rj * (3.0 / n0) * (c * d).sum(axis=1)
        got = o.get(comp)
        assert np.allclose(got[fluid], ref[fluid], rtol=1e-11, atol=1e-9 * np.abs(ref[fluid]).max())
        assert (got[~fluid] == 0).all()
    # single phase, linear pressure on the lattice: G = grad p exactly ((p_j - p_i) form)
    mm = 10
    b = scenes.fluid_blob(L0, (mm, mm, mm))
    core = _interior_mask(b, mm, 3)
    gvec = np.array([4.0, -3.0, 2.0])
    o2 = O.Oracle(b, grad_variant=3)
    o2.bin(); o2.smooth_density()
    o2.set("p", gvec[0] * b.x + gvec[1] * b.y + gvec[2] * b.z + 30.0); o2.gradient()
    for k, comp in enumerate(("gx", "gy", "gz")):
        assert np.allclose(o2.get(comp)[core], gvec[k], rtol=1e-10)


# ---- whole-step physics sanity (loose): the paper's own validation quantity (Fig. 4) ----
@pytest.mark.parametrize("route", [0, 1])
def test_dam_break_leading_edge_between_theory_bounds(route):
    # 2D column L x 2L on a floor of 4L, L = 0.18 m at l0 = 0.01.  The paper compares
    # the leading edge Z/L against t sqrt(2g/L) only in a figure; what theory fixes: the front can
    # not outrun the frictionless shallow-water (Ritter) front Z/L = 1 + 2T, and a collapsing column
    # of height 2L has passed Z/L = 2.3 by T = 2.1 (the cited experiments and methods lie near 2.8).
    c = 18
    s = scenes.dam_break_2d(L0, (4 * c, 3 * c), (c, 2 * c), seed=3)
    fl = s.type == scenes.FLUID
    o = O.Oracle(s)
    Lc, dt = c * L0, s.params["dt"]
    prev = 1.0
    for k in range(1, 5):
        o.step(100, route)
        T = 100 * k * dt * math.sqrt(2 * 9.81 / Lc)
        x, y = o.get("x"), o.get("y")
        front = x[fl & (y < 3 * L0)].max() / Lc
        assert o.stats()["n_ghost"] == 0
        assert prev - 1e-9 <= front < 1.0 + 2.0 * T
        prev = front
    assert abs(T - 2.09) < 0.01 and 2.3 <= front <= 3.3


# ---- pair viscosity nu_ij (Q9): harmonic / arithmetic mean, wall rule (unpinned branch a) ----
@pytest.mark.parametrize("mean", [1, 0])
def test_viscosity_pair_mean_shell_sum_at_a_flat_interface(mean):
    # un-jittered lattice block, lower half nu_a, upper half nu_b, u = (a z^2, 0, 0), g = 0.
    # Interior of one phase: nu * Laplacian(a z^2) = 2 a nu (T5's closed form).  In the layer just
    # below the interface the offsets with o_z > 0 reach the other phase and carry nu_ab; written
    # out as a sum over lattice offsets (Eq. 10 with nu_ij inside the sum).
    m = 16
    s = scenes.fluid_blob(L0, (m, m, m))
    ix = np.rint(s.x / L0 - 0.5).astype(int)
    iy = np.rint(s.y / L0 - 0.5).astype(int)
    iz = np.rint(s.z / L0 - 0.5).astype(int)
    s.phase[iz >= m // 2] = 1
    a = 3.0
    s.u[:] = a * s.z ** 2
    nu_a, nu_b = 0.7, 1.9
    o = O.Oracle(s, n_phases=2, nu=(nu_a, nu_b), nu_pair_mean=mean, g=(0.0, 0.0, 0.0))
    o.bin(); o.viscosity()
    ax = o.get("ax")
    core_xy = (ix >= 4) & (ix < m - 4) & (iy >= 4) & (iy < m - 4)   # layers 4..11 have their whole ball inside in z
    nu_ab = 2 * nu_a * nu_b / (nu_a + nu_b) if mean == 1 else 0.5 * (nu_a + nu_b)
    n0l, lam = GOLD["n0_3d_3.1"], GOLD["lambda_3d_3.1"] * L0 ** 2
    A = 2.0 * 3 / (n0l * lam)

    def shell_sum(zi_layer, own_phase):
        z = (zi_layer + 0.5) * L0
        tot = 0.0
        for oz in range(-3, 4):
            for oy in range(-3, 4):
                for ox in range(-3, 4):
                    r2 = ox * ox + oy * oy + oz * oz
                    if r2 == 0 or r2 >= 3.1 ** 2:
                        continue
                    other = (zi_layer + oz >= m // 2) != (own_phase == 1)
                    nu_i = nu_a if own_phase == 0 else nu_b
                    nu = nu_ab if other else nu_i
                    du = a * ((z + oz * L0) ** 2 - z ** 2)
                    tot += nu * du * (3.1 / math.sqrt(r2) - 1.0)
        return A * tot

    for layer, ph in ((m // 2 - 1, 0), (m // 2 - 2, 0), (m // 2 - 4, 0), (m // 2, 1), (m // 2 + 2, 1)):
        sel = core_xy & (iz == layer)
        assert sel.sum() > 0
        assert np.allclose(ax[sel], shell_sum(layer, ph), rtol=1e-11), (layer, ph)
    # four layers below the interface nothing reaches across: the single-nu closed form 2 a nu_a
    assert np.allclose(ax[core_xy & (iz == m // 2 - 4)], 2 * a * nu_a, rtol=1e-11)
    # the two means differ at the interface (so a swapped formula fails one of the two runs)
    assert abs(shell_sum(m // 2 - 1, 0) - 2 * a * nu_a) > 1e-3


@pytest.mark.parametrize("mean", [1, 0])
@pytest.mark.parametrize("cs", [0.0, 0.12])
def test_viscosity_brute_force_with_walls_two_phases(mean, cs):
    # jittered tank with walls present, random velocities, two viscosities: the O(N^2) definition
    # a_i = A_lap sum_j nu_ij (u_j - u_i) w + g with nu_ij = nu_i and u_j = 0 for WALL/DUMMY j (Q9),
    # nu_i = nu[phase] + nu_t (nu_t from the oracle's own field when Cs > 0: its formula is pinned by
    # test_smagorinsky_simple_shear).
    s = scenes.small_tank(shuffle=True)
    s.phase[s.z > 0.03] = 1
    rng = np.random.default_rng(12)
    fl = s.type == scenes.FLUID
    for k in "uvw":
        getattr(s, k)[fl] = rng.standard_normal(fl.sum())
        getattr(s, k)[~fl] = 7.0           # must be ignored: walls and dummies are at rest (no-slip)
    nu = np.array([0.7, 1.9])
    o = O.Oracle(s, n_phases=2, nu=tuple(nu), nu_pair_mean=mean, cs=cs)
    o.bin(); o.viscosity()
    nut = o.get("nut")
    assert (nut[~fl] == 0).all() and ((nut[fl] > 0).all() if cs > 0 else (nut == 0).all())
    re = s.params["re_lap"]
    dx = s.x[None, :] - s.x[:, None]; dy = s.y[None, :] - s.y[:, None]; dz = s.z[None, :] - s.z[:, None]
    r2 = (dx * dx + dy * dy) + dz * dz
    msk = r2 < re * re
    np.fill_diagonal(msk, False)
    w = np.where(msk, re / np.sqrt(np.where(msk, r2, 1.0)) - 1.0, 0.0)
    nui = nu[s.phase] + nut
    ni, nj = nui[:, None], nui[None, :]
    pair = 2 * ni * nj / (ni + nj) if mean == 1 else 0.5 * (ni + nj)
    solid_j = (~fl)[None, :]
    nuij = np.where(solid_j, ni, pair)
    n0l, lam = GOLD["n0_3d_3.1"], GOLD["lambda_3d_3.1"] * L0 ** 2
    A = 2.0 * 3 / (n0l * lam)
    for comp, vel, gc in (("ax", s.u, 0.0), ("ay", s.v, 0.0), ("az", s.w, -9.81)):
        uj = np.where(fl, vel, 0.0)
        ref = A * (nuij * (uj[None, :] - vel[:, None]) * w).sum(axis=1) + gc
        got = o.get(comp)
        assert np.allclose(got[fl], ref[fl], rtol=1e-11, atol=1e-9 * np.abs(ref[fl]).max()), comp
        assert (got[~fl] == 0).all()
    # the wall rule matters here: fluid next to a wall would change if nu_ij used the pair mean with nu_j
    near_wall = fl & (np.where(solid_j & msk, 1, 0).sum(axis=1) > 0)
    assert near_wall.sum() > 50


# ---- p-hat and gradient variants 0-2 by brute force, dummies carrying a non-zero p (branch b) ----
@pytest.mark.parametrize("variant", [0, 1, 2])
def test_phat_and_gradient_brute_force_skip_dummies(variant):
    # P:215 Eq. 14 / Q12, Q13: dummies have no pressure and are skipped both in p-hat and in the
    # sum.  They are given a large p here so that including them changes every wall-near value.
    s = scenes.small_tank(shuffle=True)
    rng = np.random.default_rng(21)
    p = rng.uniform(100.0, 500.0, s.n)
    dummy = s.type == scenes.DUMMY
    p[dummy] = -1.0e4                       # would win every minimum and dominate every sum
    o = O.Oracle(s, grad_variant=variant)
    o.bin(); o.set("p", p); o.phat(); o.gradient()
    re = s.params["re_n"]
    dx = s.x[None, :] - s.x[:, None]; dy = s.y[None, :] - s.y[:, None]; dz = s.z[None, :] - s.z[:, None]
    r2 = (dx * dx + dy * dy) + dz * dz
    m = (r2 < re * re) & (~dummy)[None, :]
    np.fill_diagonal(m, False)
    # p-hat: FLUID and WALL rows, minimum over i itself and its non-dummy neighbours
    ph_ref = np.minimum(p, np.where(m, p[None, :], np.inf).min(axis=1))
    on = (s.type == scenes.FLUID) | (s.type == scenes.WALL)
    ph = o.get("phat")
    assert np.array_equal(ph[on], ph_ref[on]) and (ph[~on] == 0).all()
    assert (ph[on] >= 100.0).all()          # no dummy value leaked in
    r2s = np.where(m, r2, 1.0)
    w = np.where(m, re / np.sqrt(r2s) - 1.0, 0.0)
    if variant == 0:
        coef = p[None, :] - ph_ref[:, None]
    elif variant == 1:
        phj = np.where(on, ph_ref, 0.0)
        coef = (p[:, None] + p[None, :]) - (ph_ref[:, None] + phj[None, :])
    else:
        coef = p[:, None] + p[None, :]
    c = coef / r2s * w
    n0 = GOLD["n0_3d_2.1"]
    fluid = s.type == scenes.FLUID
    touched = fluid & ((r2 < re * re) & dummy[None, :]).any(axis=1)
    assert touched.sum() > 20               # some fluid rows do have dummies in range
    for comp, d in (("gx", dx), ("gy", dy), ("gz", dz)):
        ref = (3.0 / n0) * (c * d).sum(axis=1)
        got = o.get(comp)
        assert np.allclose(got[fluid], ref[fluid], rtol=1e-11, atol=1e-9 * np.abs(ref[fluid]).max())
        assert (got[~fluid] == 0).all()


# ---- the record of neighbours kept during a solve changes no number; warm start reaches the same x ----
def test_cg_neighbour_record_and_warm_start():
    s = scenes.small_tank(shuffle=True)
    o = O.Oracle(s); o.step(3, 1); o.viscosity(); o.predict(); o.density()
    o.ppe_flags(); o.ppe_rhs()
    rows = o.get("bc") == 0
    it = o.ppe_solve(1e-8, 5000)
    x = o.get("xcg"); b = o.get("b")
    # the solve's operator (walking the record) and ppe_apply (searching the grid) are the same map
    assert np.linalg.norm(b - o.ppe_apply(x)) <= 1.5e-8 * np.linalg.norm(b)
    assert it > 10
    # warm start: from the converged pressure of the same system CG needs no iteration; from a
    # perturbed start it reaches the same solution
    w = O.Oracle(s, cg_warm_start=1)
    for k in ("x", "y", "z", "u", "v", "w", "n"):
        w.set(k, o.get(k))
    w.ppe_flags(); w.ppe_rhs()
    w.set("p", np.where(rows, x, 0.0))
    assert w.ppe_solve(1e-8, 5000) == 0
    w.set("p", np.where(rows, x * (1.0 + 0.05 * np.sin(np.arange(s.n))), 0.0))
    it_w = w.ppe_solve(1e-8, 5000)
    assert 0 < it_w <= it
    assert np.linalg.norm(w.get("xcg") - x) <= 1e-6 * np.linalg.norm(x)


# ---- key_mode 1: the Morton key (north_star "Morton- or cell-sorted") ----
def test_morton_key_table_and_sort_invariants():
    # hand table: bit k of c_x -> bit 3k, c_y -> bit 3k+1, c_z -> bit 3k+2
    table = {(0, 0, 0): 0, (1, 0, 0): 1, (0, 1, 0): 2, (0, 0, 1): 4, (1, 1, 1): 7, (2, 0, 0): 8,
             (0, 2, 0): 16, (0, 0, 2): 32, (3, 0, 0): 9, (2, 3, 1): 8 + 16 + 2 + 4,
             (5, 0, 0): 1 + 64, (0, 5, 0): 2 + 128, (0, 0, 5): 4 + 256,
             (7, 7, 7): 511, (8, 0, 0): 512, (1023, 0, 0): sum(1 << (3 * k) for k in range(10)),
             (1023, 1023, 1023): (1 << 30) - 1}
    for (cx, cy, cz), key in table.items():
        assert O.morton3(cx, cy, cz) == key, (cx, cy, cz)
    s = scenes.small_tank(shuffle=True)
    s.x[5] = 10.0                           # a ghost
    lin = O.Oracle(s)
    mor = O.Oracle(s, key_mode=1)
    kl, pl, csl = lin.bin()
    km, pm, csm = mor.bin()
    nx, ny, nz, ncl = lin.grid()
    assert mor.grid()[:3] == (nx, ny, nz)
    bits = max(nx, ny, nz).bit_length() if (max(nx, ny, nz) & (max(nx, ny, nz) - 1)) else max(nx, ny, nz).bit_length() - 1
    assert mor.grid()[3] == 8 ** bits and csm.size == 8 ** bits + 1
    # the Morton key of every particle is the interleave of the cell coordinates its linear key encodes
    live = kl < ncl
    cx, cy, cz = kl % nx, (kl // nx) % ny, kl // (nx * ny)
    ref = np.array([O.morton3(int(a), int(b), int(c)) for a, b, c in zip(cx, cy, cz)])
    assert np.array_equal(km[live], ref[live]) and (km[~live] == 8 ** bits).all() and (~live).sum() == 1
    # T12 invariants for the Morton sort
    assert np.array_equal(np.sort(pm), np.arange(s.n))
    ks = km[pm]
    assert (np.diff(ks) >= 0).all() and (np.diff(pm)[np.diff(ks) == 0] > 0).all()
    assert csm[0] == 0 and csm[-1] == s.n - 1 and (np.diff(csm) >= 0).all()
    assert np.array_equal(np.diff(csm), np.bincount(km[live], minlength=8 ** bits))
    # the neighbour sets and every field do not depend on the key
    for re in (s.params["re_n"], s.params["re_lap"]):
        a, b = lin.neighbours(re), mor.neighbours(re)
        assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])
    lin2 = O.Oracle(scenes.small_tank(shuffle=True)); mor2 = O.Oracle(scenes.small_tank(shuffle=True), key_mode=1)
    lin2.step(3, 1); mor2.step(3, 1)
    for k in ("x", "y", "z"):               # only the order of additions inside a sum differs
        assert np.abs(lin2.get(k) - mor2.get(k)).max() <= 1e-12 * 0.12


# ---- NEXT-4: preconditioned CG (P:176 ICCG) against the dense solve and against plain CG ----
@pytest.mark.parametrize("precond,degree", [(0, 0), (1, 0), (2, 0), (3, 0), (4, 3)])
def test_pcg_equals_dense_solve(precond, degree):
    # 0 none, 1 Jacobi, 2 block Jacobi on the grid cells, 3 incomplete Cholesky IC(0) -- the paper's
    # ICCG -- 4 Chebyshev polynomial.  Each must reach THE solution of A x = b (textbook LAPACK solve of
    # the matrix assembled in numpy from Listing 2's rule), whatever M is.
    s = scenes.small_tank(shuffle=True)
    o = O.Oracle(s)
    o.step(2, 0)
    o.viscosity(); o.predict(); o.density(); o.ppe_flags(); o.ppe_rhs()
    A, rows = _dense_A(o, s)
    b = o.get("b")[rows]
    xd = np.linalg.solve(A, b)
    it = o.ppe_solve_pcg(1e-12, 5000, precond, degree, 30.0)
    assert it > 0
    xp = o.get("xcg")
    assert (xp[o.get("bc") != 0] == 0).all()
    assert np.linalg.norm(xp[rows] - xd) <= 1e-9 * np.linalg.norm(xd)
    # at the default tolerance: the stated residual bound, and fewer iterations than plain CG for IC(0)
    it8 = o.ppe_solve_pcg(1e-8, 5000, precond, degree, 30.0)
    x8 = o.get("xcg")[rows]
    assert np.linalg.norm(b - A @ x8) <= 1.5e-8 * np.linalg.norm(b)
    it_cg = o.ppe_solve(1e-8, 5000)
    if precond == 0:
        assert it8 == it_cg                # the CSR path and the matrix-free path are the same iteration
    if precond == 3:
        assert it8 <= 0.5 * it_cg          # what the paper's preconditioner buys (measured: 21 -> 7)
    if precond in (1, 2):
        assert it8 <= it_cg


# ---- NEXT-3: the paper's water-drop test (section 5.1, Table 1) ----
def _drop_axes(x, y):
    # semi-axes from second moments: a uniform ellipse has <x^2> = a^2 / 4 (robust against the few
    # stray surface particles that the maximum extent follows)
    return 2.0 * math.sqrt(float((x * x).mean())), 2.0 * math.sqrt(float((y * y).mean()))


def test_water_drop_ab_invariant_and_doubling_time():
    # An incompressible drop with u = (-A x, A y) stays an ellipse with a b = R^2 (the paper's
    # criterion, after Monaghan [47]), and Euler's equations with p = 0 on the boundary give
    # A' = A^2 (a^2 - b^2)/(a^2 + b^2), so with s = b/R: A = A0 s sqrt(2/(1 + s^4)) and b doubles at
    # t2 = (1/(A0 sqrt 2)) int_1^2 sqrt(1 + s^4)/s^2 ds = 8.005e-3 s for A0 = 100 1/s.  The paper reports
    # ab constant within 0.26 % with its (unstated) default configuration; with this build's readings
    # (no surface or collision treatment, Q11; explicit route with Eq. 4 and c0 = 2000 m/s, Mach 0.09)
    # the measured figures are ab within 2.7 % and t2 = 8.3e-3 s.
    s = scenes.water_drop()
    T1 = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "water_drop_table1.txt")) as f:
        for line in f:
            w = line.split("#")[0].split()
            if len(w) == 2:
                T1[w[0]] = float(w[1])
    assert s.n == T1["particles"] == 1257
    assert s.x.max() == pytest.approx(T1["b_start"], rel=1e-12) and -s.u[0] / s.x[0] == pytest.approx(T1["rate"])
    assert T1["ab_start"] == pytest.approx(T1["b_start"] ** 2, abs=5e-4)    # the table's ab(0) is b(0)^2: a disc
    sN = np.linspace(1.0, 2.0, 20001)
    f = np.sqrt(1.0 + sN ** 4) / sN ** 2
    t2 = float(((f[1:] + f[:-1]) * 0.5 * np.diff(sN)).sum()) / (100.0 * math.sqrt(2.0))
    assert abs(t2 - 8.005e-3) < 2e-6
    o = O.Oracle(s, c0=2000.0)
    a0, b0 = _drop_axes(s.x, s.y)
    assert a0 * b0 == pytest.approx(0.875 ** 2, rel=5e-3)     # Table 1: ab(0) = 0.766
    k, worst = 0, 0.0
    while True:
        o.step(10, 0)
        k += 10
        a, b = _drop_axes(o.get("x"), o.get("y"))
        worst = max(worst, abs(a * b - a0 * b0) / (a0 * b0))
        if b >= 2.0 * b0 or k >= 2000:
            break
    t_double = k * s.params["dt"]
    print(f"water drop: b doubled after {k} steps (t = {t_double:.2e} s, theory {t2:.2e}); "
          f"ab error at the end {100 * abs(a * b - a0 * b0) / (a0 * b0):.2f} %, worst {100 * worst:.2f} % (paper: 0.26 %)")
    assert o.stats()["n_ghost"] == 0
    assert abs(t_double - t2) <= 0.06 * t2                 # measured 8.3e-3 vs 8.005e-3
    assert worst <= 0.035                                   # measured 2.7 %
    # the field stays close to the linear one: v / y = A(t) with A(t2) = A0 * 2 sqrt(2/17)
    y, v = o.get("y"), o.get("v")
    A_fit = float((y * v).sum() / (y * y).sum())
    assert A_fit == pytest.approx(100.0 * 2.0 * math.sqrt(2.0 / 17.0), rel=0.08)


def test_water_drop_on_the_ppe_route():
    # The same closed forms pin a WHOLE semi-implicit step (flags, source, solve, gradient, corrector, in
    # this order and with these signs): an incompressible drop keeps a b = R^2 and doubles b at t2.  The
    # paper does not state the configuration behind its 0.26 %; Listing 2's compressibility
    # term 1e-7 / dt^2 is sized for its dam-break step (dt ~ 1e-3), at dt = 1e-5 it would swamp
    # the Laplacian (the solve then takes 3 iterations and the drop's area grows by 19 %), so the pin
    # scales it with dt^2 (compress = 1e-10) and takes the momentum-conserving gradient (variant 2).
    # Measured: b doubles after 820 steps (8.20e-3 s, theory 8.005e-3), a b within 3.5 %.
    s = scenes.water_drop()
    o = O.Oracle(s, compress=1.0e-10, grad_variant=2)
    a0, b0 = _drop_axes(s.x, s.y)
    k, worst = 0, 0.0
    while True:
        o.step(10, 1)
        k += 10
        a, b = _drop_axes(o.get("x"), o.get("y"))
        worst = max(worst, abs(a * b - a0 * b0) / (a0 * b0))
        if b >= 2.0 * b0 or k >= 2000:
            break
    print(f"water drop, PPE route: b doubled after {k} steps, worst ab error {100 * worst:.2f} %, "
          f"cg iterations in the last step {o.stats()['cg_iters']}")
    assert o.stats()["n_ghost"] == 0 and o.stats()["cg_iters"] > 5
    assert abs(k * s.params["dt"] - 8.005e-3) <= 0.05 * 8.005e-3
    assert worst <= 0.05
