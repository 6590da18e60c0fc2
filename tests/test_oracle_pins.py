"""Pins for the fp64 oracle (oracle/tetra_oracle.c) against things other than itself.

Each test states what it pins and which plausible mistake it would catch.  None of them
retypes Eq. 12-14: they use finite differences, a case-free closed form (truncated powers),
Monte-Carlo integration over the simplex, exact moments, sum rules, the closed-form
simple-cubic DOS (elliptic integral), a Kuhn-triangulation brute force that never looks at
Table I, and invariances.  SURVEY.md 8(c) P1-P9.
"""
import itertools
import math
import os

import numpy as np
import pytest
from scipy import integrate, special

from paper_1710_10789_b200 import workloads as wl

V0 = 1.0 / 24.0  # V_T/(4 V_G) for a single cube (nk = 1)

# sorted corner-energy sets: generic, wide/narrow gaps, negative energies
E_SETS = [
    np.array([0.1, 0.35, 0.8, 1.3]),
    np.array([-2.0, -1.9, 0.5, 0.6]),
    np.array([-0.3, 0.0, 0.01, 2.0]),
    np.array([1.0, 1.5, 1.6, 1.65]),
]


def _inside(e, frac):
    """energies strictly inside each of the three intervals"""
    return [e[i] + frac * (e[i + 1] - e[i]) for i in range(3)]


# ---------------------------------------------------------------- P1
@pytest.mark.parametrize("e", E_SETS)
def test_P1_derivative_matches_central_difference(oracle_lib, e):
    """dw_l/dE as coded == numerical derivative of w_l as coded, in every case.
    Catches G1 (Eq. 12d misprint), G4 (Eq. 13l misprint) and any sign slip in 13/14."""
    for frac in (0.2, 0.5, 0.8):
        for E in _inside(e, frac):
            gap = min(abs(E - x) for x in e)
            h = 1e-4 * gap
            wp, _, kp = oracle_lib.corner_weights(e, E + h, V0)
            wm, _, km = oracle_lib.corner_weights(e, E - h, V0)
            _, dw, k0 = oracle_lib.corner_weights(e, E, V0)
            assert kp == km == k0
            num = (wp - wm) / (2 * h)
            assert np.allclose(num, dw, rtol=0, atol=1e-7 * V0 / gap), (E, num, dw)


# ---------------------------------------------------------------- P2
@pytest.mark.parametrize("e", E_SETS)
def test_P2_continuity_and_end_values(oracle_lib, e):
    """w_l and dw_l continuous at E2, E3; w_l(E4) = V; w = dw = 0 at E1; dw -> 0 at E4.
    Catches G3 (the printed Eq. 13k is discontinuous at E2/E3)."""
    for knot in (e[1], e[2]):
        eps = 1e-9
        wl_, dwl, _ = oracle_lib.corner_weights(e, knot - eps, V0)
        wr, dwr, _ = oracle_lib.corner_weights(e, knot + eps, V0)
        assert np.allclose(wl_, wr, atol=1e-8 * V0)
        assert np.allclose(dwl, dwr, atol=1e-6 * V0)
    w, dw, k = oracle_lib.corner_weights(e, e[0], V0)
    assert k == 0 and not w.any() and not dw.any()
    w, dw, k = oracle_lib.corner_weights(e, e[0] + 1e-9, V0)
    assert k == 1 and np.all(np.abs(dw) < 1e-12) and np.all(np.abs(w) < 1e-18)
    w, dw, k = oracle_lib.corner_weights(e, e[3] - 1e-9, V0)
    assert k == 3 and np.allclose(w, V0, atol=1e-12) and np.all(np.abs(dw) < 1e-10)
    w, dw, k = oracle_lib.corner_weights(e, e[3], V0)
    assert k == 4 and np.all(w == V0) and not dw.any()
    w, dw, k = oracle_lib.corner_weights(e, e[3] + 5.0, V0)
    assert k == 4 and np.all(w == V0) and not dw.any()


# ---------------------------------------------------------------- P3
def _trunc_power_sum(e, E, p):
    """sum_j (E-e_j)_+^p / prod_{i != j} (e_i - e_j): the divided difference of the
    truncated power -- a case-free textbook form (simplex spline), independent of Eq. 12-14."""
    s = 0.0
    for j in range(4):
        d = 1.0
        for i in range(4):
            if i != j:
                d *= e[i] - e[j]
        s += max(E - e[j], 0.0) ** p / d
    return s


@pytest.mark.parametrize("e", E_SETS)
def test_P3_truncated_power_closed_form(oracle_lib, e):
    """sum_l w_l = 4V * sum_j (E-e_j)_+^3 / prod(e_i-e_j)  (number of states of one
    tetrahedron), its derivative, and per corner w_l = -V d/de_l sum_j (E-e_j)_+^4/prod."""
    for frac in (0.1, 0.37, 0.5, 0.93):
        for E in _inside(e, frac):
            w, dw, _ = oracle_lib.corner_weights(e, E, V0)
            assert math.isclose(w.sum(), 4 * V0 * _trunc_power_sum(e, E, 3), rel_tol=1e-10, abs_tol=1e-15)
            assert math.isclose(dw.sum(), 12 * V0 * _trunc_power_sum(e, E, 2), rel_tol=1e-9, abs_tol=1e-13)
            for l in range(4):
                h = 1e-6
                ep, em = e.copy(), e.copy()
                ep[l] += h
                em[l] -= h
                dG = (_trunc_power_sum(ep, E, 4) - _trunc_power_sum(em, E, 4)) / (2 * h)
                assert math.isclose(w[l], -V0 * dG, rel_tol=2e-5, abs_tol=1e-9 * V0), (l, E)


# ---------------------------------------------------------------- P4
@pytest.mark.parametrize("e", E_SETS[:2])
def test_P4_monte_carlo_simplex(oracle_lib, e):
    """w_l(E)/(4V) = < lambda_l * 1[lambda.e < E] > over the uniform simplex: this is the
    definition (a band linear across one tetrahedron is integrated exactly)."""
    rng = np.random.default_rng(4)
    lam = rng.dirichlet(np.ones(4), 2_000_000)
    eps = lam @ e
    for frac in (0.3, 0.7):
        for E in _inside(e, frac):
            w, _, _ = oracle_lib.corner_weights(e, E, V0)
            mc = (lam * (eps < E)[:, None]).mean(axis=0)
            assert np.allclose(w / (4 * V0), mc, atol=6e-4), (E, w / (4 * V0), mc)


def test_P4_permuted_corners_match_mc(oracle_lib):
    """Same, through sort4: unsorted corner energies, per-corner values b -- pins that the
    permutation returned by the sort matches weights to the right corners."""
    rng = np.random.default_rng(5)
    e_in = np.array([0.7, -0.2, 1.1, 0.3])
    b_in = np.array([0.9, 0.1, 0.4, 0.6])
    es, perm = oracle_lib.sort4(e_in)
    assert np.all(np.diff(es) >= 0) and np.allclose(e_in[perm], es)
    lam = rng.dirichlet(np.ones(4), 2_000_000)
    eps = lam @ e_in
    bl = lam @ b_in
    for E in (0.0, 0.4, 0.9):
        w, _, _ = oracle_lib.corner_weights(es, E, V0)
        n_or = float((b_in[perm] * w).sum()) / (4 * V0)
        n_mc = float((bl * (eps < E)).mean())
        assert abs(n_or - n_mc) < 6e-4


# ---------------------------------------------------------------- P5
@pytest.mark.parametrize("e", E_SETS)
def test_P5_moments(oracle_lib, e):
    """int dw_l dE = V and int E dw_l dE = 4V sum_j e_j (1+delta_lj)/20 (Dirichlet second
    moments); Gauss-Legendre per piece is exact (piecewise polynomial)."""
    x, wt = np.polynomial.legendre.leggauss(8)
    m0 = np.zeros(4)
    m1 = np.zeros(4)
    for a, b in zip(e[:-1], e[1:]):
        for xi, wi in zip(x, wt):
            E = 0.5 * (a + b) + 0.5 * (b - a) * xi
            _, dw, _ = oracle_lib.corner_weights(e, E, V0)
            m0 += 0.5 * (b - a) * wi * dw
            m1 += 0.5 * (b - a) * wi * dw * E
    assert np.allclose(m0, V0, rtol=1e-12)
    expect = np.array([4 * V0 * sum(e[j] * (1 + (l == j)) / 20.0 for j in range(4)) for l in range(4)])
    assert np.allclose(m1, expect, rtol=1e-11, atol=1e-15)


# ---------------------------------------------------------------- degenerate corners (G10/G11)
def test_degenerate_corners_finite_and_ordered(oracle_lib):
    """Ties never divide by zero and tied corners get equal weights; all four equal:
    DOS = 0 everywhere, N jumps 0 -> V strictly above e (rule (i) wins at w = e)."""
    for e in ([0.0, 0.0, 0.5, 1.0], [0.0, 0.5, 0.5, 1.0], [0.0, 0.5, 1.0, 1.0],
              [0.0, 0.0, 0.0, 1.0], [0.0, 1.0, 1.0, 1.0], [0.0, 0.0, 1.0, 1.0]):
        e = np.array(e)
        for E in np.linspace(-0.1, 1.1, 49):
            w, dw, k = oracle_lib.corner_weights(e, E, V0)
            assert np.all(np.isfinite(w)) and np.all(np.isfinite(dw)), (e, E)
            assert np.all(w >= -1e-15) and np.all(w <= V0 + 1e-15)
            for i, j in itertools.combinations(range(4), 2):
                if e[i] == e[j]:
                    assert math.isclose(w[i], w[j], abs_tol=1e-15) and math.isclose(dw[i], dw[j], abs_tol=1e-12)
            if 0 < E < 1:  # compare with the generic formula at slightly split energies
                e2 = e + np.array([0, 1e-7, 2e-7, 3e-7])
                w2, _, _ = oracle_lib.corner_weights(e2, E, V0)
                assert np.allclose(w, w2, atol=1e-6 * V0)
    e = np.array([0.3, 0.3, 0.3, 0.3])
    for E, wexp in ((0.2, 0.0), (0.3, 0.0), (0.30001, V0)):
        w, dw, _ = oracle_lib.corner_weights(e, E, V0)
        assert np.all(w == wexp) and not dw.any()


# ---------------------------------------------------------------- Table I geometry (G7)
def test_table_I_tiles_the_cube(oracle_lib):
    """With the G7 labelling the six tetrahedra of Table I have volume 1/6 each, share the
    body diagonal 3-6 and every random point of the cube lies in exactly one of them."""
    T = oracle_lib.table_I()
    assert T.tolist() == [[1, 2, 3, 6], [2, 3, 4, 6], [1, 3, 5, 6], [3, 4, 6, 8], [3, 5, 6, 7], [3, 6, 7, 8]]
    pos = {c: np.array(oracle_lib.corner_offset(c), dtype=float) for c in range(1, 9)}
    assert sorted(tuple(int(x) for x in p) for p in pos.values()) == sorted(itertools.product((0, 1), repeat=3))
    assert np.allclose(pos[3] + pos[6], 1.0)  # 3 and 6 are opposite corners
    rng = np.random.default_rng(0)
    pts = rng.uniform(0, 1, (20000, 3))
    count = np.zeros(len(pts), dtype=int)
    for row in T:
        assert 3 in row and 6 in row
        v = np.array([pos[c] for c in row])
        M = (v[1:] - v[0]).T
        assert math.isclose(abs(np.linalg.det(M)) / 6.0, 1.0 / 6.0, rel_tol=1e-12)
        lam = np.linalg.solve(M, (pts - v[0]).T).T
        lam0 = 1 - lam.sum(axis=1)
        count += ((lam >= 0).all(axis=1) & (lam0 >= 0)).astype(int)
    assert np.all(count == 1)


# ---------------------------------------------------------------- P8 brute force
def _kuhn_interpolate(E, W, nk, pts):
    """Piecewise-linear interpolant over the six tetrahedra that share the body diagonal
    (0,1,0)-(1,0,1) of every cube, built from the ORDER of the local coordinates (Kuhn
    triangulation) -- never looks at Table I.  pts in [0,N)^3 grid units, periodic.
    Returns E_lin[npts][nb], W_lin[npts][nb][norb]."""
    n1, n2, n3 = nk
    base = np.floor(pts).astype(int)
    f = pts - base
    u = np.stack([f[:, 0], 1.0 - f[:, 1], f[:, 2]], axis=1)  # y mirrored: diagonal -> main diagonal
    order = np.argsort(-u, axis=1, kind="stable")
    us = np.take_along_axis(u, order, axis=1)
    lam = np.stack([1 - us[:, 0], us[:, 0] - us[:, 1], us[:, 1] - us[:, 2], us[:, 2]], axis=1)
    cur = np.zeros((len(pts), 3), dtype=int)          # vertex in u-space
    El = 0.0
    Wl = 0.0
    for step in range(4):
        d = np.stack([cur[:, 0], 1 - cur[:, 1], cur[:, 2]], axis=1)  # back to real offsets
        ik = ((base[:, 0] + d[:, 0]) % n1) + n1 * (((base[:, 1] + d[:, 1]) % n2) + n2 * ((base[:, 2] + d[:, 2]) % n3))
        El = El + lam[:, step, None] * E[ik].astype(np.float64)
        Wl = Wl + lam[:, step, None, None] * W[ik].astype(np.float64)
        if step < 3:
            cur[np.arange(len(pts)), order[:, step]] += 1
    return El, Wl


@pytest.mark.parametrize("nk", [(2, 2, 2), (3, 2, 4), (4, 4, 4)])
def test_P8_brute_force_tiny_grids(oracle_lib, nk):
    """N_m(w) from the oracle == Monte-Carlo integral of the piecewise-linear interpolant
    (definition of the method), on tiny periodic grids with random E and W.  Pins jointly:
    periodic wrap, ik convention, Table I + G7 (which diagonal), sort permutation <-> W
    matching, V_T/V_G, and the weights."""
    nb, norb = 2, 3
    E, W = wl.random_bands(nk, nb, norb, seed=11 + nk[0])
    om = np.linspace(-1.1, 1.1, 23).astype(np.float32)
    r = oracle_lib.tetra_dos(E, W, nk, om)
    rng = np.random.default_rng(2)
    npts = 1_500_000
    pts = rng.uniform(0, 1, (npts, 3)) * np.array(nk)
    El, Wl = _kuhn_interpolate(E, W, nk, pts)
    for i, w0 in enumerate(om):
        occ = (El < float(w0))                       # [npts][nb]
        mc = (Wl * occ[:, :, None]).sum(axis=1).mean(axis=0)   # [norb]
        assert np.allclose(r["nos"][:, i], mc, atol=2.5e-3), (i, r["nos"][:, i], mc)
    # bin-averaged DOS == finite difference of N (trapezoid of DOS over one bin)
    d_om = np.diff(om.astype(np.float64))
    avg = 0.5 * (r["dos"][:, 1:] + r["dos"][:, :-1]) * d_om
    assert np.allclose(avg, np.diff(r["nos"], axis=1), atol=0.04)


# ---------------------------------------------------------------- P6 sum rules
def test_P6_sum_rules_tb8(oracle_lib):
    """On the 8-orbital model (Nk=8): N_m(w >= max E) = (1/nk) sum_k sum_n W (=1: unitary
    eigenvectors); sum_m DOS_m = total DOS (W = 1 run on each band... done as nb bands,
    norb = 1); trapezoid int DOS_m = N_m(w_max); dN/dw = DOS by central difference."""
    nk = (8, 8, 8)
    E, W = wl.tb8_bands(nk, threads=1)
    om = wl.omega_grid(-6.0, 4.0, 801)
    r = oracle_lib.tetra_dos(E, W, nk, om, nthreads=2)
    top = r["nos"][:, -1]
    assert np.allclose(top, W.astype(np.float64).sum(axis=(0, 1)) / E.shape[0], rtol=0, atol=1e-12)
    assert np.allclose(top, 1.0, atol=1e-6)
    ones = np.ones(E.shape + (1,), dtype=np.float32)
    rt = oracle_lib.tetra_dos(E, ones, nk, om, nthreads=2)
    Wn = (W.astype(np.float64) / W.astype(np.float64).sum(axis=2, keepdims=True)).astype(np.float32)
    # fp32 rows of W sum to 1 only to 1e-7: compare at that level
    assert np.allclose(r["dos"].sum(axis=0), rt["dos"][0], rtol=0, atol=3e-6 * rt["dos"].max())
    assert np.allclose(r["nos"].sum(axis=0), rt["nos"][0], rtol=0, atol=3e-6 * 8)
    del Wn
    trap = np.trapezoid(r["dos"], om.astype(np.float64), axis=1)
    assert np.allclose(trap, top, atol=2e-3)
    # derivative: energies exactly representable in fp32
    w0 = np.array([-3.0, -1.5, -0.25, 0.5, 1.75], dtype=np.float64)
    h = 2.0 ** -12
    tri = np.stack([w0 - h, w0, w0 + h], axis=1).ravel().astype(np.float32)
    assert np.all(tri.astype(np.float64) == np.stack([w0 - h, w0, w0 + h], axis=1).ravel())
    rd = oracle_lib.tetra_dos(E, W, nk, tri, nthreads=2)
    num = (rd["nos"][:, 2::3] - rd["nos"][:, 0::3]) / (2 * h)
    assert np.allclose(num, rd["dos"][:, 1::3], atol=2e-4 * rd["dos"].max())


# ---------------------------------------------------------------- P7 closed-form simple cubic
def _rho2d(eps):
    a = abs(eps)
    if a >= 4.0:
        return 0.0
    # K(m) with m = 1 - eps^2/16, through ellipkm1(1-m): accurate at the log singularity eps -> 0
    return special.ellipkm1(max(eps * eps / 16.0, 1e-300)) / (2.0 * math.pi ** 2)


def _rho_sc(E):
    """Exact simple-cubic tight-binding DOS (t=1): (1/pi) int_0^pi rho2D(E + 2 cos kz) dkz,
    rho2D(e) = K(m = 1 - e^2/16)/(2 pi^2).  Textbook closed form, not the tetrahedron method."""
    if abs(E) >= 6.0:
        return 0.0
    # log singularity of rho2D at eps = 0 <-> cos kz = -E/2
    pts = []
    if abs(E) < 2.0:
        pts.append(math.acos(-E / 2.0))
    for s in (4.0, -4.0):  # support edges of rho2D
        c = (s - E) / 2.0
        if -1.0 < c < 1.0:
            pts.append(math.acos(c))
    val, _ = integrate.quad(lambda kz: _rho2d(E + 2.0 * math.cos(kz)), 0.0, math.pi,
                            points=sorted(pts) or None, limit=400, epsabs=1e-10, epsrel=1e-10)
    return val / math.pi


def _sc_reference(om):
    rho = np.array([_rho_sc(float(w)) for w in om])
    # N_exact by integrating rho between consecutive grid points
    N = np.zeros(len(om))
    prev = -6.0
    acc = 0.0
    for i, w in enumerate(om):
        w = float(w)
        hi = min(max(w, -6.0), 6.0)
        if hi > prev:
            brk = [b for b in (-2.0, 2.0) if prev < b < hi]
            acc += integrate.quad(_rho_sc, prev, hi, points=brk or None, limit=200, epsabs=1e-9)[0]
            prev = hi
        N[i] = acc
    return rho, N


def test_P7_closed_form_simple_cubic(oracle_lib):
    """Config 1 against the analytic simple-cubic DOS.  The linear tetrahedron method itself
    deviates O(1/Nk^2)..O(1/Nk) from the exact DOS, so the gates are the discretisation error
    (<= 6e-3 / 4e-3 at Nk=16, shrinking ~2x to Nk=32); the symmetry consequences
    are sharp.  A wrong V_T/V_G, a dropped tetrahedron or band of bins would fail by >> gate."""
    om = wl.omega_grid(-6.5, 6.5, 201)
    rho, Nex = _sc_reference(om)
    assert abs(rho[100] - 0.142673) < 2e-5   # rho(0), known value
    assert abs(Nex[-1] - 1.0) < 1e-6
    errs = {}
    for nkk in (16, 32):
        E, _ = wl.cosine_band((nkk,) * 3)
        r = oracle_lib.tetra_dos(E, None, (nkk,) * 3, om, windowed=True, nthreads=4)
        d, n = r["dos"][0], r["nos"][0]
        errs[nkk] = (abs(d - rho).max(), abs(n - Nex).max(), abs(d - rho).mean(), abs(n - Nex).mean())
        # sharp: particle-hole symmetry of the cosine band
        assert np.allclose(d, d[::-1], atol=1e-6)
        assert np.allclose(n + n[::-1], 1.0, atol=1e-6)
        assert abs(n[100] - 0.5) < 1e-6 and abs(n[-1] - 1.0) < 1e-9 and n[0] == 0.0
    assert errs[16][0] <= 6e-3 and errs[16][1] <= 4e-3, errs
    assert errs[32][0] <= 0.65 * errs[16][0] and errs[32][1] <= 0.65 * errs[16][1], errs
    assert errs[32][2] <= 0.5 * errs[16][2] and errs[32][3] <= 0.5 * errs[16][3], errs
    print(errs)


def test_survey_scratch_values_cfg1(oracle_lib):
    """Second opinion: values obtained by the surveyor's independent throw-away script
    (last row of the pin table), stored in tests/golden/."""
    path = os.path.join(os.path.dirname(__file__), "golden", "survey_scratch_cfg1.txt")
    rows = [l.split() for l in open(path) if l.strip() and not l.startswith("#")]
    E, _, om = wl.make_inputs("cfg1")
    r = oracle_lib.tetra_dos(E, None, (16, 16, 16), om)
    for i, dos, nos in rows:
        i = int(i)
        assert abs(r["dos"][0, i] - float(dos)) < 2e-7 and abs(r["nos"][0, i] - float(nos)) < 2e-7
    assert r["n_tb"] == 24576 and r["n_eval"] == 406053


# ---------------------------------------------------------------- P9 invariances + variants
def test_P9_invariances_and_variants(oracle_lib):
    nk = (4, 3, 5)
    nb, norb = 3, 2
    rng = np.random.default_rng(9)
    n = int(np.prod(nk))
    # energies on a 2^-10 lattice so that shifting by 1.0 is exact in fp32
    E = (rng.integers(-2048, 2048, (n, nb)) / 1024.0).astype(np.float32)
    W = rng.uniform(0, 1, (n, nb, norb)).astype(np.float32)
    om = (np.arange(-2304, 2304, 64) / 1024.0 + 2.0 ** -11).astype(np.float32)
    ref = oracle_lib.tetra_dos(E, W, nk, om)
    # periodic translation of the grid along each axis
    E3 = E.reshape(nk[2], nk[1], nk[0], nb)
    W3 = W.reshape(nk[2], nk[1], nk[0], nb, norb)
    for ax, sh in ((0, 1), (1, 2), (2, 3)):
        r = oracle_lib.tetra_dos(np.roll(E3, sh, axis=ax).reshape(n, nb), np.roll(W3, sh, axis=ax).reshape(n, nb, norb), nk, om)
        assert np.allclose(r["dos"], ref["dos"], rtol=1e-12, atol=1e-13)
        assert np.allclose(r["nos"], ref["nos"], rtol=1e-12, atol=1e-13)
    # rigid shift E -> E + 1, omega -> omega + 1 (exact in fp32 on this lattice)
    r = oracle_lib.tetra_dos(E + np.float32(1.0), W, nk, om + np.float32(1.0))
    assert np.allclose(r["dos"], ref["dos"], rtol=1e-12, atol=1e-13) and np.allclose(r["nos"], ref["nos"], rtol=1e-12, atol=1e-13)
    # SoA layout, threads, windowed variant, cube-range additivity: same numbers
    Es, Ws = wl.to_soa(E, W)
    r = oracle_lib.tetra_dos(Es, Ws, nk, om, layout=oracle_lib.SOA)
    assert np.array_equal(r["dos"], ref["dos"]) and np.array_equal(r["nos"], ref["nos"])
    r = oracle_lib.tetra_dos(E, W, nk, om, nthreads=3)
    assert np.allclose(r["dos"], ref["dos"], rtol=1e-13, atol=1e-15) and np.allclose(r["nos"], ref["nos"], rtol=1e-13, atol=1e-15)
    r = oracle_lib.tetra_dos(E, W, nk, om, windowed=True)
    assert np.allclose(r["dos"], ref["dos"], rtol=1e-13, atol=1e-15) and np.allclose(r["nos"], ref["nos"], rtol=1e-12, atol=1e-14)
    assert r["n_eval"] == ref["n_eval"] and r["n_tb"] == ref["n_tb"] == 6 * n * nb
    a = oracle_lib.tetra_dos(E, W, nk, om, cube_range=(0, 17))
    b = oracle_lib.tetra_dos(E, W, nk, om, cube_range=(17, n))
    assert np.allclose(a["dos"] + b["dos"], ref["dos"], rtol=1e-13, atol=1e-15)
    assert np.allclose(a["nos"] + b["nos"], ref["nos"], rtol=1e-13, atol=1e-15)
    # the lattice produces many exact ties and omega == corner energy never (offset 2^-11);
    # now put omega exactly ON corner energies: literal and windowed must still agree
    om2 = (np.arange(-2304, 2304, 64) / 1024.0).astype(np.float32)
    l2 = oracle_lib.tetra_dos(E, W, nk, om2)
    w2 = oracle_lib.tetra_dos(E, W, nk, om2, windowed=True)
    assert np.allclose(l2["dos"], w2["dos"], rtol=1e-13, atol=1e-15) and np.allclose(l2["nos"], w2["nos"], rtol=1e-12, atol=1e-14)


def test_windowed_oracle_equals_literal_on_configs_1_and_2(oracle_lib, cache_dir):
    """BASELINE.md 3 / SURVEY.md 8(c) step 5: the windowed variant (skips omega outside (E1, E4), Eq. 15 as step +
    prefix sum) may stand in for the literal loop at full size only once it reproduces it on the configs the literal
    loop can afford: config 1 and config 2 (Nk = 32, 8 bands, 8 orbitals, 1000 energies) -- DOS and N to 1e-12
    relative, equal work counters."""
    for name in ("cfg1", "cfg2"):
        cfg = wl.CONFIGS[name]
        E, W, om = wl.make_inputs(cfg, cache_dir)
        lit = oracle_lib.tetra_dos(E, W, cfg.nk, om, nthreads=oracle_lib.max_threads())
        win = oracle_lib.tetra_dos(E, W, cfg.nk, om, windowed=True, nthreads=oracle_lib.max_threads())
        assert lit["n_eval"] == win["n_eval"] and lit["n_tb"] == win["n_tb"] == 6 * int(np.prod(cfg.nk)) * cfg.nb
        assert list(lit["n_case"]) == list(win["n_case"])
        scale_d = np.abs(lit["dos"]).max()
        assert np.abs(lit["dos"] - win["dos"]).max() <= 1e-12 * scale_d
        pos = lit["nos"] > 0
        assert np.array_equal(pos, win["nos"] > 0)
        assert (np.abs(lit["nos"] - win["nos"])[pos] / lit["nos"][pos]).max() <= 1e-12


def test_flat_band_and_grid_outside_bands(oracle_lib):
    """Flat band: DOS = 0 at every omega (delta spike lost, inherent), N = step at e, 0 AT e.
    omega grid entirely below / above the bands: zeros / full count."""
    nk = (3, 3, 3)
    n = 27
    E = np.full((n, 1), 0.25, dtype=np.float32)
    W = np.full((n, 1, 2), 0.5, dtype=np.float32)
    om = np.array([0.0, 0.25, 0.5], dtype=np.float32)
    for windowed in (False, True):
        r = oracle_lib.tetra_dos(E, W, nk, om, windowed=windowed)
        assert not r["dos"].any() and r["n_eval"] == 0
        assert np.allclose(r["nos"], [[0, 0, 0.5], [0, 0, 0.5]], atol=1e-15)
    E, W = wl.random_bands(nk, 2, 2, seed=3)
    lo = oracle_lib.tetra_dos(E, W, nk, np.array([-5.0, -4.0], dtype=np.float32))
    hi = oracle_lib.tetra_dos(E, W, nk, np.array([4.0, 5.0], dtype=np.float32), windowed=True)
    assert not lo["dos"].any() and not lo["nos"].any() and not hi["dos"].any()
    assert np.allclose(hi["nos"], W.astype(np.float64).sum(axis=(0, 1))[:, None] / n, atol=1e-13)


def test_per_k_weights_reproduce_the_orbital_sums(oracle_lib):
    """Pin of oracle.tetra_weights (Eq. 5-7): with X = b_{n,m} the per-k weights must give back
    N_m and DOS_m of tetra_dos (Eq. 7 vs Eq. 8-9: the same sum in another order), which fixes the
    corner <-> k-point bookkeeping; every k-point is a corner of 24 tetrahedra, so above all bands each weight
    is 24 V = 1/nk (Eq. 15) and below all bands it is 0 (Eq. 11)."""
    nk, nb, norb = (4, 3, 5), 3, 4
    E, W = wl.random_bands(nk, nb, norb, seed=17)
    om = np.array([-2.0, -0.6, -0.1, 0.05, 0.4, 0.9, 2.0], dtype=np.float32)
    for layout in (oracle_lib.AOS, oracle_lib.SOA):
        Ex = E if layout == oracle_lib.AOS else np.ascontiguousarray(E.T)
        wk, dwk = oracle_lib.tetra_weights(Ex, nk, om, layout=layout)
        ref = oracle_lib.tetra_dos(E, W, nk, om)
        Wd = W.astype(np.float64)                                  # [k][n][m]
        nos = np.einsum("enk,knm->me", wk, Wd)
        dos = np.einsum("enk,knm->me", dwk, Wd)
        assert np.allclose(nos, ref["nos"], rtol=1e-12, atol=1e-15)
        assert np.allclose(dos, ref["dos"], rtol=1e-12, atol=1e-14)
        assert not wk[0].any() and not dwk[0].any()
        assert np.allclose(wk[-1], 1.0 / np.prod(nk), rtol=1e-13) and not dwk[-1].any()
        assert (wk >= 0).all()


def test_eigh_bands_pins(oracle_lib):
    """Pin of oracle.eigh_bands (Eq. 1): a closed-form 2 x 2 Hermitian matrix [[a, g], [conj(g), b]] has
    E = (a+b)/2 -+ sqrt(((a-b)/2)^2 + |g|^2) and |a_-^1|^2 = (1 + (b-a)/(2 r)) / 2 with r the square root; for the
    seeded 8-orbital Hamiltonian H a = E a holds to rounding, the weights of every band and of every orbital sum to 1,
    and the result equals what workloads.tb8_bands (an independent call path) delivers."""
    a, b, g = 0.3, -1.1, 0.4 - 0.7j
    H = np.array([[[a, g], [np.conj(g), b]]])
    E, W = oracle_lib.eigh_bands(H)
    r = np.sqrt(((a - b) / 2) ** 2 + abs(g) ** 2)
    assert np.allclose(E[0], [(a + b) / 2 - r, (a + b) / 2 + r], rtol=1e-14)
    w_lower_on_orbital0 = 0.5 * (1 + (b - a) / (2 * r))
    assert np.allclose(W[0, 0], [w_lower_on_orbital0, 1 - w_lower_on_orbital0], rtol=1e-13)
    nk = (4, 3, 5)
    H = wl.tb8_hamiltonian(nk)
    assert np.array_equal(H, H.conj().transpose(0, 2, 1))                      # exactly Hermitian after the cast
    E, W = oracle_lib.eigh_bands(H)
    assert np.all(np.diff(E, axis=1) >= 0)
    assert np.allclose(W.sum(axis=1), 1.0, atol=1e-13) and np.allclose(W.sum(axis=2), 1.0, atol=1e-13)
    w, U = np.linalg.eigh(H.astype(np.complex128))
    assert np.abs(np.einsum("kij,kjn->kin", H.astype(np.complex128), U) - U * w[:, None, :]).max() < 1e-13
    Eb, Wb = wl.tb8_bands(nk, threads=1)
    assert np.abs(E - Eb).max() < 2e-6 and np.abs(W - Wb).max() < 2e-5      # complex64 H against complex128 H


@pytest.mark.parametrize("nb,seed", [(3, 1), (8, 2)])
def test_eigh_bands_orientation_by_hellmann_feynman(oracle_lib, nb, seed):
    """Which index of W is the band and which the orbital (Eq. 1 -> E_n(k), a_n^m(k), :37-39; Eq. 3
    b_mn = a* a, :47) is pinned without reference to any eigenvector routine: by the Hellmann-Feynman theorem
    dE_n / dH_mm = |a_n^m|^2, so a central difference of the n-th EIGENVALUE returned by eigh_bands under a shift of
    the m-th diagonal element of H must reproduce W[n][m].  |U|^2 of a 2 x 2 unitary is symmetric, so only orders >= 3
    can tell W[n][m] from W[m][n]; a transposed W fails this by O(1)."""
    rng = np.random.default_rng(seed)
    M = rng.normal(size=(nb, nb)) + 1j * rng.normal(size=(nb, nb))
    H = (M + M.conj().T) / 2
    E0, W = oracle_lib.eigh_bands(H[None])
    assert np.diff(E0[0]).min() > 1e-2                         # well separated levels: the derivative exists
    h = 1e-5
    D = np.empty((nb, nb))                                     # D[n][m] = dE_n / dH_mm
    for m in range(nb):
        Hp, Hm = H.copy(), H.copy()
        Hp[m, m] += h
        Hm[m, m] -= h
        Ep, _ = oracle_lib.eigh_bands(Hp[None])
        Em, _ = oracle_lib.eigh_bands(Hm[None])
        D[:, m] = (Ep[0] - Em[0]) / (2 * h)
    assert np.abs(D - W[0]).max() < 1e-7
    assert np.abs(D - W[0].T).max() > 1e-2                     # the pin can see the orientation
