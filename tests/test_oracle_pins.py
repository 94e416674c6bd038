"""Pins of the CPU oracle against what the paper and the mathematics fix (no GPU, no CUDA path).

Each test names the passage it pins (PAPER.md:<line>).  Nothing here compares the oracle with itself:
expected values are the paper's printed numbers/tables (tests/golden/), closed forms, numpy dense algebra,
or brute-force ray counting.
"""
import math
import os

import numpy as np
import pytest

from workloads import make_field

GOLD = os.path.join(os.path.dirname(__file__), "golden")
DIRS = ["E", "W", "N", "S", "F", "B"]


# ----------------------------------------------------------------------------- constants

def test_2d_constants_eq5_6_7_17(oracle):
    """Eq. 5 (:75) A_E = 2 dy; Eq. 6 (:86) = c_xy; Eq. 7 (:89) = c_xy + c_xx; Eq. 8 (:94)."""
    dx, dy = 0.3, 0.7
    K = oracle.constants(5, 5, 1, dx, dy, 1.0)
    dd = math.hypot(dx, dy)
    assert K["F"][0] == pytest.approx(2 * dy, rel=1e-15)
    assert K["F"][1] == pytest.approx(2 * dx, rel=1e-15)
    assert K["A_tot"] == pytest.approx(4 * (dx + dy), rel=1e-15)
    assert K["c"][0, 1] == pytest.approx(dx + dy - dd, rel=1e-14)              # Eq. 6
    assert K["c"][0, 1] + K["c"][0, 0] == pytest.approx(dy - dx + dd, rel=1e-14)  # Eq. 7
    # Eq. 6 is printed as an integral too (:84): evaluate it numerically
    al = math.atan(dy / dx)
    th = np.linspace(0, al, 200001)
    i1 = np.trapezoid(dx * np.sin(th), th)
    th = np.linspace(al, math.pi / 2, 200001)
    i2 = np.trapezoid(dy * np.cos(th), th)
    assert K["c"][0, 1] == pytest.approx(i1 + i2, rel=1e-9)


def test_appendix_constants_eq45_46(oracle):
    D = 0.37
    K = oracle.constants(3, 3, 1, D, D, 1.0)
    assert K["c"][0, 0] == pytest.approx(D * (2 * math.sqrt(2) - 2), rel=1e-14)
    assert K["c"][1, 1] == pytest.approx(D * (2 * math.sqrt(2) - 2), rel=1e-14)
    assert K["c"][0, 1] == pytest.approx(D * (2 - math.sqrt(2)), rel=1e-14)
    assert K["A_tot"] == pytest.approx(8 * D, rel=1e-15)                      # :585


def test_3d_isotropic_constants_eq34_35(oracle):
    """Eq. 34-35 (:322-326) to the 13 digits printed; Eq. 24 (:262); sum rule = pi D^2 (Eq. 23)."""
    for D in (1.0, 0.25):
        K = oracle.constants(4, 4, 4, D, D, D)
        assert K["c"][0, 0] / D**2 == pytest.approx(0.6277684243304, abs=5e-14)
        assert K["c"][0, 1] / D**2 == pytest.approx(0.6284560573148, abs=5e-14)
        assert K["A_tot"] == pytest.approx(6 * math.pi * D * D, rel=1e-15)
        assert K["c"][0, 0] + 4 * K["c"][0, 1] == pytest.approx(math.pi * D * D, rel=1e-13)
    # the general-spacing quadrature (reading A7) reproduces Eq. 34 at dx=dy=dz
    assert oracle.far_face_constant(1.0, 1.0, 1.0) == pytest.approx(0.6277684243304, abs=5e-13)


def test_3d_general_constants_symmetry_and_sum_rule(oracle):
    """c_jk = c_kj (:304); every face's pieces sum to its total pi*d*d (Eq. 23 :258, Eq. 25 :266)."""
    dx, dy, dz = 1.0, 0.7, 1.9
    K = oracle.constants(4, 4, 4, dx, dy, dz)
    c, F = K["c"], K["F"]
    assert np.allclose(c, c.T, rtol=0, atol=0)
    assert np.all(c > 0)
    for a in range(3):
        b, cc = (a + 1) % 3, (a + 2) % 3
        assert c[a, a] + 2 * c[a, b] + 2 * c[a, cc] == pytest.approx(F[a], rel=1e-13)
    assert F[1] == pytest.approx(math.pi * dx * dz)
    # near-isotropic spacing must approach the closed forms continuously
    Kn = oracle.constants(4, 4, 4, 1.0, 1.0, 1.0 + 1e-9)
    Ki = oracle.constants(4, 4, 4, 1.0, 1.0, 1.0)
    assert np.allclose(Kn["c"], Ki["c"], rtol=1e-8)


# ----------------------------------------------------------------------------- general-spacing constants, pinned
# without the oracle's own quadrature and without the CUDA library.  Everything below is derived
# here from the geometric definition (Fig. 5b): the measure of the rays crossing two surface
# elements dA1, dA2 a distance r apart is cos(th1) cos(th2) / r^2 dA1 dA2 (projected area x solid angle, Eq. 22 :253;
# a whole face collects pi * area, Eq. 23 :258).

def _far_face_adaptive(da, db, dc):
    """c_aa: face a of C (db x dc) and the far face of Q = C + e_a, parallel at distance da: cos th1 = cos th2 = da / r.
    The two area integrals reduce to differences u, v (int_0^L int_0^L f(|x1 - x2|) = 2 int_0^L (L - u) f(u) du):
    c_aa = 4 int_0^db int_0^dc (db - u)(dc - v) da^2 / (u^2 + v^2 + da^2)^2 dv du.  Adaptive QUADPACK, not the
    oracle's fixed Gauss-Legendre panels."""
    from scipy import integrate
    val, err = integrate.dblquad(lambda v, u: (db - u) * (dc - v) * da * da / (u * u + v * v + da * da) ** 2,
                                 0.0, db, 0.0, dc, epsabs=1e-15, epsrel=1e-13)
    return 4.0 * val, 4.0 * err


def _far_face_mpmath(da, db, dc):
    """The same integral with mpmath's tanh-sinh quadrature at 30 digits (a second, unrelated integrator)."""
    import mpmath as mp
    mp.mp.dps = 30
    f = lambda u, v: (db - u) * (dc - v) * da * da / (u * u + v * v + da * da) ** 2
    return float(4 * mp.quad(f, [0, db], [0, dc]))


def _side_wall_1d(da, db, dc):
    """c_ab by DIRECT integration of the side-wall measure (not through the sum rule): face a of C at a = 0,
    (b, c) in [0, db] x [0, dc], normal e_a; the side wall of Q at b = db, (a, c) in [0, da] x [0, dc], normal e_b.
    With s = db - b1 and v = |c2 - c1|: cos th1 = a / r, cos th2 = s / r, r^2 = a^2 + s^2 + v^2,
      c_ab = 2 int_0^da int_0^db int_0^dc (dc - v) a s / r^4 dv ds da.
    The a and s integrals are elementary (int a / (a^2 + k)^2 = -1 / (2 (a^2 + k)), int s / (s^2 + m) = ln(s^2 + m) / 2):
      c_ab = 1/2 int_0^dc (dc - v) [ ln((db^2 + v^2) / v^2) - ln((da^2 + db^2 + v^2) / (da^2 + v^2)) ] dv,
    a 1D integral with an integrable log singularity at v = 0."""
    import mpmath as mp
    mp.mp.dps = 30
    f = lambda v: (dc - v) * (mp.log((db * db + v * v) / (v * v)) - mp.log((da * da + db * db + v * v) / (da * da + v * v)))
    return float(mp.quad(f, [0, dc / 64, dc]) / 2)


def _side_wall_3d_bruteforce(da, db, dc):
    """The unreduced kernel a s / r^4 over (a, s, c1, c2) by plain nested adaptive quadrature in the three variables
    (a, s, v) -- checks the reductions above at a looser tolerance."""
    import warnings
    from scipy import integrate
    with warnings.catch_warnings():
        warnings.simplefilter("ignore", integrate.IntegrationWarning)      # the kernel peaks along the shared edge
        val, err = integrate.tplquad(lambda v, s, a: (dc - v) * a * s / (a * a + s * s + v * v) ** 2,
                                     0.0, da, 0.0, db, 0.0, dc, epsabs=1e-9, epsrel=1e-9)
    return 2.0 * val


ANISO = [(1.0, 0.7, 1.9), (1.0 / 263, 1.0 / 15, 1.0 / 4), (0.25, 1.0 / 15, 1.0 / 263), (1.0, 1.0, 1.0)]


@pytest.mark.parametrize("sp", ANISO)
def test_far_face_constant_vs_adaptive_quadrature(oracle, sp):
    """oracle.far_face_constant (fixed Gauss-Legendre on dyadic panels) against two adaptive integrators of the defining
    integral written out in this file, for every axis ordering, at strongly anisotropic spacing (66:1).  A wrong panel
    count, a swapped db / dc or a dropped factor fails here without the CUDA library being imported."""
    for a in range(3):
        da, db, dc = sp[a], sp[(a + 1) % 3], sp[(a + 2) % 3]
        got = oracle.far_face_constant(da, db, dc)
        F = math.pi * db * dc
        ref_mp = _far_face_mpmath(da, db, dc)
        ref_qp, err = _far_face_adaptive(da, db, dc)
        assert ref_qp == pytest.approx(ref_mp, rel=1e-10, abs=1e-13 * F)          # the two integrators agree
        # what enters the stencil is c / A_tot; relative to the face total F_a the pin is 1e-11
        assert abs(got - ref_mp) <= 1e-11 * F, (a, got, ref_mp)
        assert got == pytest.approx(ref_mp, rel=1e-9)                               # and relative to c_aa itself
        # the integral is symmetric in (db, dc) but NOT in (da, db): a swapped argument is visible at these spacings
        if abs(da - db) > 1e-12:
            assert abs(oracle.far_face_constant(db, da, dc) - ref_mp) > 1e-6 * F


@pytest.mark.parametrize("sp", ANISO)
def test_cross_constants_vs_direct_side_wall_quadrature(oracle, sp):
    """The oracle obtains c_ab from the sum rules c_aa + 2 c_ab + 2 c_ac = F_a and c_ab = c_ba (:304).  Here each c_ab is
    integrated DIRECTLY over the side wall (survey probe A7 re-established): agreement to 1e-11 F_a pins the sum-rule
    construction -- and with it far_face_constant -- from a second, independent side."""
    dx, dy, dz = sp
    K = oracle.constants(4, 4, 4, dx, dy, dz)
    c, F = K["c"], K["F"]
    for a in range(3):
        for b in range(3):
            if a == b:
                continue
            cc = 3 - a - b
            direct = _side_wall_1d(sp[a], sp[b], sp[cc])
            assert abs(c[a, b] - direct) <= 1e-11 * F[a], (a, b, c[a, b], direct)
            assert c[a, b] == pytest.approx(direct, rel=1e-8)
    # the reduction to one dimension itself, against the unreduced 3D kernel (looser: nested QUADPACK near the edge)
    a, b, cc = 0, 1, 2
    assert _side_wall_1d(sp[a], sp[b], sp[cc]) == pytest.approx(_side_wall_3d_bruteforce(sp[a], sp[b], sp[cc]), rel=2e-6)
    # every ray through face a leaves Q through exactly one of its five other faces (Eq. 23 :258)
    for a in range(3):
        b, cc = (a + 1) % 3, (a + 2) % 3
        tot = _far_face_mpmath(sp[a], sp[b], sp[cc]) + 2 * _side_wall_1d(sp[a], sp[b], sp[cc]) + 2 * _side_wall_1d(sp[a], sp[cc], sp[b])
        assert tot == pytest.approx(math.pi * sp[b] * sp[cc], rel=1e-11)


# ----------------------------------------------------------------------------- brute-force ray counts (P11)

def _mc_fractions(da, db, dc, n, rng, three_d):
    """Rays leave the shared face into Q (size da along the face normal) with the cosine-weighted measure of
    Eq. 4/22 (:71, :253); returns the fractions that leave Q through far, +b, -b, +c, -c faces."""
    if not three_d:
        y0 = rng.uniform(-db / 2, db / 2, n)
        sin_t = rng.uniform(-1, 1, n)                 # pdf ~ cos(theta) d theta
        tan_t = sin_t / np.sqrt(1 - sin_t**2)
        y = y0 + da * tan_t
        return np.array([np.mean(np.abs(y) <= db / 2), np.mean(y > db / 2), np.mean(y < -db / 2), 0.0, 0.0])
    y0 = rng.uniform(-db / 2, db / 2, n)
    z0 = rng.uniform(-dc / 2, dc / 2, n)
    s2 = rng.uniform(0, 1, n)                         # sin^2(theta) uniform: pdf ~ cos sin d theta
    st, ct = np.sqrt(s2), np.sqrt(1 - s2)
    ph = rng.uniform(0, 2 * np.pi, n)
    vy, vz = st * np.cos(ph), st * np.sin(ph)
    with np.errstate(divide="ignore"):
        t_far = da / ct
        t_b = np.where(vy > 0, (db / 2 - y0) / vy, (-db / 2 - y0) / vy)
        t_c = np.where(vz > 0, (dc / 2 - z0) / vz, (-dc / 2 - z0) / vz)
    first = np.argmin(np.stack([t_far, t_b, t_c]), axis=0)
    return np.array([np.mean(first == 0), np.mean((first == 1) & (vy > 0)), np.mean((first == 1) & (vy < 0)),
                     np.mean((first == 2) & (vz > 0)), np.mean((first == 2) & (vz < 0))])


@pytest.mark.parametrize("spacing", [(1.0, 1.0, None), (0.3, 0.7, None), (1.0, 1.0, 1.0), (1.0, 0.7, 1.9)])
def test_constants_vs_monte_carlo_ray_count(oracle, spacing):
    """c_aa / F_a and c_ab / F_a are the fractions of rays through face a that crossed the far / side faces of the
    neighbour cell (Fig. 4 :185, Eq. 14 :191, Fig. 5 :245).  Statistical pin: 4e6 rays, 5 sigma."""
    dx, dy, dz = spacing
    three_d = dz is not None
    K = oracle.constants(4, 4, 4 if three_d else 1, dx, dy, dz if three_d else 1.0)
    d = [dx, dy, dz if three_d else 1.0]
    rng = np.random.default_rng(1234)
    n = 4_000_000
    for a in range(3 if three_d else 2):
        if three_d:
            b, c = (a + 1) % 3, (a + 2) % 3
        else:
            b, c = 1 - a, 2
        fr = _mc_fractions(d[a], d[b], d[c], n, rng, three_d)
        exp = np.array([K["c"][a, a], K["c"][a, b], K["c"][a, b], K["c"][a, c], K["c"][a, c]]) / K["F"][a]
        sig = np.sqrt(np.maximum(exp * (1 - exp), 1e-12) / n)
        assert np.all(np.abs(fr - exp) < 5 * sig + 1e-12), (a, fr, exp)


def test_weights_vs_monte_carlo_on_masked_grid(oracle):
    """Whole weight assembly (Eq. 15, 16, 18, 25) from first principles on a tiny masked 3D grid with anisotropic
    spacing: trace rays back one cell, classify by the validity of the cell they came from."""
    rng = np.random.default_rng(7)
    shape = (4, 5, 4)
    v = (rng.random(shape) > 0.3).astype(np.uint8)
    dx, dy, dz = 1.0, 0.8, 1.3
    d = [dx, dy, dz]
    w1, w0, w0C = oracle.weights(v, dx, dy, dz)
    K = oracle.constants(4, 5, 4, dx, dy, dz)
    nz, ny, nx = shape

    def valid(i, j, k):
        return 0 <= i < nx and 0 <= j < ny and 0 <= k < nz and v[k, j, i]

    n = 400_000
    checked = 0
    cells = [tuple(c) for c in np.argwhere(v == 1)[::5]]
    for (k, j, i) in cells:
        C = np.array([i, j, k])
        AC = 0.0
        for dd in range(6):
            a, sg = dd // 2, (1 if dd % 2 == 0 else -1)
            b, c = (a + 1) % 3, (a + 2) % 3
            e = np.zeros(3, int); e[a] = sg
            Q = C + e
            share = K["F"][a] / K["A_tot"]
            if not valid(*Q):
                AC += share
                assert w1[dd, k, j, i] == 0 and w0[dd, k, j, i] == 0
                continue
            fr = _mc_fractions(d[a], d[b], d[c], n, rng, True)
            eb = np.zeros(3, int); eb[b] = 1
            ec = np.zeros(3, int); ec[c] = 1
            origin = [Q + e, Q + eb, Q - eb, Q + ec, Q - ec]
            new = sum(f for f, o in zip(fr, origin) if valid(*o)) * share
            old = sum(f for f, o in zip(fr, origin) if not valid(*o)) * share
            tol = 5 * math.sqrt(0.25 / n) * share * 2
            assert abs(w1[dd, k, j, i] - new) < tol
            assert abs(w0[dd, k, j, i] - old) < tol
            checked += 1
        assert w0C[k, j, i] == pytest.approx(AC, rel=1e-12, abs=1e-15)
    assert checked >= 10


# ----------------------------------------------------------------------------- Table 1 (P1) and S (P2)

def _parse_table1():
    rows, fixes = {}, []
    for line in open(os.path.join(GOLD, "table1_3x3.txt")):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        t = line.split()
        if t[0] == "FIX":
            fixes.append((t[1], int(t[2]), t[3]))
        else:
            rows[t[0]] = t[1:]
            assert len(t) == 10
    return rows, fixes


def _tok(tok, D):
    s2 = math.sqrt(2)
    val = {"0": 0.0, "2D": 2 * D, "4D": 4 * D, "cxx": D * (2 * s2 - 2), "cyy": D * (2 * s2 - 2), "cxy": D * (2 - s2),
           "2cxy": 2 * D * (2 - s2)}
    return sum(val[p] for p in tok.split("+"))


def test_table1_3x3_example(oracle):
    """All ten A_j^i of all nine cells; 88 entries verbatim + the 2 of erratum A10."""
    D = 0.5
    v = np.ones((3, 3), np.uint8)
    w1, w0, w0C = oracle.weights(v, D, D)
    Atot = 8 * D
    rows, fixes = _parse_table1()
    # cell number (1..9, row-major from the top) -> numpy index (j, i) with j up
    pos = {c: (2 - (c - 1) // 3, (c - 1) % 3) for c in range(1, 10)}
    ours = {}
    for c, (j, i) in pos.items():
        ours[("A_C^n", c)] = w0C[j, i] * Atot
        ours[("A_C^n+1", c)] = 0.0                                   # Eq. 11 :113
        for dd, name in enumerate(DIRS[:4]):
            ours[(f"A_{name}^n+1", c)] = w1[dd, j, i] * Atot
            ours[(f"A_{name}^n", c)] = w0[dd, j, i] * Atot
    fixed = {(r, c): tok for r, c, tok in fixes}
    n_verbatim = 0
    for r, toks in rows.items():
        for c in range(1, 10):
            tok = fixed.get((r, c), toks[c - 1])
            assert ours[(r, c)] == pytest.approx(_tok(tok, D), abs=1e-14), (r, c, tok)
            n_verbatim += (r, c) not in fixed
    assert n_verbatim == 88 and len(fixed) == 2
    # the verbatim cell-4 entries break the table's own mirror symmetries (justifies A10)
    assert rows["A_N^n"][3] != rows["A_N^n"][5] and rows["A_N^n"][3] != rows["A_S^n"][3]
    # "all coefficients sum to A_tot, which is always required" (:631)
    for c in range(1, 10):
        assert sum(val for (r, cc), val in ours.items() if cc == c) == pytest.approx(Atot, rel=1e-14)


def test_source_eq49_50(oracle):
    """S_1 and S_5 of the 3x3 example (Eq. 49-50 :656-662): signs, 1/2 face average, missing-neighbour rule."""
    D = 0.25
    rng = np.random.default_rng(3)
    fx, fy = rng.normal(size=(3, 3)), rng.normal(size=(3, 3))
    v = np.ones((3, 3), np.uint8)
    w1, w0, _ = oracle.weights(v, D, D)
    S = oracle.source(v, w1, w0, fx, fy, None, D, D)
    pos = {c: (2 - (c - 1) // 3, (c - 1) % 3) for c in range(1, 10)}
    f_x = {c: fx[pos[c]] for c in pos}
    f_y = {c: fy[pos[c]] for c in pos}
    S1 = -(D / 8) * (f_x[2] + f_x[1] - f_y[4] - f_y[1])
    S5 = -(D / 8) * (f_x[6] - f_x[4] + f_y[2] - f_y[8])
    assert S[pos[1]] == pytest.approx(S1, rel=1e-13)
    assert S[pos[5]] == pytest.approx(S5, rel=1e-13)


# ----------------------------------------------------------------------------- invariants (P4)

@pytest.mark.parametrize("shape,sp", [((9, 11), (0.3, 0.5, 1.0)), ((6, 7, 8), (1.0, 1.0, 1.0)), ((6, 7, 8), (0.4, 1.1, 0.7)),
                                      ((1, 9), (1.0, 1.0, 1.0)), ((5, 1, 6), (1.0, 2.0, 1.0))])
def test_weights_sum_to_one_and_nonnegative(oracle, shape, sp):
    """w_C^n + sum_j (w_j^{n+1} + w_j^n) = 1 at every valid cell, any mask/spacing (:631, Eq. 8, Eq. 24)."""
    rng = np.random.default_rng(11)
    v = (rng.random(shape) > 0.25).astype(np.uint8)
    w1, w0, w0C = oracle.weights(v, *sp)
    tot = w0C + w1.sum(0) + w0.sum(0)
    assert np.allclose(tot[v == 1], 1.0, rtol=0, atol=1e-14)
    assert np.all(tot[v == 0] == 0)
    assert w1.min() >= 0 and w0.min() >= -1e-16 and w0C.min() >= 0
    # interior cell of a full box: only new-iteration weights, w = F_a / A_tot (Eq. 5)
    full = np.ones(shape, np.uint8)
    w1f, w0f, w0Cf = oracle.weights(full, *sp)
    K = oracle.constants(shape[-1], shape[-2], shape[0] if len(shape) == 3 else 1, *sp)
    if min(shape) >= 5:
        ctr = tuple(s // 2 for s in shape)
        for dd in range(2 * len(shape)):
            assert w1f[(dd,) + ctr] == pytest.approx(K["F"][dd // 2] / K["A_tot"], rel=1e-14)
            assert w0f[(dd,) + ctr] == pytest.approx(0.0, abs=1e-16)


def test_validity_eq13(oracle):
    """NaN in any used component or mask == 0 marks a cell missing (Eq. 13 :176, :158)."""
    gx, gy, gz = np.zeros((2, 3, 4)), np.zeros((2, 3, 4)), np.zeros((2, 3, 4))
    gx[0, 0, 1] = np.nan
    gz[1, 2, 3] = np.nan
    mask = np.ones((2, 3, 4), np.uint8)
    mask[1, 1, 1] = 0
    v = oracle.validity(gx, gy, gz, mask)
    exp = np.ones((2, 3, 4), np.uint8)
    exp[0, 0, 1] = exp[1, 2, 3] = exp[1, 1, 1] = 0
    assert np.array_equal(v, exp)
    # 2D ignores gz
    v2 = oracle.validity(gx[0], gy[0], None, None)
    assert v2.sum() == 11


# ----------------------------------------------------------------------------- dense algebra pins (P5, P6)

def _dense(v, w1, w0=None, w0C=None):
    """M (and W^n) as dense numpy matrices, filled entry by entry from the stored weights (Eq. 12 :119 with the
    sign convention of reading A1), then handed to numpy.linalg."""
    shape = v.shape
    N = v.size
    idx = np.arange(N).reshape(shape)
    M = np.zeros((N, N))
    W = np.zeros((N, N))
    nd = len(shape)
    for C in np.ndindex(shape):
        if not v[C]:
            continue
        r = idx[C]
        M[r, r] = 1.0
        if w0C is not None:
            W[r, r] = w0C[C]
        for dd in range(2 * nd):
            a, sg = dd // 2, (1 if dd % 2 == 0 else -1)
            Q = list(C)
            Q[nd - 1 - a] += sg
            if not (0 <= Q[nd - 1 - a] < shape[nd - 1 - a]):
                continue
            q = idx[tuple(Q)]
            M[r, q] -= w1[(dd,) + C]
            if w0 is not None:
                W[r, q] += w0[(dd,) + C]
    return M, W


@pytest.mark.parametrize("shape,sp", [((10, 12), (1.0, 0.6, 1.0)), ((5, 6, 6), (1.0, 1.0, 1.0))])
def test_inner_cg_vs_dense_lu(oracle, shape, sp):
    """Textbook CG on the non-symmetric M (reading A2) reaches the dense-LU solution on random masks."""
    rng = np.random.default_rng(5)
    v = (rng.random(shape) > 0.15).astype(np.uint8)
    w1, w0, w0C = oracle.weights(v, *sp)
    M, _ = _dense(v, w1)
    assert np.abs(M - M.T).max() > 1e-3            # the operator really is non-symmetric next to boundaries
    rhs = rng.normal(size=shape) * v
    x, k = oracle.cg(v, w1, rhs, np.zeros(shape), 1e-13 * np.linalg.norm(rhs), 2000)
    keep = v.ravel() == 1
    xs = np.linalg.solve(M[np.ix_(keep, keep)], rhs.ravel()[keep])
    assert k < 2000
    assert np.linalg.norm(x.ravel()[keep] - xs) / np.linalg.norm(xs) < 1e-10
    # apply_M agrees with the densely assembled matrix (pins the operator's indexing/signs through numpy)
    p = rng.normal(size=shape) * v
    assert np.allclose(oracle.apply_M(v, w1, p).ravel(), M @ p.ravel(), rtol=0, atol=1e-14)


@pytest.mark.parametrize("shape,sp", [((9, 10), (1.0, 0.6, 1.0)), ((5, 5, 6), (1.0, 1.3, 0.8))])
def test_outer_iteration_vs_dense_solves(oracle, shape, sp):
    """Algorithm 1 (:128-150) with numpy dense solves of Eq. 12, iteration by iteration, against oracle.solve with a
    tight inner CG; and the limit: the fixed point solves L P = S, L = weighted graph Laplacian F_a/A_tot (P5)."""
    rng = np.random.default_rng(9)
    f = make_field("gaussians2d" if len(shape) == 2 else "fourier3d", shape, seed=2, noise=0.05, kmax=2.0)
    mask = (rng.random(shape) > 0.12).astype(np.uint8)
    d = sp
    g = f["g"] + [None] * (3 - len(f["g"]))
    v = oracle.validity(g[0], g[1], g[2], mask)
    w1, w0, w0C = oracle.weights(v, *d)
    S = oracle.source(v, w1, w0, g[0], g[1], g[2], *d)
    M, W = _dense(v, w1, w0, w0C)
    keep = v.ravel() == 1
    Mk, Wk, Sk = M[np.ix_(keep, keep)], W[np.ix_(keep, keep)], S.ravel()[keep]
    P = np.zeros(keep.sum())
    for n in range(1, 6):
        P = np.linalg.solve(Mk, Wk @ P + Sk)
        Po, info = oracle.solve(g[0], g[1], g[2], mask, *d, tol=0.0, max_outer=n, max_cg=400)
        assert info["outer_iters"] == n
        assert np.linalg.norm(Po.ravel()[keep] - P) / np.linalg.norm(P) < 1e-10
        assert np.all(np.isnan(Po.ravel()[~keep]))
    # fixed point: (M - W) P = S.  L is built here from its definition, not from the oracle's weights.
    K = oracle.constants(shape[-1], shape[-2], shape[0] if len(shape) == 3 else 1, *d)
    t = K["F"] / K["A_tot"]
    N = v.size
    idx = np.arange(N).reshape(shape)
    L = np.zeros((N, N))
    nd = len(shape)
    for C in np.ndindex(shape):
        if not v[C]:
            continue
        for a in range(nd):
            for sg in (1, -1):
                Q = list(C); Q[nd - 1 - a] += sg
                if 0 <= Q[nd - 1 - a] < shape[nd - 1 - a] and v[tuple(Q)]:
                    L[idx[C], idx[C]] += t[a]
                    L[idx[C], idx[tuple(Q)]] -= t[a]
    Lk = L[np.ix_(keep, keep)]
    assert np.allclose(Lk, Mk - Wk, rtol=0, atol=1e-14)
    assert np.allclose(Lk, Lk.T)
    Pstar = np.linalg.lstsq(Lk, Sk, rcond=None)[0]
    Po, info = oracle.solve(g[0], g[1], g[2], mask, *d, tol=1e-11, max_outer=20000, max_cg=400)
    assert info["converged"]
    # compare per connected component after mean removal (reading A12)
    from scipy.sparse import csr_matrix
    from scipy.sparse.csgraph import connected_components
    ncomp, lab = connected_components(csr_matrix(np.abs(Lk) > 0), directed=False)
    a, b = Po.ravel()[keep].copy(), Pstar.copy()
    for cpt in range(ncomp):
        m = lab == cpt
        a[m] -= a[m].mean(); b[m] -= b[m].mean()
    assert np.linalg.norm(a - b) / np.linalg.norm(b) < 1e-8


def _dense_laplacian(v, t):
    """L from its definition (valid links carry t_a = F_a / A_tot), independent of the oracle's weights."""
    shape, nd = v.shape, v.ndim
    idx = np.arange(v.size).reshape(shape)
    L = np.zeros((v.size, v.size))
    for C in np.ndindex(shape):
        if not v[C]:
            continue
        for a in range(nd):
            for sg in (1, -1):
                Q = list(C); Q[nd - 1 - a] += sg
                if 0 <= Q[nd - 1 - a] < shape[nd - 1 - a] and v[tuple(Q)]:
                    L[idx[C], idx[C]] += t[a]
                    L[idx[C], idx[tuple(Q)]] -= t[a]
    return L


@pytest.mark.parametrize("shape,sp", [((9, 10), (1.0, 0.6, 1.0)), ((5, 5, 6), (1.0, 1.3, 0.8))])
def test_direct_solve_vs_dense_pseudo_inverse(oracle, shape, sp):
    """oracle.solve_direct (CG on L P = S from P = 0, SURVEY 8(f) NEXT-2 iii) returns pinv(L) S -- the solution with
    zero mean on every connected component -- with L assembled here from its definition; its truncated iterates are the
    textbook CG iterates of that dense system (numpy recurrence); and its limit is the fixed point Algorithm 1 reaches."""
    rng = np.random.default_rng(9)
    f = make_field("gaussians2d" if len(shape) == 2 else "fourier3d", shape, seed=2, noise=0.05, kmax=2.0)
    mask = (rng.random(shape) > 0.12).astype(np.uint8)
    g = f["g"] + [None] * (3 - len(f["g"]))
    v = oracle.validity(g[0], g[1], g[2], mask)
    w1, w0, w0C = oracle.weights(v, *sp)
    S = oracle.source(v, w1, w0, g[0], g[1], g[2], *sp)
    K = oracle.constants(shape[-1], shape[-2], shape[0] if len(shape) == 3 else 1, *sp)
    keep = v.ravel() == 1
    Lk = _dense_laplacian(v, K["F"] / K["A_tot"])[np.ix_(keep, keep)]
    Sk = S.ravel()[keep]
    Pstar = np.linalg.pinv(Lk, rcond=1e-12) @ Sk
    Po, info = oracle.solve_direct(g[0], g[1], g[2], mask, *sp, tol=1e-12, max_outer=5, max_cg=2000)
    assert info["converged"] and info["outer_iters"] == 1
    assert np.all(np.isnan(Po.ravel()[~keep]))
    assert np.linalg.norm(Po.ravel()[keep] - Pstar) / np.linalg.norm(Pstar) < 1e-9
    # truncated: k textbook CG steps on the dense system
    for k in (1, 3, 7):
        x = np.zeros_like(Sk); r = Sk.copy(); pv = r.copy(); rho = r @ r
        for _ in range(k):
            q = Lk @ pv
            al = rho / (pv @ q)
            x += al * pv; r -= al * q
            rho1 = r @ r
            pv = r + (rho1 / rho) * pv
            rho = rho1
        Pk, ik = oracle.solve_direct(g[0], g[1], g[2], mask, *sp, tol=0.0, max_outer=1, max_cg=k)
        assert ik["cg_iters_total"] == k
        assert np.linalg.norm(Pk.ravel()[keep] - x) / np.linalg.norm(x) < 1e-11
    # restart: max_cg = 4 with several outer iterations continues to the same limit
    Pr, ir = oracle.solve_direct(g[0], g[1], g[2], mask, *sp, tol=1e-9, max_outer=10000, max_cg=4)
    assert ir["converged"]
    # the two-level iteration converges to the same field up to a constant per connected component
    P2, i2 = oracle.solve(g[0], g[1], g[2], mask, *sp, tol=1e-11, max_outer=20000, max_cg=400)
    assert i2["converged"]
    from scipy.sparse import csr_matrix
    from scipy.sparse.csgraph import connected_components
    ncomp, lab = connected_components(csr_matrix(np.abs(Lk) > 0), directed=False)
    # a first guess (:82) only moves the constant of each component
    Pg, ig = oracle.solve_direct(g[0], g[1], g[2], mask, *sp, tol=1e-12, max_outer=5, max_cg=2000,
                                 P_init=rng.normal(size=shape))
    assert ig["converged"]
    for other, bound in ((P2, 1e-8), (Pr, 1e-6), (Pg, 1e-8)):
        a, b = other.ravel()[keep].copy(), Pstar.copy()
        for cpt in range(ncomp):
            m = lab == cpt
            a[m] -= a[m].mean(); b[m] -= b[m].mean()
        assert np.linalg.norm(a - b) / np.linalg.norm(b) < bound


# ----------------------------------------------------------------------------- analytic pins (P7, P8, P9)

@pytest.mark.parametrize("shape,sp", [((12, 10), (0.1, 0.07, 1.0)), ((7, 8, 6), (0.2, 0.15, 0.3))])
def test_exact_on_quadratics(oracle, shape, sp):
    """The face average of f is exact for quadratic P (:78 'second-order accurate'), so the converged field equals
    P up to a constant to rounding, for any mask and spacing."""
    rng = np.random.default_rng(21)
    nd = len(shape)
    ax = [np.arange(m) * s for m, s in zip(shape[::-1], sp)]          # x, y, (z)
    X = np.meshgrid(*ax[::-1], indexing="ij")[::-1]                    # X[0]=x ...
    A = rng.normal(size=(nd, nd)); A = A + A.T
    b = rng.normal(size=nd)
    P = sum(b[i] * X[i] for i in range(nd)) + 0.5 * sum(A[i, j] * X[i] * X[j] for i in range(nd) for j in range(nd))
    g = [b[i] + sum(A[i, j] * X[j] for j in range(nd)) for i in range(nd)] + [None] * (3 - nd)
    mask = np.ones(shape, np.uint8)
    mask[tuple(s // 2 for s in shape)] = 0
    mask[(1,) * nd] = 0
    Po, info = oracle.solve(g[0], g[1], g[2], mask, *sp, tol=1e-13, max_outer=50000, max_cg=500)
    assert info["converged"]
    m = mask == 1
    e = (Po[m] - Po[m].mean()) - (P[m] - P[m].mean())
    assert np.linalg.norm(e) / np.linalg.norm(P[m] - P[m].mean()) < 1e-10


def test_second_order_convergence(oracle):
    """Smooth P from exact gradients: discretisation error falls as h^2 (:78, :105)."""
    errs = []
    for n in (17, 33, 65):
        f = make_field("gaussians2d", (n, n), seed=0, noise=0.0)
        Po, info = oracle.solve(f["g"][0], f["g"][1], None, None, *f["d"], tol=1e-9, max_outer=20000, max_cg=60)
        assert info["converged"]
        e = (Po - Po.mean()) - (f["P"] - f["P"].mean())
        errs.append(np.linalg.norm(e) / np.linalg.norm(f["P"] - f["P"].mean()))
    assert 3.5 < errs[0] / errs[1] < 4.5 and 3.5 < errs[1] / errs[2] < 4.5, errs


def test_zero_gradient_gives_zero_field(oracle):
    """S = 0 -> P = 0 (constant), no iterations (Alg. 1 :139, reading A4)."""
    z = np.zeros((6, 7, 8))
    mask = np.ones(z.shape, np.uint8); mask[2, 3, 4] = 0
    Po, info = oracle.solve(z, z, z, mask, 1.0, 1.0, 1.0, tol=1e-8, max_outer=10, max_cg=10)
    assert info["outer_iters"] == 0 and info["cg_iters_total"] == 0 and info["norm_S"] == 0
    assert np.all(Po[mask == 1] == 0) and np.isnan(Po[2, 3, 4])


def test_conservation_and_residual_definition(oracle):
    """1^T S = 0 on a full box (every face term appears twice with opposite sign); eps_R (Eq. 41 :442) equals
    |S - (M - W^n) P| / |S| recomputed from the operators; eps_R^0 = 1 for P^0 = 0 (:445)."""
    f = make_field("gaussians2d", (20, 24), seed=4, noise=0.05)
    d = f["d"]
    Po, info, hist = oracle.solve(f["g"][0], f["g"][1], None, None, *d, tol=0.0, max_outer=7, max_cg=30, hist_cap=16)
    v = np.ones((20, 24), np.uint8)
    w1, w0, w0C = oracle.weights(v, *d)
    S = oracle.source(v, w1, w0, f["g"][0], f["g"][1], None, *d)
    assert abs(S.sum()) < 1e-12 * np.abs(S).sum()
    r = S - (oracle.apply_M(v, w1, Po) - oracle.apply_Wn(v, w0, w0C, Po))
    assert np.linalg.norm(r) / np.linalg.norm(S) == pytest.approx(info["eps_R_final"], rel=1e-9)
    assert hist[0] == pytest.approx(1.0, rel=1e-12)
    assert np.all(np.diff(hist[:8]) < 0)


def test_sample_matches_stored_weight_path(oracle):
    """oracle.sample (per-cell evaluation for full-size spot checks) agrees with the stored-weight operators,
    which the pins above fix."""
    rng = np.random.default_rng(17)
    shape = (7, 9, 8)
    f = make_field("fourier3d", shape, seed=6, noise=0.1, kmax=2.0)
    mask = (rng.random(shape) > 0.2).astype(np.uint8)
    d = (0.5, 0.7, 0.9)
    v = oracle.validity(*f["g"], mask)
    w1, w0, w0C = oracle.weights(v, *d)
    S = oracle.source(v, w1, w0, *f["g"], *d)
    x = rng.normal(size=shape) * v
    cells = rng.choice(v.size, 200, replace=False)
    Ss, Ms, Ws = oracle.sample(v, *f["g"], x, cells, *d)
    assert np.allclose(Ss, S.ravel()[cells], rtol=1e-14, atol=1e-16)
    assert np.allclose(Ms, oracle.apply_M(v, w1, x).ravel()[cells], rtol=1e-14, atol=1e-16)
    assert np.allclose(Ws, oracle.apply_Wn(v, w0, w0C, x).ravel()[cells], rtol=1e-14, atol=1e-16)


# ----------------------------------------------------------------------------- batched snapshots / first guess (NEXT-1)

def test_eps_R_of_field_matches_the_solver_and_the_stored_weight_path(oracle):
    """eps_R_of_field (chunked per-cell evaluation, used to certify full-size GPU fields) against (i) the eps_R the
    oracle's own solve reports for the field it returns and (ii) S + W^n P - M P through the stored-weight operators,
    on a masked anisotropic 3D grid with NaN-marked cells; chunk boundaries must not matter."""
    rng = np.random.default_rng(17)
    shape = (7, 9, 11)
    g = [rng.normal(size=shape) for _ in range(3)]
    mask = (rng.random(shape) > 0.15).astype(np.uint8)
    g[1][2, 3, 4] = np.nan
    d = (0.4, 1.1, 0.7)
    P, info = oracle.solve(g[0], g[1], g[2], mask, *d, tol=1e-6, max_outer=60, max_cg=50)     # any returned field will do
    assert 0 < info["eps_R_final"] < 1
    for chunk in (10_000_000, 97):
        eps, nr, nS = oracle.eps_R_of_field(g[0], g[1], g[2], mask, P, *d, chunk=chunk)
        assert eps == pytest.approx(info["eps_R_final"], rel=1e-9) and nS == pytest.approx(info["norm_S"], rel=1e-12)
    v = oracle.validity(g[0], g[1], g[2], mask)
    w1, w0, w0C = oracle.weights(v, *d)
    S = oracle.source(v, w1, w0, np.nan_to_num(g[0]), np.nan_to_num(g[1]), np.nan_to_num(g[2]), *d)
    Q = rng.normal(size=shape) * v
    r = S + oracle.apply_Wn(v, w0, w0C, Q) - oracle.apply_M(v, w1, Q)
    eps, nr, nS = oracle.eps_R_of_field(g[0], g[1], g[2], mask, np.where(v == 1, Q, np.nan), *d, chunk=1000)
    assert nr == pytest.approx(np.linalg.norm(r), rel=1e-12) and eps == pytest.approx(np.linalg.norm(r) / np.linalg.norm(S), rel=1e-12)


def test_batch2d_oracle_pins(oracle):
    """Stacked 2D snapshots solved as one block-diagonal system (2D constants, no coupling across planes):
    nb = 1 is bit-identical to the plain 2D solve; converged, every snapshot equals its own single solve (pinned above)
    within the tolerance; a first guess equal to the converged field needs no iteration (:82 'any other arbitrary
    value'); the fixed point does not depend on the first guess."""
    fs = [make_field("lamb_oseen2d", (26, 30), seed=s, noise=0.05) for s in range(3)]
    gx = np.stack([f["g"][0] for f in fs]); gy = np.stack([f["g"][1] for f in fs])
    m, d = fs[0]["mask"], fs[0]["d"]
    P1, i1 = oracle.solve_batch2d(gx[:1], gy[:1], m, d[0], d[1], 0.0, 5, 10)
    P2, i2 = oracle.solve(gx[0], gy[0], None, m, d[0], d[1], 1.0, tol=0.0, max_outer=5, max_cg=10)
    assert np.array_equal(P1[0], P2, equal_nan=True) and i1["eps_R_final"] == i2["eps_R_final"]
    Pb, ib = oracle.solve_batch2d(gx, gy, m, d[0], d[1], 1e-10, 100000, 400)
    assert ib["converged"]
    for b in range(3):
        Pi, ii = oracle.solve(gx[b], gy[b], None, m, d[0], d[1], 1.0, tol=1e-10, max_outer=100000, max_cg=400)
        v = ~np.isnan(Pi)
        a, c = Pb[b][v] - Pb[b][v].mean(), Pi[v] - Pi[v].mean()
        assert np.linalg.norm(a - c) / np.linalg.norm(c) < 2e-9
    Pw, iw = oracle.solve_batch2d(gx, gy, m, d[0], d[1], 1e-9, 100, 50, P_init=np.nan_to_num(Pb))
    assert iw["outer_iters"] == 0 and iw["cg_iters_total"] == 0
    rng = np.random.default_rng(0)
    Pr, ir = oracle.solve_batch2d(gx, gy, m, d[0], d[1], 1e-10, 100000, 400, P_init=rng.normal(size=gx.shape))
    v = ~np.isnan(Pb)
    for b in range(3):
        a, c = Pr[b][v[b]] - Pr[b][v[b]].mean(), Pb[b][v[b]] - Pb[b][v[b]].mean()
        assert np.linalg.norm(a - c) / np.linalg.norm(c) < 1e-7


def test_direct_batch2d_oracle_pins(oracle):
    """The stacked direct solve: nb = 1 is bit-identical to solve_direct on the 2D grid; converged, every snapshot equals
    its own direct solve (pinned to pinv(L) S above); a first guess moves nothing but the per-component constant."""
    fs = [make_field("lamb_oseen2d", (26, 30), seed=s, noise=0.05) for s in range(3)]
    gx = np.stack([f["g"][0] for f in fs]); gy = np.stack([f["g"][1] for f in fs])
    m, d = fs[0]["mask"], fs[0]["d"]
    P1, i1 = oracle.solve_batch2d(gx[:1], gy[:1], m, d[0], d[1], 0.0, 2, 9, direct=True)
    P2, i2 = oracle.solve_direct(gx[0], gy[0], None, m, d[0], d[1], 1.0, tol=0.0, max_outer=2, max_cg=9)
    assert np.array_equal(P1[0], P2, equal_nan=True) and i1["eps_R_final"] == i2["eps_R_final"]
    Pb, ib = oracle.solve_batch2d(gx, gy, m, d[0], d[1], 1e-11, 10, 2000, direct=True)
    assert ib["converged"]
    rng = np.random.default_rng(1)
    Pr, ir = oracle.solve_batch2d(gx, gy, m, d[0], d[1], 1e-11, 10, 2000, P_init=rng.normal(size=gx.shape), direct=True)
    assert ir["converged"]
    for b in range(3):
        Pi, ii = oracle.solve_direct(gx[b], gy[b], None, m, d[0], d[1], 1.0, tol=1e-11, max_outer=10, max_cg=2000)
        v = ~np.isnan(Pi)
        for other in (Pb, Pr):
            a, c = other[b][v] - other[b][v].mean(), Pi[v] - Pi[v].mean()
            assert np.linalg.norm(a - c) / np.linalg.norm(c) < 1e-8


# ----------------------------------------------------------------------------- NEXT-4: f(u) of Eq. 1 (:23)

def test_velocity_source_closed_forms(oracle):
    """oracle.velocity_source against closed forms: (i) central differences are exact on quadratics, so for a quadratic
    velocity field -rho (u . grad) u + mu lap u is reproduced to rounding at every cell with a full stencil; (ii) the 2D
    Taylor-Green vortex (steady Euler solution, P = rho/4 (cos 2x + cos 2y)): f -> grad P at second order; with
    viscosity and the matching decay rate du/dt = -2 nu u the viscous and unsteady terms cancel; (iii) missing cells
    poison exactly their stencil neighbours."""
    rng = np.random.default_rng(0)
    nz, ny, nx = 7, 8, 9
    d = (0.3, 0.5, 0.7)
    z, y, x = np.meshgrid(np.arange(nz) * d[2], np.arange(ny) * d[1], np.arange(nx) * d[0], indexing="ij")
    X = [x, y, z]
    # u_i = a_i + b_ij X_j + X^T C_i X / 2   (C_i symmetric)
    a = rng.normal(size=3); b = rng.normal(size=(3, 3)); Cq = rng.normal(size=(3, 3, 3)); Cq = Cq + Cq.transpose(0, 2, 1)
    U = [a[i] + sum(b[i, j] * X[j] for j in range(3)) + 0.5 * sum(Cq[i, j, k] * X[j] * X[k] for j in range(3) for k in range(3))
         for i in range(3)]
    grad = [[b[i, j] + sum(Cq[i, j, k] * X[k] for k in range(3)) for j in range(3)] for i in range(3)]
    rho, mu = 1.7, 0.05
    acc = [rng.normal(size=x.shape) for _ in range(3)]
    exact = [-rho * (acc[i] + sum(U[j] * grad[i][j] for j in range(3))) + mu * np.trace(Cq[i]) for i in range(3)]
    g = oracle.velocity_source(U[0], U[1], U[2], None, *d, rho=rho, mu=mu, dudt=acc)
    inner = (slice(1, -1),) * 3
    for i in range(3):
        assert np.allclose(g[i][inner], exact[i][inner], rtol=1e-12, atol=1e-12)
        edge = np.ones(x.shape, bool); edge[inner] = False
        assert np.isnan(g[i][edge]).all() and not np.isnan(g[i][inner]).any()
    # (iii) one missing cell (NaN velocity) and one masked cell: exactly the cells whose 7-point stencil touches them
    U2 = [c.copy() for c in U]; U2[1][3, 4, 4] = np.nan
    mask = np.ones(x.shape, np.uint8); mask[2, 2, 6] = 0
    g2 = oracle.velocity_source(U2[0], U2[1], U2[2], mask, *d, rho=rho, mu=mu, dudt=acc)
    expect_nan = np.ones(x.shape, bool); expect_nan[inner] = False
    for (k, j, i) in ((3, 4, 4), (2, 2, 6)):
        for dk, dj, di in ((0, 0, 0), (1, 0, 0), (-1, 0, 0), (0, 1, 0), (0, -1, 0), (0, 0, 1), (0, 0, -1)):
            expect_nan[k + dk, j + dj, i + di] = True
    assert np.array_equal(np.isnan(g2[0]), expect_nan)
    assert np.allclose(g2[2][~expect_nan], exact[2][~expect_nan], rtol=1e-12, atol=1e-12)
    # (ii) Taylor-Green, 2D, two resolutions
    errs = []
    for n in (32, 64):
        hh = 2 * np.pi / n
        yy, xx = np.meshgrid(np.arange(n) * hh, np.arange(n) * hh, indexing="ij")
        nu = 0.3
        u, v = np.sin(xx) * np.cos(yy), -np.cos(xx) * np.sin(yy)
        gP = [-0.5 * rho * np.sin(2 * xx), -0.5 * rho * np.sin(2 * yy)]
        g = oracle.velocity_source(u, v, None, None, hh, hh, rho=rho, mu=rho * nu, dudt=[-2 * nu * u, -2 * nu * v])
        inner2 = (slice(1, -1),) * 2
        errs.append(max(np.abs(g[i][inner2] - gP[i][inner2]).max() for i in range(2)))
    assert errs[0] < 2e-2 and 3.5 < errs[0] / errs[1] < 4.5


def test_rans_source_closed_forms(oracle):
    """oracle.rans_source (Eq. 42 :507) against closed forms: (i) with quadratic mean velocity and quadratic Reynolds
    stresses every central difference is exact, so -rho (ubar . grad ubar_i + d_j R_ij) is reproduced to rounding, in 3D
    and 2D, with anisotropic spacing -- a transposed stress index, a dropped term or a wrong sign fails it;
    (ii) zero stresses reduce it to the steady inviscid velocity_source (pinned above); (iii) ubar = 0, R_xx = x^2:
    f = (-2 rho x, 0, 0); (iv) a NaN in a stress component poisons exactly its stencil neighbours."""
    rng = np.random.default_rng(1)
    rho = 1.3
    for nd, shape, d in ((3, (6, 7, 8), (0.3, 0.5, 0.7)), (2, (9, 8), (0.4, 0.25))):
        coords = np.meshgrid(*[np.arange(n) * d[nd - 1 - ax] for ax, n in enumerate(shape)], indexing="ij")
        X = coords[::-1]                                        # X[a] = coordinate along axis a (x fastest)
        def quad():
            a, b = rng.normal(), rng.normal(size=nd)
            Cq = rng.normal(size=(nd, nd)); Cq = Cq + Cq.T
            f = a + sum(b[j] * X[j] for j in range(nd)) + 0.5 * sum(Cq[j, k] * X[j] * X[k] for j in range(nd) for k in range(nd))
            g = [b[j] + sum(Cq[j, k] * X[k] for k in range(nd)) for j in range(nd)]
            return f, g
        U, gU = zip(*[quad() for _ in range(nd)])
        pairs = [(0, 0), (1, 1), (0, 1)] if nd == 2 else [(0, 0), (1, 1), (2, 2), (0, 1), (0, 2), (1, 2)]
        R, gR = zip(*[quad() for _ in pairs])
        Rij = {}
        for (i, j), g in zip(pairs, gR):
            Rij[(i, j)] = g; Rij[(j, i)] = g
        exact = [-rho * (sum(U[j] * gU[i][j] for j in range(nd)) + sum(Rij[(i, j)][j] for j in range(nd))) for i in range(nd)]
        f = oracle.rans_source(U[0], U[1], U[2] if nd == 3 else None, list(R), None, *d, rho=rho)
        inner = (slice(1, -1),) * nd
        for i in range(nd):
            assert np.allclose(f[i][inner], exact[i][inner], rtol=1e-12, atol=1e-12)
            edge = np.ones(shape, bool); edge[inner] = False
            assert np.isnan(f[i][edge]).all()
        # (ii) zero stresses: the steady, inviscid form of Eq. 1
        f0 = oracle.rans_source(U[0], U[1], U[2] if nd == 3 else None, [np.zeros(shape)] * len(pairs), None, *d, rho=rho)
        v0 = oracle.velocity_source(U[0], U[1], U[2] if nd == 3 else None, None, *d, rho=rho, mu=0.0)
        for i in range(nd):
            assert np.array_equal(np.isnan(f0[i]), np.isnan(v0[i]))
            assert np.allclose(f0[i][inner], v0[i][inner], rtol=1e-13, atol=1e-13)
    # (iii) a stress gradient alone
    shape, d = (5, 6, 7), (0.5, 0.5, 0.5)
    z, y, x = np.meshgrid(*[np.arange(n) * 0.5 for n in shape], indexing="ij")
    Z = np.zeros(shape)
    f = oracle.rans_source(Z, Z, Z, [x * x, Z, Z, Z, Z, Z], None, *d, rho=rho)
    inner = (slice(1, -1),) * 3
    assert np.allclose(f[0][inner], -2 * rho * x[inner]) and np.allclose(f[1][inner], 0) and np.allclose(f[2][inner], 0)
    f = oracle.rans_source(Z, Z, Z, [Z, Z, Z, Z, Z, y * z], None, *d, rho=rho)       # R_yz = y z: f_y = -rho y, f_z = -rho z... by axis
    assert np.allclose(f[1][inner], -rho * y[inner]) and np.allclose(f[2][inner], -rho * z[inner]) and np.allclose(f[0][inner], 0)
    # (iv) NaN pattern
    Rxy = Z.copy(); Rxy[2, 3, 3] = np.nan
    f = oracle.rans_source(Z, Z, Z, [Z, Z, Z, Rxy, Z, Z], None, *d, rho=rho)
    expect = np.ones(shape, bool); expect[inner] = False
    for dk, dj, di in ((0, 0, 0), (1, 0, 0), (-1, 0, 0), (0, 1, 0), (0, -1, 0), (0, 0, 1), (0, 0, -1)):
        expect[2 + dk, 3 + dj, 3 + di] = True
    assert all(np.array_equal(np.isnan(c), expect) for c in f)


def test_compressible_rans_source_closed_forms(oracle):
    """oracle.compressible_rans_source (Eq. 43-44 :540-545).  (i) Textbook case: the compressible free vortex
    u_theta = Gamma / (2 pi r) is a steady, irrotational, homentropic Euler solution, so P / P_inf = (T / T_inf)^(gamma/(gamma-1))
    with T from the adiabatic energy equation (Eq. 43): the oracle's g must converge to gamma/(gamma-1) grad ln T at
    second order (the core is masked).  (ii) Linear mean velocity, quadratic stresses: uu_ij and T are quadratic, every
    central difference is exact, and g equals the cell-wise solve of Eq. 44 with ANALYTIC derivatives to rounding
    (catches a transposed matrix, a wrong stress index, a sign).  (iii) Fluid at rest or in uniform motion: g = 0."""
    gam = 1.4
    errs = []
    for n in (65, 129):
        h = 2.0 / (n - 1)
        y, x = np.meshgrid(-1 + np.arange(n) * h, -1 + np.arange(n) * h, indexing="ij")
        r2 = x * x + y * y
        mask = (r2 >= 0.5 ** 2).astype(np.uint8)
        G, Minf = 0.5, 0.4
        Vinf = G                                         # reference state: the streamline r = 1
        RTinf = Vinf ** 2 / (gam * Minf ** 2)            # M_inf^2 = V_inf^2 / (gamma R T_inf)
        with np.errstate(divide="ignore", invalid="ignore"):
            u, v = -G * y / r2, G * x / r2
        u[mask == 0] = np.nan; v[mask == 0] = np.nan
        g = oracle.compressible_rans_source(u, v, None, None, mask, h, h, gamma=gam, mach_inf=Minf, v_inf=Vinf, rgas_t_inf=RTinf)
        c = 0.5 * (gam - 1) * Minf ** 2 / Vinf ** 2
        with np.errstate(invalid="ignore", divide="ignore"):
            th = 1 + c * (Vinf ** 2 - G * G / r2)
            ex = [gam / (gam - 1) * c * 2 * G * G * x / r2 ** 2 / th, gam / (gam - 1) * c * 2 * G * G * y / r2 ** 2 / th]
        ok = ~np.isnan(g[0])
        assert ok.sum() > 0.5 * n * n
        errs.append(max(np.abs(g[i][ok] - ex[i][ok]).max() for i in range(2)) / max(np.abs(ex[i][ok]).max() for i in range(2)))
    assert errs[0] < 2e-2 and 3.2 < errs[0] / errs[1] < 4.8, errs      # max norm; the staircase core edge moves with n
    # (ii) exactness with analytic derivatives, 3D, anisotropic spacing, with Reynolds stresses
    rng = np.random.default_rng(2)
    shape, d = (6, 7, 8), (0.03, 0.05, 0.07)
    z, y, x = np.meshgrid(*[np.arange(n) * d[2 - ax] for ax, n in enumerate(shape)], indexing="ij")
    X = [x, y, z]
    a = rng.normal(size=3); B = 0.5 * rng.normal(size=(3, 3))
    U = [a[i] + sum(B[i, j] * X[j] for j in range(3)) for i in range(3)]
    pairs = [(0, 0), (1, 1), (2, 2), (0, 1), (0, 2), (1, 2)]
    Rq, gRq = {}, {}
    stress = []
    for (i, j) in pairs:
        b = 0.1 * rng.normal(size=3); Cq = 0.1 * rng.normal(size=(3, 3)); Cq = Cq + Cq.T
        f = 0.05 * rng.normal() + sum(b[k] * X[k] for k in range(3)) + 0.5 * sum(Cq[k, l] * X[k] * X[l] for k in range(3) for l in range(3))
        gf = [b[k] + sum(Cq[k, l] * X[l] for l in range(3)) for k in range(3)]
        Rq[(i, j)] = Rq[(j, i)] = f; gRq[(i, j)] = gRq[(j, i)] = gf
        stress.append(f)
    Minf, Vinf, RTinf = 1.5, 2.0, 3.0
    g = oracle.compressible_rans_source(U[0], U[1], U[2], stress, None, *d, gamma=gam, mach_inf=Minf, v_inf=Vinf, rgas_t_inf=RTinf)
    c = 0.5 * (gam - 1) * Minf ** 2
    th = 1 + c * (1 - sum(Ui * Ui for Ui in U) / Vinf ** 2)
    dth = [-c / Vinf ** 2 * 2 * sum(U[i] * B[i, k] for i in range(3)) for k in range(3)]
    inner = (slice(1, -1),) * 3
    for (kk, jj, ii) in ((1, 1, 1), (2, 3, 4), (4, 5, 6), (3, 2, 5)):
        A = np.zeros((3, 3)); rhs = np.zeros(3)
        for i in range(3):
            for j in range(3):
                uu = U[i][kk, jj, ii] * U[j][kk, jj, ii] + Rq[(i, j)][kk, jj, ii]
                duu = B[i, j] * U[j][kk, jj, ii] + U[i][kk, jj, ii] * B[j, j] + gRq[(i, j)][j][kk, jj, ii]
                RT = RTinf * th[kk, jj, ii]
                A[i, j] = (i == j) + uu / RT
                rhs[i] += -(duu - uu / th[kk, jj, ii] * dth[j][kk, jj, ii]) / RT
        ref = np.linalg.solve(A, rhs)
        got = np.array([g[i][kk, jj, ii] for i in range(3)])
        assert np.allclose(got, ref, rtol=1e-10, atol=1e-12), (got, ref)
    edge = np.ones(shape, bool); edge[inner] = False
    assert all(np.isnan(c_[edge]).all() and not np.isnan(c_[inner]).any() for c_ in g)
    # (iii) rest and uniform motion
    Z = np.zeros(shape)
    for Uc in ((Z, Z, Z), (Z + 0.7, Z - 0.2, Z + 0.1)):
        g = oracle.compressible_rans_source(*Uc, None, None, *d, gamma=gam, mach_inf=Minf, v_inf=Vinf, rgas_t_inf=RTinf)
        assert all(np.allclose(c_[inner], 0.0, atol=1e-13) for c_ in g)


def test_solve_guess_pins(oracle):
    """oracle.solve_guess (Alg. 1 from a first guess): (i) P_init = 0 / None is oracle.solve; (ii) started from
    its own converged field it stops at the first residual check (0 outer iterations) and returns the field; (iii) every
    row of M - W^n sums to zero (:631), so a guess shifted by a constant per connected component shifts every iterate by
    the same constants: after a fixed number of steps P(guess + c) - P(guess) = c exactly up to rounding; (iv) the fixed
    point does not depend on the guess up to that constant (compared with the dense pseudo-inverse pin via oracle.solve);
    (v) the guess at missing cells is ignored."""
    from workloads import make_field
    f = make_field("sphere3d", (10, 11, 12), seed=5, noise=0.05)
    g, m, d = f["g"], f["mask"], f["d"]
    P0, i0 = oracle.solve(*g, m, *d, tol=0.0, max_outer=4, max_cg=10)
    Pz, iz = oracle.solve_guess(*g, m, *d, tol=0.0, max_outer=4, max_cg=10, P_init=np.zeros(g[0].shape))
    assert np.array_equal(P0, Pz, equal_nan=True) and i0 == iz
    Pn, i_n = oracle.solve_guess(*g, m, *d, tol=0.0, max_outer=4, max_cg=10, P_init=None)
    assert np.array_equal(P0, Pn, equal_nan=True)
    # (ii)
    Pc, ic = oracle.solve(*g, m, *d, tol=1e-9, max_outer=100000, max_cg=200)
    assert ic["converged"]
    guess = np.where(np.isnan(Pc), 123.0, Pc)                   # (v): garbage at the missing cells
    Pr, ir = oracle.solve_guess(*g, m, *d, tol=1.0001e-9, max_outer=100000, max_cg=200, P_init=guess)
    assert ir["outer_iters"] == 0 and ir["cg_iters_total"] == 0
    assert np.array_equal(Pr, Pc, equal_nan=True)
    # (iii)
    rng = np.random.default_rng(3)
    base = rng.normal(size=g[0].shape)
    Pa, _ = oracle.solve_guess(*g, m, *d, tol=0.0, max_outer=3, max_cg=8, P_init=base)
    Pb, _ = oracle.solve_guess(*g, m, *d, tol=0.0, max_outer=3, max_cg=8, P_init=base + 2.5)
    v = ~np.isnan(Pa)
    assert np.allclose(Pb[v] - Pa[v], 2.5, rtol=0, atol=1e-11)
    # (iv)
    Pg, ig = oracle.solve_guess(*g, m, *d, tol=1e-9, max_outer=100000, max_cg=200, P_init=base)
    assert ig["converged"]
    a, b = Pg[v] - Pg[v].mean(), Pc[v] - Pc[v].mean()
    assert np.linalg.norm(a - b) / np.linalg.norm(b) < 1e-6


# ----------------------------------------------------------------------------- omni_pcg oracle (NEXT-2 ii)

def _pcg_case(oracle, shape, sp, seed=9, frac=0.12):
    rng = np.random.default_rng(seed)
    f = make_field("gaussians2d" if len(shape) == 2 else "fourier3d", shape, seed=2, noise=0.05, kmax=2.0)
    mask = (rng.random(shape) > frac).astype(np.uint8)
    g = f["g"] + [None] * (3 - len(f["g"]))
    v = oracle.validity(g[0], g[1], g[2], mask)
    w1, w0, w0C = oracle.weights(v, *sp)
    S = oracle.source(v, w1, w0, g[0], g[1], g[2], *sp)
    K = oracle.constants(shape[-1], shape[-2], shape[0] if len(shape) == 3 else 1, *sp)
    return g, mask, v, (w1, w0, w0C), S, K["F"] / K["A_tot"]


@pytest.mark.parametrize("shape,sp", [((18, 21), (1.0, 0.6, 1.0)), ((9, 10, 17), (1.0, 1.3, 0.8)), ((5, 6), (0.7, 1.0, 1.0))])
def test_pcg_oracle_vs_dense_algebra(oracle, shape, sp):
    """oracle.omni_pcg.solve_pcg (multigrid-preconditioned CG on L P = S, reading R-P1) against dense linear algebra
    written here: (a) its level-0 operator is M - W^n of the stored-weight oracle and the dense L assembled from the
    definition; (b) the V-cycle, applied to unit vectors, is a SYMMETRIC positive semi-definite matrix B (PCG needs
    that), positive on the range of L; (c) the truncated iterates are those of a dense textbook PCG with that B;
    (d) converged, the result is pinv(L) S up to a constant per component; (e) far fewer iterations than plain CG."""
    from oracle import omni_pcg as pcg
    g, mask, v, (w1, w0, w0C), S, t = _pcg_case(oracle, shape, sp)
    nd = len(shape)
    levels, plans = pcg.build_levels(v.astype(bool), pcg.face_weights(nd, *sp))
    assert np.allclose(levels[0].w, t[:nd], rtol=1e-15)
    assert len(levels) == (1 if max(shape) < 8 else len(levels)) and (max(shape) < 8 or len(levels) >= 2)
    L = _dense_laplacian(v, t)
    rng = np.random.default_rng(4)
    x = rng.normal(size=shape) * v
    Lx = oracle.apply_M(v, w1, x) - oracle.apply_Wn(v, w0, w0C, x)
    assert np.abs(levels[0].apply(x) - Lx).max() < 1e-14 and np.abs(levels[0].apply(x).ravel() - L @ x.ravel()).max() < 1e-14
    N = v.size
    B = np.zeros((N, N))
    for c in range(N):
        e = np.zeros(N); e[c] = 1.0
        B[:, c] = pcg.vcycle(levels, plans, 0, e.reshape(shape)).ravel()
    keep = v.ravel() == 1
    assert np.abs(B[~keep]).max() == 0 and np.abs(B[:, ~keep]).max() == 0
    Bk, Lk, Sk = B[np.ix_(keep, keep)], L[np.ix_(keep, keep)], S.ravel()[keep]
    assert np.abs(Bk - Bk.T).max() <= 1e-13 * np.abs(Bk).max()
    ev = np.linalg.eigvalsh(0.5 * (Bk + Bk.T))
    assert ev.min() > -1e-12 * ev.max()
    # preconditioned spectrum on the range of L: the nonzero eigenvalues of B L cluster (a usable preconditioner)
    lam = np.sort(np.linalg.eigvals(Bk @ Lk).real)
    nz = lam[lam > 1e-9]
    assert nz.max() / nz.min() < 25.0, nz.max() / nz.min()
    # dense textbook PCG with the matrix B
    for k in (1, 2, 5):
        xk = np.zeros_like(Sk); r = Sk.copy(); p = np.zeros_like(Sk); rho_old = 1.0
        for it in range(k):
            z = Bk @ r
            rho = r @ z
            p = z + ((rho / rho_old) if it else 0.0) * p
            q = Lk @ p
            al = rho / (p @ q)
            xk += al * p; r -= al * q
            rho_old = rho
        Pk, ik = pcg.solve_pcg(g[0], g[1], g[2], mask, *sp, tol=0.0, max_outer=1, max_cg=k)
        assert ik["cg_iters_total"] == k and np.all(np.isnan(Pk.ravel()[~keep]))
        assert np.linalg.norm(Pk.ravel()[keep] - xk) / np.linalg.norm(xk) < 1e-10
    Pc, ic = pcg.solve_pcg(g[0], g[1], g[2], mask, *sp, tol=1e-11, max_outer=5, max_cg=400)
    assert ic["converged"] and ic["outer_iters"] <= 2
    Pstar = np.linalg.pinv(Lk, rcond=1e-12) @ Sk
    from scipy.sparse import csr_matrix
    from scipy.sparse.csgraph import connected_components
    ncomp, lab = connected_components(csr_matrix(np.abs(Lk) > 0), directed=False)
    a, b = Pc.ravel()[keep].copy(), Pstar.copy()
    for cpt in range(ncomp):
        m = lab == cpt
        a[m] -= a[m].mean(); b[m] -= b[m].mean()
    assert np.linalg.norm(a - b) / np.linalg.norm(b) < 1e-8
    Pd, idd = oracle.solve_direct(g[0], g[1], g[2], mask, *sp, tol=1e-11, max_outer=5, max_cg=4000)
    assert idd["converged"] and (max(shape) < 8 or ic["cg_iters_total"] * 2 < idd["cg_iters_total"])


def test_pcg_oracle_pieces():
    """The pieces of the V-cycle against closed forms: restriction and prolongation are transposes (any halving plan,
    odd sizes); on a grid too small to coarsen the preconditioner is the damped-Jacobi polynomial
    sum_{j<8} (I - w D^-1 L)^j w D^-1; the coarse weights follow w * 2^m / 4 on halved axes, w * 2^m on the others."""
    from oracle import omni_pcg as pcg
    rng = np.random.default_rng(1)
    for shape, halve in (((9, 8), [True, True]), ((5, 11, 8), [False, True, True]), ((7,), [True])):
        cshape = tuple((s + 1) // 2 if h else s for s, h in zip(shape, halve))
        r, e = rng.normal(size=shape), rng.normal(size=cshape)
        assert pcg.restrict(r, halve).shape == cshape
        assert np.sum(pcg.restrict(r, halve) * e) == pytest.approx(np.sum(r * pcg.prolong(e, halve, shape)), rel=1e-13)
    assert pcg.coarsen_plan((5, 8, 17), [1.0, 1.0, 1.0]) == [False, True, True]
    # semi-coarsening: only the strongly coupled axes (weight >= 0.7 of the largest among the axes long enough) are halved
    assert pcg.coarsen_plan((40, 40, 40), [1.0, 0.69, 0.3]) == [False, False, True]       # w[0] is x = the last numpy axis
    assert pcg.coarsen_plan((40, 40, 40), [0.3, 0.71, 1.0]) == [True, True, False]
    assert pcg.coarsen_plan((40, 40, 4), [9.0, 0.71, 1.0]) == [True, True, False]         # x is too short to count
    assert pcg.coarsen_plan((4, 4), [1.0, 1.0]) == [False, False]
    # a halved axis loses a factor 4 against the others: the weak axis catches up and is halved on a later level
    lv, pl = pcg.build_levels(np.ones((32, 32, 32), bool), [1.0, 0.5, 0.2])
    assert pl[0] == [False, False, True] and np.allclose(lv[1].w, [0.5, 1.0, 0.4])
    assert pl[1] == [False, True, False] and np.allclose(lv[2].w, [1.0, 0.5, 0.8])
    assert pl[2] == [True, False, True] and np.allclose(lv[3].w, [1.0, 2.0, 0.8])
    v = rng.random((6, 7)) > 0.1
    levels, plans = pcg.build_levels(v, [0.3, 0.2])
    assert len(levels) == 1 and plans == []
    L = _dense_laplacian(v, [0.3, 0.2])
    D = np.diag(L).copy()
    Dinv = np.where(D > 0, 1.0 / np.where(D > 0, D, 1.0), 0.0)
    b = rng.normal(size=v.shape) * v
    G = np.eye(v.size) - pcg.OMEGA * Dinv[:, None] * L
    z, term = np.zeros(v.size), pcg.OMEGA * Dinv * b.ravel()
    for _ in range(pcg.NU_COARSEST):
        z, term = z + term, G @ term
    assert np.abs(pcg.vcycle(levels, plans, 0, b).ravel() - z).max() < 1e-13
    levels, plans = pcg.build_levels(np.ones((5, 16, 24), bool), [0.25, 0.25, 0.3])     # w[0] is x (24), w[2] is z (5: too short)
    assert plans[0] == [False, True, True] and np.allclose(levels[1].w, [0.25 * 4 / 4, 0.25 * 4 / 4, 0.3 * 4])
    assert levels[1].v.shape == (5, 8, 12) and plans[1] == [False, True, True] and levels[2].v.shape == (5, 4, 6)
    assert len(levels) == 3


def test_eps_P_history_eq40(oracle):
    """oracle.solve_hist records eps_P^n = ||P^n - P^(n-1)|| / ||P^n|| (Eq. 40 :438) next to eps_R (Eq. 41).  Pinned with
    fields from SEPARATE truncated solves (max_outer = n - 1 and n give P^(n-1) and P^n of the same deterministic
    iteration), and by the paper's own remark that both metrics decay at the same rate with eps_R the larger (:447)."""
    f = make_field("lamb_oseen2d", (40, 52), seed=3, noise=0.05)
    g, m, d = f["g"], f["mask"], f["d"]
    P, info, hR, hP = oracle.solve_hist(g[0], g[1], None, m, *d, tol=0.0, max_outer=12, max_cg=15, hist_cap=16)
    assert hP[0] == 0.0 and np.all(np.isnan(hP[13:])) and not np.isnan(hP[:13]).any()
    _, _, hR0 = oracle.solve(g[0], g[1], None, m, *d, tol=0.0, max_outer=12, max_cg=15, hist_cap=16)
    assert np.array_equal(hR[:13], hR0[:13])
    prev = np.zeros_like(P)
    for n in (1, 2, 5, 12):
        Pa, _ = oracle.solve(g[0], g[1], None, m, *d, tol=0.0, max_outer=n - 1, max_cg=15)
        Pb, _ = oracle.solve(g[0], g[1], None, m, *d, tol=0.0, max_outer=n, max_cg=15)
        a, b = np.nan_to_num(Pa), np.nan_to_num(Pb)
        assert hP[n] == pytest.approx(np.linalg.norm(b - a) / np.linalg.norm(b), rel=1e-10)
    late = slice(6, 13)
    rate_P = hP[late][1:] / hP[late][:-1]
    rate_R = hR[late][1:] / hR[late][:-1]
    assert np.allclose(rate_P, rate_R, rtol=0.15)


@pytest.mark.parametrize("shape,sp", [((9, 10), (1.0, 0.6, 1.0)), ((5, 5, 6), (1.0, 1.3, 0.8))])
def test_single_reduction_cg_oracle(oracle, shape, sp):
    """oracle_solve_direct_cg1 (Chronopoulos-Gear: one reduction point per iteration, NEXT-2 i) on the symmetric L:
    its truncated iterates are those of a dense textbook CG written here (the two recurrences coincide in exact
    arithmetic), it converges to pinv(L) S, and its drift from the two-reduction oracle stays at rounding level."""
    g, mask, v, _, S, t = _pcg_case(oracle, shape, sp)
    keep = v.ravel() == 1
    Lk, Sk = _dense_laplacian(v, t)[np.ix_(keep, keep)], S.ravel()[keep]
    for k in (1, 2, 5, 11):
        x = np.zeros_like(Sk); r = Sk.copy(); pv = r.copy(); rho = r @ r
        for _ in range(k):
            q = Lk @ pv
            al = rho / (pv @ q)
            x += al * pv; r -= al * q
            rho1 = r @ r
            pv = r + (rho1 / rho) * pv
            rho = rho1
        Pk, ik = oracle.solve_direct(g[0], g[1], g[2], mask, *sp, tol=0.0, max_outer=1, max_cg=k, single_reduction=True)
        assert ik["cg_iters_total"] == k
        assert np.linalg.norm(Pk.ravel()[keep] - x) / np.linalg.norm(x) < 1e-10
    P1, i1 = oracle.solve_direct(g[0], g[1], g[2], mask, *sp, tol=1e-11, max_outer=5, max_cg=2000, single_reduction=True)
    P2, i2 = oracle.solve_direct(g[0], g[1], g[2], mask, *sp, tol=1e-11, max_outer=5, max_cg=2000)
    assert i1["converged"] and i2["converged"] and abs(i1["cg_iters_total"] - i2["cg_iters_total"]) <= 3
    a, b = np.nan_to_num(P1), np.nan_to_num(P2)
    assert np.linalg.norm(a - b) / np.linalg.norm(b) < 1e-9


def test_pcg_batch2d_oracle_pins(oracle):
    """solve_pcg_batch2d (stacked 2D snapshots, joint scalars): a stack of IDENTICAL snapshots reproduces the single
    2D solve plane by plane with the same iteration counts (every inner product scales by nb, every ratio is unchanged);
    nb = 1 equals solve_pcg on the 2D grid; different snapshots converge to the fields of the unpreconditioned stacked
    solve (oracle.solve_batch2d direct=True, itself pinned to the dense pseudo-inverse)."""
    from oracle import omni_pcg as pcg
    fs = [make_field("lamb_oseen2d", (26, 41), seed=s, noise=0.05) for s in range(3)]
    m, d = fs[0]["mask"], fs[0]["d"]
    g0x, g0y = fs[0]["g"]
    P1, i1 = pcg.solve_pcg(g0x, g0y, None, m, d[0], d[1], 1.0, tol=0.0, max_outer=2, max_cg=5)
    Pb, ib = pcg.solve_pcg_batch2d(np.stack([g0x] * 3), np.stack([g0y] * 3), m, d[0], d[1], tol=0.0, max_outer=2, max_cg=5)
    assert ib["cg_iters_total"] == i1["cg_iters_total"] == 10 and ib["norm_S"] == pytest.approx(np.sqrt(3) * i1["norm_S"], rel=1e-13)
    for b in range(3):
        assert np.nanmax(np.abs(Pb[b] - P1)) <= 1e-12 * np.nanmax(np.abs(P1))
    Pn, in_ = pcg.solve_pcg_batch2d(g0x[None], g0y[None], m, d[0], d[1], tol=0.0, max_outer=2, max_cg=5)
    assert np.array_equal(np.nan_to_num(Pn[0]), np.nan_to_num(P1))
    gx = np.stack([f["g"][0] for f in fs]); gy = np.stack([f["g"][1] for f in fs])
    Pc, ic = pcg.solve_pcg_batch2d(gx, gy, m, d[0], d[1], tol=1e-10, max_outer=5, max_cg=200)
    Pd, idd = oracle.solve_batch2d(gx, gy, m, d[0], d[1], 1e-10, 5, 5000, direct=True)
    assert ic["converged"] and idd["converged"] and ic["cg_iters_total"] * 4 < idd["cg_iters_total"]
    for b in range(3):
        valid = ~np.isnan(Pd[b])
        a, c = Pc[b][valid] - Pc[b][valid].mean(), Pd[b][valid] - Pd[b][valid].mean()
        assert np.linalg.norm(a - c) / np.linalg.norm(c) < 1e-7
