"""Pins of the CPU oracle against what the paper and the mathematics fix.

None of these tests touches the CUDA path.  Each pin is chosen so that a
plausible mistake in oracle/sws_oracle.c (dropped term, wrong sign or index,
transposed operand, wrong image term) fails at least one of them.  Citations
are /root/reference/PAPER.md lines (L...), readings Q1..Q12 are DESIGN.md's.
"""
import dataclasses
from pathlib import Path

import numpy as np
import pytest

import workloads as W

GOLDEN = Path(__file__).parent / "golden"
PI = np.pi


def idx_phi1(c, l):
    return l * (c.N + 1)


def idx_phix(c, k, l):
    return l * (c.N + 1) + 1 + k


def idx_zeta1(c, l):
    return (c.N + 1) * c.M + l * (c.N + 1)


def idx_zetax(c, k, l):
    return (c.N + 1) * c.M + l * (c.N + 1) + 1 + k


def row_E1(c, k, l):
    return l * (c.N + 1) + 2 + k


def row_E2(c, k, l):
    return (c.N + 1) * c.M + l * (c.N + 1) + 2 + k


def small(N=13, M=5, h=0.4, x1=-2.2, **kw):
    return W.custom(N, M, h, x1, **kw)


# ----------------------------------------------------------------------------
# counts and ordering: eq. (18), App. A L421, L25/L189 counts
# ----------------------------------------------------------------------------
def test_counts():
    for c in W.CONFIGS:
        assert c.n == 2 * (c.N + 1) * c.M
        assert c.n == 2 * c.targets + 4 * c.M          # (N-1)M + (N-1)M + 4M equations (L189)
    assert W.CONFIGS[4].targets == 173520 and W.CONFIGS[4].sources == 173761


def test_radiation_rows_and_positions(oracle64):
    """E3-E6 (eq. (24), App. A) sit at offsets 0,1 of each line block of each half
    (L421) and read the unknowns at the positions of eq. (18) L149."""
    c = small(seed=11)
    rng = np.random.default_rng(5)
    u = W.state(c) + 0.01 * rng.standard_normal(c.n)
    E = oracle64.residual(c.params(), u, rows=[])
    n, x1, dx = c.n_rad, c.x1, c.h
    for l in range(c.M):
        p1, px1, px2 = u[idx_phi1(c, l)], u[idx_phix(c, 0, l)], u[idx_phix(c, 1, l)]
        z1, zx1, zx2 = u[idx_zeta1(c, l)], u[idx_zetax(c, 0, l)], u[idx_zetax(c, 1, l)]
        blk, blk2 = l * (c.N + 1), (c.N + 1) * c.M + l * (c.N + 1)
        assert E[blk + 0] == pytest.approx(x1 * (px1 - 1) + n * (p1 - x1), rel=1e-13, abs=1e-15)
        assert E[blk + 1] == pytest.approx(x1 * (px2 - px1) / dx + n * (px1 - 1), rel=1e-13, abs=1e-15)
        assert E[blk2 + 0] == pytest.approx(x1 * zx1 + n * z1, rel=1e-13, abs=1e-15)
        assert E[blk2 + 1] == pytest.approx(x1 * (zx2 - zx1) / dx + n * zx1, rel=1e-13, abs=1e-15)
    # rows=[] leaves every E2 entry NaN and every other entry finite
    mask = np.zeros(c.n, bool)
    for l in range(c.M):
        for k in range(c.N - 1):
            mask[row_E2(c, k, l)] = True
    assert np.isnan(E[mask]).all() and np.isfinite(E[~mask]).all()


def test_locality_of_rows(oracle64):
    """Which rows move when one unknown moves: E1_{k,l} and the radiation rows are local to line l
    (B.3/B.4 L474-483: zero for m != l); E2 is dense in zeta_x (L47)."""
    c = small(seed=3)
    u = W.state(c)
    E = oracle64.residual(c.params(), u)
    half = (c.N + 1) * c.M
    l0 = 2
    for idx in (idx_phix(c, 4, l0), idx_zetax(c, 4, l0), idx_zeta1(c, l0)):
        up = u.copy()
        up[idx] += 1e-3
        d = oracle64.residual(c.params(), up) - E
        top = d[:half].reshape(c.M, c.N + 1)
        # first half: E3/E4 only on line l0; E1 rows on neighbouring lines move only through the
        # y-spline (zeta_y*, phi_y*), never through zeta*/phi_x*: check the dominant part is on l0
        assert np.abs(top[l0]).max() > 0
        assert np.abs(top[l0]).max() >= np.abs(np.delete(top, l0, 0)).max()
    up = u.copy()
    up[idx_zetax(c, 4, l0)] += 1e-3
    d = (oracle64.residual(c.params(), up) - E)[half:].reshape(c.M, c.N + 1)
    assert (np.abs(d[:, 2:]) > 0).all()                # every E2 row feels every zeta_x (L47)
    # phi_{1,l0}: E3 on line l0 only; E1 untouched on its own line except through phi_y
    up = u.copy()
    up[idx_phi1(c, l0)] += 1e-3
    d = (oracle64.residual(c.params(), up) - E)
    assert d[l0 * (c.N + 1)] == pytest.approx(c.n_rad * 1e-3, rel=1e-9)
    assert d[l0 * (c.N + 1) + 1] == 0.0                 # E4 does not contain phi_1 (L193)


# ----------------------------------------------------------------------------
# P3 / reconstruction: eq. (19) L156 and the spline of L160
# ----------------------------------------------------------------------------
def test_x_trapezoid_expanded_form(oracle64):
    """zeta_{k,l} = zeta_1 + dx/2 zx_1 + dx sum_{i=2}^{k-1} zx_i + dx/2 zx_k (L446), same for phi (L450)."""
    c = small(N=17, M=6, seed=7)
    u = W.state(c)
    zeta, phi, _, _ = oracle64.fields(c.params(), u)
    top = u[: (c.N + 1) * c.M].reshape(c.M, c.N + 1)
    bot = u[(c.N + 1) * c.M:].reshape(c.M, c.N + 1)
    for arr, blk in ((phi, top), (zeta, bot)):
        f1, fx = blk[:, 0], blk[:, 1:]
        for k in range(c.N):
            if k == 0:
                ref = f1
            else:
                ref = f1 + c.h / 2 * fx[:, 0] + c.h * fx[:, 1:k].sum(1) + c.h / 2 * fx[:, k]
            np.testing.assert_allclose(arr[:, k], ref, rtol=1e-13, atol=1e-15)


@pytest.mark.parametrize("M", [4, 5, 11, 61])
def test_P3_spline_matches_scipy(oracle64, oracle80, M):
    from scipy.interpolate import CubicSpline
    rng = np.random.default_rng(M)
    h = 0.3
    y = h * np.arange(M)
    f = rng.standard_normal(M)
    ref = CubicSpline(y, f, bc_type=((1, 0.0), "not-a-knot"))(y, 1)
    for o in (oracle64, oracle80):
        np.testing.assert_allclose(o.dy_line(f, h, 0, True), ref, rtol=1e-11, atol=1e-12)
    # y_1 != 0: not-a-knot at both ends
    ref2 = CubicSpline(y + 1.0, f, bc_type="not-a-knot")(y + 1.0, 1)
    np.testing.assert_allclose(oracle64.dy_line(f, h, 0, False), ref2, rtol=1e-11, atol=1e-12)


def test_P3_spline_exact_on_cubics(oracle64):
    h, M = 0.25, 9
    y = h * np.arange(M)
    f = 0.7 - 1.3 * y ** 2 + 0.45 * y ** 3            # zero slope at y=0: clamped condition holds
    np.testing.assert_allclose(oracle64.dy_line(f, h, 0, True), -2.6 * y + 1.35 * y ** 2, atol=1e-13)
    g = 0.7 + 0.2 * y - 1.3 * y ** 2 + 0.45 * y ** 3  # general cubic: not-a-knot both ends exact
    np.testing.assert_allclose(oracle64.dy_line(g, h, 0, False), 0.2 - 2.6 * y + 1.35 * y ** 2, atol=1e-13)


def test_fd_scheme_exact_on_quadratics(oracle64):
    h, M = 0.25, 9
    y = h * np.arange(M)
    np.testing.assert_allclose(oracle64.dy_line(1 - 0.8 * y ** 2, h, 1, True), -1.6 * y, atol=1e-13)
    np.testing.assert_allclose(oracle64.dy_line(1 + 0.3 * y - 0.8 * y ** 2, h, 1, False), 0.3 - 1.6 * y, atol=1e-13)


def test_fields_use_spline_per_x_line(oracle64):
    from scipy.interpolate import CubicSpline
    c = small(N=9, M=7, seed=2)
    u = W.state(c)
    zeta, phi, zeta_y, phi_y = oracle64.fields(c.params(), u)
    y = W.mesh(c)[1]
    for k in (0, 3, 8):
        for f, fy in ((zeta, zeta_y), (phi, phi_y)):
            ref = CubicSpline(y, f[:, k], bc_type=((1, 0.0), "not-a-knot"))(y, 1)
            np.testing.assert_allclose(fy[:, k], ref, rtol=1e-10, atol=1e-13)


# ----------------------------------------------------------------------------
# P4 weights (L189, Q4)
# ----------------------------------------------------------------------------
def test_P4_weights_sum_to_area(oracle64):
    c = small(N=12, M=7, h=0.37)
    p = c.params()
    tot = sum(oracle64.weight(p, i, j) for i in range(c.N) for j in range(c.M))
    assert tot == pytest.approx((c.N - 1) * c.h * (c.M - 1) * c.h, rel=1e-14)
    assert oracle64.weight(p, 0, 0) == pytest.approx(c.h * c.h / 4)
    assert oracle64.weight(p, 3, c.M - 1) == pytest.approx(c.h * c.h / 2)


# ----------------------------------------------------------------------------
# P5 closed form of I (eq. (23), Q5) against tanh-sinh quadrature
# ----------------------------------------------------------------------------
def _golden_boxes():
    rows = []
    for line in (GOLDEN / "s2_box_integrals.txt").read_text().splitlines():
        if line.startswith("#") or not line.strip():
            continue
        *c, v = line.split()
        rows.append((tuple(map(float, c)), float(v)))
    return rows


def test_P5_box_integral_matches_quadrature(oracle64, oracle80):
    rows = _golden_boxes()
    assert len(rows) >= 8
    for c, v in rows:
        assert oracle64.box_integral(*c) == pytest.approx(v, rel=2e-15)
        assert oracle80.box_integral(*c) == pytest.approx(v, rel=2e-15)


def test_P5_S2_integral_is_direct_plus_image(oracle64):
    """I = direct box + image box (t' = -(y+y*)); with y_1 = 0 they merge into one box over
    t in [-(y_M + y*), y_M - y*]."""
    A, B, C = 1.09, 0.24, 1.16
    xs, ys, xa, xb, ya, yb = 0.35, 0.8, -2.0, 3.0, 0.0, 2.4
    I = oracle64.s2_integral(A, B, C, xs, ys, xa, xb, ya, yb)
    merged = oracle64.box_integral(A, B, C, xa - xs, xb - xs, -(yb + ys), yb - ys)
    assert I == pytest.approx(merged, rel=1e-14)
    # and against scipy's adaptive quadrature of the literal S2 (eqs. (21)-(22) L169-172)
    from scipy import integrate

    def S2(x, y):
        return (1 / np.sqrt(A * (x - xs) ** 2 + B * (x - xs) * (y - ys) + C * (y - ys) ** 2)
                + 1 / np.sqrt(A * (x - xs) ** 2 - B * (x - xs) * (y + ys) + C * (y + ys) ** 2))
    tot = 0.0
    for (x0, x1_) in ((xa, xs), (xs, xb)):
        for (y0, y1_) in ((ya, ys), (ys, yb)):
            v, _ = integrate.dblquad(lambda y, x: S2(x, y), x0, x1_, y0, y1_, epsabs=1e-10, epsrel=1e-10)
            tot += v
    assert I == pytest.approx(tot, rel=1e-7)


# ----------------------------------------------------------------------------
# mirror symmetry of the kernels (L107-109, L169-172; Q1)
# ----------------------------------------------------------------------------
def test_mirror_symmetry_of_kernels(oracle64):
    rng = np.random.default_rng(0)
    for _ in range(20):
        x, y, z, zx, zy, xs, ys, zs = rng.uniform(-2, 2, 8)
        y, ys = abs(y), abs(ys)
        A, B, C = 1 + 0.3 ** 2, 2 * 0.3 * 0.2, 1 + 0.2 ** 2
        K1, K2, S2 = oracle64.pair_kernels(x, y, z, zx, zy, xs, ys, zs, A, B, C)
        # y* -> -y* swaps the direct and the image term of K1 and K2
        K1m, K2m, _ = oracle64.pair_kernels(x, y, z, zx, zy, xs, -ys, zs, A, B, C)
        assert K1m == pytest.approx(K1, rel=1e-13) and K2m == pytest.approx(K2, rel=1e-13)
        # for S2 the mirror also flips zeta_y*, i.e. B -> -B
        _, _, S2m = oracle64.pair_kernels(x, y, z, zx, zy, xs, -ys, zs, A, -B, C)
        assert S2m == pytest.approx(S2, rel=1e-13)
        # explicit values: direct + image, image = same source seen from (x*, -y*)
        dx, dm, dp, dz = x - xs, y - ys, y + ys, z - zs
        Rm, Rp = np.sqrt(dx * dx + dm * dm + dz * dz), np.sqrt(dx * dx + dp * dp + dz * dz)
        assert K2 == pytest.approx(1 / Rm + 1 / Rp, rel=1e-13)
        assert K1 == pytest.approx((dz - dx * zx - dm * zy) / Rm ** 3 + (dz - dx * zx - dp * zy) / Rp ** 3, rel=1e-12)


# ----------------------------------------------------------------------------
# P1 full-plane identity: half-plane sum with images == direct-only sum over
# the evenly extended mesh y in [-y_M, y_M]  (pins the garbled K1 of L107, Q1,
# the sign of the image S2 term L172, the source-point slopes Q2, weights Q4)
# ----------------------------------------------------------------------------
def _full_plane_sums(c, u, k, l, oracle, want_star=False):
    p = c.params()
    zeta, phi, zeta_y, _ = oracle.fields(p, u)
    zeta_x = u[(c.N + 1) * c.M:].reshape(c.M, c.N + 1)[:, 1:]
    x, y = W.mesh(c)
    ext = lambda a, sgn: np.concatenate([sgn * a[:0:-1], a], 0)        # rows -(M-1)..(M-1)
    Z, P, ZX, ZY = ext(zeta, 1), ext(phi, 1), ext(zeta_x, 1), ext(zeta_y, -1)
    Yv = np.concatenate([-y[:0:-1], y])
    X, Y = np.meshgrid(x, Yv)
    cx = np.ones(c.N); cx[[0, -1]] = 0.5
    cy = np.ones(2 * c.M - 1); cy[[0, -1]] = 0.5
    Wt = c.h * c.h * np.outer(cy, cx)
    xs, ys = 0.5 * (x[k] + x[k + 1]), y[l]
    st = lambda a: 0.5 * (a[l, k] + a[l, k + 1])
    zs, ps, zxs, zys = st(zeta), st(phi), st(zeta_x), st(zeta_y)
    A, B, C = 1 + zxs ** 2, 2 * zxs * zys, 1 + zys ** 2
    dx, dy, dz = X - xs, Y - ys, Z - zs
    R = np.sqrt(dx ** 2 + dy ** 2 + dz ** 2)
    K1 = (dz - dx * ZX - dy * ZY) / R ** 3
    s1 = (Wt * (P - ps - X + xs) * K1).sum()
    s2 = (Wt * ZX / R).sum()
    s3 = (Wt / np.sqrt(A * dx ** 2 + B * dx * dy + C * dy ** 2)).sum()
    if want_star:
        return s1, s2, s3, dict(xs=xs, ys=ys, zs=zs, ps=ps, zxs=zxs, A=A, B=B, C=C)
    return s1, s2, s3


@pytest.mark.parametrize("kl", [(0, 0), (5, 2), (11, 4), (7, 0), (3, 6)])
def test_P1_full_plane_identity(oracle64, kl):
    c, u = _p1_fixture()
    k, l = kl
    t = oracle64.e2_terms(c.params(), u, k, l)
    s1, s2, s3 = _full_plane_sums(c, u, k, l, oracle64)
    assert t[2] == pytest.approx(s1, rel=1e-11, abs=1e-17)
    assert t[3] == pytest.approx(s2, rel=1e-12, abs=1e-15)
    assert t[4] == pytest.approx(s3, rel=1e-12)
    # the pin discriminates: the terms are far from zero at this state
    assert abs(s1) > 1e-5 and abs(s2) > 1e-3


def _p1_fixture():
    c = small(N=13, M=7, h=0.5, x1=-2.0, amp=0.3, seed=21)
    c = dataclasses.replace(c, eps=0.3)
    u = W.state(c)
    u[: (c.N + 1) * c.M] += 0.2 * np.random.default_rng(1).standard_normal((c.N + 1) * c.M)  # phi - x = O(1)
    return c, u


@pytest.mark.parametrize("prec", ["f64", "f80"])
def test_P1b_residual_row_is_eq12_with_its_printed_signs(oracle64, oracle80, prec):
    """The row the residual RETURNS (E2_row, not the parallel e2_terms), at a curved state with phi - x = O(1),
    against eq. (12) L101 assembled here from full-plane DIRECT-kernel sums (no images), the quadrature-pinned
    box integral (P5) and the printed signs:
        2 pi (phi* - x*) = -eps/rho* + int (phi - phi* - x + x*) K1 + int zeta_x K2,
    int zeta_x K2 -> sum w (zeta_x K2 - zeta_x* S2) + zeta_x* I (L181).  Every row of the mesh."""
    orc = oracle64 if prec == "f64" else oracle80
    c, u = _p1_fixture()
    x, y = W.mesh(c)
    E = orc.residual(c.params(), u)
    worst, k1_size = 0.0, 0.0
    for l in range(c.M):
        for k in range(c.N - 1):
            s1, s2, s3, st = _full_plane_sums(c, u, k, l, orc, want_star=True)
            I = orc.box_integral(st["A"], st["B"], st["C"], x[0] - st["xs"], x[-1] - st["xs"],
                                 -(y[-1] + st["ys"]), y[-1] - st["ys"])            # y_1 = 0: merged box
            rho = np.sqrt(st["xs"] ** 2 + st["ys"] ** 2 + (st["zs"] + 1) ** 2)
            ref = 2 * PI * (st["ps"] - st["xs"]) + c.eps / rho - s1 - (s2 - st["zxs"] * s3) - st["zxs"] * I
            worst = max(worst, abs(E[row_E2(c, k, l)] - ref))
            k1_size = max(k1_size, abs(s1))
    assert worst <= 1e-11 * np.abs(E).max(), worst
    assert k1_size > 1e-2            # the K1 sum is two orders above the tolerance: its sign and density are seen


def test_e2_terms_tie_to_residual_row(oracle64, oracle80):
    """e2_terms (the pieces the pins P1, PG1 look at) and the residual's own row are the same quantity:
    E2 = out0 + out1 - out2 - (out3 - zeta_x* out4) - zeta_x* out5."""
    c, u = _p1_fixture()
    for orc, tol in ((oracle64, 2e-12), (oracle80, 2e-14)):
        E = orc.residual(c.params(), u)
        for (k, l) in [(0, 0), (5, 2), (11, 4), (7, 0), (3, 6), (11, 6)]:
            t = orc.e2_terms(c.params(), u, k, l)
            ref = t[0] + t[1] - t[2] - (t[3] - t[6] * t[4]) - t[6] * t[5]
            assert abs(E[row_E2(c, k, l)] - ref) <= tol * max(1.0, abs(t[3])), (k, l)


# ----------------------------------------------------------------------------
# P2 Gauss flux: integral of K1 over a compact bump seen from the flat part
# vanishes when zeta_x, zeta_y are taken at the SOURCE point (Q2)
# ----------------------------------------------------------------------------
def test_P2_gauss_flux(oracle64):
    h = 0.2
    x = -6 + h * np.arange(61)
    y = h * np.arange(31)
    a, w = 0.4, 0.8
    xs, ys = -5.9 + 0.0, 0.0                      # target far upstream on the flat part
    tot = tot_wrong = 0.0
    for j, yy in enumerate(y):
        for i, xx in enumerate(x):
            z = a * np.exp(-(xx ** 2 + yy ** 2) / w ** 2)
            zx, zy = -2 * xx / w ** 2 * z, -2 * yy / w ** 2 * z
            wt = h * h * (0.5 if i in (0, 60) else 1) * (0.5 if j in (0, 30) else 1)
            K1, _, _ = oracle64.pair_kernels(xx, yy, z, zx, zy, xs, ys, 0.0, 1, 0, 1)
            tot += wt * K1
            # slopes at the target (flat: zero slopes) -- the rejected reading
            K1w, _, _ = oracle64.pair_kernels(xx, yy, z, 0.0, 0.0, xs, ys, 0.0, 1, 0, 1)
            tot_wrong += wt * K1w
    assert abs(tot) < 1e-12
    assert abs(tot_wrong) > 1e-4


# ----------------------------------------------------------------------------
# P6 uniform stream (L227 with eps = 0): E == 0
# ----------------------------------------------------------------------------
@pytest.mark.parametrize("scheme", [0, 1])
def test_P6_uniform_stream(oracle64, oracle80, scheme):
    c = dataclasses.replace(W.CONFIGS[0], eps=0.0)
    u0 = W.flat_state(c)
    for o, tol in ((oracle64, 2e-13), (oracle80, 2e-14)):  # x_k itself is an FP64-rounded input
        E = o.residual(c.params(scheme), u0)
        assert np.abs(E).max() < tol
    # first half (E1, E3, E4) and E5, E6 are exactly zero
    E = oracle64.residual(c.params(scheme), u0)
    half = (c.N + 1) * c.M
    assert np.abs(E[:half]).max() == 0.0
    assert np.abs(E[half:].reshape(c.M, c.N + 1)[:, :2]).max() == 0.0


def test_source_term_at_flat_state(oracle64):
    """Flat state, eps > 0: the only non-zero part of E2 is eps/sqrt(x*^2 + y*^2 + 1) (L101, B.1 L431)."""
    c = W.CONFIGS[0]
    E = oracle64.residual(c.params(), W.flat_state(c))
    x, y = W.mesh(c)
    xs = 0.5 * (x[:-1] + x[1:])
    ref = c.eps / np.sqrt(xs[None, :] ** 2 + y[:, None] ** 2 + 1)
    E2 = E[(c.N + 1) * c.M:].reshape(c.M, c.N + 1)[:, 2:]
    np.testing.assert_allclose(E2, ref, rtol=0, atol=3e-13)


# ----------------------------------------------------------------------------
# PH the source term of eq. (12) L101 away from zeta = 0: eps / sqrt(x*^2 + y*^2 + (zeta* + 1)^2) is the potential
# of a point source at (0, 0, -1) (L72), i.e. as a function of the surface point (x*, y*, zeta*) it is HARMONIC and
# symmetric about the plane z = -1.  At a level surface zeta = c under the uniform stream phi = x every other term
# of the row vanishes (K1 multiplies phi - phi* - x + x* = 0, the K2 / S2 / I terms multiply zeta_x = 0), so the
# rows E2 of three states c - h, c, c + h sample the source term on a 3-D lattice: its 7-point Laplacian must vanish
# at O(h^2), and the rows at c = -1 + d and c = -1 - d must coincide.  (zeta*^2 + 1 in place of (zeta* + 1)^2 has
# Laplacian -3 eps / (r^2 + 1)^(5/2) and no such symmetry.)
# ----------------------------------------------------------------------------
def _level_rows(orc, c, level):
    u = W.pack(c, np.full(c.M, c.x1), np.ones((c.M, c.N)), np.full(c.M, level), np.zeros((c.M, c.N)))
    E = orc.residual(c.params(), u)
    return E[(c.N + 1) * c.M:].reshape(c.M, c.N + 1)[:, 2:]


def test_PH_source_term_is_harmonic_and_centred_at_minus_one(oracle64):
    worst = []
    for h, N, M in ((0.2, 9, 6), (0.1, 17, 11)):
        c = dataclasses.replace(small(N=N, M=M, h=h, x1=0.45), eps=1.0)
        lo, mid, hi = (_level_rows(oracle64, c, 0.3 + d) for d in (-h, 0.0, h))
        lap = (mid[1:-1, 2:] + mid[1:-1, :-2] + mid[2:, 1:-1] + mid[:-2, 1:-1] + hi[1:-1, 1:-1] + lo[1:-1, 1:-1]
               - 6 * mid[1:-1, 1:-1]) / h ** 2
        worst.append(np.abs(lap).max())
        assert mid.min() > 0.3                                  # the term is O(eps) here, not round-off
    # discretisation error of the 7-point stencil only: small and shrinking with h (4.2e-3, 1.5e-3; the finer mesh
    # also has interior points nearer the source); zeta*^2 + 1 would leave a Laplacian of order 1 at either h
    assert worst[1] < 0.5 * worst[0] and worst[0] < 1e-2, worst
    c = dataclasses.replace(small(N=9, M=6, h=0.2, x1=0.45), eps=1.0)
    np.testing.assert_allclose(_level_rows(oracle64, c, -1 + 0.4), _level_rows(oracle64, c, -1 - 0.4), rtol=1e-13)
    assert np.abs(_level_rows(oracle64, c, -1 + 0.4) - _level_rows(oracle64, c, -1 + 0.5)).max() > 1e-2


# ----------------------------------------------------------------------------
# P7 tilted plane zeta = alpha x + beta: K1 == 0, K2 == S2 pointwise, so
#   E2 = 2 pi (phi* - x*) + eps / rho* - alpha I(A = 1 + alpha^2, B = 0, C = 1)
# with I evaluated HERE by quadrature-pinned closed form; E1 in closed form too
# ----------------------------------------------------------------------------
def test_P7_tilted_plane(oracle64):
    c = small(N=11, M=6, h=0.5, x1=-3.0, seed=4)
    c = dataclasses.replace(c, eps=0.7)
    alpha, beta, cphi = 0.15, -0.05, 1.2
    x, y = W.mesh(c)
    rng = np.random.default_rng(9)
    g = 0.1 * rng.standard_normal(c.N)                      # phi_x = cphi + g(x): any phi, constant in y
    u = W.pack(c, np.full(c.M, 0.3), np.tile(cphi + g, (c.M, 1)),
               np.full(c.M, alpha * x[0] + beta), np.full((c.M, c.N), alpha))
    E = oracle64.residual(c.params(), u)
    zeta, phi, zeta_y, phi_y = oracle64.fields(c.params(), u)
    assert np.abs(zeta_y).max() < 1e-14 and np.abs(phi_y).max() < 1e-13
    np.testing.assert_allclose(zeta, np.tile(alpha * x + beta, (c.M, 1)), atol=1e-14)
    A, B, C = 1 + alpha ** 2, 0.0, 1.0
    half = (c.N + 1) * c.M
    for l in range(c.M):
        for k in range(c.N - 1):
            xs, ys = 0.5 * (x[k] + x[k + 1]), y[l]
            zs, ps = alpha * xs + beta, 0.5 * (phi[l, k] + phi[l, k + 1])
            # I: merged box (y_1 = 0) through the quadrature-pinned box integral
            I = oracle64.box_integral(A, B, C, x[0] - xs, x[-1] - xs, -(y[-1] + ys), y[-1] - ys)
            ref = 2 * PI * (ps - xs) + c.eps / np.sqrt(xs ** 2 + ys ** 2 + (zs + 1) ** 2) - alpha * I
            assert E[half + l * (c.N + 1) + 2 + k] == pytest.approx(ref, rel=1e-12, abs=1e-13)
            pxs = cphi + 0.5 * (g[k] + g[k + 1])
            ref1 = 0.5 * pxs ** 2 / (1 + alpha ** 2) + zs / c.froude ** 2 - 0.5   # (13) L113 with phi_y = zeta_y = 0
            assert E[l * (c.N + 1) + 2 + k] == pytest.approx(ref1, rel=1e-13, abs=1e-15)


def test_E1_bernoulli_formula(oracle64):
    """eq. (13) L113 at starred values with all four slopes non-zero (FD scheme so that the y-slopes are
    simple to state here)."""
    c = small(N=9, M=6, h=0.5, x1=-1.0, amp=0.3, seed=8)
    u = W.state(c)
    zeta, phi, zeta_y, phi_y = oracle64.fields(c.params(1), u)
    E = oracle64.residual(c.params(1), u, rows=[])
    zx = u[(c.N + 1) * c.M:].reshape(c.M, c.N + 1)[:, 1:]
    px = u[: (c.N + 1) * c.M].reshape(c.M, c.N + 1)[:, 1:]
    st = lambda a: 0.5 * (a[:, :-1] + a[:, 1:])
    Z, ZX, ZY, PX, PY = st(zeta), st(zx), st(zeta_y), st(px), st(phi_y)
    ref = 0.5 * ((1 + ZX ** 2) * PY ** 2 + (1 + ZY ** 2) * PX ** 2 - 2 * ZX * ZY * PX * PY) / (1 + ZX ** 2 + ZY ** 2) \
        + Z / c.froude ** 2 - 0.5
    got = E[: (c.N + 1) * c.M].reshape(c.M, c.N + 1)[:, 2:]
    np.testing.assert_allclose(got, ref, rtol=1e-12, atol=1e-15)
    assert np.abs(PY).max() > 1e-4 and np.abs(ZY).max() > 1e-3


# ----------------------------------------------------------------------------
# PB the Bernoulli row on an EXACT potential flow (pins the nonlinear terms of eq. (13) L113 with all
# four slopes and the cross term live, by something the formula is not: the speed of a uniform stream).
#   Phi = a x + b y + c z is harmonic; the plane zeta = alpha x + beta y + gamma is a stream surface of it iff
#   Phi_x zeta_x + Phi_y zeta_y = Phi_z, i.e. c = a alpha + b beta (the kinematic condition, eq. (8)).
#   On the surface phi(x, y) = Phi(x, y, zeta(x, y)):  phi_x = a + c alpha,  phi_y = b + c beta.
#   The first term of (13) is |grad Phi|^2 / 2 written in (phi_x, phi_y, zeta_x, zeta_y) with the kinematic
#   condition eliminated, so here it must return (a^2 + b^2 + c^2) / 2 EXACTLY:
#       E1 = (a^2 + b^2 + c^2) / 2 + zeta* / F^2 - 1/2.
#   A wrong sign of the cross term, phi_x / phi_y (or zeta_x / zeta_y) transposed, a lost factor 2 or a wrong
#   denominator all change the value at O(1) of the slopes.  y_1 != 0, so that the y-derivatives of data linear
#   in y are exact in both schemes (not-a-knot spline at both ends; one-sided 3-point differences) - with
#   y_1 = 0 the even-extension end condition of reading Q3 would force zeta_y = 0 on the first line.
# ----------------------------------------------------------------------------
@pytest.mark.parametrize("scheme", [0, 1])
@pytest.mark.parametrize("flow", [(1.0, 0.35, 0.3, -0.2), (0.8, -0.5, -0.25, 0.4), (1.1, 0.0, 0.2, 0.3)])
def test_PB_bernoulli_row_on_exact_tilted_plane_flow(oracle64, oracle80, scheme, flow):
    a, b, alpha, beta = flow
    gamma = 0.07
    cz = a * alpha + b * beta                                  # kinematic condition
    c = dataclasses.replace(small(N=9, M=7, h=0.35, x1=-1.3), y1=0.6, froude=0.8)
    x, y = W.mesh(c)
    zeta1 = alpha * x[0] + beta * y + gamma
    phi1 = a * x[0] + b * y + cz * zeta1
    u = W.pack(c, phi1, np.full((c.M, c.N), a + cz * alpha), zeta1, np.full((c.M, c.N), alpha))
    for orc, tol in ((oracle64, 2e-15), (oracle80, 1e-15)):
        zeta, phi, zeta_y, phi_y = orc.fields(c.params(scheme), u)
        # the reconstruction hands the row the slopes of the exact flow (else the pin below tests nothing)
        np.testing.assert_allclose(zeta_y, beta, rtol=0, atol=1e-13)
        np.testing.assert_allclose(phi_y, b + cz * beta, rtol=0, atol=1e-13)
        E = orc.residual(c.params(scheme), u, rows=[])
        E1 = E[: (c.N + 1) * c.M].reshape(c.M, c.N + 1)[:, 2:]
        xs = 0.5 * (x[:-1] + x[1:])
        zs = alpha * xs[None, :] + beta * y[:, None] + gamma
        ref = 0.5 * (a * a + b * b + cz * cz) + zs / c.froude ** 2 - 0.5
        np.testing.assert_allclose(E1, ref, rtol=0, atol=200 * tol)
    # the pin has power: the slopes and the cross term are all of order 0.1 .. 1
    zx, zy, px, py = alpha, beta, a + cz * alpha, b + cz * beta
    assert min(abs(zx), abs(zy), abs(px)) > 0.1 and abs(2 * zx * zy * px * py) > 1e-3 or b == 0.0
    assert abs(((1 + zx * zx) * px * px + (1 + zy * zy) * py * py) - ((1 + zx * zx) * py * py + (1 + zy * zy) * px * px)) > 1e-2


# ----------------------------------------------------------------------------
# PS  A, B, C of L177: S2 is the singular part of K2.
#   L164-181: S2 = 1/sqrt(A dx^2 + B dx dy + C dy^2) is subtracted because it has the SAME singularity as
#   K2 = 1/R at the target, R^2 = dx^2 + dy^2 + (zeta - zeta*)^2.  With zeta - zeta* = zeta_x* dx + zeta_y* dy
#   + O(h^2) at a node next to the target, R^2 = Q + O(h^3) if and only if Q's coefficients are
#   A = 1 + zeta_x*^2, B = 2 zeta_x* zeta_y*, C = 1 + zeta_y*^2; then 1/R - 1/sqrt(Q) stays bounded and
#       h (K2 - S2) = O(h) -> 0   under h -> h/3 -> h/9 (the half-mesh points of mesh h are half-mesh points of
#   mesh h/3: k' = 3k + 1, l' = 3l), whereas any other coefficient leaves R^2 - Q = O(h^2) and h (K2 - S2) tends
#   to a non-zero constant.  The six nodes around the target see all three coefficients: (dx, dy) =
#   (+-h/2, 0) isolates A, (+-h/2, +-h) mixes A, B, C with both signs of dx dy.  A, B, C are the ROW'S OWN
#   (oracle.row_abc calls the helper E2_row calls), K2 and S2 are the oracle's pair kernels (pinned by P1/P2);
#   the image parts of both are smooth at the target (y* >= 2 h_0) and drop out of the limit.
# ----------------------------------------------------------------------------
def _near_field_mismatch(orc, c, k, l, abc_of=lambda A, B, C: (A, B, C)):
    """max over the six nodes around target (k, l) of h |K2 - S2|, and the row's (A, B, C)."""
    p, u = c.params(), W.state(c)
    x, y = W.mesh(c)
    zeta, _, zeta_y, _ = orc.fields(p, u)
    zeta_x = u[(c.N + 1) * c.M:].reshape(c.M, c.N + 1)[:, 1:]
    A, B, C, zs = orc.row_abc(p, u, k, l)
    A2, B2, C2 = abc_of(A, B, C)
    xs, ys = 0.5 * (x[k] + x[k + 1]), y[l]
    worst = 0.0
    for j in (l - 1, l, l + 1):
        for i in (k, k + 1):
            K1, K2, S2 = orc.pair_kernels(x[i], y[j], zeta[j, i], zeta_x[j, i], zeta_y[j, i], xs, ys, zs, A2, B2, C2)
            worst = max(worst, c.h * abs(K2 - S2))
    return worst, (A, B, C)


def test_PS_S2_is_the_singular_part_of_K2(oracle64):
    base = W.custom(N=9, M=7, h=0.6, x1=8.3, amp=0.6, seed=20, eps=0.3)
    # the interior target where zeta_x* zeta_y* is largest on the coarse mesh (B matters most there)
    best, kl = 0.0, None
    for l in range(2, base.M - 1):
        for k in range(1, base.N - 2):
            A, B, C, _ = oracle64.row_abc(base.params(), W.state(base), k, l)
            if abs(B) > best:
                best, kl = abs(B), (k, l)
    assert best > 0.05, best                  # slopes of order 0.2: the wrong-B constant is far above round-off
    got, wrong_B, wrong_AC = [], [], []
    k, l = kl
    for r in range(3):
        f = 3 ** r
        c = dataclasses.replace(base, N=(base.N - 1) * f + 1, M=(base.M - 1) * f + 1, h=base.h / f)
        d, (A, B, C) = _near_field_mismatch(oracle64, c, k, l)
        got.append(d)
        # L177 restated nowhere: what the row's own coefficients must do is make `got` vanish; for contrast,
        # the same measurement with B halved and with A, C swapped
        wrong_B.append(_near_field_mismatch(oracle64, c, k, l, lambda A, B, C: (A, B / 2, C))[0])
        wrong_AC.append(_near_field_mismatch(oracle64, c, k, l, lambda A, B, C: (C, B, A))[0])
        k, l = 3 * k + 1, 3 * l
    got, wrong_B, wrong_AC = map(np.array, (got, wrong_B, wrong_AC))
    # O(h): each refinement by 3 divides it by about 3 (measured 4.9, 4.0, then 3.4: the O(h^2) part dies out;
    # accept 2 .. 6), and it ends far below the wrong ones, which stay where they were
    assert (got[:-1] / got[1:] > 2.0).all() and (got[:-1] / got[1:] < 6.0).all(), got
    assert got[-1] < 0.15 * got[0]
    assert (wrong_B[-1] > 0.7 * wrong_B[0]) and (wrong_AC[-1] > 0.7 * wrong_AC[0]), (wrong_B, wrong_AC)
    assert got[-1] < 0.2 * min(wrong_B[-1], wrong_AC[-1]), (got, wrong_B, wrong_AC)


# ----------------------------------------------------------------------------
# P8 O(h^2) convergence of E2 under h -> h/3 (midpoints coincide: k' = 3k+1, l' = 3l, 0-based)
# ----------------------------------------------------------------------------
def test_P8_second_order_convergence(oracle64):
    base = dataclasses.replace(W.CONFIGS[0], eps=0.3, amp=0.1)
    vals = []
    pts = [(10, 0), (14, 3), (20, 5), (12, 2)]
    for r in range(4):
        f = 3 ** r
        c = dataclasses.replace(base, N=(base.N - 1) * f + 1, M=(base.M - 1) * f + 1, h=base.h / f)
        u = W.state(c)
        rows = []
        for (k, l) in pts:
            kk, ll = k, l
            for _ in range(r):
                kk, ll = 3 * kk + 1, 3 * ll
            rows.append(ll * (c.N - 1) + kk)
        x, y = W.mesh(c)
        E = oracle64.residual(c.params(), u, rows=rows)
        half = (c.N + 1) * c.M
        vals.append([E[half + (t // (c.N - 1)) * (c.N + 1) + 2 + t % (c.N - 1)] for t in rows])
    v = np.array(vals)
    d = np.abs(np.diff(v, axis=0))
    ratios = d[:-1] / d[1:]
    # ideal ratio 9; accept the asymptotic range
    assert (ratios[-1] > 5).all() and (ratios[-1] < 16).all(), ratios


# ----------------------------------------------------------------------------
# P9 linear-Jacobian closed forms (App. B) from FD columns at u_0, eps = 0
# ----------------------------------------------------------------------------
def _coeffs():
    out = {}
    for line in (GOLDEN / "linear_jacobian_coeffs.txt").read_text().splitlines():
        if line.startswith("#") or not line.strip():
            continue
        kind, case, val = line.split()
        out[(kind, case)] = float(val)
    return out


def _case(n, k):
    """paper's 1-based (n,k) case label."""
    if n == 1 and k == 1:
        return "n=1,k=1"
    if n == 1:
        return "n=1,k>1"
    if n < k:
        return "1<n<k"
    if n == k:
        return "n=k"
    if n == k + 1:
        return "n=k+1"
    return None


def test_P9_linear_jacobian(oracle80, oracle64):
    c = dataclasses.replace(small(N=13, M=5, h=0.4, x1=-2.2), eps=0.0)
    p = c.params()
    u0 = W.flat_state(c)
    co = _coeffs()
    dlt = 1e-6
    half = (c.N + 1) * c.M
    E0 = oracle80.residual(p, u0)
    x, y = W.mesh(c)

    def col(idx):
        up = u0.copy(); up[idx] += dlt
        um = u0.copy(); um[idx] -= dlt
        return (oracle80.residual(p, up) - oracle80.residual(p, um)) / (2 * dlt)

    m = 2
    # d/dphi_{1,m}: B.5 L485 (2 pi on line m), B.3 L474 (E1: 0)
    J = col(idx_phi1(c, m))
    for l in range(c.M):
        for k in range(c.N - 1):
            assert J[row_E2(c, k, l)] == pytest.approx(2 * PI if l == m else 0.0, abs=1e-7)
            assert J[row_E1(c, k, l)] == pytest.approx(0.0, abs=1e-7)
    # d/dzeta_{1,m}: B.3 L478 (1/F^2 on line m), L496 (E2: 0)
    J = col(idx_zeta1(c, m))
    for l in range(c.M):
        for k in range(c.N - 1):
            assert J[row_E1(c, k, l)] == pytest.approx(1 / c.froude ** 2 if l == m else 0.0, abs=1e-7)
            assert J[row_E2(c, k, l)] == pytest.approx(0.0, abs=1e-7)
    # d/dphix_{n,m}: B.5 L487-494 and B.3 L476
    for n0 in (0, 1, 5, c.N - 1):
        J = col(idx_phix(c, n0, m))
        for l in range(c.M):
            for k in range(c.N - 1):
                case = _case(n0 + 1, k + 1) if l == m else None
                ref2 = co[("E2_phix", case)] * PI * c.h if case else 0.0
                ref1 = 0.5 if (l == m and n0 in (k, k + 1)) else 0.0
                assert J[row_E2(c, k, l)] == pytest.approx(ref2, abs=1e-7)
                assert J[row_E1(c, k, l)] == pytest.approx(ref1, abs=1e-7)
    # d/dzetax_{n,m}: B.6 L498-501 for E2, B.4 (read from B.2 L458) for E1
    def K3(i, j, k, l):
        xs = 0.5 * (x[k] + x[k + 1])
        return 1 / np.hypot(x[i] - xs, y[j] - y[l]) + 1 / np.hypot(x[i] - xs, y[j] + y[l])
    for n0 in (0, 4, c.N - 1):
        J = col(idx_zetax(c, n0, m))
        for l in range(c.M):
            for k in range(c.N - 1):
                ref = -oracle64.weight(p, n0, m) * K3(n0, m, k, l)
                if l == m and n0 in (k, k + 1):
                    xs = 0.5 * (x[k] + x[k + 1])
                    sumwK3 = sum(oracle64.weight(p, i, j) * K3(i, j, k, l) for i in range(c.N) for j in range(c.M))
                    I = oracle64.box_integral(1.0, 0.0, 1.0, x[0] - xs, x[-1] - xs, -(y[-1] + y[l]), y[-1] - y[l])
                    ref += 0.5 * sumwK3 - 0.5 * I
                assert J[row_E2(c, k, l)] == pytest.approx(ref, abs=2e-7), (n0, k, l)
                case = _case(n0 + 1, k + 1) if l == m else None
                ref1 = co[("E1_zetax", case)] * c.h / c.froude ** 2 if case else 0.0
                assert J[row_E1(c, k, l)] == pytest.approx(ref1, abs=1e-7)
    assert np.abs(E0).max() < 1e-14


# ----------------------------------------------------------------------------
# Jv by eq. (25) L219 and the shift sigma (BASELINE.json)
# ----------------------------------------------------------------------------
def test_sigma_formula(oracle64):
    rng = np.random.default_rng(1)
    u, v = rng.standard_normal(500), rng.standard_normal(500)
    assert oracle64.sigma(u, v) == pytest.approx(1e-7 * (1 + np.linalg.norm(u)) / np.linalg.norm(v), rel=1e-14)


def test_jv_linear_rows_and_consistency(oracle80, oracle64):
    """E3-E6 are linear in u, so their JV rows are the linear formulas (L462-468) applied to v; the other
    rows must agree with a central difference at a different step; E(u_b) output is E at fma(sigma,v,u)."""
    c = W.CONFIGS[0]
    p = c.params()
    u = W.state(c)
    v = W.directions(c, 1)[0]
    s = oracle80.sigma(u, v)
    JV, Ep = oracle80.jv(p, u, v, s)
    ub = np.array([np.float64(a) for a in u])  # u_b with one rounding per entry
    import math
    ub = np.array([math.fma(s, float(b), float(a)) for a, b in zip(u, v)]) if hasattr(math, "fma") else u + s * v
    np.testing.assert_allclose(Ep, oracle80.residual(p, ub), rtol=0, atol=1e-16)
    n, x1, dx = c.n_rad, c.x1, c.h
    for l in range(c.M):
        dv = (ub - u) / s                      # the direction actually taken after rounding u_b
        p1, px1, px2 = dv[idx_phi1(c, l)], dv[idx_phix(c, 0, l)], dv[idx_phix(c, 1, l)]
        z1, zx1, zx2 = dv[idx_zeta1(c, l)], dv[idx_zetax(c, 0, l)], dv[idx_zetax(c, 1, l)]
        blk, blk2 = l * (c.N + 1), (c.N + 1) * c.M + l * (c.N + 1)
        assert JV[blk] == pytest.approx(x1 * px1 + n * p1, rel=1e-9, abs=1e-9)
        assert JV[blk + 1] == pytest.approx(x1 * (px2 - px1) / dx + n * px1, rel=1e-9, abs=1e-7)
        assert JV[blk2] == pytest.approx(x1 * zx1 + n * z1, rel=1e-9, abs=1e-9)
        assert JV[blk2 + 1] == pytest.approx(x1 * (zx2 - zx1) / dx + n * zx1, rel=1e-9, abs=1e-7)
    big = 1e-5
    cd = (oracle80.residual(p, u + big * v) - oracle80.residual(p, u - big * v)) / (2 * big)
    assert np.abs(JV - cd).max() < 1e-5 * np.abs(cd).max()
    # the double-precision oracle agrees with the long-double one at the FD rounding floor
    JV64, _ = oracle64.jv(p, u, v, s)
    assert np.abs(JV64 - JV).max() < 1e-6 * np.abs(JV).max()


def test_f64_vs_f80_residual(oracle64, oracle80):
    for c in W.CONFIGS[:2]:
        u = W.state(c)
        E64, E80 = oracle64.residual(c.params(), u), oracle80.residual(c.params(), u)
        assert np.abs(E64 - E80).max() < 1e-12 * np.abs(E80).max()


def test_row_subset_equals_full(oracle64):
    c = W.CONFIGS[0]
    u = W.state(c)
    E = oracle64.residual(c.params(), u)
    rows = [0, 17, c.targets - 1, 123]
    Es = oracle64.residual(c.params(), u, rows=rows)
    half = (c.N + 1) * c.M
    for t in rows:
        i = half + (t // (c.N - 1)) * (c.N + 1) + 2 + t % (c.N - 1)
        assert Es[i] == E[i]
    assert np.array_equal(Es[:half], E[:half])
    assert np.isnan(Es[half:]).sum() == c.targets - len(rows)


# ----------------------------------------------------------------------------
# The exact Jacobian action J(u) v (oracle c80: complex-step derivative of the SAME residual
# code, Im E(u + i h v) / h).  PJ1: closed forms of App. B; PJ2: Richardson-extrapolated
# central differences of the long-double residual at a nonlinear state; PJ3: linear rows.
# ----------------------------------------------------------------------------
def test_PJ1_exact_jacobian_reproduces_appendix_B(oracleC, oracle64):
    """Columns of J at u_0, eps = 0, to round-off (the FD pin P9 above can only reach 1e-7)."""
    c = dataclasses.replace(small(N=13, M=5, h=0.4, x1=-2.2), eps=0.0)
    p = c.params()
    u0 = W.flat_state(c)
    co = _coeffs()
    x, y = W.mesh(c)
    TOLJ = 2e-13

    def col(idx):
        e = np.zeros(c.n); e[idx] = 1.0
        return oracleC.jv_exact(p, u0, e)

    m = 2
    J = col(idx_phi1(c, m))
    for l in range(c.M):
        for k in range(c.N - 1):
            assert J[row_E2(c, k, l)] == pytest.approx(2 * PI if l == m else 0.0, abs=TOLJ)
            assert J[row_E1(c, k, l)] == pytest.approx(0.0, abs=TOLJ)
    J = col(idx_zeta1(c, m))
    for l in range(c.M):
        for k in range(c.N - 1):
            assert J[row_E1(c, k, l)] == pytest.approx(1 / c.froude ** 2 if l == m else 0.0, abs=TOLJ)
            assert J[row_E2(c, k, l)] == pytest.approx(0.0, abs=TOLJ)
    for n0 in (0, 1, 5, c.N - 1):
        J = col(idx_phix(c, n0, m))
        for l in range(c.M):
            for k in range(c.N - 1):
                case = _case(n0 + 1, k + 1) if l == m else None
                ref2 = co[("E2_phix", case)] * PI * c.h if case else 0.0
                ref1 = 0.5 if (l == m and n0 in (k, k + 1)) else 0.0
                assert J[row_E2(c, k, l)] == pytest.approx(ref2, abs=TOLJ)
                assert J[row_E1(c, k, l)] == pytest.approx(ref1, abs=TOLJ)

    def K3(i, j, k, l):
        xs = 0.5 * (x[k] + x[k + 1])
        return 1 / np.hypot(x[i] - xs, y[j] - y[l]) + 1 / np.hypot(x[i] - xs, y[j] + y[l])
    for n0 in (0, 4, c.N - 1):
        J = col(idx_zetax(c, n0, m))
        for l in range(c.M):
            for k in range(c.N - 1):
                ref = -oracle64.weight(p, n0, m) * K3(n0, m, k, l)
                if l == m and n0 in (k, k + 1):
                    xs = 0.5 * (x[k] + x[k + 1])
                    sumwK3 = sum(oracle64.weight(p, i, j) * K3(i, j, k, l) for i in range(c.N) for j in range(c.M))
                    I = oracle64.box_integral(1.0, 0.0, 1.0, x[0] - xs, x[-1] - xs, -(y[-1] + y[l]), y[-1] - y[l])
                    ref += 0.5 * sumwK3 - 0.5 * I
                assert J[row_E2(c, k, l)] == pytest.approx(ref, abs=1e-12), (n0, k, l)
                case = _case(n0 + 1, k + 1) if l == m else None
                ref1 = co[("E1_zetax", case)] * c.h / c.froude ** 2 if case else 0.0
                assert J[row_E1(c, k, l)] == pytest.approx(ref1, abs=TOLJ)


@pytest.mark.parametrize("scheme,y1", [(0, 0.0), (1, 0.0), (0, 0.6)])
def test_PJ2_exact_jv_vs_richardson_central_differences(oracleC, oracle80, scheme, y1):
    """Nonlinear state, random direction: D(s) = (E(u+sv) - E(u-sv)) / 2s in long double has error
    c2 s^2 + c4 s^4 + rounding; (4 D(s/2) - D(s)) / 3 removes the s^2 term.  Both sides use every
    term of the residual (K1, K2, S2, I, Bernoulli, spline), so a derivative that silently drops the
    dependence of anything on u (e.g. of A, B, C inside S2 or I) fails here."""
    c = W.custom(11, 6, 0.5, -2.0, y1=y1, seed=5, eps=0.4, amp=0.08)
    p = c.params(scheme)
    rng = np.random.default_rng(8)
    u = W.state(c) + 1e-2 * rng.standard_normal(c.n)
    v = rng.standard_normal(c.n)
    JV, E0 = oracleC.jv_exact(p, u, v, want_e0=True)
    assert np.abs(E0 - oracle80.residual(p, u)).max() <= 1e-15 * np.abs(E0).max()  # Re part is E(u)

    def D(s):
        return (oracle80.residual(p, u + s * v) - oracle80.residual(p, u - s * v)) / (2 * s)
    s = 2.0 ** -12   # exactly representable: u +- s v is rounded once per entry (error ~1e-16 / s)
    rich = (4 * D(s / 2) - D(s)) / 3
    scale = np.abs(JV).max()
    # remaining error: c4 s^4 (s^4 = 4e-15, large fourth derivatives near the singular pairs),
    # rounding of u +- s v in FP64 ~ 1e-16 |J| / s
    assert np.abs(JV - rich).max() / scale <= 1e-10
    # and the plain central difference converges to it at second order
    e1 = np.abs(JV - D(s)).max()
    e2 = np.abs(JV - D(s / 2)).max()
    assert 3.5 <= e1 / e2 <= 4.5


def test_PJ3_exact_jv_linear_rows_and_linearity(oracleC):
    """E3-E6 are linear in u (eq. (24)): their JV rows are the homogeneous formulas applied to
    v (B.1 L431); J(u)(a v + b w) = a J(u) v + b J(u) w to round-off; sampled rows leave NaN."""
    c = small(N=9, M=5, h=0.5, x1=-1.7)
    p = c.params()
    rng = np.random.default_rng(4)
    u = W.state(c) + 1e-2 * rng.standard_normal(c.n)
    v, w = rng.standard_normal(c.n), rng.standard_normal(c.n)
    JV = oracleC.jv_exact(p, u, v)
    half = (c.N + 1) * c.M
    n_rad, x1, dx = c.n_rad, c.x1, c.h
    for l in range(c.M):
        p1, px1, px2 = v[idx_phi1(c, l)], v[idx_phix(c, 0, l)], v[idx_phix(c, 1, l)]
        z1, zx1, zx2 = v[idx_zeta1(c, l)], v[idx_zetax(c, 0, l)], v[idx_zetax(c, 1, l)]
        b = l * (c.N + 1)
        assert JV[b] == pytest.approx(x1 * px1 + n_rad * p1, rel=1e-14)
        assert JV[b + 1] == pytest.approx(x1 * (px2 - px1) / dx + n_rad * px1, rel=1e-14)
        assert JV[half + b] == pytest.approx(x1 * zx1 + n_rad * z1, rel=1e-14)
        assert JV[half + b + 1] == pytest.approx(x1 * (zx2 - zx1) / dx + n_rad * zx1, rel=1e-14)
    JW = oracleC.jv_exact(p, u, w)
    Jc = oracleC.jv_exact(p, u, 0.3 * v - 1.7 * w)
    assert np.abs(Jc - (0.3 * JV - 1.7 * JW)).max() <= 1e-13 * np.abs(Jc).max()
    rows = np.array([0, 7, 21], dtype=np.int32)
    Js = oracleC.jv_exact(p, u, v, rows=rows)
    mask = ~np.isnan(Js)
    assert mask.sum() == half + 2 * c.M + rows.size
    assert np.array_equal(Js[mask], JV[mask])
