"""Pins of oracle/jfnk.py (linear-Jacobian preconditioner of App. B/C, right-preconditioned
GMRES, damped Newton) against what the paper and the mathematics fix.  CPU only; nothing here
touches the CUDA path.  Citations are /root/reference/PAPER.md lines.
"""
import numpy as np
import pytest
import scipy.sparse.linalg as spla

import oracle.jfnk as J
import workloads as W

PI = np.pi


def small(N=9, M=5, h=0.5, x1=-2.0, **kw):
    return W.custom(N, M, h, x1, **kw)


# ----------------------------------------------------------------------------
# PL1: the linear Jacobian of App. B is the Jacobian of the nonlinear residual at the flat
# state with eps = 0 (section 4.2: "applying our numerical scheme to the linearised
# governing equations").  Every column, against the complex-step derivative of the residual
# code (which contains no App. B formula).
# ----------------------------------------------------------------------------
@pytest.mark.parametrize("shape", [dict(N=9, M=5, h=0.5, x1=-2.0), dict(N=6, M=7, h=0.3, x1=-1.1)])
def test_linear_jacobian_is_jacobian_at_flat_state(oracle64, oracleC, shape):
    c = small(**shape, eps=0.0)
    p = c.params()
    P = J.linear_jacobian(p, oracle64.box_integral)
    u0 = W.flat_state(c)
    n = c.n
    Jc = np.empty((n, n))
    for j in range(n):
        e = np.zeros(n); e[j] = 1.0
        Jc[:, j] = oracleC.jv_exact(p, u0, e)
    assert np.abs(P - Jc).max() <= 2e-13 * np.abs(Jc).max()


def test_linear_jacobian_printed_entries(oracle64):
    """Entries exactly as printed: (B.3) 1/2; (B.5) 2 pi, pi dx/2, pi dx, 2 pi dx, 3 pi dx/2, pi dx/2
    (L474-494); (B.4) by the pattern of (B.2) L458 (reading Q8); dE2/d zeta_1 = 0 (L496); radiation
    rows (B.2) L462-468; off-diagonal (B.6) entry = -w K3 (L498-501)."""
    c = small(N=9, M=5, h=0.5, x1=-2.0)
    p = c.params()
    N, M, dx, F2 = c.N, c.M, p["dx"], p["froude"] ** 2
    n1, H = N + 1, (N + 1) * M
    P = J.linear_jacobian(p, oracle64.box_integral)
    l = 2
    r = lambda k: l * n1 + 1 + k          # E1_{k,l}; + H for E2_{k,l}
    col = lambda n: l * n1 + n            # (f_x)_{n,l}; col(0) = f_{1,l}; + H for zeta
    # (B.3)
    assert P[r(4), col(4)] == 0.5 and P[r(4), col(5)] == 0.5 and P[r(4), col(3)] == 0.0 and P[r(4), col(0)] == 0.0
    # (B.5)
    assert P[H + r(4), col(0)] == 2 * PI
    assert P[H + r(1), col(1)] == pytest.approx(PI * dx / 2, rel=1e-15)
    assert P[H + r(4), col(1)] == pytest.approx(PI * dx, rel=1e-15)
    assert P[H + r(4), col(2)] == pytest.approx(2 * PI * dx, rel=1e-15)
    assert P[H + r(4), col(4)] == pytest.approx(3 * PI * dx / 2, rel=1e-15)
    assert P[H + r(4), col(5)] == pytest.approx(PI * dx / 2, rel=1e-15)
    assert P[H + r(4), col(6)] == 0.0
    # (B.4) pattern
    assert P[r(4), H + col(0)] == pytest.approx(1 / F2)
    assert P[r(1), H + col(1)] == pytest.approx(dx / 4 / F2)
    assert P[r(4), H + col(1)] == pytest.approx(dx / 2 / F2)
    assert P[r(4), H + col(3)] == pytest.approx(dx / F2)
    assert P[r(4), H + col(4)] == pytest.approx(3 * dx / 4 / F2)
    assert P[r(4), H + col(5)] == pytest.approx(dx / 4 / F2)
    # L496 and the phi-independence of the Bernoulli row of other lines
    assert np.all(P[H + r(4), H + np.arange(M) * n1] == 0.0)
    assert np.all(P[r(4), (l + 1) * n1:(l + 2) * n1] == 0.0)
    # radiation rows
    x1, nr = p["x1"], p["n_rad"]
    for off in (0, H):
        assert P[off + l * n1, off + col(0)] == nr and P[off + l * n1, off + col(1)] == x1
        assert P[off + l * n1 + 1, off + col(1)] == pytest.approx(nr - x1 / dx)
        assert P[off + l * n1 + 1, off + col(2)] == pytest.approx(x1 / dx)
    # (B.6) off-diagonal: target (k=4, l=2) against node (n=7, m=0): weight dx dy / 2 (first y-row)
    xs, ys = x1 + (3 + 0.5) * dx, l * p["dy"]
    xn, ym = x1 + 6 * dx, 0.0
    K3 = 1 / np.hypot(xn - xs, ym - ys) + 1 / np.hypot(xn - xs, ym + ys)
    assert P[H + r(4), H + 0 * n1 + 7] == pytest.approx(-0.5 * dx * p["dy"] * K3, rel=1e-14)


def test_midpoint_coefficients_follow_eq19():
    """(B.2)'s coefficients are the trapezoid recurrence (19) L156 followed by the two-point average L454."""
    N, dx = 8, 0.3
    T = J.midpoint_coefficients(N, dx)
    for c in range(N + 1):
        f1 = 1.0 if c == 0 else 0.0
        fx = np.zeros(N)
        if c > 0:
            fx[c - 1] = 1.0
        f = np.empty(N); f[0] = f1
        for k in range(N - 1):
            f[k + 1] = f[k] + 0.5 * dx * (fx[k] + fx[k + 1])
        assert np.allclose(T[:, c], 0.5 * (f[:-1] + f[1:]), rtol=0, atol=1e-16)


def test_band_truncation_structure(oracle64):
    c = small(N=5, M=6, h=0.5, x1=-1.0)
    p = c.params()
    n1, H = c.N + 1, (c.N + 1) * c.M
    P = J.linear_jacobian(p, oracle64.box_integral)
    assert np.array_equal(J.band_truncate(P, p, 2 * c.M - 1), P)
    Q = J.band_truncate(P, p, 3)
    assert np.array_equal(Q[:H], P[:H]) and np.array_equal(Q[H:, :H], P[H:, :H])   # A, B, C untouched
    for l in range(c.M):
        for m in range(c.M):
            blk = Q[H + l * n1:H + (l + 1) * n1, H + m * n1:H + (m + 1) * n1]
            ref = P[H + l * n1:H + (l + 1) * n1, H + m * n1:H + (m + 1) * n1]
            assert np.array_equal(blk, ref if abs(l - m) <= 1 else np.zeros_like(ref))
    with pytest.raises(ValueError):
        J.band_truncate(P, p, 2)


def test_app_c_block_solve_is_a_solve(oracle64):
    """App. C: the three block steps solve P r = b."""
    c = small(N=7, M=5, h=0.5, x1=-1.5)
    p = c.params()
    P = J.band_truncate(J.linear_jacobian(p, oracle64.box_integral), p, 3)
    rng = np.random.default_rng(7)
    b = rng.standard_normal(P.shape[0])
    r = J.precond_solve_blocks(P, b)
    assert np.abs(P @ r - b).max() <= 1e-11 * np.abs(b).max()
    assert np.allclose(r, np.linalg.solve(P, b), rtol=1e-10, atol=1e-12)


# ----------------------------------------------------------------------------
# GMRES
# ----------------------------------------------------------------------------
def _system(n=60, seed=3, cond_shift=4.0):
    rng = np.random.default_rng(seed)
    A = rng.standard_normal((n, n)) / np.sqrt(n) + cond_shift * np.eye(n)
    Pm = A + 0.3 * rng.standard_normal((n, n)) / np.sqrt(n)
    b = rng.standard_normal(n)
    return A, Pm, b


def test_gmres_full_is_exact_and_monotone():
    A, Pm, b = _system()
    Pinv = np.linalg.inv(Pm)
    d, hist = J.gmres_right(lambda v: A @ v, lambda v: Pinv @ v, b, 1e-13, restart=60, maxit=60)
    assert np.allclose(d, np.linalg.solve(A, b), rtol=1e-10, atol=1e-12)
    assert all(h2 <= h1 * (1 + 1e-12) for h1, h2 in zip(hist, hist[1:]))
    assert len(hist) < 25          # the preconditioner clusters the spectrum
    # the reported history is the true residual
    assert np.linalg.norm(b - A @ d) / np.linalg.norm(b) == pytest.approx(hist[-1], rel=1e-3, abs=1e-14)


def test_gmres_minimises_over_the_krylov_space():
    """After m steps the iterate minimises ||b - A P^-1 z|| over K_m(A P^-1, b) (L213): compare
    with a least-squares solve on the explicit Krylov matrix."""
    A, Pm, b = _system(n=40, seed=5)
    Pinv = np.linalg.inv(Pm)
    B = A @ Pinv
    m = 5
    d, hist = J.gmres_right(lambda v: A @ v, lambda v: Pinv @ v, b, 0.0, restart=m, maxit=m)
    K = np.stack([np.linalg.matrix_power(B, i) @ b for i in range(m)], axis=1)
    y, *_ = np.linalg.lstsq(B @ K, b, rcond=None)
    assert np.linalg.norm(b - B @ K @ y) / np.linalg.norm(b) == pytest.approx(hist[-1], rel=1e-8)
    assert np.allclose(d, Pinv @ (K @ y), rtol=1e-7, atol=1e-10)


def test_gmres_restart_and_library():
    A, Pm, b = _system(n=80, seed=11, cond_shift=2.0)
    ident = lambda v: v
    d, hist = J.gmres_right(lambda v: A @ v, ident, b, 1e-10, restart=10, maxit=400)
    assert hist[-1] <= 1e-10
    x, info = spla.gmres(A, b, rtol=1e-12, restart=80, maxiter=10)
    assert info == 0
    assert np.allclose(d, x, rtol=1e-7, atol=1e-9)
    # maxit is a hard cap on matrix-vector products
    _, h2 = J.gmres_right(lambda v: A @ v, ident, b, 1e-30, restart=7, maxit=23)
    assert len(h2) == 23
    # zero right-hand side
    d0, h0 = J.gmres_right(lambda v: A @ v, ident, np.zeros(80), 1e-10, restart=10, maxit=10)
    assert not d0.any() and h0 == []


# ----------------------------------------------------------------------------
# Newton
# ----------------------------------------------------------------------------
def test_newton_known_root_quadratic_convergence():
    rng = np.random.default_rng(2)
    n = 30
    A = rng.standard_normal((n, n)) / np.sqrt(n) + 3 * np.eye(n)
    ustar = rng.standard_normal(n)
    rhs = A @ ustar + 0.1 * ustar ** 3
    res = lambda u: A @ u + 0.1 * u ** 3 - rhs
    jv = lambda u, v: A @ v + 0.3 * u ** 2 * v
    u, log = J.newton(res, jv, lambda v: v, np.zeros(n), ftol=1e-13, eta=1e-12, restart=30, gmres_maxit=30)
    assert np.abs(u - ustar).max() <= 1e-12
    f = [e["fnorm"] for e in log]
    assert all(e["lambda"] == 1.0 for e in log[:-1])
    assert f[-2] < 1e-3 * f[-3]                    # superlinear tail (quadratic: f_{k+1} ~ f_k^2)


def test_newton_forcing_terms_follow_the_decrease():
    """forcing = 1: the inner tolerance starts at eta_max, then is 0.9 (||E_k||/||E_{k-1}||)^2 with the
    0.9 eta^2 safeguard, clipped to [eta, eta_max]; the root is the same, with fewer Krylov iterations
    than solving every step to eta."""
    rng = np.random.default_rng(4)
    n = 40
    A = rng.standard_normal((n, n)) / np.sqrt(n) + 3 * np.eye(n)
    ustar = rng.standard_normal(n)
    rhs = A @ ustar + 0.1 * ustar ** 3
    res = lambda u: A @ u + 0.1 * u ** 3 - rhs
    jv = lambda u, v: A @ v + 0.3 * u ** 2 * v
    kw = dict(ftol=1e-12, eta=1e-8, restart=40, gmres_maxit=40)
    u0, log0 = J.newton(res, jv, lambda v: v, np.zeros(n), **kw)
    u1, log1 = J.newton(res, jv, lambda v: v, np.zeros(n), forcing=1, eta_max=0.5, **kw)
    assert np.abs(u0 - ustar).max() <= 1e-11 and np.abs(u1 - ustar).max() <= 1e-11
    assert sum(e["gmres_its"] for e in log1) < sum(e["gmres_its"] for e in log0)
    # the tolerances actually used, recomputed from the logged norms
    eta_k, f = 0.5, [e["fnorm"] for e in log1]
    for k, e in enumerate(log1[:-1]):
        assert e["gmres_rel"] <= eta_k                   # the inner solve met the tolerance of its step
        if k + 1 < len(log1):
            t = 0.9 * (f[k + 1] / f[k]) ** 2
            if 0.9 * eta_k ** 2 > 0.1:
                t = max(t, 0.9 * eta_k ** 2)
            eta_k = min(0.5, max(t, 1e-8))
    assert log1[0]["gmres_rel"] > 1e-3                   # first step solved loosely


def test_newton_line_search_damps():
    """arctan: the full Newton step from u0 = 3 overshoots and diverges; the damped iteration (2) converges."""
    res = lambda u: np.arctan(u)
    jv = lambda u, v: v / (1 + u ** 2)
    u, log = J.newton(res, jv, lambda v: v, np.array([3.0]), ftol=1e-12, eta=1e-12, restart=1, gmres_maxit=1)
    assert abs(u[0]) <= 1e-12
    assert log[0]["lambda"] < 1.0
    assert all(b["fnorm"] < a["fnorm"] for a, b in zip(log, log[1:]))   # ||E_{k+1}|| < ||E_k||, L43


def test_jfnk_reaches_the_root_of_dense_newton(oracle64, oracleC):
    """The whole method on a tiny mesh: JFNK (oracle residual, complex-step J v, linear-Jacobian
    preconditioner, flat initial guess L227) reaches the same root as Newton with the explicit
    dense Jacobian and numpy.linalg.solve."""
    c = small(N=13, M=5, h=0.8, x1=-4.0, eps=0.6)
    p = c.params()
    n = c.n
    res = lambda u: oracle64.residual(p, u)
    jv = lambda u, v: oracleC.jv_exact(p, u, v)
    P = J.band_truncate(J.linear_jacobian(p, oracle64.box_integral), p, 3)
    Pinv = np.linalg.inv(P)
    u, log = J.newton(res, jv, lambda v: Pinv @ v, W.flat_state(c), ftol=1e-11, eta=1e-4, restart=30,
                      gmres_maxit=60)
    assert log[-1]["finf"] <= 1e-11 and len(log) <= 9
    assert max(e["gmres_its"] for e in log) <= 20
    # dense Newton
    ud = W.flat_state(c)
    for _ in range(12):
        E = res(ud)
        if np.abs(E).max() <= 1e-12:
            break
        Jd = np.stack([jv(ud, np.eye(n)[j]) for j in range(n)], axis=1)
        ud = ud - np.linalg.solve(Jd, E)
    assert np.abs(res(ud)).max() <= 1e-12
    assert np.abs(u - ud).max() <= 1e-9
    assert np.abs(u - W.flat_state(c)).max() > 1e-2      # the root is not the flat state


# ----------------------------------------------------------------------------
# PW: the ORACLE's residual has the steady wave pattern of linear theory as its root.  Nothing in the
# paper prints a value of E, but the physics fixes what a root of E = 0 looks like: transverse waves of
# wavenumber 1/F^2 on the centre line (lengths scaled by the source depth, L85), i.e. wavelength
# 2 pi F^2, downstream of the source only (radiation condition (24)).  A wrong sign or factor in the
# Bernoulli row (13), in the 2 pi phi term or in the kernels of (12), or radiation rows on the wrong end,
# moves the wavelength or puts the waves upstream.
# ----------------------------------------------------------------------------
def _centreline_waves(oracle64, oracleC, N, M, h, x1, F, eps=0.3):
    import scipy.linalg as sl
    c = W.custom(N, M, h, x1, eps=eps, froude=F)
    p = c.params()
    lu = sl.lu_factor(J.linear_jacobian(p, oracle64.box_integral))
    u, log = J.newton(lambda u: oracle64.residual(p, u), lambda u, v: oracleC.jv_exact(p, u, v),
                      lambda v: sl.lu_solve(lu, v), W.flat_state(c), ftol=1e-10, eta=1e-3, restart=40, gmres_maxit=80)
    assert log[-1]["finf"] <= 1e-10
    zb = u[(N + 1) * M:].reshape(M, N + 1)
    z1, zx = zb[0, 0], zb[0, 1:]
    z = np.concatenate([[z1], z1 + np.cumsum(0.5 * h * (zx[1:] + zx[:-1]))])   # eq. (19) on y = 0
    x = x1 + h * np.arange(N)
    sel = (x > 3.0) & (x < x[-1] - 3.0)
    xs, zs = x[sel], z[sel]
    i = np.where(np.sign(zs[:-1]) != np.sign(zs[1:]))[0]
    xz = xs[i] - zs[i] * (xs[i + 1] - xs[i]) / (zs[i + 1] - zs[i])
    assert len(xz) >= 5
    return 2.0 * float(np.mean(np.diff(xz))), float(np.abs(z[x < -3.0]).max() / np.abs(z[x > 2.0]).max())


def test_oracle_root_is_the_kelvin_wave_pattern(oracle64, oracleC):
    th = 2 * PI * 0.7 ** 2
    lam3, quiet3 = _centreline_waves(oracle64, oracleC, 91, 11, 0.3, -9.0, 0.7)
    lam2, quiet2 = _centreline_waves(oracle64, oracleC, 121, 9, 0.2, -6.0, 0.7)
    assert abs(lam3 - th) <= 0.12 * th and abs(lam2 - th) <= 0.05 * th
    assert abs(lam2 - th) < abs(lam3 - th)                 # converging under refinement
    assert quiet3 <= 0.12 and quiet2 <= 0.12               # waves trail the source
    lam9, _ = _centreline_waves(oracle64, oracleC, 91, 11, 0.3, -9.0, 0.9)
    assert lam9 / lam3 == pytest.approx((0.9 / 0.7) ** 2, rel=0.10)


# ----------------------------------------------------------------------------
# Enlarged (block) GMRES: SURVEY 8(f)2 "block Krylov that actually uses b > 1"
# ----------------------------------------------------------------------------
def _groups(n, t):
    return (np.arange(n) * t) // n


def test_egmres_with_one_piece_is_gmres():
    A, Pm, b = _system(n=50, seed=7)
    Pinv = np.linalg.inv(Pm)
    d1, h1 = J.gmres_right(lambda v: A @ v, lambda v: Pinv @ v, b, 0.0, restart=8, maxit=8)
    d2, h2 = J.egmres_right(lambda Z: Z @ A.T, lambda v: Pinv @ v, b, _groups(50, 1), 1, 0.0, 8)
    assert np.allclose(h1, h2, rtol=1e-9, atol=1e-14)
    assert np.allclose(d1, d2, rtol=1e-9, atol=1e-12)


@pytest.mark.parametrize("t", [2, 4, 8])
def test_egmres_minimises_over_the_block_krylov_space(t):
    """After m block iterations the iterate minimises ||b - A P^-1 z|| over the block Krylov space
    span{(A P^-1)^i T_c b}: compared with a least-squares solve on the explicit block Krylov matrix; the
    space contains K_m(A P^-1, b), so the residual is no larger than plain GMRES's after m products; the
    reported history is the true residual; at m t = n the solve is exact."""
    n = 48
    A, Pm, b = _system(n=n, seed=13, cond_shift=2.0)
    Pinv = np.linalg.inv(Pm)
    Bm = A @ Pinv
    grp = _groups(n, t)
    m = 3
    d, hist = J.egmres_right(lambda Z: Z @ A.T, lambda v: Pinv @ v, b, grp, t, 0.0, m)
    pieces = [np.where(grp == c, b, 0.0) for c in range(t)]
    K = np.stack([np.linalg.matrix_power(Bm, i) @ pc for i in range(m) for pc in pieces], axis=1)
    y, *_ = np.linalg.lstsq(Bm @ K, b, rcond=None)
    best = np.linalg.norm(b - Bm @ K @ y) / np.linalg.norm(b)
    assert hist[-1] == pytest.approx(best, rel=1e-6, abs=1e-13)
    assert np.linalg.norm(b - A @ d) / np.linalg.norm(b) == pytest.approx(hist[-1], rel=1e-6, abs=1e-13)
    assert np.allclose(d, Pinv @ (K @ y), rtol=1e-6, atol=1e-9)
    _, hp = J.gmres_right(lambda v: A @ v, lambda v: Pinv @ v, b, 0.0, restart=m, maxit=m)
    assert hist[-1] <= hp[-1] * (1 + 1e-9)
    assert all(b2 <= b1 * (1 + 1e-12) for b1, b2 in zip(hist, hist[1:]))
    dfull, hfull = J.egmres_right(lambda Z: Z @ A.T, lambda v: Pinv @ v, b, grp, t, 1e-12, n // t)
    assert hfull[-1] <= 1e-12 and np.allclose(dfull, np.linalg.solve(A, b), rtol=1e-8, atol=1e-10)


def test_line_partition_groups_whole_lines():
    p = dict(N=5, M=7)
    g = J.line_partition(p, 3)
    assert g.shape == (2 * 6 * 7,)
    blk = g[:42].reshape(7, 6)
    assert (blk == blk[:, :1]).all() and np.array_equal(g[:42], g[42:])       # a line's phi and zeta unknowns together
    assert np.array_equal(blk[:, 0], [0, 0, 0, 1, 1, 2, 2])
