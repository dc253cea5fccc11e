"""GPU parity of libsws_jfnk (preconditioner, GMRES, Newton) against
oracle/jfnk.py, through the C-ABI binding.  All tests here need a B200.

Tolerances.  Assembled blocks: entry by entry, 1e-13 of the largest entry (same formulas, FP64,
different rounding order).  P^-1 v: the Schur complement has condition number ~1e6 (its diagonal
blocks carry the double-integration operator C A^-1 B), and the library applies explicit inverses
of the diagonal blocks, so two correct solvers differ by ~cond * eps ~ 1e-10 relative; bar 1e-8.
GMRES / Newton: iteration histories agree while they are far above that floor (1e-6 relative),
converged roots agree to 1e-8 (the Newton stopping tolerance is 1e-10 on ||E||_inf).
"""
import numpy as np
import pytest

import oracle.jfnk as OJ
import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def mods():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("gpu-marked test run without a CUDA device")
    import paper_1403_5044_b200 as sws
    import paper_1403_5044_b200.jfnk as jf
    sws.load_library()
    jf.load_jfnk()   # fails loudly if libsws_jfnk.so is missing
    return sws, jf


def dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


SHAPES = [dict(N=9, M=5, h=0.5, x1=-2.0), dict(N=6, M=7, h=0.3, x1=-1.1), dict(N=14, M=4, h=0.25, x1=-3.0, y1=0.5)]


@pytest.mark.parametrize("shape", SHAPES)
@pytest.mark.parametrize("bw", [1, 3, 0])
def test_assembled_blocks(mods, oracle64, shape, bw):
    """D blocks ((B.6) L498-501, rows E5/E6 L466-468) and Schur blocks D - C A^-1 B, every block in the band."""
    sws, jf = mods
    c = W.custom(**shape)
    p = c.params()
    n1, H, M = c.N + 1, (c.N + 1) * c.M, c.M
    P = OJ.linear_jacobian(p, oracle64.box_integral)
    A, B, C_, D = P[:H, :H], P[:H, H:], P[H:, :H], P[H:, H:]
    S = D - C_ @ np.linalg.solve(A, B)
    with jf.Preconditioner(p, bandwidth=bw, factorise=False) as pc:
        hb = (pc.bandwidth - 1) // 2
        assert pc.bandwidth == (bw if bw else 2 * M - 1)
        for l in range(M):
            for m in range(max(0, l - hb), min(M, l + hb + 1)):
                ref = D[l * n1:(l + 1) * n1, m * n1:(m + 1) * n1]
                got = pc.block(0, l, m)
                assert np.abs(got - ref).max() <= 1e-13 * np.abs(D).max(), (l, m)
                refS = S[l * n1:(l + 1) * n1, m * n1:(m + 1) * n1]
                gotS = pc.block(1, l, m)
                assert np.abs(gotS - refS).max() <= 1e-12 * np.abs(S).max(), (l, m)


def _pinv_case(mods, oracle64, c, bw, seed=0, nvec=3, tol=1e-8):
    sws, jf = mods
    p = c.params()
    P = OJ.band_truncate(OJ.linear_jacobian(p, oracle64.box_integral), p, bw if bw else 2 * c.M - 1)
    rng = np.random.default_rng(seed)
    with jf.Preconditioner(p, bandwidth=bw) as pc:
        for _ in range(nvec):
            v = rng.standard_normal(c.n)
            ref = np.linalg.solve(P, v)
            got = pc.apply(dev(v)).cpu().numpy()
            assert np.abs(got - ref).max() <= tol * np.abs(ref).max()
            # and it is a solve of the banded P itself
            assert np.abs(P @ got - v).max() <= 1e-7 * np.abs(v).max()
        # in place, deterministic
        vd = dev(v)
        r1 = pc.apply(vd).cpu().numpy()
        pc.apply(vd, out=vd)
        assert np.array_equal(vd.cpu().numpy(), r1)


@pytest.mark.parametrize("shape", SHAPES)
@pytest.mark.parametrize("bw", [1, 3, 5, 0])
def test_precond_apply_small(mods, oracle64, shape, bw):
    _pinv_case(mods, oracle64, W.custom(**shape), bw)


@pytest.mark.parametrize("bw", [1, 7, 0])
def test_precond_apply_cfg2(mods, oracle64, bw):
    _pinv_case(mods, oracle64, W.CONFIGS[1], bw, nvec=2)


def test_precond_matches_app_c_steps(mods, oracle64):
    """The oracle's literal App. C block steps and the library agree (cfg1, b = 5)."""
    sws, jf = mods
    c = W.CONFIGS[0]
    p = c.params()
    P = OJ.band_truncate(OJ.linear_jacobian(p, oracle64.box_integral), p, 5)
    v = np.random.default_rng(3).standard_normal(c.n)
    ref = OJ.precond_solve_blocks(P, v)
    with jf.Preconditioner(p, bandwidth=5) as pc:
        got = pc.apply(dev(v)).cpu().numpy()
    assert np.abs(got - ref).max() <= 1e-8 * np.abs(ref).max()


def test_error_codes(mods):
    sws, jf = mods
    c = W.CONFIGS[0]
    with pytest.raises(sws.SwsError):
        jf.Preconditioner(c.params(), bandwidth=4)
    with sws.Context(c.params(), max_batch=0) as ctx:
        with pytest.raises(sws.SwsError):
            jf.Solver(ctx, None)
    with jf.Preconditioner(c.params(), bandwidth=3, factorise=False) as pc:
        import torch
        with pytest.raises(sws.SwsError):
            pc.apply(torch.zeros(c.n, dtype=torch.float64, device="cuda"))
        with pytest.raises(sws.SwsError):
            pc.block(0, 0, 5)     # outside the band


# ---------------------------------------------------------------------------------------
def _oracle_ops(oracle64, oracleC, p, P):
    import scipy.linalg as sl
    lu = sl.lu_factor(P)
    return (lambda u: oracle64.residual(p, u), lambda u, v: oracleC.jv_exact(p, u, v), lambda v: sl.lu_solve(lu, v))


@pytest.mark.parametrize("bw,restart", [(0, 30), (3, 30), (3, 4)])
def test_gmres_parity_cfg1(mods, oracle64, oracleC, bw, restart):
    """J(u) d = -E(u) at the seeded nonlinear state of cfg1: residual history and solution."""
    sws, jf = mods
    c = W.CONFIGS[0]
    p = c.params()
    u = W.state(c)
    P = OJ.band_truncate(OJ.linear_jacobian(p, oracle64.box_integral), p, bw if bw else 2 * c.M - 1)
    res, jv, pinv = _oracle_ops(oracle64, oracleC, p, P)
    rhs = -res(u)
    d_ref, h_ref = OJ.gmres_right(lambda v: jv(u, v), pinv, rhs, 1e-9, restart, 60)
    with sws.Context(p, max_batch=1) as ctx, jf.Preconditioner(p, bandwidth=bw) as pc, jf.Solver(ctx, pc, 30) as s:
        d, st, hist = s.gmres(dev(u), dev(rhs), tol=1e-9, restart=restart, maxit=60)
        d = d.cpu().numpy()
    assert st["converged"] and st["its"] == len(h_ref)
    h_ref = np.array(h_ref)
    big = h_ref > 1e-7
    assert np.allclose(hist[big], h_ref[big], rtol=1e-5)
    assert np.abs(d - d_ref).max() <= 1e-7 * np.abs(d_ref).max()
    # it solves the system: the oracle's J applied to the library's d
    assert np.linalg.norm(jv(u, d) - rhs) <= 5e-9 * np.linalg.norm(rhs)


def test_gmres_unpreconditioned_and_fd(mods, oracle64, oracleC):
    """No preconditioner (pc = NULL) and the finite-difference J v of eq. (25) (jv_mode 1)."""
    sws, jf = mods
    c = W.CONFIGS[0]
    p = c.params()
    u = W.state(c)
    rhs = -oracle64.residual(p, u)
    jv = lambda v: oracleC.jv_exact(p, u, v)
    d_ref, h_ref = OJ.gmres_right(jv, lambda v: v, rhs, 1e-30, 20, 20)
    with sws.Context(p, max_batch=1) as ctx, jf.Solver(ctx, None, 20) as s:
        d, st, hist = s.gmres(dev(u), dev(rhs), tol=1e-30, restart=20, maxit=20)
        assert st["its"] == 20 and not st["converged"]
        assert np.allclose(hist, np.array(h_ref), rtol=1e-5)
        d2, st2, hist2 = s.gmres(dev(u), dev(rhs), tol=1e-30, restart=20, maxit=20, jv_mode=1)
        assert np.allclose(hist2, np.array(h_ref), rtol=1e-3)     # first-order difference quotient
        # jv_mode 2: the same quotient from ONE residual evaluation per product (base E(u) held by the driver)
        d3, st3, hist3 = s.gmres(dev(u), dev(rhs), tol=1e-30, restart=20, maxit=20, jv_mode=2)
        assert st3["its"] == 20
        assert np.allclose(hist3, hist2, rtol=1e-5)
        assert np.abs((d3 - d2).cpu().numpy()).max() <= 1e-5 * np.abs(d_ref).max()
        # zero right-hand side
        import torch
        d0, st0, _ = s.gmres(dev(u), torch.zeros_like(dev(u)), tol=1e-8, maxit=5)
        assert st0["converged"] and st0["its"] == 0 and not d0.cpu().numpy().any()
    assert np.abs(d.cpu().numpy() - d_ref).max() <= 1e-6 * np.abs(d_ref).max()


@pytest.mark.parametrize("bw", [0, 3])
def test_newton_parity_cfg1_mesh(mods, oracle64, oracleC, bw):
    """The whole JFNK solve on the 31x11 mesh from the flat guess (L227), eps = 1, F = 0.7: same
    Newton history and the same root as the oracle's driver."""
    sws, jf = mods
    c = W.custom(31, 11, 0.8, -8.0, eps=1.0)
    p = c.params()
    P = OJ.band_truncate(OJ.linear_jacobian(p, oracle64.box_integral), p, bw if bw else 2 * c.M - 1)
    res, jv, pinv = _oracle_ops(oracle64, oracleC, p, P)
    u0 = W.flat_state(c)
    kw = dict(ftol=1e-10, eta=1e-3, restart=30, gmres_maxit=60)
    u_ref, log_ref = OJ.newton(res, jv, pinv, u0, **kw)
    with sws.Context(p, max_batch=1) as ctx, jf.Preconditioner(p, bandwidth=bw) as pc, jf.Solver(ctx, pc, 30) as s:
        u, log, st = s.newton(dev(u0), **kw)
        u = u.cpu().numpy()
    assert st["converged"] and log_ref[-1]["finf"] <= 1e-10
    assert len(log) == len(log_ref)
    for a, b in zip(log, log_ref):
        assert a["gmres_its"] == b["gmres_its"] and a["lambda"] == b["lambda"]
        if b["fnorm"] > 1e-6:
            assert a["fnorm"] == pytest.approx(b["fnorm"], rel=1e-6)
    assert np.abs(u - u_ref).max() <= 1e-8
    assert np.abs(oracle64.residual(p, u)).max() <= 2e-10     # a root for the oracle too
    assert st["jv_products"] == sum(e["gmres_its"] for e in log)
    assert st["residual_evals"] == 1 + st["steps"]


def test_newton_forcing_parity(mods, oracle64, oracleC):
    """forcing = 1 (Eisenstat-Walker choice 2): same Newton history as the oracle's driver."""
    sws, jf = mods
    c = W.custom(31, 11, 0.8, -8.0, eps=1.0)
    p = c.params()
    P = OJ.band_truncate(OJ.linear_jacobian(p, oracle64.box_integral), p, 3)
    res, jv, pinv = _oracle_ops(oracle64, oracleC, p, P)
    u0 = W.flat_state(c)
    kw = dict(ftol=1e-10, eta=1e-4, restart=30, gmres_maxit=60, forcing=1, eta_max=0.5)
    u_ref, log_ref = OJ.newton(res, jv, pinv, u0, **kw)
    with sws.Context(p, max_batch=1) as ctx, jf.Preconditioner(p, bandwidth=3) as pc, jf.Solver(ctx, pc, 30) as s:
        u, log, st = s.newton(dev(u0), **kw)
        u_c, log_c, _ = s.newton(dev(u0), ftol=1e-10, eta=1e-4, restart=30, gmres_maxit=60)
        with pytest.raises(Exception):
            s.newton(dev(u0), ftol=1e-10, eta=0.6, forcing=1, eta_max=0.5)
    assert st["converged"] and len(log) == len(log_ref)
    for a, b in zip(log, log_ref):
        assert a["gmres_its"] == b["gmres_its"] and a["lambda"] == b["lambda"]
    assert np.abs(u.cpu().numpy() - u_ref).max() <= 1e-8
    assert sum(e["gmres_its"] for e in log) < sum(e["gmres_its"] for e in log_c)


def test_continuation_in_epsilon(mods, oracle64):
    """The bootstrapping process of L229 on the 45 x 13 mesh of Fig. 2 (L247): eps = 0.5 -> 1.0 -> 1.5, each
    from the previous solution; the eps = 1 stage is the root Newton finds from the flat guess; the final
    state is a root of the ORACLE's residual at eps = 1.5; sws_set_eps changes nothing but the source term."""
    sws, jf = mods
    c = W.custom(45, 13, 0.4, -9.0, eps=1.0)
    p = c.params()
    u0 = dev(W.flat_state(c))
    kw = dict(ftol=1e-10, eta=1e-3, restart=40, gmres_maxit=80)
    with sws.Context(p, max_batch=1) as ctx, jf.Preconditioner(p, bandwidth=5) as pc, jf.Solver(ctx, pc, 40) as s:
        u_direct, _, st_d = s.newton(u0, **kw)
        assert st_d["converged"]
        u1, stats1, n1 = s.continuation(u0, [0.5, 1.0], **kw)
        assert n1 == 2 and all(e["converged"] for e in stats1)
        assert np.abs((u1 - u_direct).cpu().numpy()).max() <= 1e-8
        u2, stats2, n2 = s.continuation(u1, [1.25, 1.5], **kw)
        assert n2 == 2
        # warm starts need fewer Newton steps than the flat guess needed
        assert stats2[0]["steps"] <= st_d["steps"]
        p15 = dict(p, eps=1.5)
        assert np.abs(oracle64.residual(p15, u2.cpu().numpy())).max() <= 1e-9
        # the context now evaluates E at eps = 1.5
        F = ctx.residual(u2).cpu().numpy()
        assert np.abs(F).max() <= 1e-9
        ctx.set_eps(1.0)
        assert np.abs(ctx.residual(u_direct).cpu().numpy()).max() <= 1e-9
        # a stage that cannot converge (one Newton step allowed) hands back the last converged solution
        u3, stats3, n3 = s.continuation(u_direct, [1.2, 1.4], max_newton=1, **kw)
        assert n3 == 0 and len(stats3) == 1 and not stats3[0]["converged"]
        assert np.array_equal(u3.cpu().numpy(), u_direct.cpu().numpy())


def test_newton_paper_mesh_91x31(mods, oracle64):
    """The paper's 'contemporary' mesh (91 x 31, dx = dy = 0.3, x0 = -9, eps = 1, F = 0.7; L259):
    converges from the flat guess with the block-banded preconditioner; the root satisfies the
    ORACLE's residual; the finite-difference Jacobian action of eq. (25) reaches the same root."""
    sws, jf = mods
    c = W.custom(91, 31, 0.3, -9.0, eps=1.0)
    p = c.params()
    u0 = dev(W.flat_state(c))
    with sws.Context(p, max_batch=1) as ctx, jf.Preconditioner(p, bandwidth=7) as pc, jf.Solver(ctx, pc, 40) as s:
        u, log, st = s.newton(u0, ftol=1e-10, eta=1e-3, restart=40, gmres_maxit=80)
        assert st["converged"] and st["steps"] <= 8
        assert max(e["gmres_its"] for e in log) <= 30
        un = u.cpu().numpy()
        assert np.abs(oracle64.residual(p, un)).max() <= 1e-9
        u2, log2, st2 = s.newton(u0, ftol=1e-8, eta=1e-3, restart=40, gmres_maxit=80, jv_mode=1)
        assert st2["converged"]
        assert np.abs(u2.cpu().numpy() - un).max() <= 1e-6
        u4, log4, st4 = s.newton(u0, ftol=1e-8, eta=1e-3, restart=40, gmres_maxit=80, jv_mode=2)
        assert st4["converged"]
        assert np.abs(u4.cpu().numpy() - un).max() <= 1e-6
        # one residual per product + one per Newton step (+ the initial one)
        assert st4["residual_evals"] == 1 + st4["steps"] + st4["jv_products"]
        # deterministic
        u3, _, _ = s.newton(u0, ftol=1e-10, eta=1e-3, restart=40, gmres_maxit=80)
        assert np.array_equal(u3.cpu().numpy(), un)
    zeta_x = un[c.n // 2:].reshape(c.M, c.N + 1)[:, 1:]
    assert np.abs(zeta_x).max() > 0.05      # a real wave pattern, not the flat state


def _centreline(u, c):
    """zeta on the line y = y_1 from the unknowns (eq. (18) layout, trapezoid rule (19))."""
    half = (c.N + 1) * c.M
    zb = u[half:].reshape(c.M, c.N + 1)
    z1, zx = zb[0, 0], zb[0, 1:]
    return np.concatenate([[z1], z1 + np.cumsum(0.5 * c.h * (zx[1:] + zx[:-1]))])


def _wavelength(x, z, lo, hi):
    sel = (x > lo) & (x < hi)
    xs, zs = x[sel], z[sel]
    i = np.where(np.sign(zs[:-1]) != np.sign(zs[1:]))[0]
    xz = xs[i] - zs[i] * (xs[i + 1] - xs[i]) / (zs[i + 1] - zs[i])
    assert len(xz) >= 8
    return 2.0 * float(np.mean(np.diff(xz)))


def test_wave_pattern_physics(mods):
    """A pin of the whole method on something neither program defines: the converged free surface carries
    the steady transverse waves of linear theory.  Their wavenumber on the centre line is 1/F^2 in the
    paper's scaling (lengths by the source depth, L85), i.e. wavelength 2 pi F^2, approached at O(h^2);
    they trail the source (radiation condition (24): nothing upstream); and the wavelength scales as F^2."""
    sws, jf = mods
    lam, quiet = {}, {}
    for key, (N, M, h, x1, F, bw) in {"h0.3": (181, 61, 0.3, -14.0, 0.7, 15), "h0.2": (241, 41, 0.2, -10.0, 0.7, 21),
                                      "F0.9": (181, 61, 0.3, -14.0, 0.9, 15)}.items():
        c = W.custom(N, M, h, x1, eps=0.3, froude=F)
        p = c.params()
        with sws.Context(p, max_batch=1) as ctx, jf.Preconditioner(p, bandwidth=bw) as pc, jf.Solver(ctx, pc, 60) as s:
            u, log, st = s.newton(dev(W.flat_state(c)), ftol=1e-10, eta=1e-3, restart=60, gmres_maxit=120, jv_mode=2)
        assert st["converged"]
        x = x1 + h * np.arange(N)
        z = _centreline(u.cpu().numpy(), c)
        lam[key] = _wavelength(x, z, 4.0, x[-1] - 4.0)
        quiet[key] = np.abs(z[x < -4.0]).max() / np.abs(z[x > 2.0]).max()
    th = 2 * np.pi * 0.7 ** 2
    e3, e2 = lam["h0.3"] - th, lam["h0.2"] - th
    assert abs(e3) <= 0.10 * th and abs(e2) <= 0.05 * th
    assert 1.6 <= e3 / e2 <= 3.2                              # (0.3 / 0.2)^2 = 2.25
    assert lam["F0.9"] / lam["h0.3"] == pytest.approx((0.9 / 0.7) ** 2, rel=0.08)
    assert max(quiet.values()) <= 0.1


def test_solve_command_line(mods, oracle64, tmp_path):
    """python -m paper_1403_5044_b200.solve on the 45 x 13 mesh of Fig. 2 (L247), eps passed through 0.5 -> 1: the
    file it writes holds a root of the ORACLE's residual and the surface rebuilt by eq. (19)."""
    import paper_1403_5044_b200.solve as cli
    out = tmp_path / "surface.npz"
    rc = cli.main(["--N", "45", "--M", "13", "--h", "0.4", "--x1", "-9", "--eps", "1.0", "--continuation", "0.5",
                   "--bandwidth", "5", "--forcing", "--ftol", "1e-10", "--out", str(out)])
    assert rc == 0
    z = np.load(out)
    c = W.custom(45, 13, 0.4, -9.0, eps=1.0)
    assert z["u"].shape == (c.n,) and z["zeta"].shape == (13, 45) and z["phi"].shape == (13, 45)
    assert np.abs(oracle64.residual(c.params(), z["u"])).max() <= 1e-9
    half = (c.N + 1) * c.M
    zb = z["u"][half:].reshape(c.M, c.N + 1)
    assert np.array_equal(z["zeta"][:, 0], zb[:, 0])                    # zeta_1 is the first unknown of each line
    assert np.allclose(np.diff(z["zeta"], axis=1), 0.5 * 0.4 * (zb[:, 2:] + zb[:, 1:-1]), atol=1e-15)
    assert np.abs(z["zeta"]).max() > 0.02


# ---------------------------------------------------------------------------------------
# Enlarged (block) GMRES: SURVEY.md 8(f)2 "block Krylov that actually uses b > 1"
def test_precond_apply_multi_equals_single(mods, oracle64):
    """One sweep over the factor panels for t vectors (tiles of 16/8/4/2/1) = t single-vector applies; the
    single-vector path still works after the internal vectors were regrown."""
    import torch
    sws, jf = mods
    c = W.CONFIGS[1]
    p = c.params()
    rng = np.random.default_rng(12)
    with jf.Preconditioner(p, bandwidth=7) as pc:
        v0 = dev(rng.standard_normal(c.n))
        r0 = pc.apply(v0).cpu().numpy()
        for t in (2, 7, 16):
            V = dev(rng.standard_normal((t, c.n)))
            R = pc.apply_multi(V).cpu().numpy()
            for q in range(t):
                ref = pc.apply(V[q].contiguous()).cpu().numpy()
                assert np.abs(R[q] - ref).max() <= 1e-11 * np.abs(ref).max(), (t, q)
        assert np.abs(pc.apply(v0).cpu().numpy() - r0).max() <= 1e-12 * np.abs(r0).max()
        with pytest.raises(sws.SwsError):
            pc.apply_multi(dev(rng.standard_normal((17, c.n))))


@pytest.mark.parametrize("t,jv_mode", [(4, 0), (2, 0), (4, 1)])
def test_egmres_parity_cfg1(mods, oracle64, oracleC, t, jv_mode):
    """Enlarged GMRES with t pieces at the seeded nonlinear state of cfg1, block-banded preconditioner: the
    residual after every block iteration and the iterate against oracle/jfnk.py's plain block Arnoldi (dense
    oracle Jacobian action, dense oracle preconditioner).  The iterate is the unique minimiser over the block
    Krylov space, so the two bases (modified vs twice-classical Gram-Schmidt) do not matter."""
    sws, jf = mods
    c = W.CONFIGS[0]
    p = c.params()
    u = W.state(c)
    P = OJ.band_truncate(OJ.linear_jacobian(p, oracle64.box_integral), p, 3)
    res, jv, pinv = _oracle_ops(oracle64, oracleC, p, P)
    rhs = -res(u)
    grp = OJ.line_partition(p, t)
    blocks = 5
    d_ref, h_ref = OJ.egmres_right(lambda Z: np.stack([jv(u, z) for z in Z]), pinv, rhs, grp, t, 0.0, blocks)
    with sws.Context(p, max_batch=t) as ctx, jf.Preconditioner(p, bandwidth=3) as pc, jf.Solver(ctx, pc, 160) as s:
        d, st, hist = s.gmres(dev(u), dev(rhs), tol=0.0, restart=blocks * t, maxit=blocks * t, jv_mode=jv_mode, block=t)
        d = d.cpu().numpy()
        # the same solve to convergence, and plain GMRES beside it
        tol = 1e-9 if jv_mode == 0 else 1e-6
        d2, st2, hist2 = s.gmres(dev(u), dev(rhs), tol=tol, restart=160, maxit=400, jv_mode=jv_mode, block=t)
        d1, st1, hist1 = s.gmres(dev(u), dev(rhs), tol=tol, restart=160, maxit=400, jv_mode=jv_mode)
    assert st["its"] == blocks * t and len(hist) == blocks
    h_ref = np.array(h_ref)
    rtol = 1e-5 if jv_mode == 0 else 2e-3           # jv_mode 1: first-order difference quotients
    big = h_ref > 1e-7
    assert np.allclose(hist[big], h_ref[big], rtol=rtol)
    assert np.abs(d - d_ref).max() <= (1e-6 if jv_mode == 0 else 1e-3) * np.abs(d_ref).max()
    assert st2["converged"] and st1["converged"]
    assert len(hist2) <= len(hist1)                 # block iterations never exceed plain iterations (nested spaces)
    if jv_mode == 0:
        assert np.linalg.norm(jv(u, d2.cpu().numpy()) - rhs) <= 5e-9 * np.linalg.norm(rhs)
        assert np.abs((d2 - d1).cpu().numpy()).max() <= 1e-6 * np.abs(d_ref).max()


def test_newton_with_enlarged_gmres_reaches_the_same_root(mods, oracle64):
    """The JFNK solve on the 45x13 paper mesh (L247) with enlarged GMRES (t = 4) as the inner solver: same root
    as with plain GMRES, and it is a root of the oracle's residual."""
    sws, jf = mods
    c = W.PAPER_BY_NAME["paper_45x13"]
    p = c.params()
    u0 = dev(W.flat_state(c))
    kw = dict(ftol=1e-10, eta=1e-3, restart=48, gmres_maxit=96)
    with sws.Context(p, max_batch=4) as ctx, jf.Preconditioner(p, bandwidth=5) as pc, jf.Solver(ctx, pc, 60) as s:
        u1, log1, st1 = s.newton(u0, **kw)
        u4, log4, st4 = s.newton(u0, block=4, **kw)
    assert st1["converged"] and st4["converged"]
    assert float((u1 - u4).abs().max()) <= 1e-8
    assert np.abs(oracle64.residual(p, u4.cpu().numpy())).max() <= 1e-9
    assert st4["jv_products"] % 4 == 0


def test_f32_panels_precondition_as_well(mods, oracle64):
    """sws_precond_create flags bit 1: factor panels stored in FP32 (half the bytes per apply).  P^-1 v moves by
    ~1e-7 x conditioning - far from a direct solve, irrelevant for a preconditioner: the Newton-GMRES histories on
    the 45x13 and 91x31 paper meshes are the FP64-panel histories, iteration for iteration, same root."""
    sws, jf = mods
    rng = np.random.default_rng(5)
    for name, bw in (("paper_45x13", 5), ("paper_91x31", 15)):
        c = W.PAPER_BY_NAME[name]
        p = c.params()
        u0 = dev(W.flat_state(c))
        kw = dict(ftol=1e-10, eta=1e-3, restart=40, gmres_maxit=120)
        V = dev(rng.standard_normal((3, c.n)))
        with sws.Context(p, max_batch=1) as ctx, jf.Preconditioner(p, bandwidth=bw) as p64, \
                jf.Preconditioner(p, bandwidth=bw, f32_panels=True) as p32:
            assert p32.bytes < 0.62 * p64.bytes
            r64, r32 = p64.apply(V[0].contiguous()), p32.apply(V[0].contiguous())
            err = float((r64 - r32).abs().max() / r64.abs().max())
            assert 0.0 < err <= 1e-3, err
            m32 = p32.apply_multi(V)
            assert float((m32[0] - r32).abs().max()) <= 1e-11 * float(r32.abs().max())
            with jf.Solver(ctx, p64, 40) as s64:
                u64, log64, st64 = s64.newton(u0, **kw)
            with jf.Solver(ctx, p32, 40) as s32:
                u32, log32, st32 = s32.newton(u0, **kw)
        assert st64["converged"] and st32["converged"]
        assert [e["gmres_its"] for e in log32] == [e["gmres_its"] for e in log64]
        assert float((u64 - u32).abs().max()) <= 1e-8
