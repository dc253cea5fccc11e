"""GPU parity at the meshes the PAPER solves on: 361x121 and 721x241 with x_0 = -14 (PAPER.md
L259, L275; F = 0.7, eps = 1) and the Fig. 7 mesh (L315 / L336: F = 1.4, 721x241, dx = dy = 0.3, x_0 = -56, so that
x reaches 160 and y 72: phi ~ x is four times larger than in any BASELINE.json config, the boxes of the closed form I
are four times longer, and the far-field switch of the S2 column sums sees dy = 0.3).

Inputs: the seeded Gaussian-sum state of the shape (workloads.PAPER_MESHES) plus seeded noise on every unknown, so
that the whole domain - not only the patch the Gaussians cover - carries non-trivial slopes.  Checked against the
long-double oracle on >= 1024 sampled integral-equation rows + corners + centre and on ALL O(NM) rows:
  sws_residual on both all-pairs paths, one slot of a finite-difference batch, one analytic sws_jv_apply direction
  (complex-step oracle), all to 1e-10; and a CONVERGED root of the Fig. 7 solve against the oracle's residual.
All tests need a B200."""
import numpy as np
import pytest

import workloads as W

pytestmark = pytest.mark.gpu

TOL = 1e-10  # BASELINE.json: "within 1e-10 relative to ||F||_inf"
SHAPES = ["paper_361x121", "paper_721x241", "paper_fig7_721x241"]


@pytest.fixture(scope="module")
def sws():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("gpu-marked test run without a CUDA device")
    import paper_1403_5044_b200 as m
    m.load_library()
    return m


def dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def noisy_state(cfg):
    rng = np.random.default_rng(cfg.seed + 1000)
    return W.state(cfg) + 2e-3 * rng.standard_normal(cfg.n)


def sample_rows(cfg, count, seed):
    rng = np.random.default_rng(seed)
    T, N, M = cfg.targets, cfg.N, cfg.M
    fixed = [0, N - 2, T - 1, T - (N - 1), (M // 2) * (N - 1) + N // 2,
             (M - 1) * (N - 1) + N // 2,          # last line (t = 0 edge of the box integral), mid x
             N // 2]                              # centre line y = 0
    return np.unique(np.concatenate([rng.integers(0, T, count), fixed])).astype(np.int32)


@pytest.mark.parametrize("path", ["const", "staged"])
@pytest.mark.parametrize("name", SHAPES)
def test_paper_shapes_residual_sampled_rows(sws, oracle80, name, path):
    cfg = W.PAPER_BY_NAME[name]
    u = noisy_state(cfg)
    pick = sample_rows(cfg, 1024, 4321)
    E = oracle80.residual(cfg.params(), u, rows=pick)
    with sws.Context(cfg.params()) as ctx:
        assert ctx.const_plan_info()["active"]                 # the default at these sizes
        if path == "staged":
            ctx.set_const_path(0)
            assert not ctx.const_plan_info()["active"]
        F = ctx.residual(dev(u)).cpu().numpy()
        F2 = ctx.residual(dev(u)).cpu().numpy()
    mask = ~np.isnan(E)
    assert mask.sum() == (cfg.N + 1) * cfg.M + 2 * cfg.M + pick.size
    assert np.isfinite(F).all() and np.array_equal(F, F2)
    half = (cfg.N + 1) * cfg.M
    scale = np.abs(E[mask]).max()
    assert np.abs(F[mask] - E[mask]).max() / scale <= TOL
    # the two halves separately, each against its own norm (E2 is 100x larger than E1 where phi - x = O(1))
    m1, m2 = mask.copy(), mask.copy()
    m1[half:] = False
    m2[:half] = False
    assert np.abs(F[m1] - E[m1]).max() / np.abs(E[m1]).max() <= TOL
    assert np.abs(F[m2] - E[m2]).max() / np.abs(E[m2]).max() <= TOL


@pytest.mark.parametrize("name", SHAPES)
def test_paper_shapes_fd_batch_slot(sws, oracle80, name):
    """One slot of a finite-difference batch (eq. (25)): E(u + sigma v) against the oracle at the same shift."""
    import torch
    cfg = W.PAPER_BY_NAME[name]
    u = noisy_state(cfg)
    V = W.directions(cfg, 2)
    pick = sample_rows(cfg, 1024, 777)
    with sws.Context(cfg.params(), max_batch=2) as ctx:
        JV, Fp, F0 = ctx.jv_batch(dev(u), dev(V), want_fpert=True, want_f0=True)
        torch.cuda.synchronize()
        sig = ctx.last_sigma(2)
        Fp, F0 = Fp.cpu().numpy(), F0.cpu().numpy()
    s_ref = oracle80.sigma(u, V[1])
    assert abs(sig[1] - s_ref) <= 1e-13 * s_ref
    _, Ep = oracle80.jv(cfg.params(), u, V[1], float(sig[1]), rows=pick)
    mask = ~np.isnan(Ep)
    assert np.abs(Fp[1][mask] - Ep[mask]).max() / np.abs(Ep[mask]).max() <= TOL


@pytest.mark.parametrize("name", SHAPES)
def test_paper_shapes_analytic_jv(sws, oracleC, name):
    """sws_linearize + sws_jv_apply (b = 1, the GMRES shape) against the complex-step oracle."""
    cfg = W.PAPER_BY_NAME[name]
    u = noisy_state(cfg)
    v = W.directions(cfg, 1)[0]
    pick = sample_rows(cfg, 256, 99)
    with sws.Context(cfg.params(), max_batch=1) as ctx:
        ctx.linearize(dev(u))
        JV = ctx.jv_apply(dev(v)).cpu().numpy()
    ref = oracleC.jv_exact(cfg.params(), u, v, rows=pick)
    mask = ~np.isnan(ref)
    assert np.abs(JV[mask] - ref[mask]).max() / np.abs(ref[mask]).max() <= TOL


def test_fig7_converged_root_satisfies_the_oracle(sws, oracle80):
    """The Fig. 7 solve (F = 1.4, 721x241, dx = 0.3, x_0 = -56) from the flat guess (L227), as bench.py runs it: the
    root the device Newton-GMRES driver returns is a root of the ORACLE's residual too (sampled integral-equation rows,
    all other rows), to 1e-9 in the max norm (the driver's own stopping tolerance is 1e-9 on the GPU residual)."""
    import torch
    import paper_1403_5044_b200.jfnk as jf
    cfg = W.PAPER_BY_NAME["paper_fig7_721x241"]
    p = cfg.params()
    with sws.Context(p, max_batch=1) as ctx, jf.Preconditioner(p, bandwidth=31, f32_panels=True) as pc, \
            jf.Solver(ctx, pc, 60) as s:
        u0 = torch.from_numpy(W.flat_state(cfg)).cuda()
        us, log, st = s.newton(u0, ftol=1e-9, eta=1e-3, restart=60, gmres_maxit=120, jv_mode=2, forcing=1, eta_max=0.5)
        torch.cuda.synchronize()
        Fg = ctx.residual(us).cpu().numpy()
    assert st["converged"], log
    u_root = us.cpu().numpy()
    # a wave pattern, not the flat state: the surface moved
    half = (cfg.N + 1) * cfg.M
    assert np.abs(u_root[half:]).max() > 1e-3
    pick = sample_rows(cfg, 1024, 2024)
    E = oracle80.residual(p, u_root, rows=pick)
    mask = ~np.isnan(E)
    assert np.abs(Fg).max() <= 1e-9
    assert np.abs(E[mask]).max() <= 1e-9, np.abs(E[mask]).max()
    assert np.abs(E[mask] - Fg[mask]).max() <= 1e-10 * max(1.0, np.abs(u_root).max())
