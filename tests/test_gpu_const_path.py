"""GPU parity and invariants of the uniform-operand ("constant-bank") form of the all-pairs quadrature
(csrc/sws_allpairs_const.cuh, sws_set_const_path): same pair arithmetic as the staged kernel, source records taken
from a 64 KB constant bank as uniform-register operands, one launch per slab of columns, two banks / two streams.
Large meshes take this path by default (tests/test_gpu_parity.py covers cfg4 / cfg5 on it); here it is FORCED on
small meshes so that every entry can be compared with the long-double oracle.  All tests need a B200."""
import numpy as np
import pytest

import workloads as W

pytestmark = pytest.mark.gpu

TOL = 1e-10  # BASELINE.json: "within 1e-10 relative to ||F||_inf"


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


def relerr(F, E):
    return float(np.abs(F - E).max() / np.abs(E).max())


@pytest.mark.parametrize("i", [0, 1, 2])
def test_const_path_full_parity(sws, oracle80, i):
    """cfg 1-3 on the constant-bank path: every entry of F against the long-double oracle; it differs from the
    staged kernel in summation order only; repeated calls are bitwise identical."""
    cfg = W.CONFIGS[i]
    u = W.state(cfg)
    E = oracle80.residual(cfg.params(), u)
    with sws.Context(cfg.params()) as ctx:
        assert not ctx.const_plan_info()["active"]      # small mesh: staged kernel by default
        F_staged = ctx.residual(dev(u)).cpu().numpy()
        ctx.set_const_path(1)
        info = ctx.const_plan_info()
        assert info["active"] and info["cols_per_slab"] == 16 and info["slabs"] == -(-cfg.N // 16)
        F = ctx.residual(dev(u)).cpu().numpy()
        assert ctx.last_launch_count == 1 + info["slabs"] + 1    # fused fields + one per slab + finish
        F_again = ctx.residual(dev(u)).cpu().numpy()
    assert np.isfinite(F).all()
    assert relerr(F, E) <= TOL
    assert relerr(F, F_staged) <= 1e-13
    assert np.array_equal(F, F_again)


SHAPES = [
    dict(N=3, M=4, h=0.5, x1=-1.0),                      # minimum sizes: one slab, one bank
    dict(N=17, M=9, h=0.45, x1=-3.0, seed=7),            # two slabs, the second of one column
    dict(N=37, M=9, h=0.45, x1=-5.0, seed=7),            # three slabs: bank 0 accumulates twice
    dict(N=131, M=7, h=0.2, x1=-6.0, seed=8),            # 910 targets: ragged last tile; 9 slabs
    dict(N=9, M=479, h=0.05, x1=-0.2, seed=9),           # longest column that fits four at a time (odd M)
    dict(N=44, M=12, h=0.4, x1=-3.0, y1=0.8, seed=11),   # y1 != 0: two boxes in I, two intervals in the far field
]


@pytest.mark.parametrize("kw", SHAPES, ids=lambda k: f"{k['N']}x{k['M']}")
@pytest.mark.parametrize("dy_scheme", [0, 1])
def test_const_path_shapes(sws, oracle80, kw, dy_scheme):
    cfg = W.custom(eps=0.3, amp=0.05, **kw)
    u = W.state(cfg) + 1e-3 * np.random.default_rng(3).standard_normal(cfg.n)
    E = oracle80.residual(cfg.params(dy_scheme), u)
    with sws.Context(cfg.params(dy_scheme)) as ctx:
        ctx.set_const_path(1)
        F = ctx.residual(dev(u)).cpu().numpy()
    assert relerr(F, E) <= TOL


@pytest.mark.parametrize("seed", range(6))
def test_const_path_random_shapes(sws, oracle80, seed):
    """seeded random meshes (dx != dy, y1 = 0 or not, either y-derivative scheme)"""
    rng = np.random.default_rng(500 + seed)
    N, M = int(rng.integers(3, 121)), int(rng.integers(4, 201))
    while N * M > 12000:
        M = max(4, M // 2)
    h = float(rng.uniform(0.05, 0.6))
    cfg = W.custom(N, M, h, float(rng.uniform(-6.0, -0.5)), y1=(0.0 if seed % 2 == 0 else float(rng.uniform(0.1, 1.0))),
                   eps=float(rng.uniform(0.0, 1.0)), froude=float(rng.uniform(0.5, 1.2)), amp=0.05, seed=600 + seed)
    p = cfg.params(seed % 2)
    p["dy"] = h * float(rng.uniform(0.5, 2.0))
    u = W.state(cfg) + 1e-3 * rng.standard_normal(cfg.n)
    E = oracle80.residual(p, u)
    with sws.Context(p) as ctx:
        ctx.set_const_path(1)
        F = ctx.residual(dev(u)).cpu().numpy()
    assert np.isfinite(F).all() and relerr(F, E) <= TOL, (N, M, p)


def test_const_path_batch_is_a_loop_of_single_evaluations(sws, oracle80):
    """sws_jv_batch on the constant-bank path (cfg3, b = 5): F0 is bitwise sws_residual(u), slot b is bitwise
    sws_residual(fma(sigma_b, v_b, u)), the perturbed residuals match the oracle at the library's shifts, the
    host-buffer calls give the device-buffer results."""
    import torch
    from fractions import Fraction
    cfg = W.CONFIGS[2]
    p, u, V = cfg.params(), W.state(cfg), W.directions(cfg, 5)
    with sws.Context(p, max_batch=5) as ctx:
        ctx.set_const_path(1)
        ud = dev(u)
        JV, Fp, F0 = ctx.jv_batch(ud, dev(V), want_fpert=True, want_f0=True)
        torch.cuda.synchronize()
        sig = ctx.last_sigma(5)
        F = ctx.residual(ud).cpu().numpy()
        JV, Fp, F0 = JV.cpu().numpy(), Fp.cpu().numpy(), F0.cpu().numpy()
        sg = Fraction(float(sig[3]))
        ub = np.array([float(sg * Fraction(float(vv)) + Fraction(float(uu))) for uu, vv in zip(u, V[3])])
        F_bit = ctx.residual(dev(ub)).cpu().numpy()
        Fh = ctx.residual_host(u)
        JVh, Fph, F0h = ctx.jv_batch_host(u, V)
    assert np.array_equal(F0, F) and np.array_equal(Fp[3], F_bit)
    assert np.array_equal(Fh, F) and np.array_equal(JVh, JV) and np.array_equal(Fph, Fp) and np.array_equal(F0h, F0)
    E0 = oracle80.residual(p, u)
    scale = np.abs(E0).max()
    assert np.abs(F - E0).max() / scale <= TOL
    for k in (0, 4):
        _, Ep = oracle80.jv(p, u, V[k], float(sig[k]))
        assert np.abs(Fp[k] - Ep).max() / scale <= TOL
        assert np.array_equal(JV[k], (Fp[k] - F0) / sig[k])


def test_const_path_two_contexts_share_the_banks(sws, oracle80):
    """The two constant banks belong to the process: calls of two contexts with different meshes, issued back to
    back on two streams without synchronisation, must not see each other's slabs or y tables."""
    import torch
    cfgA, cfgB = W.CONFIGS[1], W.custom(N=50, M=33, h=0.3, x1=-4.0, eps=0.3, amp=0.05, seed=41)
    uA, uB = W.state(cfgA), W.state(cfgB)
    sA, sB = torch.cuda.Stream(), torch.cuda.Stream()
    with sws.Context(cfgA.params()) as a, sws.Context(cfgB.params()) as b:
        a.set_const_path(1)
        b.set_const_path(1)
        refA, refB = a.residual(dev(uA)).cpu().numpy(), b.residual(dev(uB)).cpu().numpy()
        dA, dB = dev(uA), dev(uB)
        torch.cuda.synchronize()
        outs = []
        for _ in range(6):
            with torch.cuda.stream(sA):
                FA = a.residual(dA)
            with torch.cuda.stream(sB):
                FB = b.residual(dB)
            outs.append((FA, FB))
        torch.cuda.synchronize()
        for FA, FB in outs:
            assert np.array_equal(FA.cpu().numpy(), refA) and np.array_equal(FB.cpu().numpy(), refB)
    assert relerr(refA, oracle80.residual(cfgA.params(), uA)) <= TOL
    assert relerr(refB, oracle80.residual(cfgB.params(), uB)) <= TOL


def test_const_path_farfield_on_off(sws, oracle80):
    """steep state (slopes of order one): far field on / off / radius 12 agree to summation round-off"""
    cfg = W.custom(eps=0.5, amp=1.5, N=120, M=50, h=0.15, x1=-2.0, seed=22)
    u = W.state(cfg)
    E = oracle80.residual(cfg.params(), u)
    with sws.Context(cfg.params()) as ctx:
        ctx.set_const_path(1)
        F_on = ctx.residual(dev(u)).cpu().numpy()
        near = ctx.farfield_stats(1)
        ctx.set_farfield(0.0)
        F_off = ctx.residual(dev(u)).cpu().numpy()
        ctx.set_farfield(12.0)
        F_12 = ctx.residual(dev(u)).cpu().numpy()
    assert 0.0 < near < 1.0
    assert relerr(F_on, F_off) <= 2e-13 and relerr(F_12, F_off) <= 2e-13
    assert relerr(F_on, E) <= TOL and relerr(F_off, E) <= TOL


def test_const_path_refused_where_it_does_not_fit(sws):
    """a column of M = 520 records fits a bank only three at a time: the path is not offered (SWS_EINVAL), nor
    for the FP32 variant; mode values outside {-1, 0, 1} are refused"""
    cfg = W.custom(N=6, M=520, h=0.05, x1=-0.3, seed=10)
    with sws.Context(cfg.params()) as ctx:
        assert ctx.const_plan_info()["cols_per_slab"] == 0
        with pytest.raises(sws.SwsError):
            ctx.set_const_path(1)
        ctx.set_const_path(-1)
        ctx.set_const_path(0)
        with pytest.raises(sws.SwsError):
            ctx.set_const_path(2)
    with sws.Context(W.CONFIGS[0].params(), precision=1) as ctx:
        with pytest.raises(sws.SwsError):
            ctx.set_const_path(1)


def test_const_path_cuda_graph_capture_and_replay(sws):
    """sws_residual on the constant-bank path forks onto the library's two streams and joins again: a caller may
    capture it into a CUDA graph (after one eager call, which loads the modules and creates the streams) and
    replay it, also after another context has had its own y table in the banks."""
    import torch
    cfgA, cfgB = W.CONFIGS[1], W.custom(N=40, M=27, h=0.3, x1=-4.0, eps=0.3, amp=0.05, seed=43)
    with sws.Context(cfgA.params()) as a, sws.Context(cfgB.params()) as b:
        a.set_const_path(1)
        b.set_const_path(1)
        uA, uB = dev(W.state(cfgA)), dev(W.state(cfgB))
        FA = torch.empty_like(uA)
        ref = a.residual(uA).clone()
        refB = b.residual(uB).clone()
        torch.cuda.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g):
            a.residual(uA, out=FA)
        for _ in range(3):
            FA.zero_()
            assert torch.equal(b.residual(uB), refB)     # the banks now hold b's y table
            g.replay()
            torch.cuda.synchronize()
            assert torch.equal(FA, ref)
        assert torch.equal(a.residual(uA), ref)          # eager again after the capture


def test_const_path_capture_leaves_eager_calls_of_another_thread_alone(sws):
    """While host thread A has a CUDA-graph capture open that contains a constant-bank call, host thread B evaluates
    eagerly on a context and stream of its own.  A captured call keeps both banks on the capturing stream, so the
    library's two shared streams never join A's capture: B's calls run at once and are correct (they used to be
    enqueued into streams that belonged to A's open capture - swallowed into A's graph or refused), and A's graph
    holds A's work only."""
    import threading
    import torch
    cfgA, cfgB = W.CONFIGS[1], W.custom(N=47, M=29, h=0.3, x1=-4.0, eps=0.3, amp=0.05, seed=44)
    with sws.Context(cfgA.params()) as a, sws.Context(cfgB.params()) as b:
        a.set_const_path(1)
        b.set_const_path(1)
        uA, uB = dev(W.state(cfgA)), dev(W.state(cfgB))
        refA, refB = a.residual(uA).clone(), b.residual(uB).clone()
        FA1, FA2 = torch.zeros_like(uA), torch.zeros_like(uA)
        FB = [torch.zeros_like(uB) for _ in range(6)]          # B allocates nothing while A captures
        stB = torch.cuda.Stream()
        torch.cuda.synchronize()
        in_capture, b_done, errors = threading.Event(), threading.Event(), []

        def thread_b():
            try:
                torch.cuda.set_device(0)
                assert in_capture.wait(60)
                with torch.cuda.stream(stB):
                    for F in FB:
                        b.residual(uB, out=F)
                stB.synchronize()                               # B's work finishes while A's capture is still open
            except Exception as e:  # noqa: BLE001 - reported below
                errors.append(e)
            finally:
                b_done.set()

        t = threading.Thread(target=thread_b)
        t.start()
        g = torch.cuda.CUDAGraph()
        try:
            with torch.cuda.graph(g, capture_error_mode="thread_local"):
                a.residual(uA, out=FA1)
                in_capture.set()
                assert b_done.wait(120)
                a.residual(uA, out=FA2)
        finally:
            in_capture.set()
            t.join()
        assert not errors, errors
        for F in FB:
            assert torch.equal(F, refB)
        assert not FA1.any() and not FA2.any()                  # captured, not executed
        for _ in range(3):
            FA1.zero_()
            FA2.zero_()
            g.replay()
            torch.cuda.synchronize()
            assert torch.equal(FA1, refA) and torch.equal(FA2, refA)
        assert torch.equal(b.residual(uB), refB) and torch.equal(a.residual(uA), refA)


def test_const_path_host_threads(sws, oracle80):
    """Two host threads, each with a context and a stream of its own, call the constant-bank path at the same time:
    the library serialises them through its two banks (a mutex around the enqueue, stream order on the device)."""
    import threading
    import torch
    cfgs = [W.CONFIGS[1], W.custom(N=47, M=29, h=0.3, x1=-4.0, eps=0.3, amp=0.05, seed=44)]
    refs = [oracle80.residual(c.params(), W.state(c)) for c in cfgs]
    results, errors = [None, None], []

    def work(i):
        try:
            torch.cuda.set_device(0)
            st = torch.cuda.Stream()
            with sws.Context(cfgs[i].params()) as ctx, torch.cuda.stream(st):
                ctx.set_const_path(1)
                u = dev(W.state(cfgs[i]))
                outs = [ctx.residual(u) for _ in range(25)]
                st.synchronize()
                first = outs[0].cpu().numpy()
                assert all(np.array_equal(o.cpu().numpy(), first) for o in outs)
                results[i] = first
        except Exception as e:  # noqa: BLE001 - reported below
            errors.append(e)

    threads = [threading.Thread(target=work, args=(i,)) for i in range(2)]
    for t in threads:
        t.start()
    for t in threads:
        t.join()
    assert not errors, errors
    for i in range(2):
        assert relerr(results[i], refs[i]) <= TOL


def test_const_path_repeatability_stress(sws):
    """300 evaluations and 10 batches in a row on a mesh that takes the path by default (226x76, 15 slabs of 16
    columns, two banks): every result bitwise equal to the first (arrival counters return to zero, the two bank
    streams keep their slab order, no stale group sums)."""
    import torch
    cfg = W.custom(N=226, M=76, h=0.24, x1=-16.0, eps=1.0, amp=0.1, seed=5)
    u, V = dev(W.state(cfg)), dev(W.directions(cfg, 3))
    with sws.Context(cfg.params(), max_batch=3) as ctx:
        assert ctx.const_plan_info()["active"]
        F = torch.empty_like(u)
        ref = ctx.residual(u).clone()
        bad = 0
        for _ in range(300):
            ctx.residual(u, out=F)
            bad += int(not torch.equal(F, ref))
        JV0, Fp0, F00 = ctx.jv_batch(u, V, want_fpert=True, want_f0=True)
        JV0, Fp0 = JV0.clone(), Fp0.clone()
        assert torch.equal(F00, ref)
        for _ in range(10):
            JV, Fp, F0 = ctx.jv_batch(u, V, want_fpert=True, want_f0=True)
            bad += int(not (torch.equal(JV, JV0) and torch.equal(Fp, Fp0) and torch.equal(F0, ref)))
        torch.cuda.synchronize()
    assert bad == 0
