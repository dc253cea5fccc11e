"""sws_fd_shifts_noalloc: the finite-difference shifts sigma_b = 1e-7 (1 + |u|) / |v_b| of eq. (25)
computed without a context and without any device allocation inside the call.

Why the entry point exists: some users of libsws cannot call cudaMalloc at the point where they need the shifts - a
solver embedded in an application that gave all device memory to its own pool at start-up, or a continuation loop that
cannot take the device-wide stall cudaMalloc / cudaFree cause.  For them the scratch of the two-stage norm reduction
(block partial sums) is a fixed 33 KB array inside the library's device image instead of context workspace, shared by
all calls on a device and keeping the previous call's contents.  What this file checks is therefore exactly what could
go wrong with that design: the values against the existing context path (sws_jv_batch with device-computed shifts,
read back with sws_last_sigma), on TWO calls in a row of different sizes, so that a wrong scratch address, a row of
stale partial sums left by the first call, or a slot read before it was written would show.

The file is named test_zz_* so that pytest collects it last: `pytest -x` stops at the first failure and a failure here
must not hide the parity tests.  It passes alone in a fresh process (the first call then also resolves the array's
device address) and after the rest of the suite.  Needs a B200."""
import numpy as np
import pytest

import workloads as W

pytestmark = pytest.mark.gpu

TOL = 1e-13  # the tolerance tests/test_gpu_parity.py puts on the shifts


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


def context_shifts(sws, cfg, u, V):
    """The existing path: a context, sws_jv_batch with sigma_host = NULL, sws_last_sigma."""
    import torch
    with sws.Context(cfg.params(), max_batch=V.shape[0]) as ctx:
        ctx.jv_batch(dev(u), dev(V))
        torch.cuda.synchronize()
        return ctx.last_sigma(V.shape[0])


def test_fd_shifts_noalloc_two_calls_match_context_path(sws):
    import torch
    # first call: cfg 2 (61 x 21, n = 2604), its own b = 8 directions
    cfg_a = W.CONFIGS[1]
    u_a, V_a = W.state(cfg_a), W.directions(cfg_a)
    # second call: a smaller mesh (n = 704), fewer rows, other values, one zero direction (shift 0 by definition)
    cfg_b = W.CONFIGS[0]
    rng = np.random.default_rng(11)
    u_b = W.state(cfg_b) + 1e-2 * rng.standard_normal(cfg_b.n)
    V_b = 3.0 * rng.standard_normal((3, cfg_b.n))
    V_b[1] = 0.0
    ref_a = context_shifts(sws, cfg_a, u_a, V_a)
    ref_b = context_shifts(sws, cfg_b, u_b, V_b)
    assert ref_b[1] == 0.0 and (ref_a > 0).all()

    # inputs AND outputs are the caller's; the two calls follow each other on one stream with no synchronisation
    ua, Va, ub, Vb = dev(u_a), dev(V_a), dev(u_b), dev(V_b)
    out_a = torch.full((V_a.shape[0],), -1.0, dtype=torch.float64, device="cuda")
    out_b = torch.full((V_b.shape[0],), -1.0, dtype=torch.float64, device="cuda")
    sws.fd_shifts_noalloc(ua, Va, out_a)
    sws.fd_shifts_noalloc(ub, Vb, out_b)
    torch.cuda.synchronize()
    sig_a, sig_b = out_a.cpu().numpy(), out_b.cpu().numpy()

    assert np.abs(sig_a - ref_a).max() <= TOL * np.abs(ref_a).max()
    assert np.abs(sig_b - ref_b).max() <= TOL * np.abs(ref_b).max()
    assert sig_b[1] == 0.0
    # same block count and summation order as the context path: in fact bit for bit
    assert np.array_equal(sig_a, ref_a) and np.array_equal(sig_b, ref_b)
    # and the textbook formula, in numpy (not the oracle: this file must not depend on its build)
    want = 1e-7 * (1.0 + np.linalg.norm(u_a)) / np.linalg.norm(V_a, axis=1)
    assert np.abs(sig_a - want).max() <= 1e-12 * want.max()

    # the same call again after the smaller one: rows 4..8 of the scratch were not touched by call two.  By now the
    # kernels are loaded and the array's address is resolved, so the device's free memory must not move at all.
    out_a.fill_(-1.0)
    torch.cuda.synchronize()
    mem0 = torch.cuda.mem_get_info()[0]
    sws.fd_shifts_noalloc(ua, Va, out_a)
    torch.cuda.synchronize()
    mem1 = torch.cuda.mem_get_info()[0]
    assert np.array_equal(out_a.cpu().numpy(), ref_a)
    assert mem1 >= mem0, "free device memory shrank across a call: something allocated"


def test_fd_shifts_noalloc_rejects_what_the_array_cannot_hold(sws):
    import torch
    n, b = 100, sws.NOALLOC_MAX_B + 1
    u = torch.ones(n, dtype=torch.float64, device="cuda")
    V = torch.ones(b, n, dtype=torch.float64, device="cuda")
    out = torch.zeros(b, dtype=torch.float64, device="cuda")
    with pytest.raises(sws.SwsError, match="at most 64"):
        sws.fd_shifts_noalloc(u, V, out)
    # the largest batch it accepts
    sws.fd_shifts_noalloc(u, V[:-1], out[:-1])
    torch.cuda.synchronize()
    want = 1e-7 * (1.0 + np.sqrt(n)) / np.sqrt(n)
    assert np.abs(out[:-1].cpu().numpy() - want).max() <= 1e-15
    lib = sws.load_library()
    assert lib.sws_fd_shifts_noalloc(None, None, 10, 1, None, 0, None) == sws.SWS_EINVAL
    assert b"NULL" in lib.sws_noalloc_last_error()
