"""nsc_probe_static -- the probe for callers that may not allocate device memory -- against nsc_probe.

Why the entry point exists: a probe is typically read by code that watches a run and does not own it (a per-step
monitoring hook, a host program that keeps the flow state in its own tensors).  Such code often cannot call
cudaMalloc: the device has been filled on purpose (the N_r = 512 configuration holds 148 of 180 GB and the host
framework's pool owns the rest), cudaMalloc / cudaFree stall the whole device, which a once-per-step call would
pay every step, or the host program forbids allocating runtime calls where the hook runs.  nsc_probe needs a
context, and creating one allocates; nsc_probe_static takes the caller's field and output buffer and keeps its
only work space (block partial sums and an arrival counter) in a fixed 4.5 KB array inside the library.

What is checked: the value agrees with the context path (nsc_probe) within the tolerance the diagnostics
parity test uses (1e-12 x the sum of the level's coefficient magnitudes) on two calls in a row -- the second call
finds the first call's partial sums and counter still in the shared array, which must not matter -- that the
same call repeated gives the same bits, that device memory in use does not change over the calls, and that
sizes beyond the stated maximum are refused with a message that says so.

The file name sorts last on purpose: pytest -x stops at the first failure, and a failure here must not hide
the parity tests.  It does not depend on them: it passes alone in a fresh process (where its first call is the
library's first-call set-up on the device) and after the rest of the suite.
"""
import ctypes as C

import numpy as np
import pytest

from paper_1908_00587_b200 import synth


@pytest.fixture(scope="module")
def lib():
    from paper_1908_00587_b200 import build, nsc
    build.build()
    return nsc.load_library()


def test_probe_static_refuses_sizes_beyond_its_fixed_scratch(lib):
    """Argument checks come before any CUDA call, so this runs without a GPU: pointers are never dereferenced."""
    from paper_1908_00587_b200 import nsc
    dummy_in, dummy_out = C.c_void_p(4096), C.c_void_p(8192)
    ok = dict(N_r=16, M_theta=8, K_z=8, k_theta0=1, alpha=2.0, j=3, theta=0.1, z=0.2)

    def call(**over):
        a = dict(ok, **over)
        return lib.nsc_probe_static(dummy_in, a["N_r"], a["M_theta"], a["K_z"], a["k_theta0"], a["alpha"], a["j"],
                                    a["theta"], a["z"], dummy_out, None)

    for over in (dict(M_theta=513), dict(K_z=513), dict(M_theta=4096, K_z=4096)):
        assert call(**over) == nsc.NSC_EINVAL, over
        msg = lib.nsc_last_error(None).decode()
        assert "exceed the maximum" in msg and "512" in msg and "4608 bytes" in msg, msg
    for over in (dict(M_theta=0), dict(K_z=0), dict(N_r=0), dict(j=16), dict(j=-1), dict(k_theta0=0), dict(alpha=0.0),
                 dict(alpha=float("nan")), dict(theta=float("inf")), dict(z=float("nan"))):
        assert call(**over) == nsc.NSC_EINVAL, over
        assert lib.nsc_last_error(None).decode().startswith("nsc_probe_static:")
    assert lib.nsc_probe_static(None, 16, 8, 8, 1, 2.0, 3, 0.1, 0.2, dummy_out, None) == nsc.NSC_EINVAL
    assert lib.nsc_probe_static(dummy_in, 16, 8, 8, 1, 2.0, 3, 0.1, 0.2, None, None) == nsc.NSC_EINVAL


@pytest.mark.gpu
@pytest.mark.parametrize("ci,N_r,M,K", [(2, 12, 32, 40), (0, 10, 4, 8)])
def test_probe_static_matches_the_context_probe_on_two_calls_in_a_row(lib, ci, N_r, M, K):
    """(2, 12, 32, 40): heated, 33 x 81 = 2673 modes = three blocks with a ragged last one; (0, 10, 4, 8): one
    partly filled block."""
    import torch
    from paper_1908_00587_b200 import nsc
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    cfg = synth.scaled_config(ci, N_r=N_r, M=M, K=K)
    points = [(1, N_r // 2, 0.3, 0.7), (0, 1, 1.9, 0.05), (2, N_r - 2, 0.0, 0.0), (4, 3, 2.5, 1.0), (1, 0, -0.8, 4.0)]
    with nsc.Context.from_config(cfg) as ctx:
        st = synth.make_state(cfg, ctx.grid())
        rng = np.random.default_rng(cfg["seed"] + 17)        # every mode filled, not only the few of make_state
        st = [None if f is None else f + 1e-3 * (rng.standard_normal(f.shape) + 1j * rng.standard_normal(f.shape))
              for f in st]
        dev = [None if f is None else torch.from_numpy(np.ascontiguousarray(f)).cuda() for f in st]
        ctx.set_state(*dev)
        want = [ctx.probe(f, j, th, z) for f, j, th, z in points]            # the existing path (allocates on first use)

        # everything the static path needs exists before the first call: the caller's field and its output slots
        out = torch.full((2 * len(points),), float("nan"), dtype=torch.float64, device="cuda")
        f0, j0, th0, z0 = points[0]
        nsc.probe_static(dev[f0], cfg["k_theta0"], cfg["alpha"], j0, th0, z0, out[0:1])   # first call: set-up included
        torch.cuda.synchronize()
        free_before = torch.cuda.mem_get_info()[0]
        for i, (f, j, th, z) in enumerate(points):
            # two calls in a row on one stream, no synchronisation between them: the second starts from the
            # array as the first left it
            nsc.probe_static(dev[f], cfg["k_theta0"], cfg["alpha"], j, th, z, out[2 * i:2 * i + 1])
            nsc.probe_static(dev[f], cfg["k_theta0"], cfg["alpha"], j, th, z, out[2 * i + 1:2 * i + 2])
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info()[0] == free_before, "device memory in use changed over nsc_probe_static calls"
        got = out.cpu().numpy()
        for i, (f, j, th, z) in enumerate(points):
            scale = max(1.0, np.abs(st[f][j]).sum())
            assert abs(got[2 * i] - want[i]) <= 1e-12 * scale, (points[i], got[2 * i], want[i])
            assert got[2 * i + 1] == got[2 * i], "fixed summation order: the repeated call must give the same bits"
        # the context path again after the static calls: untouched by them
        assert ctx.probe(*points[0]) == pytest.approx(want[0], abs=1e-12 * max(1.0, np.abs(st[f0][j0]).sum()))
        # on a side stream of the caller's
        side = torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        nsc.probe_static(dev[2], cfg["k_theta0"], cfg["alpha"], 2, 0.4, 0.4, out[0:1], stream=side)
        side.synchronize()
        scale = max(1.0, np.abs(st[2][2]).sum())
        assert abs(out[0].item() - ctx.probe(2, 2, 0.4, 0.4)) <= 1e-12 * scale
        with pytest.raises(nsc.NscError):
            nsc.probe_static(dev[0], cfg["k_theta0"], cfg["alpha"], N_r, 0.0, 0.0, out[0:1])
