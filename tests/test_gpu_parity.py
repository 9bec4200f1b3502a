"""GPU parity (-m gpu): the CUDA path, called through the C ABI, against the oracle on the same
seeded inputs.  Tolerances are BASELINE.json north_star's: relative L2 (norm R14, all fields
concatenated, base flow included) <= 1e-11 per nonlinear evaluation, <= 1e-9 after 20 steps."""
import numpy as np
import pytest

import os

from helpers import oracle_of, nf_of
from oracle.nsc_oracle import rel_l2, rel_l2_pert
from paper_1908_00587_b200 import synth

pytestmark = pytest.mark.gpu

TOL_N = 1e-11
TOL_STEP = 1e-9
NCPU = os.cpu_count() or 1


def check_parity(got, ref, tol, K, what, mean_index="full"):
    """Asserts the R14 norm (all fields, base flow included) against ``tol`` and the same norm with the mean
    mode (0,0) left out (the base flow, 1e2..1e4 times the perturbation, sits there and would
    discount an error confined to the perturbation modes) against 10 * ``tol``; prints both."""
    e = rel_l2(got, ref)
    ep = rel_l2_pert(got, ref, K) if mean_index == "full" else rel_l2_pert(got, ref, K, mean_index=mean_index)
    print(f"{what}: rel-L2 {e:.2e}, without mode (0,0) {ep:.2e}")
    assert e <= tol, (what, e)
    assert ep <= 10 * tol, (what, "without (0,0)", ep)


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1908_00587_b200 import build
    build.build()
    return torch


def _ctx(cfg, **over):
    from paper_1908_00587_b200 import nsc
    return nsc.Context.from_config(cfg, **over)


def _dev(torch, arrs):
    return [None if a is None else torch.from_numpy(a).cuda() for a in arrs]


def _random_fields(cfg, seed, n):
    rng = np.random.default_rng(seed)
    shp = (cfg["N_r"], cfg["M"] + 1, 2 * cfg["K"] + 1)
    out = []
    for _ in range(n):
        f = rng.standard_normal(shp) + 1j * rng.standard_normal(shp)
        out.append(np.ascontiguousarray(f))
    return out


# (config index, N_r, M, K, oracle DFT backend): spans every transform length 12 .. 1536, several
# line tiles per CTA with ragged tails (N_r * (M+1) and N_r * N_z not multiples of the tile)
NL_CASES = [
    (0, 32, 8, 8, "naive"),       # cfg 1 as is
    (2, 11, 4, 16, "naive"),      # heated; lengths 12 / 48
    (1, 13, 32, 32, "naive"),     # lengths 96 / 96
    (2, 10, 64, 8, "naive"),      # heated; 192 / 24
    (3, 9, 128, 4, "naive"),      # 384 / 12
    (3, 12, 256, 8, "naive"),     # 768 / 24  (cfg 4's theta length)
    (1, 10, 8, 256, "naive"),     # 24 / 768  (cfg 4's z length)
    (4, 9, 512, 4, "naive"),      # heated; 1536 / 12 (cfg 5's theta length)
    (4, 9, 4, 512, "naive"),      # heated; 12 / 1536
    (2, 10, 128, 128, "naive"),   # heated; 384 / 384 (cfg 3's lengths)
    (4, 9, 512, 512, "naive"),    # heated; 1536 / 1536 (cfg 5's lengths: warp-pair kernels in both directions)
    (3, 9, 512, 8, "naive"),      # no temperature; 1536 / 24
]


@pytest.mark.parametrize("ci,N_r,M,K,dft", NL_CASES)
def test_nonlinear_matches_oracle(torch_cuda, ci, N_r, M, K, dft):
    torch = torch_cuda
    cfg = synth.scaled_config(ci, N_r=N_r, M=M, K=K)
    o = oracle_of(cfg, dft=dft)
    with _ctx(cfg) as ctx:
        np.testing.assert_array_equal(ctx.grid(), o.r)        # same nodes, bit for bit
        st = synth.make_state(cfg, ctx.grid())
        ctx.set_state(*_dev(torch, st))
        got = ctx.nonlinear_to_host()
    ref = o.nonlinear(*st[:nf_of(cfg)])
    check_parity(got, ref, TOL_N, K, f"nonlinear {N_r}x{M}x{K}")


@pytest.mark.parametrize("ci,N_r,M,K,n_theta,n_z", [(3, 9, 128, 8, 768, 0), (1, 9, 8, 128, 0, 768), (3, 10, 64, 64, 768, 768)])
def test_nonlinear_length_768_kernels_on_a_padded_grid(torch_cuda, ci, N_r, M, K, n_theta, n_z):
    """The length-768 kernels with fewer than 256 modes (a physical grid padded beyond the 3/2 rule through
    n_theta_phys / n_z_phys = 768): more zero slots on input, fewer kept on output."""
    torch = torch_cuda
    cfg = synth.scaled_config(ci, N_r=N_r, M=M, K=K)
    o = oracle_of(cfg, dft="naive", n_theta=n_theta, n_z=n_z)
    with _ctx(cfg, n_theta=n_theta, n_z=n_z) as ctx:
        st = synth.make_state(cfg, ctx.grid())
        ctx.set_state(*_dev(torch, st))
        got = ctx.nonlinear_to_host()
    check_parity(got, o.nonlinear(*st[:3]), TOL_N, K, f"nonlinear {N_r}x{M}x{K} on {n_theta or 3 * M} x {n_z or 3 * K}")


@pytest.mark.parametrize("ci,N_r,M,K", [(3, 9, 256, 256), (2, 9, 128, 128), (3, 9, 512, 512)])
def test_nonlinear_white_noise_through_the_long_transforms(torch_cuda, ci, N_r, M, K):
    """Full-band white-noise fields with a non-Hermitian m = 0 row (reading R6) through the length-768 and
    length-384 kernels, against the naive-DFT oracle."""
    torch = torch_cuda
    cfg = synth.scaled_config(ci, N_r=N_r, M=M, K=K)
    nf = nf_of(cfg)
    o = oracle_of(cfg, dft="naive")
    fs = _random_fields(cfg, 6, nf)
    with _ctx(cfg) as ctx:
        ctx.set_state(*(_dev(torch, fs) + [None] * (5 - nf)))
        got = ctx.nonlinear_to_host()
    check_parity(got, o.nonlinear(*fs), TOL_N, K, f"white-noise nonlinear {N_r}x{M}x{K}")


@pytest.mark.parametrize("ci,N_r,M,K,n_theta,n_z", [(0, 12, 5, 6, 24, 24), (2, 10, 100, 50, 384, 192), (1, 9, 1, 3, 12, 12)])
def test_mode_counts_that_are_not_powers_of_two(torch_cuda, ci, N_r, M, K, n_theta, n_z):
    """Any 1 <= M, K <= 512: the default physical grid is the shortest supported transform length that holds the
    3/2 rule; nonlinear term and two steps against the oracle on that grid."""
    torch = torch_cuda
    cfg = synth.scaled_config(ci, N_r=N_r, M=M, K=K)
    nf = nf_of(cfg)
    o = oracle_of(cfg, dft="fft", n_theta=n_theta, n_z=n_z)
    with _ctx(cfg) as ctx:
        st = synth.make_state(cfg, ctx.grid())
        ctx.set_state(*_dev(torch, st))
        got = ctx.nonlinear_to_host()
        check_parity(got, o.nonlinear(*st[:nf]), TOL_N, K, f"nonlinear {N_r}x{M}x{K} on the default grid")
        for _ in range(2):
            ctx.step(cfg["dt"])
        end = ctx.state_to_host()
    ref = st
    for _ in range(2):
        ref = o.step(ref, cfg["dt"])
    check_parity(end[:nf], ref[:nf], TOL_STEP, K, f"two steps {N_r}x{M}x{K}")


def test_nonlinear_broadband_random_fields_and_chunking(torch_cuda):
    """Full-band random (non-smooth, non-Hermitian m = 0 row) fields; radial chunking of the
    transform pipeline must not change a bit."""
    torch = torch_cuda
    cfg = synth.scaled_config(2, N_r=21, M=16, K=8)
    o = oracle_of(cfg)
    fs = _random_fields(cfg, 5, 4)
    ref = o.nonlinear(*fs)
    res = []
    for chunk in (0, 4, 1):
        with _ctx(cfg, radial_chunk=chunk) as ctx:
            ctx.set_state(*_dev(torch, fs), None)
            res.append(ctx.nonlinear_to_host())
    check_parity(res[0], ref, TOL_N, cfg["K"], "broadband random fields")
    for other in res[1:]:
        for a, b in zip(res[0], other):
            np.testing.assert_array_equal(a, b)


def test_nonlinear_padded_grid_variant(torch_cuda):
    """cfg 1 on the 24 x 48 grid BASELINE.json quotes (reading R4): equal to the oracle on that
    grid, and equal to the 24 x 24 result away from |k| = K."""
    torch = torch_cuda
    cfg = synth.config(0)
    o = oracle_of(cfg, n_z=48)
    with _ctx(cfg, n_z=48) as ctx:
        st = synth.make_state(cfg, ctx.grid())
        ctx.set_state(*_dev(torch, st))
        got = ctx.nonlinear_to_host()
    check_parity(got, o.nonlinear(*st[:3]), TOL_N, cfg["K"], "cfg 1 on the 24 x 48 grid")


SUB_CASES = [(0, 32, 8, 8), (2, 24, 4, 8), (1, 64, 8, 4), (3, 40, 4, 4), (2, 9, 4, 4)]


@pytest.mark.parametrize("ci,N_r,M,K", SUB_CASES)
def test_substep_matches_oracle(torch_cuda, ci, N_r, M, K):
    torch = torch_cuda
    cfg = synth.scaled_config(ci, N_r=N_r, M=M, K=K)
    nf = nf_of(cfg)
    o = oracle_of(cfg)
    with _ctx(cfg) as ctx:
        st = synth.make_state(cfg, ctx.grid())
        rng = np.random.default_rng(3)
        st[4] = 10.0 * (rng.standard_normal(st[0].shape) + 1j * rng.standard_normal(st[0].shape))
        U = max(abs(cfg["Re_i"]), abs(cfg["Re_o"]))
        E = [U * U * 0.1 * f for f in _random_fields(cfg, 8, nf)]
        ctx.set_state(*_dev(torch, st))
        Ed = _dev(torch, E) + [None] * (4 - nf)
        ctx.substep(*Ed, cfg["dt"])
        got = ctx.state_to_host()
    ref = o.substep(st, E, cfg["dt"])
    check_parity(got[:nf], ref[:nf], 1e-11, cfg["K"], f"sub-step {ci, N_r, M, K}")
    assert rel_l2([got[4]], [ref[4]]) <= 1e-7       # pressure: parity unpinned (phi / dt amplifies round-off)


@pytest.mark.parametrize("ci,N_r,M,K,nsteps", [(0, 32, 8, 8, 20), (2, 32, 8, 8, 20), (1, 64, 32, 32, 5)])
def test_steps_match_oracle(torch_cuda, ci, N_r, M, K, nsteps):
    torch = torch_cuda
    cfg = synth.scaled_config(ci, N_r=N_r, M=M, K=K)
    nf = nf_of(cfg)
    o = oracle_of(cfg, dft="fft")
    with _ctx(cfg) as ctx:
        st = synth.make_state(cfg, ctx.grid())
        ctx.set_state(*_dev(torch, st))
        for _ in range(nsteps):
            ctx.step(cfg["dt"])
        got = ctx.state_to_host()
    ref = st
    for _ in range(nsteps):
        ref = o.step(ref, cfg["dt"])
    check_parity(got[:nf], ref[:nf], TOL_STEP, K, f"{nsteps} steps {N_r}x{M}x{K}")


def _twenty_steps_full(torch, ci, side_stream, nsteps=20):
    """20 nsc_step calls at a full BASELINE.json configuration against 20 oracle steps (the north-star
    criterion; fewer where said).  Oracle: library FFT (pinned to the naive sums at these lengths, tests/test_oracle_transforms.py)
    and the plain-C banded elimination (pinned to the dense one, tests/test_oracle_banded.py)."""
    cfg = synth.config(ci)
    nf = nf_of(cfg)
    o = oracle_of(cfg, dft="fft", solve="c")
    with _ctx(cfg) as ctx:
        if side_stream:                       # a non-default stream: the steps are CUDA-graph replays
            s = torch.cuda.Stream()
            ctx.set_stream(s)
        st = synth.make_state(cfg, ctx.grid())
        ctx.set_state(*_dev(torch, st))
        for _ in range(nsteps):
            ctx.step(cfg["dt"])
        got = ctx.state_to_host()
        replays = ctx.graph_replays()
    assert replays == (nsteps if side_stream else 0)
    ref = st
    for _ in range(nsteps):
        ref = o.step(ref, cfg["dt"], workers=NCPU)
    check_parity(got[:nf], ref[:nf], TOL_STEP, cfg["K"], f"{nsteps} steps at full cfg {ci + 1}")


@pytest.mark.parametrize("ci", [1, 2])
def test_twenty_steps_at_full_size(torch_cuda, ci):
    """BASELINE.json configs[1] (64 x 33 x 65 modes) and configs[2] (heated, 128 x 129 x 257 modes; the oracle
    takes ~10 s per step on 16 cores)."""
    _twenty_steps_full(torch_cuda, ci, side_stream=(ci == 2))


@pytest.mark.parametrize("N_r,M,K,chunk,nsteps", [(12, 512, 16, 5, 20), (12, 16, 512, 5, 20), (9, 512, 512, 4, 6)])
def test_steps_on_the_1536_kernels_in_several_radial_chunks(torch_cuda, N_r, M, K, chunk, nsteps):
    """What stands in for the unpinned full steps at cfg 5: cfg 5's physics (heated) and its
    code path -- the length-1536 warp-pair kernels, the radial pipeline forced into several chunks (spectral k_dr +
    three z transforms per line) and CUDA-graph replays on a side stream -- at radial sizes where the oracle can
    step.  20 steps with the 1536 transform in theta only and in z only (0.3 s of oracle time per step), 6 steps
    with both (9 x 513 x 1025 modes, 1536 x 1536 grid: 10 s per oracle step on the GPU box's host, 30 s on 8 cores;
    measured in round 3: 3.6e-15 / 3.8e-15 after 20 steps, 5.2e-16 after 3 with both)."""
    torch = torch_cuda
    cfg = synth.scaled_config(4, N_r=N_r, M=M, K=K)
    nf = nf_of(cfg)
    assert nf == 4
    o = oracle_of(cfg, dft="fft", solve="c")
    with _ctx(cfg, radial_chunk=chunk) as ctx:
        s = torch.cuda.Stream()
        ctx.set_stream(s)
        st = synth.make_state(cfg, ctx.grid())
        ctx.set_state(*_dev(torch, st))
        for _ in range(nsteps):
            ctx.step(cfg["dt"])
        got = ctx.state_to_host()
        assert ctx.graph_replays() == nsteps
    ref = st
    for _ in range(nsteps):
        ref = o.step(ref, cfg["dt"], workers=NCPU)
    check_parity(got[:nf], ref[:nf], TOL_STEP, K, f"{nsteps} steps at {N_r} x {M + 1} x {2 * K + 1} modes, radial chunk {chunk}")


@pytest.mark.skipif(not os.environ.get("NSC_TEST_CFG4_20STEPS"), reason="opt-in: the oracle takes ~2 min per step at cfg 4")
def test_twenty_steps_at_full_cfg4(torch_cuda):
    """BASELINE.json configs[3] (N_r = 256, 257 x 513 modes; bench.py's workload, graph replays on a side
    stream).  Opt-in (NSC_TEST_CFG4_20STEPS=1); the last recorded figures are in DESIGN.md section 9."""
    _twenty_steps_full(torch_cuda, 3, side_stream=True)


@pytest.mark.skipif(not os.environ.get("NSC_TEST_CFG5_STEPS"), reason="opt-in: the oracle needs > 200 GB of host memory for a full step at cfg 5")
def test_steps_at_full_cfg5(torch_cuda):
    """BASELINE.json configs[4] (N_r = 512, 513 x 1025 modes, heated; the warp-pair kernels in several radial chunks):
    NSC_TEST_CFG5_STEPS full steps against the oracle.  Opt-in and so far never completed: on the 196 GB host of the
    round-2 box the oracle's step was killed for lack of memory, so full steps at cfg 5 remain unpinned (DESIGN.md
    section 9); the nonlinear term and the sub-step are checked there on samples."""
    _twenty_steps_full(torch_cuda, 4, side_stream=True, nsteps=int(os.environ["NSC_TEST_CFG5_STEPS"]))


def test_couette_flow_is_a_fixed_point_on_the_gpu(torch_cuda):
    torch = torch_cuda
    cfg = synth.scaled_config(0, N_r=32, M=4, K=4)
    o = oracle_of(cfg)
    base = o.base_state_discrete()
    with _ctx(cfg) as ctx:
        ctx.set_state(*_dev(torch, base))
        for _ in range(3):
            ctx.step(1e-2)
        got = ctx.state_to_host()
    assert rel_l2(got[:3], base[:3]) <= 1e-13


def test_host_buffer_entry_points_and_errors(torch_cuda):
    from paper_1908_00587_b200 import nsc
    cfg = synth.scaled_config(0, N_r=16, M=4, K=4)
    with _ctx(cfg) as ctx:
        with pytest.raises(nsc.NscError) as ei:
            ctx.step(1e-3)
        assert ei.value.code == nsc.NSC_ESTATE
        st = synth.make_state(cfg, ctx.grid())
        ctx.set_state(*st)                         # numpy arrays -> nsc_set_state_host
        back = ctx.state_to_host()
        for a, b in zip(st, back):
            if a is not None:
                np.testing.assert_array_equal(a, b)
        n0 = ctx.launch_count()                    # set_state may launch (D1 p of the new state)
        with pytest.raises(nsc.NscError) as ei:
            ctx.step(-1.0)
        assert ei.value.code == nsc.NSC_EINVAL
        assert ctx.launch_count() == n0
        ctx.step(1e-3)
        assert ctx.launch_count() > n0


@pytest.mark.parametrize("ci", [3, 2])
def test_full_size_sampled(torch_cuda, ci):
    """BASELINE.json configs[3] (N_r = 256, M = K = 256, 768 x 768 grid: bench.py's workload, length-768
    transform pipeline + fused linear sweeps) and configs[2] (heated, 128^3, generic transform kernels) at full
    size: the nonlinear term at sampled radial nodes and one sub-step at sampled modes against the oracle, then
    the divergence of the stepped state at round-off (a property that holds at any size)."""
    torch = torch_cuda
    cfg = synth.config(ci)
    nf = nf_of(cfg)
    N_r = cfg["N_r"]
    o = oracle_of(cfg, dft="naive")      # the naive sums decide at the sampled nodes; the sub-step uses no transform
    nodes = [0, 1, 4, N_r // 2 - 1, (3 * N_r) // 4, N_r - 5, N_r - 2, N_r - 1]
    rng = np.random.default_rng(11)
    im = np.concatenate([[0, 0, 0, cfg["M"], cfg["M"], 1], rng.integers(0, cfg["M"] + 1, 26)])
    ik = np.concatenate([[cfg["K"], cfg["K"] + 1, 0, 0, 2 * cfg["K"], cfg["K"] - 1], rng.integers(0, 2 * cfg["K"] + 1, 26)])
    with _ctx(cfg) as ctx:
        st = synth.make_state(cfg, ctx.grid())
        ctx.set_state(*_dev(torch, st))
        got = ctx.nonlinear_to_host()
        ref = o.nonlinear(*st[:nf], nodes=nodes)
        check_parity([g[nodes] for g in got], ref, TOL_N, cfg["K"], f"cfg {ci + 1} nonlinear at {len(nodes)} nodes")
        # sub-step with the nonlinear term just computed as the explicit term
        E = got
        ctx.substep(*(_dev(torch, E) + [None] * (4 - nf)), cfg["dt"])
        sub = ctx.state_to_host()
        ref_s = o.substep(st, E, cfg["dt"], modes=(im, ik))
        got_s = [f[:, im, ik] for f in sub[:nf]]
        mean = np.nonzero((im == 0) & (ik == cfg["K"]))[0]
        check_parity(got_s, ref_s[:nf], 1e-11, cfg["K"], f"cfg {ci + 1} sub-step at {len(im)} modes", mean_index=mean)
        # scaled divergence of the new state (formula of SURVEY.md section 8(c), pin T5)
        ur, ut, uz = sub[:3]
        r = o.r[:, None, None]
        n = o.n[None, :, None]
        kap = o.kappa[None, None, :]
        d = o.divergence(ur, ut, uz)[1:-1]
        scale = (np.abs(o.D1) @ np.abs(ur).reshape(N_r, -1)).reshape(ur.shape) + np.abs(ur) / r \
            + np.abs(n / r * ut) + np.abs(kap * uz)
        scale = scale[1:-1]
        mask = scale > 0
        # SURVEY T5 quotes <= 1e-9 for single modes at N_r = 256; over all 3.3e7 interior mode-points of the
        # broadband state the maximum is a few 1e-9 (cond(P) ~ 1e13 on the Chebyshev grid): bar 1e-8
        assert np.max(np.abs(d[mask]) / scale[mask]) <= 1e-8


@pytest.mark.parametrize("ci,N_r,M,K", [(3, 12, 256, 256), (2, 17, 8, 16)])
def test_step_is_deterministic(torch_cuda, ci, N_r, M, K):
    """Two contexts, same state, three steps each: bit-identical results (R15: one deterministic result per
    input).  A shared-memory race in the transform tiles or in the cp.async row pipelines of the marching
    sweeps would show up here as run-to-run differences; (3, 12, 256, 256) runs the length-768 kernels."""
    torch = torch_cuda
    cfg = synth.scaled_config(ci, N_r=N_r, M=M, K=K)
    res = []
    for _ in range(2):
        with _ctx(cfg) as ctx:
            st = synth.make_state(cfg, ctx.grid())
            ctx.set_state(*_dev(torch, st))
            for _ in range(3):
                ctx.step(cfg["dt"])
            res.append(ctx.state_to_host())
    for a, b in zip(*res):
        if a is not None:
            assert np.isfinite(a).all()
            np.testing.assert_array_equal(a, b)


@pytest.mark.parametrize("grid,c", [(0, 0.5), (1, 0.7), (1, 1.0), (0, 0.3)])
def test_substep_uniform_grid_and_other_implicitness(torch_cuda, grid, c):
    """The rewrite of L1 as u/c - gamma A u for gamma = (1-c)/c != 1 and gamma = 0,
    and the uniform radial grid (R2 type 0): one sub-step and two full steps against the oracle."""
    torch = torch_cuda
    cfg = dict(synth.scaled_config(2, N_r=20, M=4, K=8), grid=grid)
    nf = nf_of(cfg)
    o = oracle_of(cfg, c=c)
    with _ctx(cfg, c=c) as ctx:
        np.testing.assert_array_equal(ctx.grid(), o.r)
        st = synth.make_state(cfg, ctx.grid())
        rng = np.random.default_rng(4)
        st[4] = 5.0 * (rng.standard_normal(st[0].shape) + 1j * rng.standard_normal(st[0].shape))
        U = max(abs(cfg["Re_i"]), abs(cfg["Re_o"]))
        E = [U * U * 0.1 * f for f in _random_fields(cfg, 9, nf)]
        ctx.set_state(*_dev(torch, st))
        ctx.substep(*_dev(torch, E), cfg["dt"])
        got = ctx.state_to_host()
        ref = o.substep(st, E, cfg["dt"])
        check_parity(got[:nf], ref[:nf], 1e-11, cfg["K"], f"sub-step, grid {grid}, c = {c}")
        ctx.set_state(*_dev(torch, st))
        for _ in range(2):
            ctx.step(cfg["dt"])
        got = ctx.state_to_host()
    ref = st
    for _ in range(2):
        ref = o.step(ref, cfg["dt"])
    check_parity(got[:nf], ref[:nf], TOL_STEP, cfg["K"], f"two steps, grid {grid}, c = {c}")


@pytest.mark.parametrize("ci,N_r,M,K,mult,amp,kmin", [(0, 24, 8, 8, 4.0, 5e-2, 2), (2, 20, 4, 8, 20.0, None, 1)])
def test_iterated_corrector_matches_oracle(torch_cuda, ci, N_r, M, K, mult, amp, kmin):
    """NEXT-1 (R16): nsc_step_iterated against the oracle's step_iterated -- same number of corrector
    passes, same convergence norm, same state; one pass is bit-identical to nsc_step; a following plain
    step still agrees (the accepted pressure and its radial derivative became the state)."""
    torch = torch_cuda
    cfg = synth.scaled_config(ci, N_r=N_r, M=M, K=K)
    if amp is not None:
        cfg["amp"] = amp
    nf = nf_of(cfg)
    dt = mult * cfg["dt"]
    o = oracle_of(cfg, dft="fft")
    with _ctx(cfg) as ctx:
        st = synth.make_state(cfg, ctx.grid())
        # one pass == nsc_step
        ctx.set_state(*_dev(torch, st))
        ctx.step(dt)
        plain = ctx.state_to_host()
        ctx.set_state(*_dev(torch, st))
        k1, e1 = ctx.step_iterated(dt, 0.0, 1)
        one = ctx.state_to_host()
        assert k1 == 1 and np.isfinite(e1)
        for a, b in zip(plain, one):
            if a is not None:
                np.testing.assert_array_equal(a, b)
        # iterate to tol, then one plain step
        tol = 1e-6
        ctx.set_state(*_dev(torch, st))
        k, err = ctx.step_iterated(dt, tol, 30)
        got = ctx.state_to_host()
        ref, k_ref, err_ref = o.step_iterated(st, dt, tol, 30)
        assert k == k_ref and kmin <= k < 30
        assert abs(err - err_ref) <= 1e-3 * err_ref + 1e-15
        check_parity(got[:nf], ref[:nf], TOL_STEP, cfg["K"], f"iterated corrector, {k} passes")
        ctx.step(dt)
        got2 = ctx.state_to_host()
    ref2 = o.step(ref, dt)
    check_parity(got2[:nf], ref2[:nf], TOL_STEP, cfg["K"], "plain step after the iterated one")


@pytest.mark.parametrize("ci,N_r,M,K", [(2, 24, 8, 8), (0, 20, 4, 8)])
def test_diagnostics_match_oracle(torch_cuda, ci, N_r, M, K):
    """NEXT-3: nsc_nusselt and nsc_probe against the oracle's nusselt / probe, before and after steps."""
    torch = torch_cuda
    cfg = synth.scaled_config(ci, N_r=N_r, M=M, K=K)
    nf = nf_of(cfg)
    o = oracle_of(cfg, dft="fft")
    with _ctx(cfg) as ctx:
        st = synth.make_state(cfg, ctx.grid())
        ctx.set_state(*_dev(torch, st))
        for it in range(2):
            got = np.array(ctx.nusselt())
            ref = np.array(o.nusselt(st))
            assert np.array_equal(np.isnan(got), np.isnan(ref))
            np.testing.assert_allclose(got[~np.isnan(ref)], ref[~np.isnan(ref)], rtol=1e-11, atol=1e-12)
            for field, j, th, z in [(1, N_r // 2, 0.3, 0.7), (0, 1, 1.9, 0.05), (2, N_r - 2, 0.0, 0.0), (4, 3, 2.5, 1.0)]:
                ref_v = o.probe(st[field], j, th, z)
                scale = max(1.0, np.abs(st[field][j]).sum())
                assert abs(ctx.probe(field, j, th, z) - ref_v) <= 1e-12 * scale
            if nf == 4:
                assert abs(ctx.probe(3, 2, 0.4, 0.4) - o.probe(st[3], 2, 0.4, 0.4)) <= 1e-12
            ctx.step(cfg["dt"])
            st = o.step(st, cfg["dt"])
        with pytest.raises(Exception):
            ctx.probe(3 if nf == 3 else 5, 0, 0.0, 0.0)


@pytest.mark.parametrize("ci,N_r,M,K,chunk", [(1, 10, 8, 256, 4), (3, 12, 256, 8, 5), (3, 11, 256, 256, 3), (1, 10, 8, 512, 3),
                                             (1, 10, 8, 128, 4)])
def test_nonlinear_length_768_in_several_radial_chunks(torch_cuda, ci, N_r, M, K, chunk):
    """The multi-chunk form of the length-768 pipeline (spectral k_dr + three z transforms per line, used when
    the work arrays of the whole radius do not fit) against the oracle, and against the single-chunk form."""
    torch = torch_cuda
    cfg = synth.scaled_config(ci, N_r=N_r, M=M, K=K)
    o = oracle_of(cfg, dft="naive")
    res = []
    for rc in (chunk, 0):
        with _ctx(cfg, radial_chunk=rc) as ctx:
            st = synth.make_state(cfg, ctx.grid())
            ctx.set_state(*_dev(torch, st))
            res.append(ctx.nonlinear_to_host())
    ref = o.nonlinear(*st[:3])
    check_parity(res[0], ref, TOL_N, K, "768 pipeline, several chunks")
    check_parity(res[1], ref, TOL_N, K, "768 pipeline, one chunk")
    assert rel_l2(res[0], res[1]) <= 1e-13


def test_full_size_cfg5_sampled(torch_cuda):
    """BASELINE.json configs[4] (the paper's Fig. 1 problem size: N_r = 512, 513 x 1025 modes, heated; 131 GB on
    the device, ~20 GB of host arrays) at full size: the nonlinear term at sampled radial nodes against the
    naive-DFT oracle (70 s), then one sub-step with that term as the explicit term at sampled modes against the
    oracle's plain-C backend (per listed mode: seconds; the dense backend forms the right-hand sides of all 5e5
    modes with 512 x 512 operators, 28 min, which is why this leg used to be opt-in)."""
    import gc
    torch = torch_cuda
    free_dev = torch.cuda.mem_get_info()[0]
    try:
        free_host = os.sysconf("SC_AVPHYS_PAGES") * os.sysconf("SC_PAGE_SIZE")
    except (ValueError, OSError):
        free_host = 1 << 62
    if free_dev < 155e9 or free_host < 48e9:
        pytest.skip(f"cfg 5 needs 148 GB on the device and ~40 GB of host memory (free: {free_dev / 1e9:.0f} / {free_host / 1e9:.0f} GB)")
    cfg = synth.config(4)
    o = oracle_of(cfg, dft="naive")
    N_r = cfg["N_r"]
    nodes = [0, N_r // 2 + 3, N_r - 1]
    rng = np.random.default_rng(12)
    im = np.concatenate([[0, 0, cfg["M"], 1], rng.integers(0, cfg["M"] + 1, 28)])
    ik = np.concatenate([[cfg["K"], cfg["K"] + 1, 0, cfg["K"] - 1], rng.integers(0, 2 * cfg["K"] + 1, 28)])
    with _ctx(cfg) as ctx:
        st = synth.make_state(cfg, ctx.grid())
        ctx.set_state(*st)
        E = ctx.nonlinear_to_host()
        ref = o.nonlinear(*st[:4], nodes=nodes)
        check_parity([g[nodes] for g in E], ref, TOL_N, cfg["K"], "cfg 5 nonlinear at sampled nodes")
        ctx.substep(*_dev(torch, E), cfg["dt"])
        sub = ctx.state_to_host()
    got_s = [f[:, im, ik].copy() for f in sub[:4]]
    del sub
    gc.collect()
    ref_s = oracle_of(cfg, dft="naive", solve="c").substep(st, E, cfg["dt"], modes=(im, ik))
    mean = np.nonzero((im == 0) & (ik == cfg["K"]))[0]
    # the bar of the sub-step at cfg 3 / 4 is 1e-11 (1e-10 without (0,0)); cond(P) grows like N_r^4 on the clustered grid,
    # so at N_r = 512 the bar is ten times that -- still ten times below the 1e-9 this leg asserted while it was opt-in
    check_parity(got_s, ref_s[:4], 1e-10, cfg["K"], f"cfg 5 sub-step at {len(im)} modes", mean_index=mean)


def test_step_graph_replay_equals_plain_launches(torch_cuda):
    """On a non-default stream nsc_step captures its kernel sequence into a CUDA graph and replays it; on the
    legacy default stream (no capture possible) it launches kernel by kernel.  Same bits, same launch count;
    a change of dt or an nsc_step_iterated in between (buffer swap) re-captures."""
    torch = torch_cuda
    cfg = synth.scaled_config(1, N_r=20, M=8, K=8)
    dt = cfg["dt"]
    res, counts = [], []
    for side in (False, True):
        with _ctx(cfg) as ctx:
            s = torch.cuda.Stream() if side else None
            if side:
                ctx.set_stream(s)
            st = synth.make_state(cfg, ctx.grid())
            ctx.set_state(*_dev(torch, st))
            torch.cuda.synchronize()
            n0 = ctx.launch_count()
            for _ in range(3):
                ctx.step(dt)
            ctx.step(0.5 * dt)
            ctx.step_iterated(dt, 0.0, 2)
            for _ in range(2):
                ctx.step(dt)
            torch.cuda.synchronize()
            counts.append(ctx.launch_count() - n0)
            res.append(ctx.state_to_host())
            assert ctx.graph_replays() == (6 if side else 0)     # every nsc_step on the side stream was a replay
    assert counts[0] == counts[1]
    for a, b in zip(*res):
        if a is not None:
            np.testing.assert_array_equal(a, b)


def test_graph_replay_after_a_substep_with_another_dt(torch_cuda):
    """nsc_step(dt), nsc_substep(E, dt / 2), nsc_step(dt) on a side stream: the sub-step rebuilds the Helmholtz
    factors in place for dt / 2, so the cached step graph must see factors for dt again before it is replayed.
    Compared bit for bit with a context that never uses a graph (nsc_params.no_graph)."""
    torch = torch_cuda
    cfg = synth.scaled_config(2, N_r=18, M=8, K=8)
    nf = nf_of(cfg)
    dt = cfg["dt"]
    res = []
    for no_graph in (1, 0):
        with _ctx(cfg, no_graph=no_graph) as ctx:
            s = torch.cuda.Stream()
            ctx.set_stream(s)
            st = synth.make_state(cfg, ctx.grid())
            ctx.set_state(*_dev(torch, st))
            E = _dev(torch, [1e3 * f for f in _random_fields(cfg, 2, nf)])
            ctx.step(dt)
            ctx.substep(*E, 0.5 * dt)
            ctx.step(dt)
            ctx.step(dt)
            torch.cuda.synchronize()
            assert ctx.graph_replays() == (0 if no_graph else 3)
            res.append(ctx.state_to_host())
    for a, b in zip(*res):
        if a is not None:
            assert np.isfinite(a).all()
            np.testing.assert_array_equal(a, b)


@pytest.mark.parametrize("ci,N_r,M,K", [(0, 20, 4, 4), (2, 12, 16, 32), (1, 11, 64, 8), (3, 9, 256, 256), (2, 10, 128, 128),
                                       (4, 9, 512, 16)])
def test_cfl_rate_matches_oracle(torch_cuda, ci, N_r, M, K):
    """NEXT-1 (R17): nsc_cfl_rate (maxima of |u| per radial level gathered inside the theta kernels, generic and
    warp-transform forms) against the oracle's cfl_rate on the physical grid."""
    torch = torch_cuda
    cfg = synth.scaled_config(ci, N_r=N_r, M=M, K=K)
    o = oracle_of(cfg, dft="fft")
    with _ctx(cfg) as ctx:
        st = synth.make_state(cfg, ctx.grid())
        st[0] = st[0] + 0.3 * st[1]                      # radial velocity of the size of the rotation: all three terms matter
        ctx.set_state(*_dev(torch, st))
        got = ctx.cfl_rate()
        again = ctx.cfl_rate()
    ref, _ = o.cfl_rate(st)
    assert got == again
    assert abs(got - ref) <= 1e-12 * ref


@pytest.mark.parametrize("heated", [False, True])
def test_step_size_controller_follows_the_oracle(torch_cuda, heated):
    """NEXT-1 (R17): nsc_advance after an impulsive change of the rotation rate against the oracle's
    advance: the same sequence of attempts (step sizes bit for bit, corrector passes, accept / reject), the same
    corrector norms, the same state at t_end; rejected attempts leave the state untouched."""
    torch = torch_cuda
    cfg = synth.scaled_config(2 if heated else 0, N_r=20, M=4, K=4)
    if heated:
        cfg = dict(cfg, Re_i=100.0, Re_o=0.0, Ra=2.0e3, dt=1e-3)
    nf = nf_of(cfg)
    cfg2 = dict(cfg, Re_i=400.0)
    o1 = oracle_of(cfg, dft="fft")
    st = synth.make_state(cfg, o1.r)
    o2 = oracle_of(cfg2, dft="fft")
    args = (8e-3, 200, 4e-3, 1e-7, 0.5, 2)
    ref, t_ref, rlog = o2.advance(st, *args)
    assert any(not ok for (_, _, _, ok) in rlog) and t_ref == args[0]
    with _ctx(cfg2) as ctx:
        ctx.set_state(*_dev(torch, st))
        # one attempt only: rejected, nothing moves
        info1, log1 = ctx.advance(args[0], 1, *args[2:])
        assert info1["t"] == 0.0 and info1["rejected"] == 1 and info1["accepted"] == 0 and not log1[0][3]
        for a, b in zip(ctx.state_to_host(), st):
            if b is not None:
                np.testing.assert_array_equal(a, b)
        info, log = ctx.advance(*args)
        got = ctx.state_to_host()
    assert len(log) == len(rlog)
    for (dt, k, err, ok), (rdt, rk, rerr, rok) in zip(log, rlog):
        assert dt == rdt and k == rk and ok == rok
        assert abs(err - rerr) <= 1e-4 * rerr + 1e-14
    assert info["t"] == t_ref and info["accepted"] == sum(ok for (_, _, _, ok) in rlog)
    assert info["rejected"] == len(rlog) - info["accepted"] and info["passes"] == sum(k for (_, k, _, _) in rlog)
    assert info["dt_min"] == min(d for (d, _, _, ok) in rlog if ok) and info["dt_max"] == max(d for (d, _, _, ok) in rlog if ok)
    check_parity(got[:nf], ref[:nf], TOL_STEP, cfg["K"], f"controller, {len(log)} attempts")


def test_wave_speed_matches_oracle(torch_cuda):
    """NEXT-3: nsc_wave_speed / nsc_mode_coefficient against the oracle's wave_speed on the pinned case (a
    temperature disturbance carried by solid-body rotation, speed -> Omega) and on a velocity mode of cfg 1."""
    torch = torch_cuda
    Omega = 40.0
    cfg = dict(synth.scaled_config(2, N_r=16, M=4, K=4), eta=0.5, Re_i=Omega * 1.0, Re_o=Omega * 2.0, Ra=1e-9, Pr=0.7)
    o = oracle_of(cfg, dft="fft")
    st = o.base_state_discrete()
    x = o.r - o.r[0]
    st[3][:, 2, 1 + o.p.K] += 1e-3 * x * (1 - x) * (1 + 0.5j)
    ref, ref_state = o.wave_speed(st, 3, 7, 2, 1, 2.5e-4, 8)
    with _ctx(cfg) as ctx:
        ctx.set_state(*_dev(torch, st))
        assert ctx.mode_coefficient(3, 7, 2, 1) == complex(st[3][7, 2, 1 + o.p.K])
        got = ctx.wave_speed(3, 7, 2, 1, 2.5e-4, 8)
        end = ctx.state_to_host()
        with pytest.raises(Exception):
            ctx.wave_speed(3, 7, 0, 1, 2.5e-4, 2)        # m = 0 has no azimuthal phase speed
    assert abs(got - ref) <= 1e-9 * abs(ref) and abs(got - Omega) <= 3e-4 * Omega
    check_parity(end[:4], ref_state[:4], TOL_STEP, cfg["K"], "state after the wave-speed steps")
    cfg = synth.scaled_config(0, N_r=24, M=8, K=8)
    o = oracle_of(cfg, dft="fft")
    st = synth.make_state(cfg, o.r)
    ref, _ = o.wave_speed(st, 1, 12, 1, 2, cfg["dt"], 5)
    with _ctx(cfg) as ctx:
        ctx.set_state(*_dev(torch, st))
        got = ctx.wave_speed(1, 12, 1, 2, cfg["dt"], 5)
    assert abs(got - ref) <= 1e-8 * abs(ref)


@pytest.mark.parametrize("src,dst", [((0, 20, 4, 8, 1), (0, 33, 8, 4, 0)), ((2, 24, 8, 8, 1), (2, 16, 4, 16, 1)),
                                     ((2, 18, 4, 4, 0), (0, 18, 4, 4, 0))])
def test_regrid_matches_oracle(torch_cuda, src, dst):
    """NEXT-4 (R18): nsc_regrid against the oracle's regrid -- radial interpolation onto another
    grid family and node count, mode padding and truncation, pressure included, temperature kept or dropped;
    regridding onto the same resolution is the identity; the regridded context steps on in parity."""
    torch = torch_cuda
    ca = dict(synth.scaled_config(src[0], N_r=src[1], M=src[2], K=src[3]), grid=src[4])
    cb = dict(synth.scaled_config(dst[0], N_r=dst[1], M=dst[2], K=dst[3]), grid=dst[4])
    for key in ("eta", "alpha", "k_theta0"):
        cb[key] = ca[key]
    oa, ob = oracle_of(ca, dft="fft"), oracle_of(cb, dft="fft")
    nfb = nf_of(cb)
    st = synth.make_state(ca, oa.r)
    rng = np.random.default_rng(7)
    st[4] = 3.0 * (rng.standard_normal(st[0].shape) + 1j * rng.standard_normal(st[0].shape))
    ref = ob.regrid(st, oa)
    with _ctx(ca) as a, _ctx(cb) as b, _ctx(ca) as a2:
        with pytest.raises(Exception):
            b.regrid_from(a)                         # the source has no state yet
        a.set_state(*_dev(torch, st))
        b.regrid_from(a)
        got = b.state_to_host()
        for g, r_ in zip(got, ref):
            assert (g is None) == (r_ is None)
        keep = [i for i in range(5) if ref[i] is not None]
        scale = max(np.abs(ref[i]).max() for i in keep)
        for i in keep:
            assert np.abs(got[i] - ref[i]).max() <= 1e-13 * scale
            assert np.array_equal(got[i] == 0, ref[i] == 0)      # padded modes are exactly zero
        a2.regrid_from(a)                            # same resolution: the identity
        for g, s_ in zip(a2.state_to_host(), st):
            if s_ is not None:
                np.testing.assert_array_equal(g, s_)
        with pytest.raises(Exception, match="two contexts"):
            a.regrid_from(a)                         # in place: refused, the kernel would read rows it is overwriting
        for g, s_ in zip(a.state_to_host(), st):
            if s_ is not None:
                np.testing.assert_array_equal(g, s_)
        b.step(cb["dt"])
        nxt = b.state_to_host()
    check_parity(nxt[:nfb], ob.step(ref, cb["dt"])[:nfb], TOL_STEP, cb["K"], "one step after the regrid")


@pytest.mark.parametrize("ci,N_r,M,K", [(2, 12, 128, 128), (0, 14, 8, 8), (3, 11, 256, 8)])
def test_nonlinear_window_shorter_than_the_stencil_at_either_wall(torch_cuda, ci, N_r, M, K):
    """nsc_set_window with one or two levels at j0 = 0 and at the outer wall: the nine-point stencil there is
    one-sided (s0 = clamp(j - 4, 0, N_r - 9)), so the window reads nine levels, not its own plus four.  Before every
    windowed evaluation the work arrays are filled by an evaluation of another state, so a level the windowed
    pass forgets to transform shows up as a wrong result.  (2, 12, 128, 128) runs the single-chunk warp kernels
    (D1 applied inside the work array), (0, 14, 8, 8) the generic ones, (3, 11, 256, 8) a mix."""
    torch = torch_cuda
    cfg = synth.scaled_config(ci, N_r=N_r, M=M, K=K)
    nf = nf_of(cfg)
    n_modes = (M + 1) * (2 * K + 1)
    with _ctx(cfg) as ctx:
        st = synth.make_state(cfg, ctx.grid())
        rng = np.random.default_rng(cfg["seed"] + 5)
        other = [None if f is None else f + 0.5 * (rng.standard_normal(f.shape) + 1j * rng.standard_normal(f.shape))
                 for f in st]
        ctx.set_state(*_dev(torch, st))
        full = ctx.nonlinear_to_host()
        for j0, nj in [(0, 1), (N_r - 1, 1), (0, 2), (N_r - 2, 2), (3, 1), (N_r - 5, 1), (N_r // 2, 1), (2, 4)]:
            ctx.set_window()
            ctx.set_state(*_dev(torch, other))
            ctx.nonlinear_to_host()                      # the work arrays now hold the other state's lines
            ctx.set_state(*_dev(torch, st))
            ctx.set_window(j0, nj, 0, n_modes)
            bufs = [torch.full(ctx.shape, float("nan"), dtype=torch.complex128, device="cuda") for _ in range(nf)]
            ctx.nonlinear(*bufs)
            torch.cuda.synchronize()
            for i in range(nf):
                g = bufs[i].cpu().numpy()
                np.testing.assert_array_equal(g[j0:j0 + nj], full[i][j0:j0 + nj], err_msg=f"window ({j0}, {nj}), field {i}")
                assert np.isnan(g[:j0]).all() and np.isnan(g[j0 + nj:]).all(), "levels outside the window were written"


@pytest.mark.parametrize("ci,N_r,M,K,world", [(0, 24, 8, 8, 3), (2, 16, 4, 16, 2), (3, 16, 256, 8, 2), (2, 12, 128, 128, 2),
                                              (0, 16, 8, 8, 4), (2, 12, 128, 128, 3)])
def test_slab_decomposed_step_equals_the_single_context_step(torch_cuda, ci, N_r, M, K, world):
    """NEXT-2 on one GPU: `world` contexts play the ranks of a slab-decomposed run (paper_1908_00587_b200.slabs.
    SlabStepper: windowed phases of the step), the exchanges between them are done here by slicing (their
    torch.distributed form is tested over gloo in tests/test_slabs_gloo.py).  Every mode of the assembled result
    equals the plain nsc_step of one context bit for bit: levels and modes are independent."""
    from paper_1908_00587_b200.slabs import SlabPlan, SlabStepper
    torch = torch_cuda
    cfg = synth.scaled_config(ci, N_r=N_r, M=M, K=K)
    nf = nf_of(cfg)
    dt = cfg["dt"]
    n_modes = (M + 1) * (2 * K + 1)
    plan = SlabPlan(N_r=N_r, n_modes=n_modes, world=world)
    nsteps = 3
    with _ctx(cfg) as one:
        st = synth.make_state(cfg, one.grid())
        one.set_state(*_dev(torch, st))
        for _ in range(nsteps):
            one.step(dt)
        ref = one.state_to_host()
    ranks = [_ctx(cfg) for _ in range(world)]
    try:
        steppers = []
        for r, c in enumerate(ranks):
            c.set_state(*_dev(torch, st))
            steppers.append(SlabStepper(c, plan, r))
        for _ in range(nsteps):
            for phase in range(4):
                for s in steppers:
                    s.run_phase(phase, dt)
                torch.cuda.synchronize()
                bufs = [s.written(phase) for s in steppers]
                for dst in range(world):
                    e0, e1 = plan.modes(dst)
                    h0, h1 = plan.levels_with_halo(dst)
                    for src in range(world):
                        if src == dst:
                            continue
                        p0, p1 = plan.modes(src)
                        j0, j1 = plan.levels(src)
                        for f in range(nf):
                            if phase in (0, 2):       # rows of src -> columns of dst
                                bufs[dst][f][j0:j1, e0:e1] = bufs[src][f][j0:j1, e0:e1]
                            else:                     # columns of src -> rows (+ halo) of dst
                                bufs[dst][f][h0:h1, p0:p1] = bufs[src][f][h0:h1, p0:p1]
                torch.cuda.synchronize()
        shape = ref[0].shape
        for r, c in enumerate(ranks):
            e0, e1 = plan.modes(r)
            got = c.state_to_host()
            for i in list(range(nf)) + [4]:
                a = got[i].reshape(N_r, -1)[:, e0:e1]
                b = ref[i].reshape(N_r, -1)[:, e0:e1]
                assert np.isfinite(a).all()
                np.testing.assert_array_equal(a, b)
        assert shape == (N_r, M + 1, 2 * K + 1)
        # a window can be lifted again
        ranks[0].set_window()
        with pytest.raises(Exception):
            ranks[0].set_window(0, N_r + 1, 0, 1)
    finally:
        for c in ranks:
            c.destroy()


def test_slab_stepper_with_one_rank_is_the_plain_step(torch_cuda):
    """SlabStepper.step (phases + in-place exchanges through paper_1908_00587_b200.slabs) with a single rank."""
    from paper_1908_00587_b200.slabs import SlabPlan, SlabStepper
    torch = torch_cuda
    cfg = synth.scaled_config(2, N_r=18, M=8, K=8)
    res = []
    for slab in (False, True):
        with _ctx(cfg) as ctx:
            ctx.set_stream(torch.cuda.current_stream())
            st = synth.make_state(cfg, ctx.grid())
            ctx.set_state(*_dev(torch, st))
            stepper = SlabStepper(ctx, SlabPlan(N_r=18, n_modes=9 * 17, world=1), 0) if slab else None
            for _ in range(2):
                stepper.step(cfg["dt"]) if slab else ctx.step(cfg["dt"])
            res.append(ctx.state_to_host())
    for a, b in zip(*res):
        if a is not None:
            np.testing.assert_array_equal(a, b)


def test_double_buffered_host_transfers_equal_the_synchronous_ones(torch_cuda):
    """nsc_set_state_host_async + nsc_get_state_host_async + nsc_host_copies_wait: three rounds of (state in from the host, step, state out) with
    the read-out of round k overlapping round k + 1; every round's host buffers hold what the synchronous call gives."""
    torch = torch_cuda
    cfg = synth.scaled_config(2, N_r=20, M=16, K=16)
    with _ctx(cfg) as ctx:
        states = []
        for seed in range(3):
            st = synth.make_state(dict(cfg, seed=cfg["seed"] + seed), ctx.grid())
            states.append(st)
        sync_out, async_out = [], []
        for st in states:
            ctx.set_state(*st)
            ctx.step(cfg["dt"])
            sync_out.append(ctx.state_to_host())
        pinned = [[torch.empty(st[0].shape, dtype=torch.complex128, pin_memory=True).numpy() for _ in range(5)] for _ in states]
        pin_in = []
        for st in states:
            row = []
            for a in st:
                if a is None:
                    row.append(None)
                else:
                    t = torch.empty(a.shape, dtype=torch.complex128, pin_memory=True).numpy()
                    t[...] = a
                    row.append(t)
            pin_in.append(row)
        for k, (st, out) in enumerate(zip(pin_in, pinned)):
            if k % 2 == 0:
                ctx.set_state_host_async(*st)       # read-in through the staging set
            else:
                ctx.set_state(*st)                  # ... mixed with the synchronous call
            ctx.step(cfg["dt"])
            ctx.get_state_host_async(*out)
        ctx.host_copies_wait()
        for ref, out in zip(sync_out, pinned):
            for a, b in zip(ref, out):
                np.testing.assert_array_equal(a, b)
    # a temperature buffer handed to a context without temperature would stay unwritten: refused, not skipped
    cold = synth.scaled_config(0, N_r=12, M=4, K=4)
    with _ctx(cold) as ctx:
        st = synth.make_state(cold, ctx.grid())
        ctx.set_state(*st)
        bufs = [np.full(st[0].shape, 7.0 + 0j) for _ in range(5)]
        with pytest.raises(Exception, match="temperature"):
            ctx.get_state_host_async(*bufs)
        ctx.get_state_host_async(bufs[0], bufs[1], bufs[2], None, bufs[4])
        ctx.host_copies_wait()
        for i in (0, 1, 2, 4):
            np.testing.assert_array_equal(bufs[i], st[i])
        assert (bufs[3] == 7.0).all()


def test_measured_fp64_peaks_are_sane_and_leave_the_current_device_alone(torch_cuda):
    """nsc_fp64_peak (bench.py's roofline denominators): a positive finite rate below the nominal 148 SM x 64 lanes
    x 2 flop x 2.1 GHz = 40 TFLOP/s, add/mul at about half the FMA rate, bad ordinals refused, and the calling
    thread's current device unchanged."""
    import ctypes as C
    torch = torch_cuda
    from paper_1908_00587_b200 import nsc
    before = torch.cuda.current_device()
    fma, addmul = nsc.fp64_peak(0, 0), nsc.fp64_peak(1, -1)
    assert torch.cuda.current_device() == before
    assert np.isfinite(fma) and 10.0 < fma < 40.0, fma
    assert np.isfinite(addmul) and 0.4 * fma < addmul < 0.6 * fma, (fma, addmul)
    lib, v = nsc.load_library(), C.c_double(-1.0)
    assert lib.nsc_fp64_peak(0, torch.cuda.device_count(), C.byref(v)) == nsc.NSC_EINVAL
    assert lib.nsc_fp64_peak(2, 0, C.byref(v)) == nsc.NSC_EINVAL and v.value == -1.0
