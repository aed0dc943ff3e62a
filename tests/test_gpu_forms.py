"""GPU parity for the SURVEY.md 8(f) rows built after the hot path: the rotational form omega x u (row f1,
dns_plan_set_form), the ensemble-coupled streamwise-mean flow (row f2, dns_plan_set_coupling / dns_plan_set_exchange,
PAPER.md:286-292) and dns_add_increment, element by element against the oracle with the same switches, through the C ABI.
Tolerances as in test_gpu_parity.py (BASELINE.json: 1e-10 after 1 step, 1e-8 after 20).  Run with `pytest -m gpu`.
"""
import numpy as np
import pytest

from oracle.dns_oracle import ROTATIONAL, STREAMWISE_MEAN, Oracle
from paper_2306_12739_b200 import binding, inputs
from test_gpu_parity import PI, TOL_1, TOL_20, assert_errs, field_err, lane_cover, run_pair

pytestmark = pytest.mark.gpu
ROT, COUPLED = binding.DNS_FORM_ROTATIONAL, binding.DNS_COUPLING_STREAMWISE_MEAN
assert (ROT, COUPLED) == (ROTATIONAL, STREAMWISE_MEAN)


# ------------------------------------------------------------------------------------------------ f1: rotational form
def test_rotational_config1_all_members_1_and_20_steps():
    cfg = inputs.CONFIGS[1]
    errs, _, _ = run_pair(cfg, range(cfg.E), 20, check_at=(1, 20), form=ROT)
    assert_errs(errs, 1, TOL_1)
    assert_errs(errs, 20, TOL_20)


@pytest.mark.parametrize("cid,m1,m20", [(2, None, [0, 37, 63]), (3, [0, 7, 15], [15]), (4, None, [3, 255])])
def test_rotational_full_size_configs(cid, m1, m20):
    cfg = inputs.CONFIGS[cid]
    errs, _, _ = run_pair(cfg, lane_cover(cfg.E) if m1 is None else m1, 1, form=ROT)
    assert_errs(errs, 1, TOL_1)
    errs, _, _ = run_pair(cfg, m20, 20, check_at=(20,), form=ROT)
    assert_errs(errs, 20, TOL_20)


@pytest.mark.parametrize("cid,members", [(3, [4]), (4, [17, 250])])
def test_rotational_broadband_state_at_full_size(cid, members):
    cfg = inputs.CONFIGS[cid]
    errs, _, _ = run_pair(cfg, members, 1, state=inputs.make_broadband_state(cfg), form=ROT)
    assert_errs(errs, 1, TOL_1)
    assert errs[1]["v_mode"] < 1e-9 and errs[1]["eta_mode"] < 1e-9, errs[1]


@pytest.mark.parametrize("Nx,Nz,E", [(12, 16, 3), (16, 12, 3), (18, 24, 5), (24, 18, 3), (32, 36, 17), (36, 32, 9),
                                     (48, 54, 3), (54, 48, 17), (64, 72, 3), (72, 64, 3), (16, 48, 17), (16, 64, 17)])
def test_rotational_every_transform_length(Nx, Nz, E):
    """Every padded length as x and as z length in the rotational kernels (6-field ring of the line kernel, 6-field z
    inverse in the register and the shared-memory family), member tiles of 4, 8 and 16 lanes with a ragged last tile."""
    cfg = inputs.Config(1, inputs.COUETTE, 350.0, 1.9 * PI, 1.1 * PI, Nx, 13, Nz, E, 0.01, 1, 0.1, 0, box=3)
    errs, _, _ = run_pair(cfg, sorted({0, E // 2, E - 1}), 2, check_at=(1, 2), form=ROT)
    assert_errs(errs, 1, TOL_1)
    assert_errs(errs, 2, TOL_1 * 10)


@pytest.mark.parametrize("E,Ny,flow", [(1, 17, 0), (5, 20, 1), (7, 5, 1), (2, 66, 1), (3, 129, 0)])
def test_rotational_odd_even_ny_both_flows(E, Ny, flow):
    cfg = inputs.Config(3 if flow else 1, flow, 500.0, 2 * PI, PI, 16, Ny, 12, E, 0.01, 1, 0.1, 0, box=2)
    errs, _, _ = run_pair(cfg, range(E), 3, check_at=(1, 3), form=ROT)
    assert_errs(errs, 1, TOL_1)
    assert_errs(errs, 3, TOL_1 * 10)


def test_rotational_stage_pieces_against_oracle():
    """Per-kernel parity through the debug hook: omega_z, omega_x of the reconstruction kernel, the spectral H = omega x u
    and F^0, G^0 of the first stage, the stage-1 eta written for the next transform."""
    cfg = inputs.CONFIGS[2].with_E(5)
    st = inputs.make_state(cfg)
    plan = binding.Plan(*inputs.plan_args(cfg), form=ROT)
    plan.set_state(st["vhat"], st["etahat"], st["U00"], st["W00"])
    o = Oracle(*inputs.plan_args(cfg), form=ROTATIONAL)
    o.set_state(st["vhat"], st["etahat"], st["U00"], st["W00"])
    u, v, w, Du, Dv, Dw = o.velocities(o.v, o.eta, o.U, o.W)
    ikx, ikz = 1j * o.kx[None, :, None, None], 1j * o.kz[None, None, :, None]
    for which, ref in ((0, u), (1, w), (2, ikx * v - Du), (3, Dw - ikz * v)):
        assert field_err(plan.debug_fetch(which)[..., 1:-1], ref[..., 1:-1]) < 1e-12, which
    F, G, Su, Sw = o.nonlinear(o.v, o.eta, o.U, o.W)
    plan.debug_stage(0)
    assert field_err(plan.debug_fetch(5)[..., 1:-1], F) < 1e-11
    assert field_err(plan.debug_fetch(6)[..., 1:-1], G) < 1e-11
    s1 = o.stage(o.v, o.eta, o.U, o.W, 0.5, F, G, Su, Sw)
    assert field_err(plan.debug_fetch(10), s1[1]) < 1e-12
    assert field_err(plan.debug_fetch(8), s1[2]) < 1e-12
    plan.close()


def test_rotational_laminar_fixed_points_and_switch_errors():
    for cid, prof in ((2, lambda y: y), (3, lambda y: 1.5 * (1 - y * y))):
        cfg = inputs.CONFIGS[cid].with_E(6)
        plan = binding.Plan(*inputs.plan_args(cfg), form=ROT)
        st = inputs.make_state(cfg)
        plan.set_state(0 * st["vhat"], 0 * st["etahat"], st["U00"], st["W00"])
        plan.step(5)
        v, eta, U, W = plan.get_state()
        assert np.abs(U - prof(inputs.grid_y(cfg.Ny))).max() < 1e-13
        assert np.abs(v).max() < 1e-15 and np.abs(eta).max() < 1e-15      # H_y = -U dU/dy leaks at FFT round-off only
        assert binding.dns_plan_set_form(plan.h, 0) == binding.DNS_ESTATE    # a state is set
        assert binding.dns_plan_set_coupling(plan.h, 1, cfg.E) == binding.DNS_ESTATE
        plan.close()
    st_, h = binding.dns_plan_create(*inputs.plan_args(inputs.CONFIGS[1]))
    assert binding.dns_plan_set_form(h, 7) == binding.DNS_EINVAL
    assert binding.dns_plan_set_coupling(h, 1, 1) == binding.DNS_EINVAL     # E_total < E
    assert binding.dns_plan_set_coupling(h, 3, 2) == binding.DNS_EINVAL
    assert binding.dns_plan_set_form(h, ROT) == binding.DNS_OK
    binding.dns_plan_destroy(h)


# ------------------------------------------------------------------------------------------------ f2: coupled ensemble
@pytest.mark.parametrize("form", [0, ROT])
@pytest.mark.parametrize("cid,E", [(1, 5), (2, 21), (3, 4)])
def test_coupled_ensemble_against_oracle(cid, E, form):
    """All members through the oracle (the coupling is a sum over ALL members), 1 and 5 steps."""
    cfg = inputs.CONFIGS[cid].with_E(E)
    errs, _, _ = run_pair(cfg, range(E), 5, check_at=(1, 5), form=form, coupling=COUPLED, share_mean=True)
    assert_errs(errs, 1, TOL_1)
    assert_errs(errs, 5, TOL_1 * 10)


def test_coupled_ensemble_shares_its_streamwise_mean_and_is_deterministic():
    cfg = inputs.CONFIGS[2].with_E(40)
    st = inputs.make_state(cfg)
    v0, e0, U0, W0 = st["vhat"].copy(), st["etahat"].copy(), st["U00"].copy(), st["W00"].copy()
    v0[:, 0], e0[:, 0] = v0[0, 0], e0[0, 0]
    outs = []
    for rep in range(2):
        plan = binding.Plan(*inputs.plan_args(cfg), coupling=COUPLED)
        plan.set_state(v0, e0, U0, W0)
        plan.step(6)
        outs.append(plan.get_state())
        assert plan.launches_per_step() == 18
        plan.close()
    v, eta, U, W = outs[0]
    for f in (v[:, 0], eta[:, 0], U, W):                      # a common streamwise-mean flow
        assert np.array_equal(f, np.broadcast_to(f[0], f.shape))
    assert np.abs(v[:, 1:] - v[0, 1:][None]).max() > 1e-4     # distinct perturbations
    for a, b in zip(*outs):
        assert np.array_equal(a, b)


def test_coupled_exchange_callback_matches_single_launch():
    """The exchange path (sums -> callback -> apply, direct launches) with an identity 'all-reduce' equals the fused
    one-GPU path bit for bit; with a callback that doubles the buffer and E_total = 2 E it does so again (two ranks
    holding the same members); a failing callback surfaces as DNS_ECUDA."""
    import torch
    cfg = inputs.CONFIGS[2].with_E(12)
    st = inputs.make_state(cfg)
    res, calls = [], []
    for mode in ("fused", "identity", "double"):
        kw = {}
        if mode == "identity":
            kw = dict(allreduce=lambda t: calls.append(t.numel()))
        if mode == "double":
            kw = dict(allreduce=lambda t: t.mul_(2.0), E_total=2 * cfg.E)
        plan = binding.Plan(*inputs.plan_args(cfg), coupling=COUPLED, **kw)
        plan.set_state(st["vhat"], st["etahat"], st["U00"], st["W00"])
        plan.step(2)
        res.append(plan.get_state())
        if mode != "fused":
            assert plan.launches_per_step() == 21
        plan.close()
    assert len(calls) == 6 and calls[0] == 2 * (3 * cfg.Ny * (cfg.Nz - 1) + cfg.Ny * (3 * cfg.Nz // 2))
    for r in res[1:]:
        for a, b in zip(res[0], r):
            assert np.array_equal(a, b)

    def boom(t):
        raise RuntimeError("exchange failed")
    plan = binding.Plan(*inputs.plan_args(cfg), coupling=COUPLED, allreduce=boom)
    plan.set_state(st["vhat"], st["etahat"], st["U00"], st["W00"])
    with pytest.raises(binding.DnsError):
        plan.step(1)
    plan.close()
    torch.cuda.synchronize()


def test_add_increment_against_oracle():
    """dns_add_increment (stochastic-forcing realisations are the caller's): state += increment with the set_state
    normalisation, time and flux target kept; then two more steps."""
    cfg = inputs.CONFIGS[3].with_E(3)
    cfg = inputs.Config(**{**cfg.__dict__, "Nx": 16, "Nz": 16, "Ny": 33})
    st = inputs.make_state(cfg)
    rng = np.random.default_rng(11)
    shape = st["vhat"].shape
    dv = 1e-3 * (rng.standard_normal(shape) + 1j * rng.standard_normal(shape))
    de = 1e-3 * (rng.standard_normal(shape) + 1j * rng.standard_normal(shape))
    plan = binding.Plan(*inputs.plan_args(cfg))
    o = Oracle(*inputs.plan_args(cfg))
    for x in (plan, o):
        x.set_state(st["vhat"], st["etahat"], st["U00"], st["W00"])
        x.step(1)
        x.add_increment(dv, de)
    gv, ge, gU, gW = plan.get_state()
    assert field_err(gv, o.v) < TOL_1 and field_err(ge, o.eta) < TOL_1
    assert np.all(gv[..., 0] == 0) and np.all(gv[:, 0, 0] == 0)
    plan.step(2)
    o.step(2)
    gv, ge, gU, gW = plan.get_state()
    assert field_err(gv, o.v) < TOL_1 * 10 and field_err(ge, o.eta) < TOL_1 * 10 and field_err(gU, o.U) < TOL_1 * 10
    d = plan.diagnostics()
    assert np.abs(d[:, 5] - 3 * cfg.dt).max() < 1e-15 and np.abs(d[:, 3] - 1.0).max() < 1e-13
    plan.close()


def test_fp64_peak_microbenchmark_runs():
    got = {}
    for kind in (0, 1, 2):
        st, tf = binding.dns_debug_fp64_peak(kind, 0.05)
        assert st == binding.DNS_OK and 5.0 < tf < 80.0, (kind, tf)
        got[kind] = tf
    # DFMA and DMMA chains interleaved in one kernel do not add up: one fp64 pipe
    assert got[2] < 1.1 * max(got[0], got[1]), got
    assert binding.dns_debug_fp64_peak(3, 0.05)[0] == binding.DNS_EINVAL
    assert binding.dns_debug_set_option("no_such_option", 1) == binding.DNS_EINVAL


def test_shared_memory_z_kernels_both_forms():
    """Option "zreg" = 0 forces the shared-memory z transforms for lengths the register kernels normally take."""
    assert binding.dns_debug_set_option("zreg", 0) == binding.DNS_OK
    try:
        for form in (0, ROT):
            cfg = inputs.Config(1, inputs.COUETTE, 350.0, 1.9 * PI, 1.1 * PI, 16, 13, 32, 9, 0.01, 1, 0.1, 0, box=3)
            errs, _, _ = run_pair(cfg, [0, 8], 2, check_at=(1, 2), form=form)
            assert_errs(errs, 1, TOL_1)
    finally:
        binding.dns_debug_set_option("zreg", -1)


@pytest.mark.parametrize("Nx,Nz", [(36, 16), (48, 16), (16, 48)])
def test_line_kernel_round_variants(Nx, Nz):
    """Mx = 54 and 72 in the 16-lane family (ragged second member tile): the default line kernel runs two transforms per
    round with four exchange buffers (6-slot ring in the convective form); options "line_pair" = 0 / 1 / 5 select one
    transform per round, two exchange buffers, four buffers with a half ring; "pdl" = 1 adds programmatic dependent launch;
    "zinv_tp" = 0 takes the L2 prefetch out of the two-pass z inverse and, for Mz = 72 (third case), selects the one-pass
    z inverse instead of the two-pass one.
    Every variant against the oracle, and all variants bit-identical to each other (same arithmetic per line)."""
    cfg = inputs.Config(1, inputs.COUETTE, 350.0, 1.9 * PI, 1.1 * PI, Nx, 13, Nz, 17, 0.01, 1, 0.1, 0, box=3)
    st = inputs.make_state(cfg)
    idx = [0, 8, 15, 16]
    for form in (0, ROT):
        o = Oracle(*inputs.plan_args(cfg, E=len(idx)), form=form)
        o.set_state(st["vhat"][idx], st["etahat"][idx], st["U00"][idx], st["W00"][idx])
        o.step(2)
        ref = None
        for name, val in (("line_pair", -1), ("line_pair", 0), ("line_pair", 1), ("line_pair", 5), ("pdl", 1), ("zinv_tp", 0)):
            assert binding.dns_debug_set_option(name, val) == binding.DNS_OK
            try:
                plan = binding.Plan(*inputs.plan_args(cfg), form=form)
                plan.set_state(st["vhat"], st["etahat"], st["U00"], st["W00"])
                plan.step(2)
                got = plan.get_state()
                plan.close()
            finally:
                binding.dns_debug_set_option(name, -1)
            assert field_err(got[0][idx], o.v) < TOL_1 * 10 and field_err(got[1][idx], o.eta) < TOL_1 * 10, (name, val, form)
            assert field_err(got[2][idx], o.U) < TOL_1 * 10
            if ref is None:
                ref = got
            else:
                for a, b in zip(ref, got):
                    assert np.array_equal(a, b), (name, val, form)


def test_exchange_callback_runs_on_the_plans_stream():
    """include/dns.h orders the exchange on the plan's stream.  The plan is bound inside a side-stream block and stepped
    OUTSIDE it (torch's current stream is then the default one, as in bench.measure_e2e): the callback must still see the
    plan's stream as the current stream, so that an all-reduce enqueued there is ordered between the two halves of the
    coupled mean; the result equals the fused one-GPU path bit for bit."""
    import torch
    cfg = inputs.CONFIGS[2].with_E(12)
    st = inputs.make_state(cfg)
    ref = binding.Plan(*inputs.plan_args(cfg), coupling=COUPLED)
    ref.set_state(st["vhat"], st["etahat"], st["U00"], st["W00"])
    ref.step(3)
    want = ref.get_state()
    ref.close()

    side = torch.cuda.Stream()
    seen = []

    def allreduce(t):
        seen.append(torch.cuda.current_stream().cuda_stream)
        t.mul_(1.0)                                           # a device operation enqueued on the current stream

    with torch.cuda.stream(side):
        plan = binding.Plan(*inputs.plan_args(cfg), coupling=COUPLED, allreduce=allreduce)
        plan.set_state(st["vhat"], st["etahat"], st["U00"], st["W00"])
    assert torch.cuda.current_stream().cuda_stream != side.cuda_stream
    plan.step(3)
    got = plan.get_state()
    assert len(seen) == 9 and all(s == side.cuda_stream for s in seen), (seen, side.cuda_stream)
    for a, b in zip(want, got):
        assert np.array_equal(a, b)
    plan.close()
    torch.cuda.synchronize()
