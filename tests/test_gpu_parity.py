"""GPU parity: the CUDA library (through the C ABI binding) against the CPU oracle, element by element on the
same seeded inputs.  Tolerances are BASELINE.json's: relative 1e-10 in every spectral coefficient after 1 step,
1e-8 after 20 steps, where "relative" is the reading A14 of DESIGN.md: |a_gpu - a_or| <= tol * s, s = the
max-modulus of that field of that member.  At the full BASELINE sizes the GPU advances every member and the oracle
a fixed subset (members are independent, pin P12).  Run with `pytest -m gpu` on a B200.
"""
import numpy as np
import pytest

from oracle.dns_oracle import Oracle
from paper_2306_12739_b200 import binding, inputs

pytestmark = pytest.mark.gpu
TOL_1, TOL_20 = 1e-10, 1e-8
PI = np.pi


def field_err(a, b):
    """max over members of  max|a-b| / max|b|  (per member, per field)."""
    E = b.shape[0]
    num = np.abs(a - b).reshape(E, -1).max(axis=1)
    den = np.abs(b).reshape(E, -1).max(axis=1)
    den = np.where(den == 0, 1.0, den)
    return float((num / den).max())


def mode_err(a, b, floor=1e-6):
    """Largest per-(n,m) relative error: max_y |a - b| / max_y |b| over the modes whose oracle modulus exceeds `floor`
    of that member's field maximum (a check that small, high-wavenumber coefficients are right in relative terms)."""
    num = np.abs(a - b).max(axis=-1)
    den = np.abs(b).max(axis=-1)
    big = den > floor * den.reshape(den.shape[0], -1).max(axis=1)[:, None, None]
    return float((num[big] / den[big]).max()) if big.any() else 0.0


def run_pair(cfg, members, steps, check_at=(1,), tol=None, zero_pert=False, form=0, coupling=0, state=None, share_mean=False):
    """GPU on all cfg.E members, oracle on `members`; returns the errors at the requested step counts."""
    plan = binding.Plan(*inputs.plan_args(cfg), form=form, coupling=coupling)
    full = state if state is not None else inputs.make_state(cfg)
    s = 0.0 if zero_pert else 1.0
    v0, e0, U0, W0 = s * full["vhat"], s * full["etahat"], full["U00"].copy(), full["W00"].copy()
    if share_mean:                                  # coupled ensembles: every member starts from member 0's kx = 0 part
        v0[:, 0], e0[:, 0], U0[:], W0[:] = v0[0, 0], e0[0, 0], U0[0], W0[0]
    plan.set_state(v0, e0, U0, W0)
    o = Oracle(*inputs.plan_args(cfg, E=len(members)), form=form, coupling=coupling)
    idx = list(members)
    o.set_state(v0[idx], e0[idx], U0[idx], W0[idx])
    out = {}
    done = 0
    for n in sorted(check_at):
        plan.step(n - done)
        o.step(n - done)
        done = n
        v, eta, U, W = plan.get_state()
        dg, do = plan.diagnostics()[idx], o.diagnostics()
        out[n] = dict(v=field_err(v[idx], o.v), eta=field_err(eta[idx], o.eta), U=field_err(U[idx], o.U),
                      W=float(np.abs(W[idx] - o.W).max() / max(np.abs(o.U).max(), 1e-300)),
                      diag=float(np.abs(dg - do).max()),
                      v_mode=mode_err(v[idx], o.v), eta_mode=mode_err(eta[idx], o.eta))
    plan.close()
    return out, plan, o


def assert_errs(errs, n, tol):
    e = errs[n]
    assert e["v"] < tol and e["eta"] < tol and e["U"] < tol and e["W"] < tol, (n, e)
    assert e["diag"] < 100 * tol, (n, e)


# ------------------------------------------------------------------------------------------------ BASELINE configs
def test_config1_all_members_1_and_20_steps():
    cfg = inputs.CONFIGS[1]
    errs, _, _ = run_pair(cfg, range(cfg.E), 20, check_at=(1, 20))
    assert_errs(errs, 1, TOL_1)
    assert_errs(errs, 20, TOL_20)


def lane_cover(E, T=16):
    """16 members that sit on every lane position of a T-lane member tile, spread over the tiles, and include the
    last member (the ragged or last tile)."""
    ntile = (E + T - 1) // T
    m = sorted({min(E - 1, ((k * 7) % ntile) * T + k) for k in range(T)} | {E - 1})
    return m


def test_config2_all_members_1_step_and_16_members_20_steps():
    cfg = inputs.CONFIGS[2]                       # E = 64
    errs, _, _ = run_pair(cfg, range(cfg.E), 1)
    assert_errs(errs, 1, TOL_1)
    errs, _, _ = run_pair(cfg, lane_cover(cfg.E)[::2], 20, check_at=(20,))
    assert_errs(errs, 20, TOL_20)


def test_config3_all_members_1_step_and_sampled_20_steps():
    cfg = inputs.CONFIGS[3]                       # Poiseuille, constant mass flux, 64 x 97 x 64, E = 16
    errs, _, _ = run_pair(cfg, range(cfg.E), 1)
    assert_errs(errs, 1, TOL_1)
    errs, _, _ = run_pair(cfg, [2, 15], 20, check_at=(20,))
    assert_errs(errs, 20, TOL_20)


def test_config4_lane_covering_members_1_step_and_sampled_20_steps():
    cfg = inputs.CONFIGS[4]                       # E = 256, per-member amplitudes: the configuration bench.py times
    errs, _, _ = run_pair(cfg, lane_cover(cfg.E), 1)
    assert_errs(errs, 1, TOL_1)
    errs, _, _ = run_pair(cfg, [3, 77, 200, 255], 20, check_at=(20,))
    assert_errs(errs, 20, TOL_20)


@pytest.mark.parametrize("E", inputs.SWEEP_E)
def test_config5_sweep_one_step(E):
    cfg = inputs.CONFIGS[5].with_E(E)
    members = lane_cover(E) if E >= 16 else range(E)
    errs, _, _ = run_pair(cfg, members, 1)
    assert_errs(errs, 1, TOL_1)


@pytest.mark.parametrize("cid,members", [(3, [0, 9]), (4, [5, 100, 255])])
def test_broadband_state_at_full_size(cid, members):
    """Every retained (n,m) energised (amplitude ~ (1 + n^2 + m^2)^(-5/6)) with rough wall-normal profiles (Chebyshev
    coefficients up to degree Ny - 5 under the no-slip envelopes): high-kx / high-kz handling and the full y resolution
    are exercised at the BASELINE sizes.  Besides the A14 metric every mode above 1e-6 of the field maximum must be
    right to 1e-9 RELATIVE to its own modulus."""
    cfg = inputs.CONFIGS[cid]
    st = inputs.make_broadband_state(cfg)
    errs, _, _ = run_pair(cfg, members, 1, state=st)
    assert_errs(errs, 1, TOL_1)
    assert errs[1]["v_mode"] < 1e-9 and errs[1]["eta_mode"] < 1e-9, errs[1]


# ------------------------------------------------------------------------------------------------ edge cases
@pytest.mark.parametrize("Nx,Nz", [(12, 16), (16, 12), (18, 24), (24, 18), (32, 36), (36, 32), (48, 54), (54, 48),
                                   (64, 72), (72, 64)])
def test_every_transform_length_both_directions(Nx, Nz):
    """All 3N/2 = 2^a 3^b lengths in 16..128 (18..108), as x and as z length; ragged member tile E = 3."""
    cfg = inputs.Config(1, inputs.COUETTE, 350.0, 1.9 * PI, 1.1 * PI, Nx, 13, Nz, 3, 0.01, 1, 0.1, 0, box=3)
    errs, _, _ = run_pair(cfg, range(3), 2, check_at=(1, 2))
    assert_errs(errs, 1, TOL_1)
    assert_errs(errs, 2, TOL_1 * 10)


@pytest.mark.parametrize("Nx", [12, 16, 18, 24, 36, 54, 72])
def test_sixteen_lane_line_kernel_for_every_x_length(Nx):
    """Every padded x length with an ensemble large enough for the 16-lane member tiles (E = 17: one full tile and a
    ragged one); oracle on the first and the last member."""
    cfg = inputs.Config(1, inputs.COUETTE, 350.0, 1.9 * PI, 1.1 * PI, Nx, 13, 16, 17, 0.01, 1, 0.1, 0, box=3)
    errs, _, _ = run_pair(cfg, [0, 16], 2, check_at=(1, 2))
    assert_errs(errs, 1, TOL_1)
    assert_errs(errs, 2, TOL_1 * 10)


@pytest.mark.parametrize("Nz", [12, 16, 18, 24, 32, 36, 48, 54, 64, 72])
def test_every_z_length_with_sixteen_member_tiles(Nz):
    """Every padded z length (register z transforms for Mz = 24, 36, 48, 72, 96, shared-memory ones otherwise) against
    the 16-member tiles of the mixed layout, ragged last tile (E = 17)."""
    cfg = inputs.Config(1, inputs.COUETTE, 350.0, 1.9 * PI, 1.1 * PI, 16, 13, Nz, 17, 0.01, 1, 0.1, 0, box=3)
    errs, _, _ = run_pair(cfg, [0, 16], 2, check_at=(1, 2))
    assert_errs(errs, 1, TOL_1)
    assert_errs(errs, 2, TOL_1 * 10)


@pytest.mark.parametrize("Nx,Nz,E", [(48, 32, 17), (32, 48, 9), (32, 32, 21), (64, 16, 19)])
def test_ragged_member_tiles_of_the_wide_layouts(Nx, Nz, E):
    """Member tiles of 8 and 16 lanes (line kernel, mixed layout) and the two-thread register z transforms with a
    ragged last tile / a lane count that is not a multiple of the block; oracle on first, middle and last member."""
    cfg = inputs.Config(1, inputs.COUETTE, 350.0, 1.9 * PI, 1.1 * PI, Nx, 13, Nz, E, 0.01, 1, 0.1, 0, box=3)
    members = sorted({0, E // 2, E - 1})
    errs, _, _ = run_pair(cfg, members, 2, check_at=(1, 2))
    assert_errs(errs, 1, TOL_1)
    assert_errs(errs, 2, TOL_1 * 10)


@pytest.mark.parametrize("E,Ny,flow", [(1, 17, 0), (5, 20, 1), (33, 12, 0), (7, 5, 1), (2, 66, 1), (6, 75, 0),
                                       (3, 129, 0), (2, 257, 1)])       # 257 = the largest Ny dns_plan_create accepts
def test_ragged_members_and_odd_even_ny(E, Ny, flow):
    cfg = inputs.Config(3 if flow else 1, flow, 500.0, 2 * PI, PI, 16, Ny, 12, E, 0.01, 1, 0.1, 0, box=2)
    errs, _, _ = run_pair(cfg, range(E), 3, check_at=(1, 3))
    assert_errs(errs, 1, TOL_1)
    assert_errs(errs, 3, TOL_1 * 10)


def test_laminar_fixed_points_on_gpu_at_full_size():
    for cid, prof in ((2, lambda y: y), (3, lambda y: 1.5 * (1 - y * y))):
        cfg = inputs.CONFIGS[cid]
        plan = binding.Plan(*inputs.plan_args(cfg))
        st = inputs.make_state(cfg)
        plan.set_state(0 * st["vhat"], 0 * st["etahat"], st["U00"], st["W00"])
        plan.step(5)
        v, eta, U, W = plan.get_state()
        y = inputs.grid_y(cfg.Ny)
        assert np.abs(U - prof(y)).max() < 1e-13 and np.abs(v).max() == 0 and np.abs(eta).max() == 0
        d = plan.diagnostics()
        if cid == 3:
            assert np.abs(d[:, 4] - 3.0 / cfg.Re).max() < 1e-15 * cfg.Re     # gamma = 2c/Re, c = 1.5
            assert np.abs(d[:, 3] - 1.0).max() < 1e-13
        plan.close()


def test_flux_conservation_and_noslip_at_full_size():
    cfg = inputs.CONFIGS[3]
    plan = binding.Plan(*inputs.plan_args(cfg))
    st = inputs.make_state(cfg)
    plan.set_state(st["vhat"], st["etahat"], st["U00"], st["W00"])
    q0 = plan.diagnostics()[:, 3]
    plan.step(10)
    d = plan.diagnostics()
    assert np.abs(d[:, 3] - q0).max() < 1e-13                                 # pin P5 on the GPU
    v, eta, U, W = plan.get_state()
    assert np.all(v[..., 0] == 0) and np.all(v[..., -1] == 0) and np.all(eta[..., 0] == 0)
    assert np.all(v[:, 0, 0] == 0) and np.all(eta[:, 0, 0] == 0)
    assert np.all(U[:, 0] == 0) and np.all(U[:, -1] == 0) and np.all(W[:, 0] == 0)
    assert np.all(np.isfinite(d))
    plan.close()


def test_member_independence_bitwise():
    """P12 on the GPU: a member's result does not depend on E or on the other members."""
    cfg5 = inputs.CONFIGS[1].with_E(5)
    full = inputs.make_state(cfg5)
    plan = binding.Plan(*inputs.plan_args(cfg5))
    plan.set_state(full["vhat"], full["etahat"], full["U00"], full["W00"])
    plan.step(3)
    v5, e5, U5, W5 = plan.get_state()
    plan.close()
    idx = [4, 1]
    plan2 = binding.Plan(*inputs.plan_args(cfg5, E=2))
    plan2.set_state(full["vhat"][idx], full["etahat"][idx], full["U00"][idx], full["W00"][idx])
    plan2.step(3)
    v2, e2, U2, W2 = plan2.get_state()
    plan2.close()
    assert np.array_equal(v2, v5[idx]) and np.array_equal(e2, e5[idx]) and np.array_equal(U2, U5[idx])


def test_step_n_equals_n_steps_and_is_deterministic():
    cfg = inputs.CONFIGS[1]
    st = inputs.make_state(cfg)
    res = []
    for chunks in ((4,), (1, 1, 2), (4,)):
        plan = binding.Plan(*inputs.plan_args(cfg))
        plan.set_state(st["vhat"], st["etahat"], st["U00"], st["W00"])
        for c in chunks:
            plan.step(c)
        res.append(plan.get_state())
        assert plan.diagnostics()[0, 5] == pytest.approx(4 * cfg.dt)
        plan.close()
    for r in res[1:]:
        for a, b in zip(r, res[0]):
            assert np.array_equal(a, b)


def test_graph_replay_equals_direct_launches_bitwise():
    """dns_step replays a CUDA graph of one time step; option "graph" = 0 and dns_step_profile launch the same kernels directly.
    All three must give bit-identical states (same kernels, same order, the mean-flow kernel joined before its readers)."""
    cfg = inputs.CONFIGS[2].with_E(9)
    st = inputs.make_state(cfg)
    outs = []
    for mode in ("graph", "direct", "profile"):
        assert binding.dns_debug_set_option("graph", 0 if mode == "direct" else -1) == binding.DNS_OK
        try:
            plan = binding.Plan(*inputs.plan_args(cfg))
            plan.set_state(st["vhat"], st["etahat"], st["U00"], st["W00"])
            if mode == "profile":
                plan.step_profile(4)
            else:
                plan.step(3)
                plan.step(1)
            outs.append(plan.get_state())
            plan.close()
        finally:
            binding.dns_debug_set_option("graph", -1)
    for o in outs[1:]:
        for a, b in zip(outs[0], o):
            assert np.array_equal(a, b)


def test_set_state_normalisation_matches_oracle():
    cfg = inputs.CONFIGS[1]
    st = inputs.make_state(cfg)
    rng = np.random.default_rng(7)
    v = st["vhat"] + 0.01 * (rng.standard_normal(st["vhat"].shape) + 1j * rng.standard_normal(st["vhat"].shape))
    eta = st["etahat"] + 0.01 * rng.standard_normal(st["vhat"].shape)
    U = st["U00"] + 0.3
    W = st["W00"] + 0.1
    plan = binding.Plan(*inputs.plan_args(cfg))
    plan.set_state(v, eta, U, W)
    o = Oracle(*inputs.plan_args(cfg))
    o.set_state(v, eta, U, W)
    gv, ge, gU, gW = plan.get_state()
    assert np.array_equal(gv, o.v) and np.array_equal(ge, o.eta) and np.array_equal(gU, o.U) and np.array_equal(gW, o.W)
    plan.step(1)
    o.step(1)
    gv, ge, gU, gW = plan.get_state()
    assert field_err(gv, o.v) < TOL_1 and field_err(ge, o.eta) < TOL_1 and field_err(gU, o.U) < TOL_1
    plan.close()


def test_device_pointer_io():
    import torch
    cfg = inputs.CONFIGS[1]
    st = inputs.make_state(cfg)
    plan = binding.Plan(*inputs.plan_args(cfg))
    dev = [torch.from_numpy(np.ascontiguousarray(st[k])).cuda() for k in ("vhat", "etahat", "U00", "W00")]
    plan.set_state(*dev)
    plan.step(2)
    outs = [torch.empty_like(t) for t in dev]
    plan.get_state(outs)
    plan2 = binding.Plan(*inputs.plan_args(cfg))
    plan2.set_state(st["vhat"], st["etahat"], st["U00"], st["W00"])
    plan2.step(2)
    host = plan2.get_state()
    for a, b in zip(outs, host):
        assert np.array_equal(a.cpu().numpy(), b)
    plan.close()
    plan2.close()


def test_error_paths_on_device():
    cfg = inputs.CONFIGS[1]
    st, h = binding.dns_plan_create(*inputs.plan_args(cfg))
    assert st == binding.DNS_OK
    assert binding.dns_step(h, 1) == binding.DNS_ESTATE                      # nothing bound
    import torch
    n = binding.dns_plan_workspace_bytes(h)
    assert n > 0
    small = torch.empty(1024, dtype=torch.uint8, device="cuda")
    assert binding.dns_plan_bind(h, small.data_ptr(), 1024) == binding.DNS_EINVAL
    ws = torch.empty(n + 256, dtype=torch.uint8, device="cuda")
    base = (ws.data_ptr() + 255) & ~255
    assert binding.dns_plan_bind(h, base + 8, n) == binding.DNS_EINVAL       # misaligned
    assert binding.dns_plan_bind(h, base, n) == binding.DNS_OK
    assert binding.dns_step(h, 1) == binding.DNS_ESTATE                      # no state yet
    assert binding.dns_step(h, -1) == binding.DNS_EINVAL
    assert binding.dns_launches_per_step(h) > 0
    assert binding.dns_plan_destroy(h) == binding.DNS_OK


def test_nonfinite_energy_is_reported():
    cfg = inputs.CONFIGS[1]
    st = inputs.make_state(cfg)
    v = st["vhat"].copy()
    v[1, 2, 3, 5] = np.nan
    plan = binding.Plan(*inputs.plan_args(cfg))
    plan.set_state(v, st["etahat"], st["U00"], st["W00"])
    out = np.empty((cfg.E, 6))
    assert binding.dns_diagnostics(plan.h, out) == binding.DNS_ENONFINITE
    assert np.isfinite(out[0, 0]) and not np.isfinite(out[1, 0])
    plan.close()


def test_stage_pieces_against_oracle():
    """Per-kernel parity through the debug hook: reconstruction (Eq. 17-18), the spectral advection terms and
    F^0, G^0 (Eq. 4-5) of the first stage."""
    cfg = inputs.CONFIGS[2].with_E(5)
    st = inputs.make_state(cfg)
    plan = binding.Plan(*inputs.plan_args(cfg))
    plan.set_state(st["vhat"], st["etahat"], st["U00"], st["W00"])
    o = Oracle(*inputs.plan_args(cfg))
    o.set_state(st["vhat"], st["etahat"], st["U00"], st["W00"])
    u, v, w, Du, Dv, Dw = o.velocities(o.v, o.eta, o.U, o.W)
    for which, ref in ((0, u), (1, w), (2, Du), (3, Dw)):
        got = plan.debug_fetch(which)
        assert field_err(got[..., 1:-1], ref[..., 1:-1]) < 1e-12, which
    F, G, Su, Sw = o.nonlinear(o.v, o.eta, o.U, o.W)
    plan.debug_stage(0)                       # after stage 0 the history buffers hold F^0, G^0
    assert field_err(plan.debug_fetch(5)[..., 1:-1], F) < 1e-11
    assert field_err(plan.debug_fetch(6)[..., 1:-1], G) < 1e-11
    plan.close()


def test_one_point_statistics_against_oracle():
    """Row f4: running one-point statistics (Parseval sums on the GPU) against the oracle's plane averages on the
    padded physical grid, accumulated over the same three samples; reset and sample count."""
    cfg = inputs.CONFIGS[2].with_E(5)
    st = inputs.make_state(cfg)
    plan = binding.Plan(*inputs.plan_args(cfg))
    plan.set_state(st["vhat"], st["etahat"], st["U00"], st["W00"])
    o = Oracle(*inputs.plan_args(cfg))
    o.set_state(st["vhat"], st["etahat"], st["U00"], st["W00"])
    s0, n0 = plan.stats()
    assert n0 == 0 and np.all(s0 == 0.0)
    acc = np.zeros((cfg.E, cfg.Ny, 5))
    for _ in range(3):
        plan.step(2)
        o.step(2)
        plan.stats_accumulate()
        acc += o.one_point_stats()
    s, n = plan.stats()
    assert n == 3
    ref = acc / 3
    for k in range(5):
        scale = max(np.abs(ref[:, :, k]).max(), 1e-300)
        assert np.abs(s[:, :, k] - ref[:, :, k]).max() < 1e-10 * max(scale, np.abs(ref[:, :, 1]).max()), k
    plan.stats_reset()
    s1, n1 = plan.stats()
    assert n1 == 0 and np.all(s1 == 0.0)
    plan.close()


def test_rebinding_the_workspace_rebuilds_graph_and_tensor_maps():
    """dns_plan_bind on a second buffer after steps have been taken: the captured step graph and the TMA descriptors
    hold pointers into the first buffer and must be rebuilt; results equal those of the first run bit for bit."""
    import torch
    cfg = inputs.CONFIGS[2].with_E(6)
    st = inputs.make_state(cfg)
    plan = binding.Plan(*inputs.plan_args(cfg))
    plan.set_state(st["vhat"], st["etahat"], st["U00"], st["W00"])
    plan.step(2)
    first = plan.get_state()
    n = plan.workspace_bytes
    ws2 = torch.empty(n + 256, dtype=torch.uint8, device="cuda")
    base = (ws2.data_ptr() + 255) & ~255
    assert binding.dns_plan_bind(plan.h, base, n) == binding.DNS_OK
    assert binding.dns_step(plan.h, 1) == binding.DNS_ESTATE                 # the state went with the old workspace
    plan.workspace.fill_(0xFF)                                               # poison the old buffer
    plan.set_state(st["vhat"], st["etahat"], st["U00"], st["W00"])
    plan.step(1)
    plan.step(1)
    second = plan.get_state()
    for a, b in zip(first, second):
        assert np.array_equal(a, b)
    plan.close()
    del ws2


def test_plan_on_a_non_default_stream():
    """The plan works on whatever stream it is bound to (here a torch side stream): graph replay, the internal
    mean-flow stream and the copies are all ordered on it; same bits as on the default stream."""
    import torch
    cfg = inputs.CONFIGS[2].with_E(6)
    st = inputs.make_state(cfg)
    outs = []
    for use_side in (False, True):
        s = torch.cuda.Stream() if use_side else torch.cuda.current_stream()
        with torch.cuda.stream(s):
            plan = binding.Plan(*inputs.plan_args(cfg))
            plan.set_state(st["vhat"], st["etahat"], st["U00"], st["W00"])
            plan.step(3)
            outs.append(plan.get_state())
            d = plan.diagnostics()
            assert np.all(np.isfinite(d))
            plan.close()
    for a, b in zip(*outs):
        assert np.array_equal(a, b)


def test_four_plans_on_four_host_threads_equal_the_serial_run_bitwise():
    """One plan per host thread is the supported concurrent use (bench.measure_e2e drives four).  Four threads each create,
    bind (own stream), load and step their own plan for 50 steps at the same time -- different grids, so that they reach
    different kernel instantiations and shared-memory grants concurrently -- and every final state equals, bit for bit, the
    one the same plan produces when run alone."""
    import threading
    import torch

    cfgs = [inputs.CONFIGS[1],
            inputs.CONFIGS[2].with_E(8),
            inputs.Config(3, inputs.POISEUILLE_CMF, 2000.0, 1.75 * PI, 1.2 * PI, 24, 41, 16, 5, 0.01, 1, 0.2, 0, box=3),
            inputs.Config(1, inputs.COUETTE, 400.0, 1.75 * PI, 1.2 * PI, 16, 129, 24, 3, 0.01, 1, 0.2, 0, box=3)]
    states = [inputs.make_state(c) for c in cfgs]

    def run(i, out, stream=None):
        try:
            with torch.cuda.stream(stream if stream is not None else torch.cuda.current_stream()):
                p = binding.Plan(*inputs.plan_args(cfgs[i]))
                st = states[i]
                p.set_state(st["vhat"], st["etahat"], st["U00"], st["W00"])
                for _ in range(10):
                    p.step(5)
                out[i] = p.get_state() + (p.diagnostics(),)
                p.close()
        except Exception as exc:                              # surfaces in the main thread
            out[i] = exc

    serial = [None] * 4
    for i in range(4):
        run(i, serial)
    for rep in range(2):
        par = [None] * 4
        threads = [threading.Thread(target=run, args=(i, par, torch.cuda.Stream())) for i in range(4)]
        for t in threads:
            t.start()
        for t in threads:
            t.join()
        for i in range(4):
            assert not isinstance(par[i], Exception) and not isinstance(serial[i], Exception), (par[i], serial[i])
            for a, b in zip(serial[i], par[i]):
                assert np.array_equal(a, b), (rep, i)
    torch.cuda.synchronize()
