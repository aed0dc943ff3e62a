"""GPU parity for the linearised forward / adjoint ensemble (Appendix B): the
dns_lin_* calls against oracle/dns_linear_oracle.py on the same seeded inputs, element by element (BASELINE.json's
tolerances: 1e-10 relative after 1 step; looser by the step count after more).  Run with `pytest -m gpu`."""
import numpy as np
import pytest

from oracle.dns_linear_oracle import LinearEnsemble
from paper_2306_12739_b200 import binding, inputs
from test_gpu_parity import PI, TOL_1, field_err

pytestmark = pytest.mark.gpu


def setup(cfg, n_list, Eg, dt_lin, seed_member=0, rough=False):
    """A DNS plan holding the base state (member seed_member's streamwise mean is the base flow), the linear GPU plan and
    the linear oracle with the same base flow and the same seeded disturbances."""
    st = inputs.make_state(cfg)
    dns = binding.Plan(*inputs.plan_args(cfg))
    dns.set_state(st["vhat"], st["etahat"], st["U00"], st["W00"])
    lin = binding.LinPlan(cfg.Nx, cfg.Ny, cfg.Nz, n_list, Eg, cfg.Re, cfg.Lx, cfg.Lz, dt_lin)
    lin.set_base(dns, seed_member)
    o = LinearEnsemble(cfg.Nx, cfg.Ny, cfg.Nz, n_list, Eg, cfg.Re, cfg.Lx, cfg.Lz, dt_lin, cfg.flow)
    o.set_base(st["vhat"][seed_member, 0], st["etahat"][seed_member, 0], st["U00"][seed_member], st["W00"][seed_member])
    E = len(n_list) * Eg
    gen = inputs.make_broadband_state if rough else inputs.make_state
    pert = gen(inputs.Config(**{**cfg.__dict__, "E": E}), range(20, 20 + E))
    v = np.stack([pert["vhat"][e, n] for e, n in enumerate(o.n_of)])
    eta = np.stack([pert["etahat"][e, n] for e, n in enumerate(o.n_of)])
    lin.set_state(v, eta)
    o.set_state(v, eta)
    return dns, lin, o


def compare(lin, o, tol):
    gv, ge = lin.get_state()
    assert field_err(gv, o.v) < tol and field_err(ge, o.eta) < tol, (field_err(gv, o.v), field_err(ge, o.eta))


@pytest.mark.parametrize("flow", [inputs.COUETTE, inputs.POISEUILLE_CMF])
@pytest.mark.parametrize("adjoint", [False, True])
def test_linear_forward_and_adjoint_steps_small(flow, adjoint):
    cfg = inputs.Config(3 if flow else 1, flow, 400.0, 1.75 * PI, 1.2 * PI, 16, 25, 16, 2, 0.02, 1, 0.3, 0, box=3)
    dns, lin, o = setup(cfg, [1, 2, 3], 5, 5 * cfg.dt, seed_member=1)
    compare(lin, o, 1e-14)                                   # set_state round trip (wall rows zeroed on both sides)
    assert np.abs(lin.energy() - o.energy()).max() < 1e-12 * o.energy().max()
    lin.step(1, adjoint)
    o.step(1, adjoint)
    compare(lin, o, TOL_1)
    lin.step(3, adjoint)
    o.step(3, adjoint)
    compare(lin, o, TOL_1 * 10)
    assert np.abs(lin.energy() - o.energy()).max() < 1e-9 * o.energy().max()
    lin.close()
    dns.close()


def test_linear_ensemble_at_the_papers_size():
    """C1 resolution (48 x 65 x 48) with 45 disturbances = kx/alpha in {1, 2, 3} x 15 (Fig. 7) and the
    time-step factor t_f = 5 (:315); the base flow is the streamwise mean of a config-4 member.  Rough (broadband)
    disturbances; forward and adjoint step against the oracle on every member."""
    cfg = inputs.CONFIGS[4].with_E(2)
    dns, lin, o = setup(cfg, [1, 2, 3], 15, 5 * cfg.dt, seed_member=1, rough=True)
    lin.step(1, False)
    o.step(1, False)
    compare(lin, o, TOL_1)
    lin.step(1, True)
    o.step(1, True)
    compare(lin, o, TOL_1 * 10)
    lin.close()
    dns.close()


@pytest.mark.parametrize("Nz,Eg", [(12, 3), (24, 17), (32, 33), (36, 4), (54, 9)])
def test_linear_every_z_kernel_family_and_ragged_groups(Nz, Eg):
    """Register (Mz = 36, 48, 72) and shared-memory (Mz = 18, 81) z transforms with a single kx row, member tiles that end
    inside a kx group (Eg not a multiple of the tile), more than 32 members per group in Gram-Schmidt."""
    cfg = inputs.Config(1, inputs.COUETTE, 350.0, 1.9 * PI, 1.1 * PI, 16, 13, Nz, 1, 0.01, 1, 0.2, 0, box=3)
    dns, lin, o = setup(cfg, [2, 1], Eg, 0.03)
    for adj in (False, True):
        lin.step(2, adj)
        o.step(2, adj)
        compare(lin, o, TOL_1 * 10)
    lin.close()
    dns.close()


def test_gram_schmidt_against_oracle_and_orthonormality():
    cfg = inputs.Config(1, inputs.COUETTE, 400.0, 1.75 * PI, 1.2 * PI, 16, 25, 16, 1, 0.02, 1, 0.3, 0, box=3)
    dns, lin, o = setup(cfg, [1, 3], 7, 0.1)
    lin.orthonormalise()
    o.orthonormalise()
    compare(lin, o, 1e-11)
    assert np.abs(lin.energy() - 1.0).max() < 1e-12
    lin.step(2, False)                                       # the transform inputs were refreshed: stepping still agrees
    o.step(2, False)
    compare(lin, o, 1e-9)
    lin.close()
    dns.close()


def test_optimal_disturbance_loop_against_oracle():
    """dns_lin_optimals = the oracle's power iteration: same gains and the same converged vectors; the
    leading gain is real transient growth."""
    cfg = inputs.Config(1, inputs.COUETTE, 300.0, 8 * PI, 1.2 * PI, 16, 21, 16, 1, 0.25, 1, 0.3, 0, box=2)
    dns, lin, o = setup(cfg, [1, 2], 3, 0.25)
    g_gpu = lin.optimals(12, 6)
    g_or = o.optimals(12, 6)
    assert np.abs(g_gpu - g_or).max() < 1e-7 * g_or.max(), (g_gpu, g_or)
    assert g_or.max() > 5.0
    compare(lin, o, 1e-6)
    lin.close()
    dns.close()


def test_linear_error_paths():
    cfg = inputs.CONFIGS[1]
    assert binding.dns_lin_plan_create(16, 33, 16, [0], 2, 400.0, 5.0, 3.0, 0.02)[0] == binding.DNS_EINVAL   # n = 0: a mean flow
    assert binding.dns_lin_plan_create(16, 33, 16, [8], 2, 400.0, 5.0, 3.0, 0.02)[0] == binding.DNS_EINVAL   # n >= Nx/2
    assert binding.dns_lin_plan_create(16, 33, 16, [], 2, 400.0, 5.0, 3.0, 0.02)[0] == binding.DNS_EINVAL
    st = inputs.make_state(cfg)
    dns = binding.Plan(*inputs.plan_args(cfg))
    lin = binding.LinPlan(cfg.Nx, cfg.Ny, cfg.Nz, [1], 2, cfg.Re, cfg.Lx, cfg.Lz, 0.1)
    assert binding.dns_lin_set_base(lin.h, dns.h, 0) == binding.DNS_ESTATE            # the DNS plan has no state yet
    dns.set_state(st["vhat"], st["etahat"], st["U00"], st["W00"])
    assert binding.dns_lin_set_base(lin.h, dns.h, 5) == binding.DNS_EINVAL            # no such member
    assert binding.dns_lin_step(lin.h, 1, 0) == binding.DNS_ESTATE                    # no base, no state
    assert binding.dns_step(lin.h, 1) == binding.DNS_EINVAL                           # a linear plan is not a DNS plan
    assert binding.dns_lin_step(dns.h, 1, 0) == binding.DNS_EINVAL
    assert binding.dns_plan_set_form(lin.h, 1) == binding.DNS_EINVAL
    rot = binding.Plan(*inputs.plan_args(cfg), form=binding.DNS_FORM_ROTATIONAL)
    rot.set_state(st["vhat"], st["etahat"], st["U00"], st["W00"])
    assert binding.dns_lin_set_base(lin.h, rot.h, 0) == binding.DNS_EINVAL
    other = binding.Plan(16, 33, 24, 1, 400.0, cfg.Lx, cfg.Lz, 0.02, 0)
    assert binding.dns_lin_set_base(lin.h, other.h, 0) == binding.DNS_EINVAL          # another grid
    lin.set_base(dns, 0)
    assert binding.dns_lin_step(lin.h, 1, 0) == binding.DNS_ESTATE                    # still no state
    assert binding.dns_lin_step(lin.h, 1, 2) in (binding.DNS_ESTATE, binding.DNS_EINVAL)
    for p in (lin, dns, rot, other):
        p.close()


def test_gram_schmidt_with_a_zero_member_stays_finite():
    """A member with no energy has no direction: dns_lin_orthonormalise sets it to zero instead of dividing by zero, the
    other members of its kx group come out exactly as if it were not there, and every call still returns DNS_OK."""
    cfg = inputs.Config(1, inputs.COUETTE, 400.0, 1.75 * PI, 1.2 * PI, 16, 25, 16, 1, 0.02, 1, 0.3, 0, box=3)
    dns, lin, o = setup(cfg, [1, 2], 4, 0.1)
    v, eta = lin.get_state()
    v[1], eta[1] = 0.0, 0.0                                   # second member of the first group
    lin.set_state(v, eta)
    lin.orthonormalise()
    gv, ge = lin.get_state()
    en = lin.energy()
    assert np.isfinite(gv).all() and np.isfinite(ge).all() and np.isfinite(en).all()
    assert en[1] == 0.0 and np.abs(np.delete(en, 1) - 1.0).max() < 1e-12
    # the oracle on the same vectors without the zero member (3 + 4 members would not fit its equal groups: group 0 alone)
    o3 = LinearEnsemble(cfg.Nx, cfg.Ny, cfg.Nz, [1], 3, cfg.Re, cfg.Lx, cfg.Lz, 0.1, cfg.flow)
    o3.set_state(v[[0, 2, 3]], eta[[0, 2, 3]])
    o3.orthonormalise()
    assert field_err(gv[[0, 2, 3]], o3.v) < 1e-11 and field_err(ge[[0, 2, 3]], o3.eta) < 1e-11
    lin.step(1, False)                                        # and it keeps stepping
    assert np.isfinite(lin.energy()).all()
    lin.close()
    dns.close()


def test_linear_step_graph_replay_equals_direct_launches_bitwise():
    """dns_lin_step replays one CUDA graph per direction; with the test option "graph" = 0 it launches directly.  Same bits,
    forward and adjoint, also after the base flow has been replaced (the graphs hold pointers, not contents)."""
    cfg = inputs.Config(1, inputs.COUETTE, 400.0, 1.75 * PI, 1.2 * PI, 16, 33, 16, 2, 0.02, 1, 0.3, 0, box=3)
    outs = []
    for graph in (-1, 0):
        assert binding.dns_debug_set_option("graph", graph) == binding.DNS_OK
        try:
            dns, lin, o = setup(cfg, [1, 2, 3], 5, 5 * cfg.dt, seed_member=1)
            lin.step(3, False)
            lin.step(2, True)
            lin.set_base(dns, 0)
            lin.step(2, False)
            outs.append(lin.get_state())
            lin.close()
            dns.close()
        finally:
            binding.dns_debug_set_option("graph", -1)
    for a, b in zip(*outs):
        assert np.array_equal(a, b)
