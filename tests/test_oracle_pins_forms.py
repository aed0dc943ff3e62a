"""Pins for the oracle's two SURVEY.md 8(f) extensions: the rotational form omega x u of the nonlinear term (row f1,
pins P17) and the ensemble-coupled streamwise-mean flow (row f2, pins P18).  As in
test_oracle_pins.py the oracle is checked against what the mathematics fixes, not against itself:
  P17a  the vector identity (u.grad)u = omega x u + grad(|u|^2/2): on a state whose products are exactly representable
        (no dealiasing truncation, polynomial degrees below Ny) the two forms give the same F, G, S_u, S_w to round-off;
  P17b  u . (omega x u) = 0 at every grid point (the rotational term does no work);
  P17c  Orr-Sommerfeld / Squire growth rates against the independent eigen-solve (P7 in the rotational form);
  P17d  laminar Couette and Poiseuille are fixed points although omega x u does not vanish at a moving wall;
  P17e  the energy budget across a step (P11) and the Kutta polynomial (P16) in the rotational form;
  P18a  an ensemble of identical members is unchanged by the coupling;
  P18b  members that share their kx = 0 components keep sharing them, and only the kx = 0 forcing is touched, with its
        ensemble mean conserved;
  P18c  the ensemble-averaged energy obeys the budget dE/dt = -eps + input although single members do not.
All tests run on CPU (`-m "not gpu"`).
"""
import numpy as np
import pytest

from oracle.dns_oracle import (CONVECTIVE, COUETTE, POISEUILLE_CMF, ROTATIONAL, STREAMWISE_MEAN, UNCOUPLED, Oracle)
from paper_2306_12739_b200 import inputs

import test_oracle_pins as base

PI = np.pi


def make(cfg, form=CONVECTIVE, coupling=UNCOUPLED, share_mean=False):
    o = Oracle(*inputs.plan_args(cfg), form=form, coupling=coupling)
    st = inputs.make_state(cfg)
    v, eta, U, W = st["vhat"].copy(), st["etahat"].copy(), st["U00"].copy(), st["W00"].copy()
    if share_mean:                                  # every member gets member 0's streamwise-mean (kx = 0) components
        v[:, 0], eta[:, 0], U[:], W[:] = v[0, 0], eta[0, 0], U[0], W[0]
    o.set_state(v, eta, U, W)
    return o


# ------------------------------------------------------------------------------------------------ P17
@pytest.mark.parametrize("flow", [COUETTE, POISEUILLE_CMF])
def test_P17a_vector_identity_links_the_two_forms(flow):
    """Modes |n|,|m| <= 2 on a 12 x 25 x 12 grid (retained |n|,|m| <= 5), y-profiles of degree <= 6: every product has
    wavenumbers <= 4 and degree <= 12 < Ny, so nothing is truncated and grad(|u|^2/2) drops out of Eq. 4-7 exactly."""
    cfg = base.small_cfg(flow, rms=0.3, cid=3 if flow else 1)
    oc, orot = make(cfg, CONVECTIVE), make(cfg, ROTATIONAL)
    a = oc.nonlinear(oc.v, oc.eta, oc.U, oc.W)
    b = orot.nonlinear(orot.v, orot.eta, orot.U, orot.W)
    for name, x, y in zip("F G Su Sw".split(), a, b):
        if name[0] == "S":                           # mean-flow sources: only interior rows enter Eq. 14-15
            x, y = x[:, 1:-1], y[:, 1:-1]
        assert np.abs(x - y).max() < 2e-12 * max(np.abs(x).max(), 1e-3), name
    assert np.abs(a[0]).max() > 1e-3                 # the comparison is not between zeros
    # the two nonlinear vectors themselves differ by the gradient term, at O(1)
    Nc, Hr = oc.advection(oc.v, oc.eta, oc.U, oc.W), orot.advection(orot.v, orot.eta, orot.U, orot.W)
    assert np.abs(Nc[0] - Hr[0]).max() > 1e-2


def test_P17a_forms_differ_only_at_wall_normal_truncation_level():
    """The 3/2 rule keeps the product rule exact on the retained Fourier modes whatever the spectrum, so the two forms
    differ only through the wall-normal collocation: with Ny = 11 the degree-12 products of the degree-6 profiles are no
    longer representable and the forms must differ, by little (P17a is not vacuous; the switch really switches).
    With energy up to the Fourier cut-off but Ny = 25 they still agree to round-off."""
    cfg = base.small_cfg(COUETTE, Ny=11, rms=0.3)
    oc, orot = make(cfg, CONVECTIVE), make(cfg, ROTATIONAL)
    a = oc.nonlinear(oc.v, oc.eta, oc.U, oc.W)
    b = orot.nonlinear(orot.v, orot.eta, orot.U, orot.W)
    d = np.abs(a[0] - b[0]).max() / np.abs(a[0]).max()
    assert 1e-9 < d < 0.5, d
    cfg = base.small_cfg(COUETTE, rms=0.3, box=5)
    oc, orot = make(cfg, CONVECTIVE), make(cfg, ROTATIONAL)
    a = oc.nonlinear(oc.v, oc.eta, oc.U, oc.W)
    b = orot.nonlinear(orot.v, orot.eta, orot.U, orot.W)
    assert np.abs(a[0] - b[0]).max() < 1e-12 * np.abs(a[0]).max()


def test_P17b_rotational_term_does_no_work_pointwise():
    cfg = base.small_cfg(COUETTE, rms=0.3, box=5)
    o = make(cfg, ROTATIONAL)
    Hx, Hy, Hz, _, _ = o.advection(o.v, o.eta, o.U, o.W)
    u, v, w, *_ = o.velocities(o.v, o.eta, o.U, o.W)
    pu, pv, pw = o.to_physical(u), o.to_physical(v), o.to_physical(w)
    work = pu * Hx + pv * Hy + pw * Hz
    scale = np.abs(pu).max() * max(np.abs(Hx).max(), np.abs(Hy).max(), np.abs(Hz).max())
    assert np.abs(work).max() < 1e-14 * scale
    assert np.abs(Hy).max() > 1e-2
    # H_x and H_z vanish on both walls exactly, H_y = omega_z U_w does not (Couette): wall planes of H_y are never used
    assert np.abs(Hx[:, [0, -1]]).max() == 0.0 and np.abs(Hz[:, [0, -1]]).max() == 0.0
    assert np.abs(Hy[:, [0, -1]]).max() > 1e-3


@pytest.mark.parametrize("flow,Re,n,m", [(POISEUILLE_CMF, 3000.0, 1, 1), (COUETTE, 800.0, 1, 2)])
def test_P17c_growth_rates_in_the_rotational_form(flow, Re, n, m, monkeypatch):
    """P7 with the rotational oracle: same independent eigen-solve, same tolerance."""
    class RotOracle(Oracle):
        def __init__(self, *a, **k):
            super().__init__(*a, form=ROTATIONAL, **k)
    monkeypatch.setattr(base, "Oracle", RotOracle)
    base.test_P7_oracle_growth_rate_matches_orr_sommerfeld_squire(flow, Re, n, m)


def test_P17d_laminar_fixed_points_rotational():
    cfg = base.small_cfg(COUETTE)
    o = Oracle(*inputs.plan_args(cfg), form=ROTATIONAL)
    z = np.zeros((cfg.E, cfg.Nx // 2, cfg.Nz - 1, cfg.Ny), complex)
    o.set_state(z, z, np.tile(o.y, (cfg.E, 1)), np.zeros((cfg.E, cfg.Ny)))
    o.step(20)
    # H_y = -U dU/dy is a function of y only; its image on the (n,m) != (0,0) modes is DFT round-off, not exactly 0
    assert np.abs(o.U - o.y).max() < 1e-13 and np.abs(o.v).max() < 1e-15 and np.abs(o.eta).max() < 1e-15
    cfg = base.small_cfg(POISEUILLE_CMF, Re=2800.0, dt=0.005, cid=3)
    o = Oracle(*inputs.plan_args(cfg), form=ROTATIONAL)
    U = np.tile(1.5 * (1 - o.y ** 2), (cfg.E, 1))
    o.set_state(z, z, U, np.zeros_like(U))
    o.step(20)
    assert np.abs(o.U - U).max() < 1e-13
    assert np.abs(o.gamma - 3.0 / cfg.Re).max() < 1e-13 * cfg.Re


@pytest.mark.parametrize("flow", [COUETTE, POISEUILLE_CMF])
def test_P17e_energy_budget_rotational(flow):
    res = []
    for dt in (0.02, 0.01):
        cfg = base.small_cfg(flow, Re=200.0, dt=dt, rms=0.3, cid=3 if flow else 1)
        o = make(cfg, ROTATIONAL)
        o.step(2)
        E0, r0 = o.energy(), base._budget_rhs(o)
        o.step(1)
        E1, r1 = o.energy(), base._budget_rhs(o)
        res.append(np.abs((E1 - E0) - 0.5 * dt * (r0 + r1)).max())
        assert res[-1] < 5e-3 * np.abs(dt * r0).max() + 1e-9
    assert res[0] / res[1] > 5.0, res


def test_P17e_kutta_polynomial_rotational(monkeypatch):
    class RotOracle(Oracle):
        def __init__(self, *a, **k):
            super().__init__(*a, form=ROTATIONAL, **k)
    monkeypatch.setattr(base, "Oracle", RotOracle)
    base.test_P16_rk3_weights_kutta_amplification_polynomial()


# ------------------------------------------------------------------------------------------------ P18
@pytest.mark.parametrize("form", [CONVECTIVE, ROTATIONAL])
def test_P18a_identical_members_are_unchanged_by_the_coupling(form):
    cfg = base.small_cfg(COUETTE, E=3, rms=0.2)
    st = inputs.make_state(cfg, [1, 1, 1])
    a = Oracle(*inputs.plan_args(cfg), form=form, coupling=UNCOUPLED)
    b = Oracle(*inputs.plan_args(cfg), form=form, coupling=STREAMWISE_MEAN)
    for o in (a, b):
        o.set_state(st["vhat"], st["etahat"], st["U00"], st["W00"])
        o.step(2)
    for x, y in zip(a.get_state(), b.get_state()):
        assert np.abs(x - y).max() < 1e-15 * max(np.abs(x).max(), 1.0)


@pytest.mark.parametrize("flow", [COUETTE, POISEUILLE_CMF])
def test_P18b_shared_streamwise_mean_stays_shared_and_only_kx0_forcing_changes(flow):
    cfg = base.small_cfg(flow, E=4, rms=0.2, cid=3 if flow else 1)
    oc, ou = make(cfg, coupling=STREAMWISE_MEAN, share_mean=True), make(cfg, coupling=UNCOUPLED, share_mean=True)
    Fc, Gc, Suc, Swc = oc.nonlinear(oc.v, oc.eta, oc.U, oc.W)
    Fu, Gu, Suu, Swu = ou.nonlinear(ou.v, ou.eta, ou.U, ou.W)
    # n != 0 untouched; n = 0 and the mean-flow sources replaced by their ensemble mean (which is conserved)
    assert np.array_equal(Fc[:, 1:], Fu[:, 1:]) and np.array_equal(Gc[:, 1:], Gu[:, 1:])
    for c, u in ((Fc[:, 0], Fu[:, 0]), (Gc[:, 0], Gu[:, 0]), (Suc, Suu), (Swc, Swu)):
        assert np.abs(c - u.mean(axis=0)[None]).max() < 1e-14 * max(np.abs(u).max(), 1.0)
        assert np.abs(u - u.mean(axis=0)[None]).max() > 1e-6 * np.abs(u).max()        # members did differ
    oc.step(3)
    ou.step(3)
    for f in (oc.v[:, 0], oc.eta[:, 0], oc.U, oc.W):          # common streamwise-mean flow
        assert np.abs(f - f[0][None]).max() < 1e-14 * max(np.abs(f).max(), 1.0)
    assert np.abs(oc.v[:, 1:] - oc.v[0, 1:][None]).max() > 1e-4                      # perturbations stay distinct
    assert np.abs(ou.v[:, 0] - ou.v[0, 0][None]).max() > 1e-8                        # uncoupled members drift apart
    if flow == POISEUILLE_CMF:                                                       # the flux constraint is unaffected
        assert np.abs(oc.diagnostics()[:, 3] - 1.0).max() < 1e-13
    assert np.array_equal(oc.U[:, [0, -1]], ou.U[:, [0, -1]])                        # and so are the wall values


@pytest.mark.parametrize("form", [CONVECTIVE, ROTATIONAL])
def test_P18c_ensemble_mean_energy_budget(form):
    """With a shared streamwise-mean flow U and perturbations u'_e (kx != 0), E_e = E(U) + E(u'_e) and the transfers
    between U and <u'u'> cancel in the ensemble mean, while the kx != 0 self-interaction of each member does no net
    work on it: d<E>/dt = <-eps + input> holds for the ensemble average (trapezoid residual ~ dt^3), but not member by
    member."""
    res, single = [], []
    for dt in (0.02, 0.01):
        cfg = base.small_cfg(COUETTE, E=4, Re=200.0, dt=dt, rms=0.3)
        o = make(cfg, form=form, coupling=STREAMWISE_MEAN, share_mean=True)
        o.step(2)
        E0, r0 = o.energy(), base._budget_rhs(o)
        o.step(1)
        E1, r1 = o.energy(), base._budget_rhs(o)
        resid = (E1 - E0) - 0.5 * dt * (r0 + r1)
        res.append(abs(resid.mean()))
        single.append(np.abs(resid).max())
        assert res[-1] < 5e-3 * np.abs(dt * r0).max() + 1e-9
    assert res[0] / res[1] > 5.0, res
    assert single[1] > 20 * res[1], (single, res)        # single members exchange energy through the shared mean
