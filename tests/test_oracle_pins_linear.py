"""Pins P19 for the oracle of the linearised forward / adjoint ensemble (oracle/dns_linear_oracle.py; SURVEY.md 8(f) row
f3; PAPER.md:296-317 and Appendix B :390-417), against what the mathematics fixes:
  P19a  B.2 is the linearisation of the momentum equation: the forward linear vector equals the central difference of the
        PINNED nonlinear oracle about the base flow, which is exact for a quadratic nonlinearity (round-off only);
  P19b  B.5 is the adjoint of B.2 in the energy inner product of B.1: <lam, N_fwd(u)> = <N_adj(lam), u> on states whose
        products are resolved;
  P19c  the forward-adjoint power iteration of :417 converges to the leading singular values of the explicitly assembled
        forward propagator (energy norm), first and second optimal;
  P19d  Gram-Schmidt leaves an energy-orthonormal set and only normalises the first vector of every kx group;
  P19e  on a laminar base flow a forward step amplifies an Orr-Sommerfeld eigenmode by exp(lambda dt) (independent
        eigen-solve of test_oracle_pins.py), with a time-step factor t_f = 5 as in :315;
  P19f  the stage weights of LinearEnsemble.step and the reversed time of the adjoint leg (:411-417):
        one inviscid step multiplies a Squire mode by Kutta's polynomial in z (forward) and in -z (adjoint); three wrong
        weightings are kept red;
  P19g  the 1/(2V) of LinearEnsemble.inner (Eq. B.1, :396) against the pinned Oracle.energy of the same disturbance.
All tests run on CPU (`-m "not gpu"`).
"""
import numpy as np
import pytest
from numpy.polynomial import chebyshev as C

from oracle.dns_linear_oracle import LinearEnsemble
from oracle.dns_oracle import COUETTE, POISEUILLE_CMF, Oracle
from paper_2306_12739_b200 import inputs

import test_oracle_pins as base

PI = np.pi


def base_and_members(flow=COUETTE, Nx=12, Ny=25, Nz=12, n_list=(1, 2), Eg=2, dt=0.02, Re=400.0, rms=0.3, seed=5):
    """A streamwise-mean base flow = the kx = 0 plane of a seeded DNS state, and polynomial disturbances at single kx."""
    cfg = inputs.Config(3 if flow else 1, flow, Re, 1.75 * PI, 1.2 * PI, Nx, Ny, Nz, 1, dt, 1, rms, 0, box=2)
    st = inputs.make_state(cfg)
    L = LinearEnsemble(Nx, Ny, Nz, n_list, Eg, Re, cfg.Lx, cfg.Lz, dt, flow)
    L.set_base(st["vhat"][0, 0], st["etahat"][0, 0], st["U00"][0], st["W00"][0])
    pert = inputs.make_state(inputs.Config(**{**cfg.__dict__, "E": L.E}), range(10, 10 + L.E))
    v = np.stack([pert["vhat"][e, n] for e, n in enumerate(L.n_of)])
    eta = np.stack([pert["etahat"][e, n] for e, n in enumerate(L.n_of)])
    L.set_state(v, eta)
    return cfg, st, L


@pytest.mark.parametrize("flow", [COUETTE, POISEUILLE_CMF])
def test_P19a_forward_vector_is_the_linearisation_of_the_pinned_nonlinear_term(flow):
    cfg, st, L = base_and_members(flow)
    o = Oracle(*inputs.plan_args(cfg))
    eps = 1e-3
    for e in range(L.E):
        n = L.n_of[e]
        F_lin, G_lin = L.forcing(e, adjoint=False)
        out = []
        for sgn in (+1.0, -1.0):
            v = np.zeros((1, o.nkx, o.nkz, o.Ny), complex)
            eta = np.zeros_like(v)
            v[0, 0], eta[0, 0] = st["vhat"][0, 0], st["etahat"][0, 0]
            v[0, n], eta[0, n] = sgn * eps * L.v[e], sgn * eps * L.eta[e]
            o.set_state(v, eta, st["U00"], st["W00"])
            F, G, _, _ = o.nonlinear(o.v, o.eta, o.U, o.W)
            out.append((F[0, n], G[0, n]))
        F_fd = (out[0][0] - out[1][0]) / (2 * eps)          # exact for a quadratic term: no O(eps^2) remainder
        G_fd = (out[0][1] - out[1][1]) / (2 * eps)
        assert np.abs(F_lin - F_fd).max() < 1e-10 * np.abs(F_fd).max()
        assert np.abs(G_lin - G_fd).max() < 1e-10 * np.abs(G_fd).max()
        assert np.abs(F_fd).max() > 1e-3


def _inner_vec(L, e, a, b):
    """Energy inner product (B.1) of two velocity vectors given as spectral [3][nkz][Ny] arrays at member e's kx."""
    return 0.5 * np.einsum("cmj,j->", np.conj(a) * b, L.o.w)


@pytest.mark.parametrize("flow", [COUETTE, POISEUILLE_CMF])
def test_P19b_adjoint_identity_in_the_energy_inner_product(flow):
    """<lam, (U.grad)u + (u.grad)U> = <-(U.grad)lam - U_j grad lam_j, u> for divergence-free no-slip u, lam and a
    divergence-free base flow with V = 0 on the walls (integration by parts; exact for the resolved polynomial states)."""
    cfg, st, L = base_and_members(flow, Eg=2, n_list=(1, 2))
    for g in range(2):
        a, b = g * L.Eg, g * L.Eg + 1                       # u = member a, lam = member b (same kx)
        ua = np.stack(L._velocities(a))
        lb = np.stack(L._velocities(b))
        lhs = _inner_vec(L, a, lb, L.linear_vector(a, adjoint=False))
        rhs = _inner_vec(L, a, L.linear_vector(b, adjoint=True), ua)
        assert abs(lhs - rhs) < 1e-11 * abs(lhs), (lhs, rhs)
        assert abs(lhs) > 1e-4


def test_P19d_gram_schmidt_orthonormal_in_energy_norm():
    cfg, st, L = base_and_members(COUETTE, Eg=3, n_list=(1, 2))
    v0 = L.v.copy()
    e0 = L.energy()
    L.orthonormalise()
    for g in range(2):
        idx = range(g * L.Eg, (g + 1) * L.Eg)
        gram = np.array([[L.inner(a, b) for b in idx] for a in idx])
        assert np.abs(gram - np.eye(L.Eg)).max() < 1e-12
        first = g * L.Eg
        assert np.abs(L.v[first] - v0[first] / np.sqrt(e0[first])).max() < 1e-13      # only normalised
    assert np.abs(L.energy() - 1.0).max() < 1e-12


def test_P19c_power_iteration_finds_the_optimal_gains_of_the_forward_propagator():
    """Tiny case (8 x 17 x 8, kx = 0.25, Couette Re = 300 with a roll/streak base flow, T_opt = 16 steps of dt_lin = 0.25).
    Reference: the forward oracle applied to a basis of smooth clamped profiles ((1-y^2)^2 T_k for v, (1-y^2) T_k for eta,
    k < 7, every kz) gives the Gram matrices of the initial and final energies; their generalised eigenvalues are the
    optimal gains over that subspace (converged in k: 11.69, 10.13, 9.33).  (The full nodal space is not usable here: a
    unit vector at one collocation point is not a clamped function, and the first implicit solve 'gains' energy on it.)
    The forward-adjoint loop with Gram-Schmidt must converge to the same leading gains although it uses the
    CONTINUOUS adjoint B.5: first gain to 0.1 %, second to 1 %, and the gains never decrease along the iteration."""
    import scipy.linalg as sla
    Nx, Ny, Nz, n, nst = 8, 17, 8, 1, 16
    flow, Re, dt, Lx, Lz = COUETTE, 300.0, 0.25, 8 * PI, 1.2 * PI
    cfg = inputs.Config(1, flow, Re, Lx, Lz, Nx, Ny, Nz, 1, dt, 1, 0.3, 0, box=2)
    st = inputs.make_state(cfg)
    nkz, K = Nz - 1, 7
    y = inputs.grid_y(Ny)
    vs, es = [], []
    for mi in range(nkz):
        for k in range(K):
            T = np.cos(k * np.arccos(np.clip(y, -1, 1)))
            z = np.zeros((nkz, Ny), complex)
            a, b = z.copy(), z.copy()
            a[mi], b[mi] = (1 - y * y) ** 2 * T, (1 - y * y) * T
            vs += [a, z]
            es += [z, b]
    nb = len(vs)
    L = LinearEnsemble(Nx, Ny, Nz, [n], nb, Re, Lx, Lz, dt, flow)
    L.set_base(st["vhat"][0, 0], st["etahat"][0, 0], st["U00"][0], st["W00"][0])
    L.set_state(np.stack(vs), np.stack(es))
    M0 = np.array([[L.inner(a, b) for b in range(nb)] for a in range(nb)])
    L.step(nst)
    MT = np.array([[L.inner(a, b) for b in range(nb)] for a in range(nb)])
    ref = sla.eigh(MT, M0, eigvals_only=True)[::-1]
    assert ref[0] > 10.0 and ref[1] < 0.9 * ref[0]                  # real transient growth, separated leading gain

    Lo = LinearEnsemble(Nx, Ny, Nz, [n], 3, Re, Lx, Lz, dt, flow)
    Lo.set_base(st["vhat"][0, 0], st["etahat"][0, 0], st["U00"][0], st["W00"][0])
    rng = np.random.default_rng(3)
    c = rng.standard_normal((3, nb)) + 1j * rng.standard_normal((3, nb))
    Lo.set_state(np.einsum("ek,kmj->emj", c, np.stack(vs)), np.einsum("ek,kmj->emj", c, np.stack(es)))
    hist = [Lo.optimals(nst, 8) for _ in range(5)]
    gains = hist[-1]
    assert abs(gains[0] - ref[0]) < 1e-3 * ref[0], (gains, ref[:3])
    assert abs(gains[1] - ref[1]) < 1e-2 * ref[1], (gains, ref[:3])
    top = [h[0] for h in hist]
    assert all(b >= a * (1 - 1e-6) for a, b in zip(top, top[1:])), top


def test_P19e_laminar_base_flow_orr_sommerfeld_growth_with_time_step_factor():
    """Base flow = laminar Poiseuille (no roll): the linear forward step must amplify the least-stable Orr-Sommerfeld mode
    of the independent eigen-solve by exp(lambda T); dt_lin = t_f dt with t_f = 5."""
    Re, Lx, Lz, n, m, Ny = 3000.0, 2 * PI, 2 * PI, 1, 1, 57
    dt_lin, nsteps = 5 * 0.004, 20
    Uf, dUf, d2Uf = (lambda y: 1 - y * y), (lambda y: -2 * y), (lambda y: -2 + 0 * y)
    kx, kz = 2 * PI * n / Lx, 2 * PI * m / Lz
    Neig = Ny + 24
    yE, lam, vec = base._os_squire_eig(Neig, Re, kx, kz, Uf, dUf, d2Uf)
    vnorm = np.linalg.norm(vec[:Neig], axis=0) / np.linalg.norm(vec, axis=0)
    cand = np.where(vnorm > 1e-3)[0]
    k = cand[np.argmax(lam[cand].real)]
    Vinv = np.linalg.inv(C.chebvander(yE, Neig - 1))
    L = LinearEnsemble(12, Ny, 12, [n], 1, Re, Lx, Lz, dt_lin, POISEUILLE_CMF)
    z = np.zeros((11, Ny), complex)
    L.set_base(z, z, Uf(L.o.y), np.zeros(Ny))
    v0 = C.chebval(L.o.y, Vinv @ vec[:Neig, k])
    e0 = C.chebval(L.o.y, Vinv @ vec[Neig:, k])
    vh, eh = np.zeros((1, 11, Ny), complex), np.zeros((1, 11, Ny), complex)
    mi = inputs.m_index(m, 12)
    vh[0, mi], eh[0, mi] = v0, e0
    L.set_state(vh, eh)
    vi = L.v[0, mi].copy()
    L.step(nsteps)
    fac = np.vdot(vi, L.v[0, mi]) / np.vdot(vi, vi)
    expect = np.exp(lam[k] * nsteps * dt_lin)
    assert abs(fac - expect) < 2e-5 * abs(expect), (fac, expect)


# ------------------------------------------------------------------------------------------------ P19f / P19g
def _lin_inviscid_squire_step(adjoint, dt=0.15, Ny=25, n=2, step=None):
    """One step of the LINEAR oracle on a Squire mode (v = 0, kz = 0, eta = 1e-9 g(y)) over the parabola U = 1 - y^2 at
    Re = 1e12 (Crank-Nicolson part switched off).  Eq. 17-18 give u = 0, w = i eta / kx, so the forward vector of B.2 is
    N_w = i kx U w and Eq. 5 gives G = i kx U eta: every collocation point obeys d eta_j/dt = -i kx U(y_j) eta_j.  In B.5
    (v = 0, kz = 0: U_i grad lam_i vanishes with u) the reversed-time equation is d eta_j/d tau = +i kx U(y_j) eta_j.
    Returns (eta_0, eta_1, z_j) with z_j = -i kx U(y_j) dt, the FORWARD exponent."""
    Lx = 2 * PI
    L = LinearEnsemble(12, Ny, 12, [n], 1, 1e12, Lx, PI, dt, POISEUILLE_CMF)
    if step is not None:
        L.step = step.__get__(L)
    y = L.o.y
    z0 = np.zeros((11, Ny), complex)
    L.set_base(z0, z0, 1 - y ** 2, np.zeros(Ny))
    eh = np.zeros((1, 11, Ny), complex)
    eh[0, 0] = 1e-9 * (1 - y ** 2) * (1 + 0.3 * y) * np.exp(0.7j * y)
    L.set_state(np.zeros_like(eh), eh)
    e0 = L.eta[0, 0].copy()
    L.step(1, adjoint)
    assert np.abs(L.v).max() < 1e-16
    return e0, L.eta[0, 0].copy(), -1j * (2 * PI * n / Lx) * (1 - y ** 2) * dt


def _mutated_lin_step(mutation):
    """LinearEnsemble.step with one wrong stage weighting (the three the round-2 review found invisible to P19a-e)."""
    def step(self, nsteps=1, adjoint=False):
        for _ in range(int(nsteps)):
            v_t, e_t = self.v, self.eta
            F0, G0 = self._forcing_all(adjoint)
            self.v, self.eta = self._stage(v_t, e_t, 0.5, F0, G0)
            F1, G1 = self._forcing_all(adjoint)
            c2 = (F1, G1) if mutation == "stage2_F1" else (2.0 * F1 - F0, 2.0 * G1 - G0)
            self.v, self.eta = self._stage(v_t, e_t, 1.0, *c2)
            F2, G2 = self._forcing_all(adjoint)
            if mutation == "stage3_quarter":
                c3 = ((F0 + 2.0 * F1 + F2) / 4.0, (G0 + 2.0 * G1 + G2) / 4.0)
            elif mutation == "stage3_F1":
                c3 = (F1, G1)
            else:
                c3 = ((F0 + 4.0 * F1 + F2) / 6.0, (G0 + 4.0 * G1 + G2) / 6.0)
            self.v, self.eta = self._stage(v_t, e_t, 1.0, *c3)
    return step


@pytest.mark.parametrize("adjoint", [False, True])
def test_P19f_rk3_weights_of_the_linear_step_kutta_polynomial(adjoint):
    """LinearEnsemble.step re-states the stage weights of PAPER.md:120-126 (F^0 with h = 1/2; 2 F^1 - F^0; (F^0 + 4 F^1 +
    F^2)/6) and does not call the pinned Oracle.step, so it gets the pin P16 gives that one: one inviscid step multiplies
    eta(y_j) by EXACTLY Kutta's polynomial 1 + z + z^2/2 + z^3/6 -- with z = -i kx U(y_j) dt forward (B.2) and with -z for
    the adjoint, which runs in reversed time (B.5, reading L1; "evolved backwards").  kx dt = 0.3 makes the
    cubic term 4.5e-3 against a tolerance of 1e-10 (measured on the oracle: 1e-12).  The sign of the exponent also pins the
    direction of time of the adjoint leg, which P19b (an identity at one instant) cannot see.  Red on: stage 2 <- F^1,
    stage 3 <- (F^0 + 2 F^1 + F^2)/4, stage 3 <- F^1 (test_P19f_detects_wrong_rk3_weights), all of which passed P19a-e."""
    e0, e1, z = _lin_inviscid_squire_step(adjoint)
    if adjoint:
        z = -z
    kutta = 1 + z + z ** 2 / 2 + z ** 3 / 6
    assert np.abs(z ** 3 / 6).max() > 4e-3
    err = np.abs(e1 - kutta * e0).max() / np.abs(e0).max()
    assert err < 1e-10, err
    wrong = 1 - z + z ** 2 / 2 - z ** 3 / 6                   # the other direction of time misses by ~2|z| = 0.6
    assert np.abs(e1 - wrong * e0).max() / np.abs(e0).max() > 0.1


@pytest.mark.parametrize("adjoint", [False, True])
@pytest.mark.parametrize("mutation", ["stage2_F1", "stage3_quarter", "stage3_F1"])
def test_P19f_detects_wrong_rk3_weights(mutation, adjoint):
    e0, e1, z = _lin_inviscid_squire_step(adjoint, step=_mutated_lin_step(mutation))
    if adjoint:
        z = -z
    kutta = 1 + z + z ** 2 / 2 + z ** 3 / 6
    assert np.abs(e1 - kutta * e0).max() / np.abs(e0).max() > 1e-3


def test_P19f_mutation_harness_reproduces_the_real_step():
    """The mutation harness with no mutation is LinearEnsemble.step: the red results above are due to the weights alone."""
    a = _lin_inviscid_squire_step(False)
    b = _lin_inviscid_squire_step(False, step=_mutated_lin_step("none"))
    assert np.array_equal(a[1], b[1])


def test_P19g_energy_normalisation_of_B1_against_the_pinned_dns_energy():
    """LinearEnsemble.inner carries the 1/(2V) of Eq. B.1 as the factor 0.5 on the sum over the stored
    kx > 0 modes (a stored mode stands for the pair +-kx).  Pin: a DNS state that holds the same single-kx disturbance and
    nothing else (U00 = W00 = 0, Poiseuille walls at rest) has, by Oracle.energy -- itself pinned by the generator's closed
    form and by P11 -- the same energy.  P19c/P19d use inner() on both sides of their comparisons, so its constant cancels
    there; here 0.5 -> 1.0 (or 0.25) is off by a factor 2."""
    cfg, st, L = base_and_members(POISEUILLE_CMF, n_list=(1, 2), Eg=2)
    o = Oracle(cfg.Nx, cfg.Ny, cfg.Nz, L.E, cfg.Re, cfg.Lx, cfg.Lz, cfg.dt, POISEUILLE_CMF)
    v = np.zeros((L.E, o.nkx, o.nkz, o.Ny), complex)
    eta = np.zeros_like(v)
    for e, n in enumerate(L.n_of):
        v[e, n], eta[e, n] = L.v[e], L.eta[e]
    o.set_state(v, eta, np.zeros((L.E, o.Ny)), np.zeros((L.E, o.Ny)))
    want, got = o.energy(), L.energy()
    assert (want > 1e-6).all()
    assert np.abs(got - want).max() < 1e-13 * want.max(), (got, want)
    # and the cross terms: <a, b> is conjugate-symmetric and linear in b with the same constant
    ab, ba = L.inner(0, 1), L.inner(1, 0)
    assert abs(ab - np.conj(ba)) < 1e-15 * want.max()
    L.v[1], L.eta[1] = L.v[0] + L.v[1], L.eta[0] + L.eta[1]
    assert abs(L.inner(0, 1) - (L.inner(0, 0) + ab)) < 1e-14 * want.max()
