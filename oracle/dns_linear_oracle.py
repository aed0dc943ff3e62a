"""ORACLE for the linearised forward / adjoint ensemble of arXiv 2306.12739 (section 4.1.1, and
Appendix B, Eq. B.1-B.6, :390-417) -- TEST INFRASTRUCTURE ONLY.

A plain, slow, fp64 CPU restatement written from the paper, for parity-checking the CUDA path.  Only `tests/`,
`__graft_entry__.smoke()` and `bench.py`'s cpu legs may import it; it imports nothing from the product.

What it computes.  E = nmodes * Eg disturbance vectors; vector e has ONE streamwise wavenumber kx = 2 pi n_e / Lx
("we may specify the streamwise wavenumber of each disturbance") and no mean flow, so only Eq. 12-13 are
solved, with the precomputed single-kx operators of that vector (:304) and a time step dt_lin = t_f dt (:315).  The base
flow (U, V, W)(y, z) is a frozen streamwise-mean flow, i.e. the kx = 0 part of a DNS state (Fig. 7(a), :302).
  forward  (B.2):  d u'/dt     = -[(U.grad)u' + (u'.grad)U] - grad p' + (1/Re) Lap u'
  adjoint  (B.5):  d lam/d tau = +[(U.grad)lam + U_i grad lam_i] - grad b + (1/Re) Lap lam,   tau = T - t
Both have the form of the momentum equation with a "nonlinear vector" N that is linear in the disturbance, so F, G of
Eq. 4-5 and the CN/RK3 stages of Eq. 11-13 are reused unchanged, with the operators and LU factors
of oracle.dns_oracle.Oracle, which are pinned by tests/test_oracle_pins.py ("The matrices are also valid for the adjoint
equations", :304).  Products are formed on the 3/2-padded z grid (x is analytic: d/dx = i kx).
Energy inner product (B.1): <a, b> = 1/(2V) int conj(a).b dV over the pair of modes +-kx
                                   = (1/2) sum_m sum_j w_j (conj(u_a) u_b + conj(v_a) v_b + conj(w_a) w_b).
Optimal disturbances (:417): forward over T_opt, adjoint back from the forward final state, the adjoint final state
re-orthonormalised by Gram-Schmidt within each kx (modes of different kx are orthogonal already) is the next initial
condition; the gains E(T_opt)/E(0) of the converged vectors are the leading optimal growths.

Readings (L1-L4).  L1: B.5 is printed with d/dt on the left and all signs positive; it is read as
the adjoint in reversed time tau = T - t (the paper integrates it "backwards over the same time interval", :417), and its
second term U_i grad lam_i equals the textbook -lam_j grad U_j up to a gradient absorbed in b.  L2: the adjoint variable
satisfies the forward boundary conditions (no-slip, :85) and is represented by (lam_2, d lam_1/dz - d lam_3/dx) exactly as
(v, eta).  L3: the base flow is frozen over the optimisation window (:296 "the constant mean flow").  L4: Gram-Schmidt is
the modified (sequential) variant in member order within a kx group.

Pins (tests/test_oracle_pins_linear.py): P19a the forward linear vector is the exact central difference of the pinned
nonlinear oracle about the base flow; P19b the discrete adjoint identity <lam, N_fwd(u)> = <N_adj(lam), u> on resolved
states; P19c the power iteration against the generalised eigenvalues (final vs initial energy Gram matrices) of the forward
oracle on a basis of smooth clamped profiles; P19d Gram-Schmidt orthonormality; P19e Orr-Sommerfeld growth on a laminar base
flow; P19f the RK3 stage weights that step() re-states and the direction of time of the adjoint leg,
against Kutta's amplification polynomial 1 + z + z^2/2 + z^3/6 in the inviscid limit, forward (z) and adjoint (-z); P19g the
1/(2V) of inner() (B.1) against the pinned Oracle.energy of a DNS state holding the same single-kx disturbance.
Parity with the author's MATLAB output: UNPINNED.
"""
from __future__ import annotations

import numpy as np

from oracle.dns_oracle import Oracle


class LinearEnsemble:
    """State layout = the C-ABI layout of dns_lin_*: vhat, etahat [E][nkz][Ny] complex128, member e = g * Eg + i belongs to
    kx group g with streamwise mode n_list[g]; m in FFT order; y ascending."""

    def __init__(self, Nx, Ny, Nz, n_list, Eg, Re, Lx, Lz, dt_lin, flow):
        self.o = Oracle(Nx, Ny, Nz, 1, Re, Lx, Lz, dt_lin, flow)      # operators, LU factors and stage() for dt_lin
        self.n_list = [int(n) for n in n_list]
        assert all(1 <= n < self.o.nkx for n in self.n_list)
        self.Eg, self.E = int(Eg), int(Eg) * len(self.n_list)
        self.n_of = np.repeat(self.n_list, self.Eg)
        o = self.o
        self.v = np.zeros((self.E, o.nkz, o.Ny), np.complex128)
        self.eta = np.zeros_like(self.v)
        self.base = None

    # ---------------------------------------------------------------- base flow (frozen streamwise mean, reading L3)
    def set_base(self, vhat0, etahat0, U00, W00):
        """vhat0, etahat0 [nkz][Ny]: the kx = 0 plane of a DNS state; U00, W00 [Ny].  Stores U, V, W and their y and z
        derivatives on the padded z grid, real [Ny][Mz] each."""
        o = self.o
        v = np.zeros((1, o.nkx, o.nkz, o.Ny), np.complex128)
        e = np.zeros_like(v)
        v[0, 0], e[0, 0] = vhat0, etahat0
        o.set_state(v, e, np.asarray(U00, float)[None], np.asarray(W00, float)[None])   # normalises like dns_set_state
        u, v0, w, Du, Dv, Dw = o.velocities(o.v, o.eta, o.U, o.W)
        ikz = 1j * o.kz[:, None]
        phys = lambda f: np.einsum("mj,mq->jq", f, o.Ez_inv).real          # kx = 0: a real function of (y, z)
        U, V, W = u[0, 0], v0[0, 0], w[0, 0]
        self.base = {"U": phys(U), "V": phys(V), "W": phys(W),
                     "Uy": phys(Du[0, 0]), "Vy": phys(Dv[0, 0]), "Wy": phys(Dw[0, 0]),
                     "Uz": phys(ikz * U), "Vz": phys(ikz * V), "Wz": phys(ikz * W)}

    def set_state(self, vhat, etahat):
        v = np.array(vhat, dtype=np.complex128).reshape(self.v.shape)
        eta = np.array(etahat, dtype=np.complex128).reshape(self.v.shape)
        for f in (v, eta):
            f[..., 0] = 0.0
            f[..., -1] = 0.0                                                # PAPER.md:82 Eq. 8
        self.v, self.eta = v, eta

    # ---------------------------------------------------------------- velocities of one member (Eq. 17-18)
    def _velocities(self, e):
        o, n = self.o, self.n_of[e]
        ikx, ikz = 1j * o.kx[n], 1j * o.kz[:, None]
        al = o.alpha[n][:, None]
        v = self.v[e]
        Dv = v @ o.D.T
        u = (ikx * Dv - ikz * self.eta[e]) / al                             # Eq. 17
        w = (ikz * Dv + ikx * self.eta[e]) / al                             # Eq. 18
        u[:, [0, -1]] = 0.0
        w[:, [0, -1]] = 0.0
        return u, v, w

    def linear_vector(self, e, adjoint):
        """The vector N (spectral, [3][nkz][Ny]) that takes the place of u.grad u in Eq. 4-5:
        forward (B.2)  N_i = (U.grad) u_i + (u.grad) U_i ;  adjoint (B.5, reversed time)  N_i = -(U.grad) lam_i - U_j d_i lam_j."""
        o, n, B = self.o, self.n_of[e], self.base
        ikx, ikz = 1j * o.kx[n], 1j * o.kz[:, None]
        u, v, w = self._velocities(e)
        P = lambda f: np.einsum("mj,mq->jq", f, o.Ez_inv)                   # complex amplitude on the padded z grid
        pu, pv, pw = P(u), P(v), P(w)
        ux, vx, wx = ikx * pu, ikx * pv, ikx * pw                           # x is analytic
        uy, vy, wy = P(u @ o.D.T), P(v @ o.D.T), P(w @ o.D.T)
        uz, vz, wz = P(ikz * u), P(ikz * v), P(ikz * w)
        U, V, W = B["U"], B["V"], B["W"]
        adv = lambda fx, fy, fz: U * fx + V * fy + W * fz                   # (U.grad) f
        if not adjoint:
            Nu = adv(ux, uy, uz) + pv * B["Uy"] + pw * B["Uz"]              # + (u.grad) U ; dU/dx = 0
            Nv = adv(vx, vy, vz) + pv * B["Vy"] + pw * B["Vz"]
            Nw = adv(wx, wy, wz) + pv * B["Wy"] + pw * B["Wz"]
        else:
            Nu = -adv(ux, uy, uz) - (U * ux + V * vx + W * wx)              # - U_j d lam_j/dx
            Nv = -adv(vx, vy, vz) - (U * uy + V * vy + W * wy)              # - U_j d lam_j/dy
            Nw = -adv(wx, wy, wz) - (U * uz + V * vz + W * wz)              # - U_j d lam_j/dz
        S = lambda f: np.einsum("jq,mq->mj", f, o.Ez_fwd) / o.Mz            # back to the retained kz
        return np.stack([S(Nu), S(Nv), S(Nw)])

    def forcing(self, e, adjoint):
        """F, G of Eq. 4-5 at interior rows with the linear vector in place of u.grad u: [nkz][Ni] each."""
        o, n = self.o, self.n_of[e]
        ikx, ikz = 1j * o.kx[n], 1j * o.kz[:, None]
        Nu, Nv, Nw = self.linear_vector(e, adjoint)
        F = -o.alpha[n][:, None] * Nv - ikx * (Nu @ o.D.T) - ikz * (Nw @ o.D.T)
        G = ikz * Nu - ikx * Nw
        return F[:, 1:-1], G[:, 1:-1]

    # ---------------------------------------------------------------- CN/RK3 step of Eq. 12-13
    def _stage(self, v_t, eta_t, h, F, G):
        """Eq. 12-13 for every member and every kz of its own kx row, with the LU factors of the pinned Oracle (the same
        statements as Oracle.stage, restricted to the rows that are not identically zero):
          [I - g T] v' = [I + g T] v_t - h dt Delta^-1 F          (Eq. 12)
          [I - g Delta] eta' = [I + g Delta] eta_t - h dt G        (Eq. 13)"""
        import scipy.linalg as sla
        o = self.o
        hdt = h * o.dt
        v_n, eta_n = np.zeros_like(v_t), np.zeros_like(eta_t)
        for e in range(self.E):
            n = self.n_of[e]
            for m in range(o.nkz):
                a = o.alpha[n, m]
                Lf, luDel = o.lu[(h, a)], o.ops[a][2]
                rhs = Lf["B"] @ v_t[e, m, 1:-1] - hdt * sla.lu_solve(luDel, F[e, m])
                v_n[e, m, 1:-1] = sla.lu_solve(Lf["A"], rhs)
                rhs = Lf["Sp"] @ eta_t[e, m, 1:-1] - hdt * G[e, m]
                eta_n[e, m, 1:-1] = sla.lu_solve(Lf["Sm"], rhs)
        return v_n, eta_n

    def _forcing_all(self, adjoint):
        FG = [self.forcing(e, adjoint) for e in range(self.E)]
        return np.stack([f for f, _ in FG]), np.stack([g for _, g in FG])

    def step(self, nsteps=1, adjoint=False):
        for _ in range(int(nsteps)):
            v_t, e_t = self.v, self.eta
            F0, G0 = self._forcing_all(adjoint)
            self.v, self.eta = self._stage(v_t, e_t, 0.5, F0, G0)                                   # h = 1/2 with F^0
            F1, G1 = self._forcing_all(adjoint)
            self.v, self.eta = self._stage(v_t, e_t, 1.0, 2.0 * F1 - F0, 2.0 * G1 - G0)             # h = 1, 2 F^1 - F^0
            F2, G2 = self._forcing_all(adjoint)
            self.v, self.eta = self._stage(v_t, e_t, 1.0, (F0 + 4.0 * F1 + F2) / 6.0, (G0 + 4.0 * G1 + G2) / 6.0)

    # ---------------------------------------------------------------- energy inner product (B.1) and Gram-Schmidt
    def inner(self, a, b):
        ua, va, wa = self._velocities(a)
        ub, vb, wb = self._velocities(b)
        return 0.5 * np.einsum("mj,j->", np.conj(ua) * ub + np.conj(va) * vb + np.conj(wa) * wb, self.o.w)

    def energy(self):
        return np.array([self.inner(e, e).real for e in range(self.E)])

    def orthonormalise(self):
        """Modified Gram-Schmidt in member order within each kx group (reading L4), energy inner product."""
        for g in range(len(self.n_list)):
            for a in range(g * self.Eg, (g + 1) * self.Eg):
                nrm = np.sqrt(self.inner(a, a).real)
                self.v[a] /= nrm
                self.eta[a] /= nrm
                for b in range(a + 1, (g + 1) * self.Eg):
                    c = self.inner(a, b)
                    self.v[b] -= c * self.v[a]
                    self.eta[b] -= c * self.eta[a]

    def optimals(self, nsteps, niter):
        """Power iteration of PAPER.md:417.  Returns the gains E(T_opt)/E(0) of the last forward leg, [E]."""
        gains = None
        self.orthonormalise()
        for _ in range(int(niter)):
            self.step(nsteps, adjoint=False)
            gains = self.energy()                                           # initial energy is 1
            self.step(nsteps, adjoint=True)
            self.orthonormalise()
        return gains
