"""ORACLE for the ensemble CN/RK3 step of arXiv 2306.12739 -- TEST INFRASTRUCTURE ONLY.

A plain, slow, fp64 CPU restatement of the paper's time step, written from PAPER.md in the paper's
order and notation, for parity-checking the CUDA library.  Only `tests/`, `__graft_entry__.smoke()` and
`bench.py`'s cpu_baseline / `--impl reference` legs may import this file; the product path
(`paper_2306_12739_b200`) never does, and this file imports nothing from the product.

Primitives are the slowest obvious ones: dense DFT sums (matrices of exp(+-2 pi i n p / M) built from the
integer n*p mod M, applied with matmul), dense Chebyshev differentiation matrices, dense LU with partial
pivoting (scipy.linalg.lu_factor / lu_solve) for every solve.  The oracle never forms the inverse matrices
the GPU path multiplies with; it factors each left-hand side once and solves per stage.

What pins it (tests/test_oracle_pins.py, `-m "not gpu"`): P1 D exact on polynomials; P2 laminar
Couette/Poiseuille are fixed points (gamma = 2c/Re); P3 manufactured solves for Delta and the clamped
fourth derivative; P4 divergence / vorticity identities and exact no-slip; P5 flux conservation; P6 the
closed-form Crank-Nicolson amplification of a Squire mode; P7 Orr-Sommerfeld growth rate and phase speed
against an independent generalised eigen-solve and Orszag's published eigenvalue; P8 temporal order;
P9 the dealiasing cut-off; P10 translation / reflection covariance; P11 the kinetic-energy budget;
P12 member independence; P13 LU path vs explicitly inverted matrices; P14 single-harmonic DFT;
P15 one-point statistics against Parseval sums and the closed form of a single spanwise mode;
P16 the RK3 stage weights of PAPER.md:126 against Kutta's amplification polynomial 1 + z + z^2/2 + z^3/6 of an
inviscid pointwise-advection Squire mode (and third-order convergence in that limit).
Rows f1 / f2 of SURVEY.md 8(f) (tests/test_oracle_pins_forms.py): P17 the rotational form omega x u against the vector
identity (u.grad)u = omega x u + grad(|u|^2/2), pointwise orthogonality to u, the Orr-Sommerfeld growth rates, the laminar
fixed points, the energy budget and the Kutta polynomial; P18 the ensemble-coupled streamwise-mean flow
against the identical-member limit, the shared-mean invariant and the ensemble-mean energy budget.
Parity with the author's MATLAB output: UNPINNED (code and data are not available here); in particular
reading A7 (only d^4/dy^4 uses the clamped matrix) is pinned against the PDE, not against that code.

Citations are PAPER.md:<line>.  Readings of silent / garbled passages (A1..A17) are listed in DESIGN.md.
"""
from __future__ import annotations

import numpy as np
import scipy.linalg as sla

COUETTE = 0
POISEUILLE_CMF = 1
CONVECTIVE = 0        # nonlinear term u . grad u_i, the paper's form
ROTATIONAL = 1        # omega x u (reading F1 of DESIGN.md)
UNCOUPLED = 0         # independent members
STREAMWISE_MEAN = 1   # members share the streamwise-mean flow (row f2, reading F2 of DESIGN.md)


# --------------------------------------------------------------------------------------------------
# O-setup: Chebyshev collocation (PAPER.md:95-96 Listing 1, :112)
# --------------------------------------------------------------------------------------------------
def cheb_points(Ny: int) -> np.ndarray:
    """y_j = -cos(pi j/(Ny-1)): Gauss-Lobatto points ascending from the lower wall (the
    paper flips `cheb` so that the grid ascends)."""
    return -np.cos(np.pi * np.arange(Ny) / (Ny - 1))


def cheb_D(Ny: int) -> np.ndarray:
    """First-derivative collocation matrix on cheb_points (PAPER.md:95 `cheb(N+1)`, ref. [26]):
    D_ij = (c_i/c_j) (-1)^(i+j) / (y_i - y_j), c = 2 at the two ends else 1; D_ii = -sum_{j!=i} D_ij."""
    y = cheb_points(Ny)
    c = np.ones(Ny)
    c[0] = c[-1] = 2.0
    D = np.zeros((Ny, Ny))
    for i in range(Ny):
        for j in range(Ny):
            if i != j:
                D[i, j] = (c[i] / c[j]) * (-1.0) ** (i + j) / (y[i] - y[j])
    for i in range(Ny):
        D[i, i] = -(np.sum(D[i, :i]) + np.sum(D[i, i + 1:]))
    return D


def clamped_D4(Ny: int) -> np.ndarray:
    """Fourth derivative at the interior nodes with BOTH v = dv/dy = 0 built in (`cheb4bc`
    [25]): the interpolant is p(y) = (1-y^2) q(y) with q(+-1) = 0, q_j = v_j/(1-y_j^2); the product rule
    gives p'''' = (1-y^2) q'''' - 8 y q''' - 12 q''  (restated from the definition, reading A7)."""
    y = cheb_points(Ny)
    D = cheb_D(Ny)
    D2 = D @ D
    D3 = D2 @ D
    D4 = D3 @ D
    full = np.diag(1.0 - y * y) @ D4 - 8.0 * np.diag(y) @ D3 - 12.0 * D2
    return full[1:-1, 1:-1] @ np.diag(1.0 / (1.0 - y[1:-1] ** 2))


def clenshaw_curtis(Ny: int) -> np.ndarray:
    """Quadrature weights on cheb_points from their definition: sum_j w_j T_k(y_j) = int_{-1}^{1} T_k dy
    for k = 0..Ny-1 (= 2/(1-k^2) for even k, 0 for odd k)."""
    y = cheb_points(Ny)
    k = np.arange(Ny)
    T = np.cos(np.outer(k, np.arccos(np.clip(y, -1.0, 1.0))))
    mom = np.zeros(Ny)
    mom[0::2] = 2.0 / (1.0 - k[0::2].astype(float) ** 2)
    return np.linalg.solve(T, mom)


# --------------------------------------------------------------------------------------------------
# naive DFT (PAPER.md:225 `fft2_cuben`; convention f = sum fhat exp(+i(kx x + kz z)), reading A5)
# --------------------------------------------------------------------------------------------------
def dft_matrix(modes: np.ndarray, M: int, sign: int) -> np.ndarray:
    """exp(sign * 2 pi i * mode * p / M) for p = 0..M-1, angle taken from the integer (mode*p mod M)."""
    modes = np.asarray(modes, dtype=np.int64)
    r = (modes[:, None] * np.arange(M, dtype=np.int64)[None, :]) % M
    ang = 2.0 * np.pi * r.astype(float) / M
    return np.cos(ang) + 1j * sign * np.sin(ang)


class Oracle:
    """CN/RK3 ensemble step in the v-eta formulation (PAPER.md:68-87 Eq. 4-9, :114-126, :149-167 Eq. 12-15).

    State layout = the C-ABI layout: vhat, etahat [E][nkx][nkz][Ny] complex128 (n = 0..Nx/2-1; m in FFT order
    0..Nz/2-1, -(Nz/2-1)..-1), U00, W00 [E][Ny].
    """

    def __init__(self, Nx, Ny, Nz, E, Re, Lx, Lz, dt, flow, form=CONVECTIVE, coupling=UNCOUPLED):
        self.Nx, self.Ny, self.Nz, self.E = int(Nx), int(Ny), int(Nz), int(E)
        self.Re, self.Lx, self.Lz, self.dt, self.flow = float(Re), float(Lx), float(Lz), float(dt), int(flow)
        self.form, self.coupling = int(form), int(coupling)
        self.Mx, self.Mz = 3 * self.Nx // 2, 3 * self.Nz // 2          # 3/2 rule
        self.nkx, self.nkz = self.Nx // 2, self.Nz - 1                 # retained |n| <= Nx/2-1 (reading A2, A3)
        self.Ni = self.Ny - 2
        self.Uw = 1.0 if flow == COUETTE else 0.0                      # PAPER.md:85 Eq. 9
        self.y = cheb_points(self.Ny)
        self.D = cheb_D(self.Ny)
        self.D2F = self.D @ self.D
        self.D2 = self.D2F[1:-1, 1:-1]                                 # interior block (reading A1)
        self.D4c = clamped_D4(self.Ny)
        self.w = clenshaw_curtis(self.Ny)
        self.n_of = np.arange(self.nkx)
        h2 = self.Nz // 2
        self.m_of = np.concatenate([np.arange(0, h2), np.arange(-(h2 - 1), 0)])
        self.kx = 2.0 * np.pi * self.n_of / self.Lx
        self.kz = 2.0 * np.pi * self.m_of / self.Lz
        self.alpha = self.kx[:, None] ** 2 + self.kz[None, :] ** 2     # [nkx][nkz]
        self._setup_solvers()
        # DFT matrices over the retained modes only (the sums in SURVEY 8(c) O-nonlinear)
        self.n_full = np.arange(-(self.nkx - 1), self.nkx)             # Hermitian-completed n range
        self.Ex_inv = dft_matrix(self.n_full, self.Mx, +1)             # [2nkx-1][Mx]
        self.Ez_inv = dft_matrix(self.m_of, self.Mz, +1)               # [nkz][Mz]
        self.Ex_fwd = dft_matrix(self.n_of, self.Mx, -1)               # [nkx][Mx]
        self.Ez_fwd = dft_matrix(self.m_of, self.Mz, -1)               # [nkz][Mz]
        self.t = 0.0
        self.gamma = np.zeros(self.E)
        self.v = np.zeros((self.E, self.nkx, self.nkz, self.Ny), np.complex128)
        self.eta = np.zeros_like(self.v)
        self.U = np.tile(self.Uw * self.y, (self.E, 1))
        self.W = np.zeros((self.E, self.Ny))
        self.Qstar = np.zeros(self.E)

    # ---------------------------------------------------------------- O-setup item 3
    def _setup_solvers(self):
        I = np.eye(self.Ni)
        self.lu = {}      # (h, alpha) -> dict of LU factors
        self.ops = {}     # alpha -> (Delta, T)
        for a in np.unique(self.alpha):
            if a == 0.0:
                continue
            Del = self.D2 - a * I                                       # Delta
            DelDel = self.D4c - 2.0 * a * self.D2 + a * a * I           # Delta Delta
            luDel = sla.lu_factor(Del)
            T = sla.lu_solve(luDel, DelDel)                             # Delta^-1 Delta Delta (Eq. 12)
            self.ops[a] = (Del, T, luDel)
            for h in (0.5, 1.0):
                g = h * self.dt / (2.0 * self.Re)
                self.lu[(h, a)] = {
                    "A": sla.lu_factor(I - g * T), "B": I + g * T,          # Eq. 12
                    "Sm": sla.lu_factor(I - g * Del), "Sp": I + g * Del,    # Eq. 13 (Listing 3)
                }
        self.mean = {}
        IF = np.eye(self.Ny)
        for h in (0.5, 1.0):
            g = h * self.dt / (2.0 * self.Re)
            S0m = IF - g * self.D2F                                     # Eq. 14-15 lhs
            S0p = IF + g * self.D2F
            self.mean[h] = {"S0m": S0m, "S0p": S0p, "lu": sla.lu_factor(S0m[1:-1, 1:-1])}

    # ---------------------------------------------------------------- state I/O (SURVEY 8(b) input normalisation)
    def set_state(self, vhat, etahat, U00, W00):
        v = np.array(vhat, dtype=np.complex128).reshape(self.E, self.nkx, self.nkz, self.Ny)
        eta = np.array(etahat, dtype=np.complex128).reshape(v.shape)
        U = np.array(U00, dtype=float).reshape(self.E, self.Ny)
        W = np.array(W00, dtype=float).reshape(self.E, self.Ny)
        for f in (v, eta):
            f[..., 0] = 0.0
            f[..., -1] = 0.0                                            # PAPER.md:82 Eq. 8
            f[:, 0, 0, :] = 0.0                                         # V00 = eta00 = 0
            for i, m in enumerate(self.m_of):                           # reading A13: m > 0 authoritative on n = 0
                if m < 0:
                    f[:, 0, i, :] = np.conj(f[:, 0, -m, :])
        U[:, 0], U[:, -1] = -self.Uw, self.Uw                           # PAPER.md:85 Eq. 9
        W[:, 0] = W[:, -1] = 0.0
        self.v, self.eta, self.U, self.W = v, eta, U, W
        self.Qstar = 0.5 * U @ self.w                                   # target bulk flux (reading A6)
        self.t = 0.0
        self.gamma = np.zeros(self.E)

    def get_state(self):
        return self.v.copy(), self.eta.copy(), self.U.copy(), self.W.copy()

    def add_increment(self, dv, deta):
        """state += (dv, deta) between two steps: how a caller applies one realisation of a stochastic forcing
        (the realisations themselves are the caller's, reading F2).  Wall rows, the (0,0) column and
        the m < 0 half of the n = 0 plane of the result are normalised as in set_state."""
        v = self.v + np.asarray(dv, dtype=np.complex128).reshape(self.v.shape)
        eta = self.eta + np.asarray(deta, dtype=np.complex128).reshape(self.eta.shape)
        t, g, Q = self.t, self.gamma, self.Qstar
        self.set_state(v, eta, self.U, self.W)
        self.t, self.gamma, self.Qstar = t, g, Q

    # ---------------------------------------------------------------- a1-a3: velocities from (v, eta) (Eq. 17-18)
    def velocities(self, v, eta, U, W):
        """u, w (and Dv, Du, Dw) in spectral space; wall rows imposed (reading A10); (0,0) = mean profiles."""
        ikx = 1j * self.kx[None, :, None, None]
        ikz = 1j * self.kz[None, None, :, None]
        al = self.alpha.copy()
        al[0, 0] = 1.0
        al = al[None, :, :, None]
        v = v.copy()
        v[:, 0, 0, :] = 0.0
        Dv = v @ self.D.T                                               # a1: D v (y is the last axis)
        u = (ikx * Dv - ikz * eta) / al                                 # Eq. 17
        w = (ikz * Dv + ikx * eta) / al                                 # Eq. 18
        u[..., 0] = u[..., -1] = 0.0
        w[..., 0] = w[..., -1] = 0.0
        u[:, 0, 0, :] = U
        w[:, 0, 0, :] = W
        Du = u @ self.D.T                                               # a3
        Dw = w @ self.D.T
        return u, v, w, Du, Dv, Dw

    # ---------------------------------------------------------------- a4 / a6: naive DFTs
    def to_physical(self, fh):
        """f(x_p, z_q) = sum_{n,m} fhat(n,m) exp(2 pi i (n p/Mx + m q/Mz)) over the Hermitian-completed
        retained modes, fhat(-n,-m) = conj fhat(n,m).  fh: [E][nkx][nkz][Ny] -> real [E][Ny][Mx][Mz]."""
        E = fh.shape[0]
        full = np.zeros((E, 2 * self.nkx - 1, self.nkz, self.Ny), np.complex128)
        full[:, self.nkx - 1:, :, :] = fh
        mneg = np.array([int(np.where(self.m_of == -m)[0][0]) for m in self.m_of])
        for n in range(1, self.nkx):
            full[:, self.nkx - 1 - n, :, :] = np.conj(fh[:, n, mneg, :])
        g = np.einsum("enmj,mq->enqj", full, self.Ez_inv, optimize=True)
        f = np.einsum("enqj,np->ejpq", g, self.Ex_inv, optimize=True)
        return f.real

    def to_spectral(self, f):
        """Nhat(n,m) = (Mx Mz)^-1 sum_{p,q} N(p,q) exp(-2 pi i (n p/Mx + m q/Mz)) on retained modes.
        f: real [E][Ny][Mx][Mz] -> [E][nkx][nkz][Ny]."""
        g = np.einsum("ejpq,np->ejnq", f.astype(np.complex128), self.Ex_fwd, optimize=True)
        fh = np.einsum("ejnq,mq->enmj", g, self.Ez_fwd, optimize=True)
        return fh / (self.Mx * self.Mz)

    # ---------------------------------------------------------------- O-nonlinear (a1-a7)
    def advection(self, v, eta, U, W):
        """The nonlinear vector in physical space on the padded grid, real [E][Ny][Mx][Mz] each, and the two mean-flow
        sources S_u, S_w [E][Ny] of Eq. 6-7.
        CONVECTIVE (the paper's form): N_i = u . grad u_i; S_u = d/dy [uv]00, S_w = d/dy [wv]00 with the
        plane means of the products (reading A9).
        ROTATIONAL (row f1): H = omega x u with omega = curl u = (dw/dy - dv/dz, du/dz - dw/dx, dv/dx - du/dy).
        Since (u . grad)u = omega x u + grad(|u|^2/2) and Eq. 4-5 are what is left of the momentum equation once
        gradients are eliminated, F and G keep their form with H in place of N; the plane mean of
        d/dx(|u|^2/2) vanishes, so the mean-flow sources are the plane means of H_x and H_z themselves."""
        ikx = 1j * self.kx[None, :, None, None]
        ikz = 1j * self.kz[None, None, :, None]
        u, v0, w, Du, Dv, Dw = self.velocities(v, eta, U, W)
        P = self.to_physical
        pu, pv, pw = P(u), P(v0), P(w)
        if self.form == CONVECTIVE:
            Nu = pu * P(ikx * u) + pv * P(Du) + pw * P(ikz * u)            # u . grad u   (a5)
            Nv = pu * P(ikx * v0) + pv * P(Dv) + pw * P(ikz * v0)          # u . grad v
            Nw = pu * P(ikx * w) + pv * P(Dw) + pw * P(ikz * w)            # u . grad w
            uv00 = np.mean(pu * pv, axis=(2, 3))                           # plane means [uv]00(y) (reading A9)
            wv00 = np.mean(pw * pv, axis=(2, 3))
            Su = uv00 @ self.D.T                                           # d/dy [uv]00 (Eq. 6)
            Sw = wv00 @ self.D.T                                           # d/dy [wv]00 (Eq. 7)
            return Nu, Nv, Nw, Su, Sw
        ox = P(Dw - ikz * v0)                                              # omega_x = dw/dy - dv/dz
        oy = P(ikz * u - ikx * w)                                          # omega_y = du/dz - dw/dx (= eta)
        oz = P(ikx * v0 - Du)                                              # omega_z = dv/dx - du/dy
        Hx = oy * pw - oz * pv
        Hy = oz * pu - ox * pw
        Hz = ox * pv - oy * pu
        return Hx, Hy, Hz, np.mean(Hx, axis=(2, 3)), np.mean(Hz, axis=(2, 3))

    def nonlinear(self, v, eta, U, W):
        """F, G at interior rows for all (n,m) and the mean-flow sources S_u, S_w (PAPER.md:72-78 Eq. 4-7, :108).
        With coupling = STREAMWISE_MEAN (row f2: "Each ensemble member shares a common streamwise
        mean flow, which is updated at every time-step by the perturbation Reynolds stresses averaged over the
        ensemble members") the kx = 0 part of the nonlinear vector -- all that forces the streamwise-mean flow -- and
        the two mean-flow sources are replaced by their average over the members; n != 0 is untouched."""
        ikx = 1j * self.kx[None, :, None, None]
        ikz = 1j * self.kz[None, None, :, None]
        Nu, Nv, Nw, Su, Sw = self.advection(v, eta, U, W)
        Nuh, Nvh, Nwh = self.to_spectral(Nu), self.to_spectral(Nv), self.to_spectral(Nw)   # a6
        if self.coupling == STREAMWISE_MEAN:
            for f in (Nuh, Nvh, Nwh):
                f[:, 0, :, :] = np.sum(f[:, 0, :, :], axis=0) / f.shape[0]
            Su = np.tile(np.sum(Su, axis=0) / Su.shape[0], (Su.shape[0], 1))
            Sw = np.tile(np.sum(Sw, axis=0) / Sw.shape[0], (Sw.shape[0], 1))
        al = self.alpha[None, :, :, None]
        F = -al * Nvh - ikx * (Nuh @ self.D.T) - ikz * (Nwh @ self.D.T)   # a7 (Eq. 4 with Eq. 10's sign)
        G = ikz * Nuh - ikx * Nwh                                          # a7 (Eq. 5)
        F = F[..., 1:-1].copy()
        G = G[..., 1:-1].copy()
        F[:, 0, 0, :] = 0.0
        G[:, 0, 0, :] = 0.0
        return F, G, Su, Sw

    # ---------------------------------------------------------------- O-stage (a9, a10)
    def stage(self, v_t, eta_t, U_t, W_t, h, Fc, Gc, Suc, Swc):
        E = v_t.shape[0]
        v_n = np.zeros_like(v_t)
        eta_n = np.zeros_like(eta_t)
        hdt = h * self.dt
        for n in range(self.nkx):
            for m in range(self.nkz):
                a = self.alpha[n, m]
                if a == 0.0:
                    continue
                L = self.lu[(h, a)]
                luDel = self.ops[a][2]
                # Eq. 12: [I - g T] v' = [I + g T] v_t - h dt Delta^-1 F
                rhs = L["B"] @ v_t[:, n, m, 1:-1].T - hdt * sla.lu_solve(luDel, Fc[:, n, m, :].T)
                v_n[:, n, m, 1:-1] = sla.lu_solve(L["A"], rhs).T
                # Eq. 13: [I - g Delta] eta' = [I + g Delta] eta_t - h dt G
                rhs = L["Sp"] @ eta_t[:, n, m, 1:-1].T - hdt * Gc[:, n, m, :].T
                eta_n[:, n, m, 1:-1] = sla.lu_solve(L["Sm"], rhs).T
        Mh = self.mean[h]
        S0m, S0p = Mh["S0m"], Mh["S0p"]
        U_n = np.zeros_like(U_t)
        W_n = np.zeros_like(W_t)
        gam = np.zeros(E)
        for e in range(E):
            U_lo, U_hi = -self.Uw, self.Uw
            # Eq. 14 with the boundary columns moved to the rhs (f+-)
            r = (S0p @ U_t[e])[1:-1] - hdt * Suc[e, 1:-1] - S0m[1:-1, 0] * U_lo - S0m[1:-1, -1] * U_hi
            Up = np.zeros(self.Ny)
            Up[1:-1] = sla.lu_solve(Mh["lu"], r)
            Up[0], Up[-1] = U_lo, U_hi
            if self.flow == POISEUILLE_CMF:
                Ug = np.zeros(self.Ny)
                Ug[1:-1] = sla.lu_solve(Mh["lu"], hdt * np.ones(self.Ni))
                gam[e] = (self.Qstar[e] - 0.5 * self.w @ Up) / (0.5 * self.w @ Ug)   # reading A6
                Up = Up + gam[e] * Ug
            U_n[e] = Up
            r = (S0p @ W_t[e])[1:-1] - hdt * Swc[e, 1:-1]               # Eq. 15
            W_n[e, 1:-1] = sla.lu_solve(Mh["lu"], r)
        return v_n, eta_n, U_n, W_n, gam

    # ---------------------------------------------------------------- O-step
    def step(self, nsteps=1):
        for _ in range(int(nsteps)):
            s_t = (self.v, self.eta, self.U, self.W)
            N0 = self.nonlinear(*s_t)
            s1 = self.stage(*s_t, 0.5, *N0)                                        # h = 1/2 with F^0
            N1 = self.nonlinear(*s1[:4])
            c2 = tuple(2.0 * a - b for a, b in zip(N1, N0))                        # 2 F^1 - F^0, h = 1
            s2 = self.stage(*s_t, 1.0, *c2)
            N2 = self.nonlinear(*s2[:4])
            c3 = tuple((a + 4.0 * b + c) / 6.0 for a, b, c in zip(N0, N1, N2))     # (F^0 + 4 F^1 + F^2)/6, h = 1
            s3 = self.stage(*s_t, 1.0, *c3)
            self.v, self.eta, self.U, self.W, self.gamma = s3
            self.t += self.dt

    # ---------------------------------------------------------------- diagnostics
    def energy(self, v=None, eta=None, U=None, W=None):
        """E = 1/(2V) int |u|^2 dV by Parseval over the Hermitian-completed modes and
        Clenshaw-Curtis in y."""
        if v is None:
            v, eta, U, W = self.v, self.eta, self.U, self.W
        u, v0, w, _, _, _ = self.velocities(v, eta, U, W)
        dens = np.abs(u) ** 2 + np.abs(v0) ** 2 + np.abs(w) ** 2         # [E][nkx][nkz][Ny]
        cn = np.where(self.n_of == 0, 1.0, 2.0)[None, :, None, None]
        return 0.25 * np.einsum("enmj,j->e", cn * dens, self.w)

    def one_point_stats(self):
        """One-point statistics of the current state ("the time-averaged streamwise- and
        spanwise-mean velocity profile U(y), the rms profile of the velocity fluctuations from the mean profile
        (u', v', w') and the tangential Reynolds stress u'v'"): for one instant, the plane averages over the
        padded physical grid, written out as the definition -- [E][Ny][5] = U, <u'u'>, <v'v'>, <w'w'>, <u'v'>,
        primes = deviations from the (x, z) plane mean.  A time average is the mean of these over samples."""
        u, v, w, _, _, _ = self.velocities(self.v, self.eta, self.U, self.W)
        up, vp, wp = self.to_physical(u), self.to_physical(v), self.to_physical(w)      # [E][Ny][Mx][Mz]
        out = np.zeros((self.E, self.Ny, 5))
        Um, Vm, Wm = up.mean(axis=(2, 3)), vp.mean(axis=(2, 3)), wp.mean(axis=(2, 3))
        uf, vf, wf = up - Um[:, :, None, None], vp - Vm[:, :, None, None], wp - Wm[:, :, None, None]
        out[:, :, 0] = Um
        out[:, :, 1] = (uf * uf).mean(axis=(2, 3))
        out[:, :, 2] = (vf * vf).mean(axis=(2, 3))
        out[:, :, 3] = (wf * wf).mean(axis=(2, 3))
        out[:, :, 4] = (uf * vf).mean(axis=(2, 3))
        return out

    def diagnostics(self):
        out = np.zeros((self.E, 6))
        out[:, 0] = self.energy()
        dU = self.U @ self.D.T
        out[:, 1] = dU[:, 0]
        out[:, 2] = dU[:, -1]
        out[:, 3] = 0.5 * self.U @ self.w
        out[:, 4] = self.gamma
        out[:, 5] = self.t
        return out
