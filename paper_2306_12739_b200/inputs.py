"""Seeded synthetic inputs for the ensemble DNS step (shared by oracle tests, GPU tests and bench.py).

This module holds NONE of the method's arithmetic: no Chebyshev matrices, no transforms, no time
stepping.  It only (i) tabulates the five BASELINE.json configs, (ii) draws polynomial wall-normal
profiles with a seeded generator and (iii) scales them with exact polynomial integrals.

Recipe ("Perturbation recipe"; shapes follow PAPER.md:359 Table A.4):
  rng = numpy.random.default_rng([20230612, config, e]) per member e;
  for every listed (n, m):  vhat(y) = (1-y^2)^2 (a0 + a1 y + a2 y^2),  etahat(y) = (1-y^2)(b0 + b1 y + b2 y^2),
  a_i, b_i complex standard normal  ->  v = dv/dy = eta = 0 at the walls (Eq. 8), so the
  field is no-slip and (being built from v, eta) divergence-free by construction;
  on n = 0 the entries with m < 0 are the conjugates of m > 0 (real field);
  all coefficients of the member are scaled by one factor so that sqrt(2 E') = rms, where
  E' = 1/(2V) int |u'|^2 dV (definition) is evaluated in closed form by polynomial algebra.

State layout is the C-ABI layout of include/dns.h:  vhat, etahat [E][nkx][nkz][Ny] complex128,
nkx = Nx/2 (n = 0..Nx/2-1), nkz = Nz-1 with m in FFT order 0..Nz/2-1, -(Nz/2-1)..-1
(the paper's `mrange`);  y_j = -cos(pi j/(Ny-1));  U00, W00 [E][Ny] float64.
"""
from __future__ import annotations

import hashlib
from dataclasses import dataclass

import numpy as np
from numpy.polynomial import polynomial as npoly

COUETTE = 0
POISEUILLE_CMF = 1


@dataclass(frozen=True)
class Config:
    cid: int
    flow: int
    Re: float
    Lx: float
    Lz: float
    Nx: int
    Ny: int
    Nz: int
    E: int
    dt: float
    nsteps: int
    rms: float          # target perturbation rms (or lower bound when rms_hi is set)
    kcut2: int          # modes with n^2 + m^2 <= kcut2 (config 1 uses the box |n|,|m| <= 3 instead)
    box: int = 0        # if > 0: modes 0 <= n <= box, |m| <= box
    rms_hi: float = 0.0  # if > 0: per-member rms ~ U(rms, rms_hi)

    def with_E(self, E: int) -> "Config":
        return Config(**{**self.__dict__, "E": int(E)})

    @property
    def name(self) -> str:
        f = "couette" if self.flow == COUETTE else "poiseuille_cmf"
        return f"config{self.cid}:{f}_Re{self.Re:g}_{self.Nx}x{self.Ny}x{self.Nz}_E{self.E}"


_PI = np.pi
CONFIGS = {
    1: Config(1, COUETTE, 400.0, 1.75 * _PI, 1.2 * _PI, 16, 33, 16, 2, 0.02, 20, 0.05, 0, box=3),
    2: Config(2, COUETTE, 1000.0, 2 * _PI, _PI, 32, 49, 32, 64, 0.01, 200, 0.1, 16),
    3: Config(3, POISEUILLE_CMF, 2800.0, _PI, _PI / 2, 64, 97, 64, 16, 0.005, 100, 0.1, 36),
    4: Config(4, POISEUILLE_CMF, 1400.0, 2 * _PI, _PI, 48, 65, 48, 256, 0.01, 100, 0.05, 36, rms_hi=0.2),
    # config 5 = config 2's grid with E swept over {1,4,16,64,256,1024}, 50 steps
    5: Config(5, COUETTE, 1000.0, 2 * _PI, _PI, 32, 49, 32, 64, 0.01, 50, 0.1, 16),
}
SWEEP_E = (1, 4, 16, 64, 256, 1024)


def grid_y(Ny: int) -> np.ndarray:
    """Chebyshev-Gauss-Lobatto points, ascending from the lower wall (PAPER.md:95 flips cheb)."""
    return -np.cos(np.pi * np.arange(Ny) / (Ny - 1))


def m_index(m: int, Nz: int) -> int:
    """Position of spanwise mode m in the stored FFT order (PAPER.md:188 `mrange`)."""
    return m if m >= 0 else (Nz - 1) + m


def m_of_index(Nz: int) -> np.ndarray:
    h = Nz // 2
    return np.concatenate([np.arange(0, h), np.arange(-(h - 1), 0)])


def mode_list(cfg: Config):
    """Independent (n, m) pairs that receive random coefficients (n = 0 only with m > 0)."""
    out = []
    if cfg.box:
        ns, ms = range(0, cfg.box + 1), range(-cfg.box, cfg.box + 1)
        keep = lambda n, m: True
    else:
        r = int(np.sqrt(cfg.kcut2)) + 1
        ns, ms = range(0, r + 1), range(-r, r + 1)
        keep = lambda n, m: n * n + m * m <= cfg.kcut2
    for n in ns:
        for m in ms:
            if (n, m) == (0, 0) or not keep(n, m):
                continue
            if n == 0 and m < 0:
                continue
            if n > cfg.Nx // 2 - 1 or abs(m) > cfg.Nz // 2 - 1:
                continue
            out.append((n, m))
    return out


def _abs2_integral(c: np.ndarray) -> float:
    """int_{-1}^{1} |p(y)|^2 dy for a complex polynomial with ascending coefficients c (exact algebra)."""
    sq = npoly.polymul(c.real, c.real) + npoly.polymul(c.imag, c.imag)
    k = np.arange(sq.size)
    return float(np.sum(sq[k % 2 == 0] * 2.0 / (k[k % 2 == 0] + 1)))


def laminar_profile(cfg: Config, y: np.ndarray) -> np.ndarray:
    """Couette u = y (walls at +-1); Poiseuille u = 1.5 (1 - y^2), bulk velocity 1."""
    return y.copy() if cfg.flow == COUETTE else 1.5 * (1.0 - y * y)


def member_state(cfg: Config, e: int):
    """State of ensemble member e in ABI layout (without the leading member axis)."""
    Nx, Ny, Nz = cfg.Nx, cfg.Ny, cfg.Nz
    nkx, nkz = Nx // 2, Nz - 1
    y = grid_y(Ny)
    rng = np.random.default_rng([20230612, cfg.cid, e])
    rms = cfg.rms if cfg.rms_hi <= 0 else float(rng.uniform(cfg.rms, cfg.rms_hi))
    vhat = np.zeros((nkx, nkz, Ny), np.complex128)
    ehat = np.zeros((nkx, nkz, Ny), np.complex128)
    env_v = np.array([1.0, 0.0, -2.0, 0.0, 1.0])   # (1-y^2)^2
    env_e = np.array([1.0, 0.0, -1.0])             # (1-y^2)
    energy = 0.0
    for (n, m) in mode_list(cfg):
        a = rng.standard_normal(3) + 1j * rng.standard_normal(3)
        b = rng.standard_normal(3) + 1j * rng.standard_normal(3)
        pv = npoly.polymul(env_v, a)
        pe = npoly.polymul(env_e, b)
        vhat[n, m_index(m, Nz)] = npoly.polyval(y, pv)
        ehat[n, m_index(m, Nz)] = npoly.polyval(y, pe)
        if n == 0:
            vhat[0, m_index(-m, Nz)] = np.conj(vhat[0, m_index(m, Nz)])
            ehat[0, m_index(-m, Nz)] = np.conj(ehat[0, m_index(m, Nz)])
        alpha = (2 * np.pi * n / cfg.Lx) ** 2 + (2 * np.pi * m / cfg.Lz) ** 2
        # |u|^2 + |w|^2 = (|dv/dy|^2 + |eta|^2)/alpha for one Fourier mode; every listed pair stands for
        # itself and its Hermitian partner, hence the factor 2;  E' = (1/4) int sum_modes |.|^2 dy
        dens = _abs2_integral(pv) + (_abs2_integral(npoly.polyder(pv)) + _abs2_integral(pe)) / alpha
        energy += 2.0 * 0.25 * dens
    scale = rms / np.sqrt(2.0 * energy)
    vhat *= scale
    ehat *= scale
    vhat[..., 0] = 0.0
    vhat[..., -1] = 0.0
    ehat[..., 0] = 0.0
    ehat[..., -1] = 0.0
    U00 = laminar_profile(cfg, y)
    W00 = np.zeros(Ny)
    return vhat, ehat, U00, W00, rms


def make_state(cfg: Config, members=None):
    """Arrays for members `members` (default: all E) in ABI layout, plus a SHA-256 of the bytes."""
    if members is None:
        members = range(cfg.E)
    members = list(members)
    nkx, nkz = cfg.Nx // 2, cfg.Nz - 1
    vhat = np.empty((len(members), nkx, nkz, cfg.Ny), np.complex128)
    ehat = np.empty_like(vhat)
    U00 = np.empty((len(members), cfg.Ny))
    W00 = np.empty_like(U00)
    rms = np.empty(len(members))
    for i, e in enumerate(members):
        vhat[i], ehat[i], U00[i], W00[i], rms[i] = member_state(cfg, e)
    h = hashlib.sha256()
    for a in (vhat, ehat, U00, W00):
        h.update(np.ascontiguousarray(a).tobytes())
    return {"vhat": vhat, "etahat": ehat, "U00": U00, "W00": W00, "rms": rms, "sha256": h.hexdigest()}


def broadband_member_state(cfg: Config, e: int, amp: float = 0.01):
    """A second, rough family of inputs for parity tests at the full sizes: EVERY retained pair (n, m) != (0, 0) carries
    energy, amplitude amp (1 + n^2 + m^2)^(-5/6) (a k^(-5/3)-like spectrum), and the wall-normal profiles are Chebyshev
    series of degree Ny - 5 with slowly decaying random coefficients c_k ~ N(0,1)/sqrt(1 + k) under the no-slip
    envelopes:  vhat = (1-y^2)^2 sum c_k T_k(y),  etahat = (1-y^2) sum c'_k T_k(y)  (Eq. 8).  No scaling by
    the energy (that would need the method's arithmetic): amp sets the level directly."""
    Nx, Ny, Nz = cfg.Nx, cfg.Ny, cfg.Nz
    nkx, nkz = Nx // 2, Nz - 1
    y = grid_y(Ny)
    rng = np.random.default_rng([20230612, 100 + cfg.cid, e])
    deg = Ny - 5
    decay = 1.0 / np.sqrt(1.0 + np.arange(deg + 1))
    T = np.cos(np.outer(np.arange(deg + 1), np.arccos(np.clip(y, -1.0, 1.0))))     # T_k(y_j)
    mo = m_of_index(Nz)
    a = amp * (1.0 + np.arange(nkx)[:, None] ** 2 + mo[None, :] ** 2) ** (-5.0 / 6.0)
    cv = (rng.standard_normal((nkx, nkz, deg + 1)) + 1j * rng.standard_normal((nkx, nkz, deg + 1))) * decay
    ce = (rng.standard_normal((nkx, nkz, deg + 1)) + 1j * rng.standard_normal((nkx, nkz, deg + 1))) * decay
    vhat = a[:, :, None] * (cv @ T) * ((1.0 - y * y) ** 2)[None, None, :]
    ehat = a[:, :, None] * (ce @ T) * (1.0 - y * y)[None, None, :]
    vhat[0, 0] = 0.0
    ehat[0, 0] = 0.0
    for i, m in enumerate(mo):                     # real field: the m < 0 half of the n = 0 plane mirrors m > 0
        if m < 0:
            vhat[0, i] = np.conj(vhat[0, m_index(-int(m), Nz)])
            ehat[0, i] = np.conj(ehat[0, m_index(-int(m), Nz)])
    for f in (vhat, ehat):
        f[..., 0] = 0.0
        f[..., -1] = 0.0
    return vhat, ehat, laminar_profile(cfg, y), np.zeros(Ny)


def make_broadband_state(cfg: Config, members=None, amp: float = 0.01):
    members = list(range(cfg.E) if members is None else members)
    nkx, nkz = cfg.Nx // 2, cfg.Nz - 1
    vhat = np.empty((len(members), nkx, nkz, cfg.Ny), np.complex128)
    ehat = np.empty_like(vhat)
    U00 = np.empty((len(members), cfg.Ny))
    W00 = np.empty_like(U00)
    for i, e in enumerate(members):
        vhat[i], ehat[i], U00[i], W00[i] = broadband_member_state(cfg, e, amp)
    return {"vhat": vhat, "etahat": ehat, "U00": U00, "W00": W00}


def plan_args(cfg: Config, E=None):
    """Positional arguments of dns_plan_create / the oracle constructor."""
    return (cfg.Nx, cfg.Ny, cfg.Nz, cfg.E if E is None else int(E), cfg.Re, cfg.Lx, cfg.Lz, cfg.dt, cfg.flow)
