"""Free-propagator lookup tables (input data).

Convention (readings G17-G19; the paper fixes only
g_sigma(0^-) = -<n_sigma>_0):

    g(r, tau) = (1/N_k) sum_k e^{i k.r} e^{-xi_k tau} (1 - f(xi_k)),   0 <= tau <= beta,

tabulated on `n_tau` nodes tau_k = k beta / (n_tau - 1), both ends included.
Anti-periodic continuation, the 0^- rule and the linear interpolation belong to
the *method* (tabulation step A2) and are therefore NOT in this file.

square    : xi_k = -2t (cos kx + cos ky) - mu_eff
honeycomb : 2x2 Bloch matrix [[-mu_eff, eps],[eps*, -mu_eff]],  eps(k) = -t (1 + e^{i k.b1} + e^{i k.b2})
            (Eq. 48 with Delta_sigma = 0), bands xi_pm = +-|eps| - mu_eff, projectors
            P_pm = 1/2 [[1, +-eps/|eps|],[+-eps*/|eps|, 1]]  (1/2 * identity at a Dirac point).

Table layout (C-contiguous fp64):  T[block][s * n_sub + s'][dx * L + dy][k]
with dx, dy in [0, L) the displacement r = r_from - r_to modulo L.
"""
from dataclasses import dataclass
import numpy as np


@dataclass
class PropTable:
    lattice: int
    L: int
    n_sub: int
    beta: float
    n_tau: int
    mu_eff: tuple
    data: np.ndarray        # [n_blocks][n_sub^2][L*L][n_tau] fp64

    @property
    def n_blocks(self) -> int:
        return self.data.shape[0]


def _occupation_factor(xi, tau, beta):
    """e^{-xi tau} (1 - f(xi)) = e^{-xi tau} / (1 + e^{-beta xi}), overflow-free."""
    xi = np.asarray(xi, dtype=np.float64)
    pos = xi >= 0
    out = np.empty(np.broadcast(xi, tau).shape, dtype=np.float64)
    xi_b = np.broadcast_to(xi, out.shape)
    tau_b = np.broadcast_to(tau, out.shape)
    p = np.broadcast_to(pos, out.shape)
    out[p] = np.exp(-xi_b[p] * tau_b[p]) / (1.0 + np.exp(-beta * xi_b[p]))
    q = ~p
    out[q] = np.exp(xi_b[q] * (beta - tau_b[q])) / (1.0 + np.exp(beta * xi_b[q]))
    return out


def build_table(lattice: int, L: int, t: float, mu_eff, beta: float, n_tau: int = 1024) -> PropTable:
    mu_eff = tuple(float(m) for m in mu_eff)
    taus = np.arange(n_tau, dtype=np.float64) * (beta / (n_tau - 1))
    k1 = 2.0 * np.pi * np.arange(L) / L
    K1, K2 = np.meshgrid(k1, k1, indexing="ij")             # [L][L]
    n_sub = 2 if lattice == 1 else 1
    data = np.zeros((len(mu_eff), n_sub * n_sub, L * L, n_tau), dtype=np.float64)
    # phase e^{i k.r} for r = (dx, dy): use inverse FFT over the k grid.
    for b, mu in enumerate(mu_eff):
        if lattice == 0:
            xi = -2.0 * t * (np.cos(K1) + np.cos(K2)) - mu    # [L][L]
            w = _occupation_factor(xi[:, :, None], taus[None, None, :], beta)   # [L][L][n_tau]
            # (1/N) sum_k e^{i k.r} w_k  ==  ifft2 over the two k axes
            g = np.fft.ifft2(w, axes=(0, 1))
            data[b, 0] = g.real.reshape(L * L, n_tau)
        else:
            eps = -t * (1.0 + np.exp(1j * K1) + np.exp(1j * K2))
            a = np.abs(eps)
            dirac = a < 1e-13
            ph = np.where(dirac, 0.0, eps / np.where(dirac, 1.0, a))           # eps/|eps|, 0 at Dirac points
            wp = _occupation_factor((a - mu)[:, :, None], taus[None, None, :], beta)
            wm = _occupation_factor((-a - mu)[:, :, None], taus[None, None, :], beta)
            diag = 0.5 * (wp + wm)
            off = 0.5 * (wp - wm)
            gk = {
                0: diag,                                  # AA
                1: ph[:, :, None] * off,                  # AB
                2: np.conj(ph)[:, :, None] * off,         # BA
                3: diag,                                  # BB
            }
            for ss, w in gk.items():
                g = np.fft.ifft2(w, axes=(0, 1))
                data[b, ss] = g.real.reshape(L * L, n_tau)
    return PropTable(lattice=lattice, L=L, n_sub=n_sub, beta=float(beta), n_tau=n_tau,
                     mu_eff=mu_eff, data=np.ascontiguousarray(data))


def table_for(w) -> PropTable:
    """Table of a `Workload`."""
    return build_table(w.lattice, w.L, w.t, w.mu_eff(), w.beta, w.n_tau)
