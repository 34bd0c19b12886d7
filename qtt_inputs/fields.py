"""Dense seeded fields and random site tensors (no MPS algebra here).

Conventions: N = 2**n, x_j = y_j = j/N, arrays are ``F[x][y]`` (row index = x),
fp64.  Every function is deterministic in (n, seed).
"""
from __future__ import annotations

import numpy as np

# BASELINE.json configs, as parameters only.
CONFIGS = {
    # cfg: n, chi, Re, dt, steps
    1: dict(n=5, chi=8, Re=None, dt=None, steps=0),
    2: dict(n=8, chi=32, Re=1.0e4, dt=1.0e-4, steps=1),
    3: dict(n=10, chi=64, Re=2.0e5, dt=5.0e-5, steps=100),
    4: dict(n=11, chi=128, Re=1.0e6, dt=0.1 / 2**10, steps=20),
    5: dict(n=12, chi=(16, 32, 64, 128, 256), Re=None, dt=None, steps=0),
}


def grid(n: int):
    """Return (X, Y) with X[x][y] = x/N and Y[x][y] = y/N."""
    N = 1 << n
    t = np.arange(N, dtype=np.float64) / N
    return np.meshgrid(t, t, indexing="ij")


def config1_field(n: int = 5, seed: int = 0) -> np.ndarray:
    """BASELINE config 1: u_x = tanh((y-0.5)/0.05) + 1e-3*N(0,1)."""
    N = 1 << n
    _, Y = grid(n)
    Z = np.random.default_rng(seed).standard_normal((N, N))
    return np.tanh((Y - 0.5) / 0.05) + 1e-3 * Z


def shear_layer(n: int = 8):
    """BASELINE config 2: periodic double shear layer (u_x, u_y)."""
    X, Y = grid(n)
    ux = np.where(Y < 0.5, np.tanh((Y - 0.25) / 0.02), np.tanh((0.75 - Y) / 0.02))
    uy = 0.05 * np.sin(2.0 * np.pi * X)
    return ux, uy


def _wavenumbers(N: int):
    k = np.fft.fftfreq(N, d=1.0 / N)  # integers -N/2..N/2-1
    return np.meshgrid(k, k, indexing="ij")


def _from_streamfunction(psi_hat: np.ndarray):
    """u = (d psi/dy, -d psi/dx) by spectral derivative; real part."""
    N = psi_hat.shape[0]
    KX, KY = _wavenumbers(N)
    ux = np.real(np.fft.ifft2(2j * np.pi * KY * psi_hat))
    uy = np.real(np.fft.ifft2(-2j * np.pi * KX * psi_hat))
    return ux, uy


def decaying_jet(n: int = 10, seed: int = 0, kmax: float = 16.0, rms: float = 1e-3):
    """BASELINE config 3: jet 0.5*(tanh((y-.4)/.005) - tanh((y-.6)/.005)), u_y = 0,
    plus a divergence-free random-Fourier perturbation: psi_hat(k) = exp(i phi_k)/|k|
    for 0 < |k| <= kmax, phi ~ U[0, 2pi) drawn on the full N x N FFT grid, scaled
    to RMS speed ``rms``."""
    N = 1 << n
    _, Y = grid(n)
    ux = 0.5 * (np.tanh((Y - 0.4) / 0.005) - np.tanh((Y - 0.6) / 0.005))
    uy = np.zeros_like(ux)
    phi = np.random.default_rng(seed).uniform(0.0, 2.0 * np.pi, size=(N, N))
    KX, KY = _wavenumbers(N)
    K = np.sqrt(KX**2 + KY**2)
    mask = (K > 0) & (K <= kmax)
    psi_hat = np.zeros((N, N), dtype=np.complex128)
    psi_hat[mask] = np.exp(1j * phi[mask]) / K[mask]
    px, py = _from_streamfunction(psi_hat)
    scale = rms / np.sqrt(np.mean(px**2 + py**2))
    return ux + scale * px, uy + scale * py


def decaying_turbulence(n: int = 11, seed: int = 0, k0: float = 16.0):
    """BASELINE config 4: divergence-free random-phase field from a streamfunction
    with E(k) ~ k^4 exp(-2 (k/k0)^2); |u_hat|^2 = E(k)/(pi k); unit RMS speed."""
    N = 1 << n
    phi = np.random.default_rng(seed).uniform(0.0, 2.0 * np.pi, size=(N, N))
    KX, KY = _wavenumbers(N)
    K = np.sqrt(KX**2 + KY**2)
    mask = K > 0
    E = np.zeros_like(K)
    E[mask] = K[mask] ** 4 * np.exp(-2.0 * (K[mask] / k0) ** 2)
    amp_u = np.zeros_like(K)
    amp_u[mask] = np.sqrt(E[mask] / (np.pi * K[mask]))
    psi_hat = np.zeros((N, N), dtype=np.complex128)
    # |u_hat| = 2 pi |k| |psi_hat|
    psi_hat[mask] = amp_u[mask] / (2.0 * np.pi * K[mask]) * np.exp(1j * phi[mask])
    ux, uy = _from_streamfunction(psi_hat)
    scale = 1.0 / np.sqrt(np.mean(ux**2 + uy**2))
    return ux * scale, uy * scale


def taylor_green_3d(n: int = 4, seed: int = 0, noise: float = 1e-3):
    """3D stand-in workload (PAPER.md:320-322 names the 3D Taylor-Green vortex of ref. [13]): arrays F[x][y][z] on
    [0, 1)^3, u = (sin X cos Y cos Z, -cos X sin Y cos Z, 0) with X = 2 pi x etc., plus ``noise`` * N(0,1) (seeded) on
    every component so that the bonds are not the closed-form ones."""
    N = 1 << n
    t = 2.0 * np.pi * np.arange(N, dtype=np.float64) / N
    X, Y, Z = np.meshgrid(t, t, t, indexing="ij")
    rng = np.random.default_rng(seed)
    u1 = np.sin(X) * np.cos(Y) * np.cos(Z) + noise * rng.standard_normal((N, N, N))
    u2 = -np.cos(X) * np.sin(Y) * np.cos(Z) + noise * rng.standard_normal((N, N, N))
    u3 = noise * rng.standard_normal((N, N, N))
    return u1, u2, u3


def bond_profile(n: int, chi: int, d: int = 4):
    """Bonds r_0..r_n with r_0 = r_n = 1 and r_l = min(d^l, d^(n-l), chi)."""
    return [1] + [int(min(d**l, d ** (n - l), chi)) for l in range(1, n)] + [1]


def random_cores(n: int, chi: int, seed: int = 0, d: int = 4):
    """BASELINE config 5 raw material: N(0,1) site tensors [r_{l-1}][d][r_l] with
    the full bond profile.  (Canonicalisation/normalisation is the consumer's
    business: it is method arithmetic and does not belong here.)"""
    rng = np.random.default_rng(seed)
    r = bond_profile(n, chi, d)
    return [rng.standard_normal((r[l], d, r[l + 1])) for l in range(n)]


def config_fields(cfg: int, seed: int = 0):
    """(u_x, u_y) dense fields of BASELINE config ``cfg`` (2, 3 or 4)."""
    if cfg == 2:
        return shear_layer(CONFIGS[2]["n"])
    if cfg == 3:
        return decaying_jet(CONFIGS[3]["n"], seed)
    if cfg == 4:
        return decaying_turbulence(CONFIGS[4]["n"], seed)
    raise ValueError(f"config {cfg} has no velocity-field recipe")
