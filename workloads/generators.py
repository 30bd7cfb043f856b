"""Seeded generators for psi, V_loc(r), beta, D and k-points.

All randomness comes from numpy ``Generator(PCG64)`` seeded by
``SeedSequence(SEED, spawn_key=(config ordinal, stream ordinal))`` so every
consumer (oracle, CUDA path, CPU baseline) sees identical arrays.  The
generators return INPUTS only; nothing here evaluates a term of H.
Recipe and the readings A9/A11/A18 are written down in DESIGN.md section 4.
"""
from __future__ import annotations

import numpy as np

from .configs import Config, CONFIGS

SEED = 230807277
_STREAMS = {"k": 0, "psi": 1, "vloc": 2, "d": 3, "aux": 4}


def rng_for(cfg: Config, stream: str, sub: int = 0) -> np.random.Generator:
    ordinal = list(CONFIGS).index(cfg.name) if cfg.name in CONFIGS else 99
    ss = np.random.SeedSequence(SEED, spawn_key=(ordinal, _STREAMS[stream], sub))
    return np.random.Generator(np.random.PCG64(ss))


def make_kpoints(cfg: Config) -> np.ndarray:
    """k in crystal coordinates (fractions of b_i).  Gamma, or U[-1/2,1/2)^3 draws (A18)."""
    if cfg.nk == 1:
        return np.zeros((1, 3))
    return rng_for(cfg, "k").uniform(-0.5, 0.5, size=(cfg.nk, 3))


def make_psi(cfg: Config, ik: int, ng: int, nbands: int | None = None,
             orthonormalise: bool = True) -> np.ndarray:
    """psi[nb][ng] complex128: i.i.d. N(0,1) real+imag, rows orthonormalised by QR."""
    nb = cfg.nbands if nbands is None else nbands
    rng = rng_for(cfg, "psi", ik)
    a = rng.standard_normal((nb, ng)) + 1j * rng.standard_normal((nb, ng))
    if not orthonormalise:
        return np.ascontiguousarray(a)
    q, r = np.linalg.qr(a.T)                 # (ng, nb), (nb, nb)
    d = np.diagonal(r)
    q = q * (d / np.abs(d))                  # make R's diagonal positive
    return np.ascontiguousarray(q.T)


def _recip(lattice: np.ndarray) -> np.ndarray:
    return 2.0 * np.pi * np.linalg.inv(lattice).T


def make_vloc(cfg: Config, lattice: np.ndarray) -> np.ndarray:
    """Real V(r) on the FFT box, flat C order, Hartree (reading A9).

    Coefficients c(G) ~ N(0,1)+iN(0,1) on |G|^2 <= 4*ecutwfc [bohr^-2 vs Ry],
    c(-G) = conj c(G), c(0) real, damped by exp(-|G|^2/8); synthesised with a
    library inverse FFT and scaled so max|V| = 1 Ha.
    """
    n1, n2, n3 = cfg.grid
    rng = rng_for(cfg, "vloc")
    a = rng.standard_normal(cfg.grid) + 1j * rng.standard_normal(cfg.grid)
    m1 = np.fft.fftfreq(n1, 1.0 / n1).astype(np.int64)
    m2 = np.fft.fftfreq(n2, 1.0 / n2).astype(np.int64)
    m3 = np.fft.fftfreq(n3, 1.0 / n3).astype(np.int64)
    M1, M2, M3 = np.meshgrid(m1, m2, m3, indexing="ij")
    B = _recip(lattice)
    G = M1[..., None] * B[0] + M2[..., None] * B[1] + M3[..., None] * B[2]
    g2 = np.sum(G * G, axis=-1)
    # Hermitian symmetry: the partner of box index (i,j,k) is (-i,-j,-k) mod n.
    i1 = (-np.arange(n1)) % n1
    i2 = (-np.arange(n2)) % n2
    i3 = (-np.arange(n3)) % n3
    partner = a[np.ix_(i1, i2, i3)]
    flat = np.arange(n1 * n2 * n3).reshape(cfg.grid)
    pflat = flat[np.ix_(i1, i2, i3)]
    c = np.where(flat < pflat, a, np.conj(partner))
    c = np.where(flat == pflat, a.real + 0j, c)
    c = c * np.exp(-g2 / 8.0)
    c[g2 > 4.0 * cfg.ecutwfc_ry] = 0.0
    v = np.fft.ifftn(c) * (n1 * n2 * n3)
    assert np.max(np.abs(v.imag)) < 1e-9 * np.max(np.abs(v.real))
    v = v.real
    v = v / np.max(np.abs(v))
    return np.ascontiguousarray(v.reshape(-1))


def make_beta(cfg: Config, lattice: np.ndarray, positions: np.ndarray,
              k_cryst: np.ndarray, miller: np.ndarray) -> np.ndarray:
    """beta[nproj][ng] complex128 (reading A11).

    ``miller`` (ng x 3 integers) is supplied by the caller from its own sphere.
    q = (k+m).B Cartesian; per atom tau: s = Om^-1/2 e^{-q^2/4} e^{-i q.tau};
    p_alpha = (-i) Om^-1/2 q_alpha e^{-q^2/4} e^{-i q.tau}, alpha = x,y,z.
    """
    B = _recip(lattice)
    vol = abs(np.linalg.det(lattice))
    q = (np.asarray(k_cryst, dtype=np.float64)[None, :] + miller.astype(np.float64)) @ B
    q2 = np.sum(q * q, axis=1)
    radial = np.exp(-q2 / 4.0) / np.sqrt(vol)
    ng = miller.shape[0]
    nat = positions.shape[0]
    beta = np.empty((nat, 4, ng), dtype=np.complex128)
    for ia in range(nat):
        sf = np.exp(-1j * (q @ positions[ia])) * radial
        beta[ia, 0] = sf
        beta[ia, 1] = -1j * q[:, 0] * sf
        beta[ia, 2] = -1j * q[:, 1] * sf
        beta[ia, 3] = -1j * q[:, 2] * sf
    return beta.reshape(4 * nat, ng)


def make_dmatrix(cfg: Config) -> np.ndarray:
    """D as per-atom blocks: array [natoms][4][4] real symmetric, Hartree."""
    nat = cfg.natoms
    d = np.zeros((nat, 4, 4))
    if not cfg.dense_d:
        d[:] = np.diag([1.0, 0.5, 0.5, 0.5])
        return d
    rng = rng_for(cfg, "d")
    for ia in range(nat):
        qm, _ = np.linalg.qr(rng.standard_normal((4, 4)))
        lam = rng.uniform(0.1, 1.0, size=4)
        blk = (qm * lam) @ qm.T
        d[ia] = 0.5 * (blk + blk.T)
    return d
