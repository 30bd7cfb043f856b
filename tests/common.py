"""Shared helpers for the GPU parity tests: build a config's inputs once and hand them to both sides."""
from __future__ import annotations

import functools

import numpy as np

from oracle import gsphere as og
from oracle import hpsi as oh
from workloads import CONFIGS, cell_for, make_beta, make_dmatrix, make_kpoints, make_psi, make_vloc

TOL = 1e-11   # BASELINE.json north_star: max relative error per band (A13)


@functools.lru_cache(maxsize=None)
def problem(name: str, ik: int = 0, nbands: int | None = None, orthonormalise: bool = True):
    cfg = CONFIGS[name]
    lat, pos = cell_for(cfg)
    kpts = make_kpoints(cfg)
    k = kpts[ik]
    miller, idx, g2 = og.gsphere(lat, cfg.ecutwfc_ry, cfg.grid, k)
    v = make_vloc(cfg, lat)
    beta = make_beta(cfg, lat, pos, k, miller)
    dblk = make_dmatrix(cfg)
    psi = make_psi(cfg, ik, idx.size, nbands=nbands, orthonormalise=orthonormalise)
    return dict(cfg=cfg, lat=lat, pos=pos, kpts=kpts, k=k, miller=miller, idx=idx, g2=g2, v=v,
                vhat=oh.vhat_box(v, cfg.grid), beta=beta, dblk=dblk, psi=psi)


def band_errors(got: np.ndarray, ref: np.ndarray):
    """A13: per band max|d|/max|ref| and ||d||2/||ref||2; returns the worst of each."""
    d = np.abs(got - ref)
    e_inf = np.max(d, axis=1) / np.max(np.abs(ref), axis=1)
    e_2 = np.linalg.norm(got - ref, axis=1) / np.linalg.norm(ref, axis=1)
    return float(np.max(e_inf)), float(np.max(e_2))
