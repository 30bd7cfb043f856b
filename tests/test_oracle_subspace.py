"""Pins of the subspace-product oracle (oracle/subspace.py) against what the mathematics fixes.

None of these re-type the oracle's formula: closed forms on plane waves and geometric sequences, the defining
properties of an inner product, the library routine it reduces to (np.vdot / BLAS zgemm, allowed as a check of the
oracle), and its tie to the H oracle (Hermiticity of <psi_i|H psi_j>).
"""
import numpy as np

from oracle import subspace as osub
from oracle import gsphere as og
from oracle import hpsi as oh
from workloads import CONFIGS, cell_for, make_beta, make_dmatrix, make_psi, make_vloc


def test_unit_vectors_pick_out_conjugated_components():
    # <e_p | phi_j> = phi_j[p]   and   <psi_i | e_p> = conj(psi_i[p]): fixes which side is conjugated
    rng = np.random.default_rng(1)
    ng = 37
    phi = rng.standard_normal((3, ng)) + 1j * rng.standard_normal((3, ng))
    e = np.zeros((2, ng), dtype=complex); e[0, 5] = 1.0; e[1, 30] = 1.0
    s = osub.vdot_matrix(e, phi)
    np.testing.assert_array_equal(s, np.array([phi[:, 5], phi[:, 30]]))
    s2 = osub.vdot_matrix(phi, e)
    np.testing.assert_array_equal(s2, np.conj(np.array([phi[:, 5], phi[:, 30]])).T)


def test_geometric_sequences_closed_form():
    # psi(G_n) = z^n, phi(G_n) = w^n  =>  S = sum (conj(z) w)^n = (1 - q^N) / (1 - q), q = conj(z) w
    n = 200
    z, w = 0.97 * np.exp(0.3j), 1.01 * np.exp(-0.7j)
    k = np.arange(n)
    s = osub.vdot_matrix((z ** k)[None, :], (w ** k)[None, :])[0, 0]
    q = np.conj(z) * w
    want = (1 - q ** n) / (1 - q)
    assert abs(s - want) <= 1e-13 * abs(want)


def test_inner_product_axioms():
    rng = np.random.default_rng(2)
    ng = 300
    a = rng.standard_normal((4, ng)) + 1j * rng.standard_normal((4, ng))
    b = rng.standard_normal((5, ng)) + 1j * rng.standard_normal((5, ng))
    s_ab, s_ba, s_aa = osub.vdot_matrix(a, b), osub.vdot_matrix(b, a), osub.vdot_matrix(a, a)
    np.testing.assert_allclose(s_ab, np.conj(s_ba.T), rtol=0, atol=1e-13)              # conjugate symmetry
    assert np.all(np.abs(s_aa.imag.diagonal()) == 0.0) and np.all(s_aa.real.diagonal() > 0)   # positive norms
    np.testing.assert_allclose(s_aa.real.diagonal(), np.linalg.norm(a, axis=1) ** 2, rtol=1e-14)
    lam = 0.3 - 1.1j                                                                     # linear in the ket,
    np.testing.assert_allclose(osub.vdot_matrix(a, lam * b), lam * s_ab, rtol=0, atol=1e-12)
    np.testing.assert_allclose(osub.vdot_matrix(lam * a, b), np.conj(lam) * s_ab, rtol=0, atol=1e-12)  # antilinear in the bra


def test_reduces_to_library_vdot_and_gemm():
    rng = np.random.default_rng(3)
    ng = 1234
    a = rng.standard_normal((6, ng)) + 1j * rng.standard_normal((6, ng))
    b = rng.standard_normal((7, ng)) + 1j * rng.standard_normal((7, ng))
    s = osub.vdot_matrix(a, b)
    assert abs(s[2, 4] - np.vdot(a[2], b[4])) <= 1e-12 * np.linalg.norm(a[2]) * np.linalg.norm(b[4])
    np.testing.assert_allclose(s, np.conj(a) @ b.T, rtol=0, atol=1e-11)


def test_orthonormal_block_gives_identity_and_h_subspace_is_hermitian():
    cfg = CONFIGS["cfg1"]
    lat, pos = cell_for(cfg)
    miller, idx, g2 = og.gsphere(lat, cfg.ecutwfc_ry, cfg.grid, np.zeros(3))
    psi = make_psi(cfg, 0, idx.size)                      # rows orthonormalised by the generator (QR)
    np.testing.assert_allclose(osub.vdot_matrix(psi, psi), np.eye(cfg.nbands), rtol=0, atol=1e-13)
    v = make_vloc(cfg, lat)
    beta = make_beta(cfg, lat, pos, np.zeros(3), miller)
    hpsi = oh.apply_h_rows(psi, miller, g2, oh.vhat_box(v, cfg.grid), cfg.grid, beta, oh.expand_d(make_dmatrix(cfg)))
    h = osub.vdot_matrix(psi, hpsi)                       # <psi_i|H psi_j>: Hermitian because H is
    assert np.max(np.abs(h - np.conj(h.T))) <= 1e-12 * np.max(np.abs(h))
    # Rayleigh quotients lie inside the spectrum of H: at least the kinetic lower bound min(V) and finite
    assert np.all(h.real.diagonal() > np.min(v) - 1e-9)
