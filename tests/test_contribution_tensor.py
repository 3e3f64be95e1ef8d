"""Eq. 23: H = ((C*)^-1 - (C1)^-1)/phi.  CPU only: dr_contribution_tensor is host code of libdr."""
import numpy as np
import pytest

from oracle import post


def hooke(K, G):
    C = np.zeros((6, 6))
    C[:3, :3] = K - 2.0 * G / 3.0
    C[np.arange(3), np.arange(3)] = K + 4.0 * G / 3.0
    C[np.arange(3, 6), np.arange(3, 6)] = G
    return C


@pytest.fixture(scope="module")
def binding():
    from paper_2410_20441_b200 import build, binding
    build.build()
    return binding


def dilute_pore_compliance_H(K, G):
    """closed form for dry spherical pores in the non-interaction approximation (Eshelby 1957; Kachanov & Sevostianov
    2018 cited P:189): 1/K* = (1/K)(1 + phi a), 1/G* = (1/G)(1 + phi b) => H is the isotropic compliance with
    bulk part a/K and shear part b/G."""
    nu = (3 * K - 2 * G) / (2 * (3 * K + G))
    a = 3 * (1 - nu) / (2 * (1 - 2 * nu))
    b = 15 * (1 - nu) / (7 - 5 * nu)
    # isotropic compliance from (1/K, 1/G): S11 = 1/(9K) + 1/(3G), S12 = 1/(9K) - 1/(6G), S44 = 1/G
    def iso(invK, invG):
        S = np.zeros((6, 6))
        S[:3, :3] = invK / 9 - invG / 6
        S[np.arange(3), np.arange(3)] = invK / 9 + invG / 3
        S[np.arange(3, 6), np.arange(3, 6)] = invG
        return S
    return iso(a / K, b / G), iso


def test_oracle_post_pinned_by_closed_form_round_trip():
    K, G, phi = 70.2, 29.0, 0.0168
    H_exact, iso = dilute_pore_compliance_H(K, G)
    S1 = iso(1 / K, 1 / G)
    assert np.allclose(S1 @ hooke(K, G), np.eye(6), atol=1e-14)            # iso() really is the inverse of Hooke
    C_eff = np.linalg.inv(S1 + phi * H_exact)
    H = post.contribution_tensor(C_eff, hooke(K, G), phi)
    assert np.max(np.abs(H - H_exact)) <= 1e-11 * np.max(np.abs(H_exact))
    # and the effective moduli are the dilute formulas of the pins file (App. A3 of the survey), compliance form
    nu = (3 * K - 2 * G) / (2 * (3 * K + G))
    Ks = 1 / (C_eff[:3, :3].sum() / 9) if False else (C_eff[0, 0] + 2 * C_eff[0, 1]) / 3
    assert Ks == pytest.approx(K / (1 + phi * 3 * (1 - nu) / (2 * (1 - 2 * nu))), rel=1e-12)


def test_libdr_matches_oracle_on_anisotropic_tensors(binding):
    rng = np.random.default_rng(3)
    for _ in range(5):
        A = rng.normal(size=(6, 6))
        C1 = hooke(36.0, 44.0)
        Ce = C1 - 0.05 * (A @ A.T) - 0.3 * np.diag(rng.uniform(0, 1, 6))     # SPD, softer, fully anisotropic
        phi = float(rng.uniform(0.01, 0.2))
        H = binding.contribution_tensor(Ce, C1, phi)
        Ho = post.contribution_tensor(Ce, C1, phi)
        assert np.max(np.abs(H - Ho)) <= 1e-12 * np.max(np.abs(Ho))
    # unsymmetric input (the solver's C is not symmetrised) and pivoting
    P = np.eye(6)[[3, 4, 5, 0, 1, 2]]
    Ce = P @ Ce + 1e-3 * rng.normal(size=(6, 6))
    C1p = P @ C1
    assert np.max(np.abs(binding.contribution_tensor(Ce, C1p, 0.1) - post.contribution_tensor(Ce, C1p, 0.1))) <= 1e-11 * 10


def test_libdr_argument_checks(binding):
    C1 = hooke(36.0, 44.0)
    with pytest.raises(binding.DrError):
        binding.contribution_tensor(C1, C1, 0.0)
    with pytest.raises(binding.DrError):
        binding.contribution_tensor(np.zeros((6, 6)), C1, 0.1)
    assert np.max(np.abs(binding.contribution_tensor(C1, C1, 0.5))) == 0.0
