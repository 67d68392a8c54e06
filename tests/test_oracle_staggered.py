"""Pins of the improved staggered oracle (oracle/staggered_oracle.cpp), against what
the paper and the mathematics fix -- none of them re-types the oracle's own loop:
  * "the staggered fermion matrix is anti-Hermitian": <x, D y> = -<D x, y>;
  * "the even and odd lattices are decoupled" in M^dag M;
  * free field (fat = c1, lng = c3): M^dag M e^{ipx} u = [m^2 + sum_mu (c1 sin p_mu + c3 sin 3 p_mu)^2] e^{ipx} u,
    with half-integer momenta in antiperiodic directions (pins phases, signs, the 3-hop and R15);
  * gauge covariance under a random SU(3) transformation of the fat and long links;
  * dense LU of (M^dag M + sigma) on 4^4 (pins the CG, Eq. 4)."""
import numpy as np
import pytest

import oracle
from paper_1109_2935_b200 import inputs

BC = (1, 1, 1, -1)


def _rel(a, b):
    return np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel())


@pytest.fixture(scope="module")
def small():
    dims = (4, 6, 4, 8)
    fat, lng = inputs.staggered_links(dims, 0.4, 1)
    return dims, fat, lng


def test_anti_hermitian_and_parity_structure(small):
    dims, fat, lng = small
    x = inputs.gaussian_colour_vector(dims, 2)
    y = inputs.gaussian_colour_vector(dims, 3)
    Dy, Dx = oracle.stag_dslash(y, fat, lng, BC), oracle.stag_dslash(x, fat, lng, BC)
    assert abs(np.vdot(x, Dy) + np.vdot(Dx, y)) <= 1e-13 * np.linalg.norm(x) * np.linalg.norm(Dy)
    # M^dag is the adjoint of M, and M^dag M = m^2 - D^2/4
    m = 0.05
    assert abs(np.vdot(x, oracle.stag_M(y, fat, lng, BC, m)) - np.vdot(oracle.stag_M(x, fat, lng, BC, m, dagger=True), y)) <= 1e-13 * np.linalg.norm(x) * np.linalg.norm(y)
    want = m * m * y - 0.25 * oracle.stag_dslash(Dy, fat, lng, BC)
    assert _rel(oracle.stag_MdagM(y, fat, lng, BC, m), want) <= 1e-14
    # D couples opposite parities only (1 and 3 hops are odd), so M^dag M keeps the parities apart
    par = inputs.parity_mask(dims)
    ye = y * (par == 0)[..., None]
    assert np.max(np.abs(oracle.stag_dslash(ye, fat, lng, BC)[par == 0])) == 0.0
    # (the cross terms +m D/2 - m D/2 cancel to rounding, not bitwise, in the two-application form)
    assert np.max(np.abs(oracle.stag_MdagM(ye, fat, lng, BC, m, 0.3)[par == 1])) <= 1e-15 * np.max(np.abs(ye))


@pytest.mark.parametrize("dims,bc,n", [((4, 6, 8, 10), (1, 1, 1, -1), (1, 2, 3, 4)), ((8, 4, 6, 4), (-1, 1, -1, 1), (3, 1, 0, 2)),
                                       ((6, 8, 4, 12), (1, -1, 1, -1), (0, 5, 1, 7))])
def test_free_field_closed_form(dims, bc, n):
    c1, c3, m, sigma = 1.125, -1.0 / 24.0, 0.07, 0.4
    X, Y, Z, T = dims
    one = inputs.unit_gauge(dims)
    p = 2 * np.pi * (np.array(n) + np.where(np.array(bc) < 0, 0.5, 0.0)) / np.array(dims)
    t, z, y, x = np.meshgrid(np.arange(T), np.arange(Z), np.arange(Y), np.arange(X), indexing="ij")
    phase = np.exp(1j * (p[0] * x + p[1] * y + p[2] * z + p[3] * t))
    u = np.array([0.3 - 1.0j, 2.0, -0.5 + 0.25j])
    chi = phase[..., None] * u
    got = oracle.stag_MdagM(chi, c1 * one, c3 * one, bc, m, sigma)
    lam = m * m + sigma + np.sum((c1 * np.sin(p) + c3 * np.sin(3 * p)) ** 2)
    assert _rel(got, lam * chi) <= 1e-13
    # D itself on the plane wave: (D chi)(x) = sum_mu eta_mu(x) 2i (c1 sin p_mu + c3 sin 3p_mu) chi(x)
    eta = [np.ones_like(x), (-1.0) ** x, (-1.0) ** (x + y), (-1.0) ** (x + y + z)]
    want = sum(eta[mu] * 2j * (c1 * np.sin(p[mu]) + c3 * np.sin(3 * p[mu])) for mu in range(4))[..., None] * chi
    assert _rel(oracle.stag_dslash(chi, c1 * one, c3 * one, bc), want) <= 1e-13


def test_gauge_covariance(small):
    """fat'_mu(x) = g(x) fat_mu(x) g(x+mu)^dag, lng'_mu(x) = g(x) lng_mu(x) g(x+3mu)^dag, chi' = g chi  =>  D' chi' = g D chi.
    Periodic boundaries (a transformation is periodic)."""
    dims, fat, lng = small
    bc = (1, 1, 1, 1)
    g = inputs.random_su3_field(dims, 3)
    chi = inputs.gaussian_colour_vector(dims, 4)
    axis = {0: 3, 1: 2, 2: 1, 3: 0}
    fat2, lng2 = np.empty_like(fat), np.empty_like(lng)
    for mu in range(4):
        g1 = np.roll(g, -1, axis=axis[mu])
        g3 = np.roll(g, -3, axis=axis[mu])
        fat2[mu] = g @ fat[mu] @ np.conj(np.swapaxes(g1, -1, -2))
        lng2[mu] = g @ lng[mu] @ np.conj(np.swapaxes(g3, -1, -2))
    gchi = np.einsum("...ij,...j->...i", g, chi)
    want = np.einsum("...ij,...j->...i", g, oracle.stag_dslash(chi, fat, lng, bc))
    assert _rel(oracle.stag_dslash(gchi, fat2, lng2, bc), want) <= 1e-13


def test_dense_lu_shifted_systems():
    dims = (4, 4, 4, 4)
    fat, lng = inputs.staggered_links(dims, 0.5, 5)
    b = inputs.gaussian_colour_vector(dims, 6)
    m = 0.1
    n = b.size
    A = np.zeros((n, n), dtype=np.complex128)
    e = np.zeros(n, dtype=np.complex128)
    for k in range(n):
        e[:] = 0
        e[k] = 1
        A[:, k] = oracle.stag_MdagM(e.reshape(b.shape), fat, lng, BC, m, 0.0).ravel()
    assert np.linalg.norm(A - A.conj().T) <= 1e-13 * np.linalg.norm(A)
    assert np.min(np.linalg.eigvalsh(A)) >= m * m * (1 - 1e-10)              # M^dag M = m^2 - D^2/4 >= m^2
    for sigma in (0.0, 0.02, 0.5):
        x_lu = np.linalg.solve(A + sigma * np.eye(n), b.ravel()).reshape(b.shape)
        x, info = oracle.stag_cg(b, fat, lng, BC, m, sigma, tol=1e-12)
        assert info["status"] == 0 and info["true_residual"] <= 2e-12
        assert _rel(x, x_lu) <= 1e-10
