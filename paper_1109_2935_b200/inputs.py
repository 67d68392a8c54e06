"""Seeded synthetic inputs shared by the oracle-side tests and the CUDA-side tests/bench.

This module holds NONE of the method's arithmetic (no Dslash, clover, solver, layout or
compression code); it only draws the random SU(3) gauge fields and Gaussian spinors of
BASELINE.json's configs (recipe in DESIGN.md "Inputs"):

    U_mu(x) = reunitarize(exp(i * eps * sum_a w_a T_a)),  w_a ~ N(0,1),  T_a = lambda_a / 2
    psi     = complex Gaussian, re and im ~ N(0, 1/2)

They stand in for the paper's production gauge configurations (V=32^3x256
anisotropic clover), which are not available here.

Canonical layouts (include/lqcd.h): U[mu][t][z][y][x][3][3], psi[t][z][y][x][4][3], complex128.
"""
import numpy as np

_GELL_MANN = np.zeros((8, 3, 3), dtype=np.complex128)
_GELL_MANN[0][0, 1] = _GELL_MANN[0][1, 0] = 1
_GELL_MANN[1][0, 1] = -1j
_GELL_MANN[1][1, 0] = 1j
_GELL_MANN[2][0, 0] = 1
_GELL_MANN[2][1, 1] = -1
_GELL_MANN[3][0, 2] = _GELL_MANN[3][2, 0] = 1
_GELL_MANN[4][0, 2] = -1j
_GELL_MANN[4][2, 0] = 1j
_GELL_MANN[5][1, 2] = _GELL_MANN[5][2, 1] = 1
_GELL_MANN[6][1, 2] = -1j
_GELL_MANN[6][2, 1] = 1j
_GELL_MANN[7][0, 0] = _GELL_MANN[7][1, 1] = 1 / np.sqrt(3)
_GELL_MANN[7][2, 2] = -2 / np.sqrt(3)


def _reunitarize(U):
    """Project to SU(3): normalise row 0, Gram-Schmidt row 1, row 2 = conj(row0 x row1)."""
    r0 = U[..., 0, :]
    r0 = r0 / np.linalg.norm(r0, axis=-1, keepdims=True)
    r1 = U[..., 1, :]
    r1 = r1 - np.sum(np.conj(r0) * r1, axis=-1, keepdims=True) * r0
    r1 = r1 / np.linalg.norm(r1, axis=-1, keepdims=True)
    r2 = np.conj(np.cross(r0, r1))
    return np.stack([r0, r1, r2], axis=-2)


def random_gauge(dims, eps, seed):
    """Random SU(3) links U[mu][t][z][y][x][3][3] (numpy path; any size that fits host memory)."""
    X, Y, Z, T = dims
    rng = np.random.default_rng(seed)
    out = np.empty((4, T, Z, Y, X, 3, 3), dtype=np.complex128)
    for mu in range(4):                      # one direction at a time keeps the peak memory low
        w = rng.standard_normal((T, Z, Y, X, 8))
        H = eps * 0.5 * np.einsum("...a,aij->...ij", w, _GELL_MANN)
        ev, V = np.linalg.eigh(H)
        E = np.einsum("...ik,...k,...jk->...ij", V, np.exp(1j * ev), np.conj(V))
        out[mu] = _reunitarize(E)
    return out


def unit_gauge(dims):
    X, Y, Z, T = dims
    out = np.zeros((4, T, Z, Y, X, 3, 3), dtype=np.complex128)
    out[..., 0, 0] = out[..., 1, 1] = out[..., 2, 2] = 1
    return out


def gaussian_spinor(dims, seed):
    """psi[t][z][y][x][4][3], re and im ~ N(0, 1/2)."""
    X, Y, Z, T = dims
    rng = np.random.default_rng(seed)
    a = rng.standard_normal((T, Z, Y, X, 4, 3, 2)) / np.sqrt(2.0)
    return np.ascontiguousarray(a[..., 0] + 1j * a[..., 1])


def random_su3_field(dims, seed):
    """One random SU(3) matrix per site g[t][z][y][x][3][3] (for gauge-covariance tests)."""
    X, Y, Z, T = dims
    rng = np.random.default_rng(seed)
    w = rng.standard_normal((T, Z, Y, X, 8))
    H = 0.5 * np.einsum("...a,aij->...ij", w, _GELL_MANN)
    ev, V = np.linalg.eigh(H)
    E = np.einsum("...ik,...k,...jk->...ij", V, np.exp(1j * ev), np.conj(V))
    return _reunitarize(E)


def parity_mask(dims):
    """p[t][z][y][x] = (x+y+z+t) mod 2."""
    X, Y, Z, T = dims
    t, z, y, x = np.meshgrid(np.arange(T), np.arange(Z), np.arange(Y), np.arange(X), indexing="ij")
    return (x + y + z + t) & 1


def random_gauge_torch(dims, eps, seed, device="cpu"):
    """Same distribution as random_gauge, drawn with a seeded torch generator and a batched
    matrix exponential (fast path for 32^3x64 and 48^3x96; not bit-identical to the numpy path).
    Returns a torch complex128 tensor U[mu][t][z][y][x][3][3] on `device`."""
    import torch
    X, Y, Z, T = dims
    g = torch.Generator(device=device)
    g.manual_seed(seed)
    lam = torch.from_numpy(_GELL_MANN).to(device)
    out = torch.empty((4, T, Z, Y, X, 3, 3), dtype=torch.complex128, device=device)
    for mu in range(4):
        w = torch.randn((T, Z, Y, X, 8), generator=g, dtype=torch.float64, device=device)
        H = (eps * 0.5) * torch.einsum("...a,aij->...ij", w.to(torch.complex128), lam)
        E = torch.linalg.matrix_exp(1j * H)
        r0 = E[..., 0, :]
        r0 = r0 / torch.linalg.vector_norm(r0, dim=-1, keepdim=True)
        r1 = E[..., 1, :]
        r1 = r1 - torch.sum(torch.conj(r0) * r1, dim=-1, keepdim=True) * r0
        r1 = r1 / torch.linalg.vector_norm(r1, dim=-1, keepdim=True)
        r2 = torch.conj(torch.linalg.cross(r0, r1, dim=-1))
        out[mu] = torch.stack([r0, r1, r2], dim=-2)
    return out


def gaussian_spinor_torch(dims, seed, device="cpu"):
    import torch
    X, Y, Z, T = dims
    g = torch.Generator(device=device)
    g.manual_seed(seed)
    a = torch.randn((T, Z, Y, X, 4, 3, 2), generator=g, dtype=torch.float64, device=device) / (2.0 ** 0.5)
    return torch.view_as_complex(a.contiguous())


def staggered_links(dims, eps, seed, c1=1.125, c3=-1.0 / 24.0, smear=0.05):
    """Synthetic fat and long link fields for the improved staggered operator: general
    complex 3x3 matrices per link, as smeared links are.  fat = c1 * (random SU(3) + smear * complex
    Gaussian noise) stands in for the asqtad fat links (sums of paths, not unitary); lng = c3 * (an
    independent random SU(3)) for the three-link Naik term.  Both are inputs of the operator; no
    smearing or link product is computed here.  Returns (fat, lng), each [mu][t][z][y][x][3][3]."""
    X, Y, Z, T = dims
    rng = np.random.default_rng(seed + 7919)
    fat = c1 * random_gauge(dims, eps, seed)
    n = rng.standard_normal((4, T, Z, Y, X, 3, 3, 2)) * (smear / np.sqrt(2.0))
    fat = fat + c1 * (n[..., 0] + 1j * n[..., 1])
    lng = c3 * random_gauge(dims, eps, seed + 104729)
    return np.ascontiguousarray(fat), np.ascontiguousarray(lng)


def gaussian_colour_vector(dims, seed):
    """chi[t][z][y][x][3], re and im ~ N(0, 1/2): a staggered "spinor"."""
    X, Y, Z, T = dims
    rng = np.random.default_rng(seed)
    a = rng.standard_normal((T, Z, Y, X, 3, 2)) / np.sqrt(2.0)
    return np.ascontiguousarray(a[..., 0] + 1j * a[..., 1])
