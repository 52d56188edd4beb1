"""Seeded synthetic inputs (gauge links and sources) shaped like the paper's workloads.

This module is the ONLY code shared by the CUDA path's callers and the oracle's callers.  It
holds none of the method's arithmetic (no hop operator, no BLAS, no solver): it only draws
random SU(3) matrices, folds the staggered phases and the long-link coefficient into them,
and draws Gaussian sources.  It stands in for the MILC HISQ ensembles of PAPER.md:313-320
(Table 1), which are not available; the recipe is BASELINE.json's.

Canonical layouts (what the C ABI and the oracle both take), complex128:
    links   (4, V, 3, 3)  [mu][s = x + X(y + Y(z + Z t))][row][col]
    sources (N, Vh, 3)    [rhs][even-odd index e = s // 2 of an even site][colour]

Everything is torch so the large lattices (32^3x64, 48^3x96) can be drawn directly on the GPU;
the small ones are drawn on the CPU.  A given (seed, device type) always gives the same bits.
"""
import math

import torch

C1_FREE = 9.0 / 8.0
C3 = -1.0 / 24.0


def volume(dims):
    v = 1
    for d in dims:
        v *= int(d)
    return v


def site_coords(dims, device="cpu"):
    """(4, V) int64: coordinates x, y, z, t of every lexicographic site."""
    X, Y, Z, T = [int(d) for d in dims]
    s = torch.arange(X * Y * Z * T, device=device, dtype=torch.int64)
    x = s % X
    y = (s // X) % Y
    z = (s // (X * Y)) % Z
    t = s // (X * Y * Z)
    return torch.stack([x, y, z, t])


def staggered_phases(dims, device="cpu"):
    """(4, V) float64 of +-1: eta_x = 1, eta_y = (-1)^x, eta_z = (-1)^(x+y), eta_t = (-1)^(x+y+z)."""
    c = site_coords(dims, device)
    one = torch.ones_like(c[0], dtype=torch.float64)
    sgn = lambda n: 1.0 - 2.0 * (n % 2).to(torch.float64)
    return torch.stack([one, sgn(c[0]), sgn(c[0] + c[1]), sgn(c[0] + c[1] + c[2])])


def _randn_complex(shape, gen, device):
    re = torch.randn(shape, generator=gen, device=device, dtype=torch.float64)
    im = torch.randn(shape, generator=gen, device=device, dtype=torch.float64)
    return torch.complex(re, im)


def _det3(m):
    return (m[..., 0, 0] * (m[..., 1, 1] * m[..., 2, 2] - m[..., 1, 2] * m[..., 2, 1])
            - m[..., 0, 1] * (m[..., 1, 0] * m[..., 2, 2] - m[..., 1, 2] * m[..., 2, 0])
            + m[..., 0, 2] * (m[..., 1, 0] * m[..., 2, 1] - m[..., 1, 1] * m[..., 2, 0]))


def _inv3(m):
    """closed-form inverse of (..., 3, 3) matrices (adjugate / determinant)."""
    a, b, c = m[..., 0, 0], m[..., 0, 1], m[..., 0, 2]
    d, e, f = m[..., 1, 0], m[..., 1, 1], m[..., 1, 2]
    g, h, i = m[..., 2, 0], m[..., 2, 1], m[..., 2, 2]
    A, B, C = e * i - f * h, c * h - b * i, b * f - c * e
    D, E, F = f * g - d * i, a * i - c * g, c * d - a * f
    G, H, I = d * h - e * g, b * g - a * h, a * e - b * d
    det = a * A + b * D + c * G
    adj = torch.stack([torch.stack([A, B, C], -1), torch.stack([D, E, F], -1), torch.stack([G, H, I], -1)], -2)
    return adj / det[..., None, None]


def _remove_det_phase(u):
    """divide a unitary matrix by the principal cube root of its determinant -> det = 1."""
    theta = torch.angle(_det3(u))
    ph = torch.polar(torch.ones_like(theta), -theta / 3.0)
    return u * ph[..., None, None]


def su3_gram_schmidt(g):
    """Gaussian complex 3x3 -> Gram-Schmidt on the columns -> det phase removed (config 1)."""
    a0, a1, a2 = g[..., :, 0], g[..., :, 1], g[..., :, 2]
    dot = lambda u, v: (u.conj() * v).sum(-1, keepdim=True)
    nrm = lambda u: u / torch.sqrt(dot(u, u).real)
    u0 = nrm(a0)
    u1 = nrm(a1 - u0 * dot(u0, a1))
    w2 = a2 - u0 * dot(u0, a2)
    u2 = nrm(w2 - u1 * dot(u1, w2))
    return _remove_det_phase(torch.stack([u0, u1, u2], -1))


def su3_polar(w, max_iter=60):
    """proj_SU3(W): unitary polar factor of W by Newton's iteration X <- (X + X^-dag)/2, then
    det phase removed (configs 2-5 with W = 1 + 0.3 G)."""
    x = w
    eye = torch.eye(3, dtype=w.dtype, device=w.device)
    for _ in range(max_iter):
        x = 0.5 * (x + _inv3(x).conj().transpose(-1, -2))
        err = (x.conj().transpose(-1, -2) @ x - eye).abs().max()
        if float(err) < 1e-14:
            break
    return _remove_det_phase(x)


def make_links(dims, kind, seed, device="cpu", c1=1.0, c3=C3, eps=0.3):
    """fat, lng: (4, V, 3, 3) complex128 with the staggered phases and coefficients folded in.

    kind = "free"      : fat = c1 * eta * 1,            lng = c3 * eta * 1   (closed-form check)
           "random"    : fat = c1 * eta * GS-SU3(G),    lng = c3 * eta * GS-SU3(G')  (configs 1, 5)
           "perturbed" : fat = c1 * eta * proj(1+eps G), lng = c3 * eta * proj(1+eps G')  (configs 2-4)
    """
    V = volume(dims)
    gen = torch.Generator(device=device)
    gen.manual_seed(int(seed))
    eta = staggered_phases(dims, device)
    eye = torch.eye(3, dtype=torch.complex128, device=device)
    out = []
    for coeff in (c1, c3):
        u = torch.empty((4, V, 3, 3), dtype=torch.complex128, device=device)
        for mu in range(4):  # one direction at a time bounds the temporaries on the big lattices
            if kind == "free":
                m = eye.expand(V, 3, 3)
            elif kind == "random":
                m = su3_gram_schmidt(_randn_complex((V, 3, 3), gen, device))
            elif kind == "perturbed":
                m = su3_polar(eye + eps * _randn_complex((V, 3, 3), gen, device))
            else:
                raise ValueError(kind)
            u[mu] = m * (coeff * eta[mu])[:, None, None]
        out.append(u)
    return out[0], out[1]


def make_sources(dims, N, seed, device="cpu"):
    """(N, Vh, 3) complex128, real and imaginary parts i.i.d. N(0,1), on even sites."""
    gen = torch.Generator(device=device)
    gen.manual_seed(int(seed) + 7919)
    return _randn_complex((int(N), volume(dims) // 2, 3), gen, device)


CONFIGS = {
    # BASELINE.json configs: lattice, link generator, mass, N
    1: dict(dims=(4, 4, 4, 4), kind="random", mass=0.1, N=4),
    2: dict(dims=(16, 16, 16, 16), kind="perturbed", mass=0.05, N=8),
    3: dict(dims=(32, 32, 32, 64), kind="perturbed", mass=0.01, N=16),
    4: dict(dims=(48, 48, 48, 96), kind="perturbed", mass=0.005, N=32),
    5: dict(dims=(32, 32, 32, 32), kind="random", mass=0.05, N=16),
}
