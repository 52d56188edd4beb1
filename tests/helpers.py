"""Test-only helpers: code that is independent of BOTH the oracle and the CUDA path.

* dense assembly of the hop matrix entry by entry from the definition (eq. 2 in
  the sign convention of DESIGN.md U1) -- the brute-force pin P5;
* gauge rotation of links and fields (pin P4);
* plane waves and the free-field closed form lambda(p) (pin P3, from BASELINE.json's north_star).
"""
import numpy as np
import torch

from paper_1710_09745_b200 import synth


def np_links(dims, kind, seed, **kw):
    fat, lng = synth.make_links(dims, kind, seed, device="cpu", **kw)
    return fat.numpy(), lng.numpy()


def np_sources(dims, N, seed):
    return synth.make_sources(dims, N, seed, device="cpu").numpy()


def coords(dims):
    return synth.site_coords(dims).numpy()  # (4, V)


def parity_sites(dims):
    """lexicographic indices of even and of odd sites, each in even-odd order (e = s // 2)."""
    c = coords(dims)
    par = c.sum(0) % 2
    s = np.arange(par.size)
    ev, od = s[par == 0], s[par == 1]
    assert np.array_equal(ev // 2, np.arange(ev.size)) and np.array_equal(od // 2, np.arange(od.size))
    return ev, od


def dense_D(dims, fat, lng):
    """(3V x 3V) dense hop matrix, row/col index = 3*s + colour, built entry by entry."""
    c = coords(dims)
    V = c.shape[1]
    D = np.zeros((3 * V, 3 * V), dtype=np.complex128)
    ext = [int(d) for d in dims]
    stride = [1, ext[0], ext[0] * ext[1], ext[0] * ext[1] * ext[2]]
    for s in range(V):
        for mu in range(4):
            for h, U in ((1, fat), (3, lng)):
                xf = (c[mu, s] + h) % ext[mu]
                xb = (c[mu, s] - h) % ext[mu]
                sf = s + (xf - c[mu, s]) * stride[mu]
                sb = s + (xb - c[mu, s]) * stride[mu]
                D[3 * s:3 * s + 3, 3 * sf:3 * sf + 3] += U[mu, s]
                D[3 * s:3 * s + 3, 3 * sb:3 * sb + 3] -= U[mu, sb].conj().T
    return D


def dense_blocks(dims, fat, lng, mass):
    """D_oe, D_eo (3Vh x 3Vh each) and M_ee = 4 m^2 - D_eo D_oe, in even-odd order."""
    D = dense_D(dims, fat, lng)
    ev, od = parity_sites(dims)
    ie = (3 * ev[:, None] + np.arange(3)[None, :]).ravel()
    io = (3 * od[:, None] + np.arange(3)[None, :]).ravel()
    assert np.abs(D[np.ix_(ie, ie)]).max() == 0 and np.abs(D[np.ix_(io, io)]).max() == 0
    Doe, Deo = D[np.ix_(io, ie)], D[np.ix_(ie, io)]
    M = 4 * mass * mass * np.eye(ie.size) - Deo @ Doe
    return Doe, Deo, M


def random_su3_field(dims, seed):
    g = torch.Generator().manual_seed(seed)
    V = synth.volume(dims)
    z = torch.complex(torch.randn((V, 3, 3), generator=g, dtype=torch.float64),
                      torch.randn((V, 3, 3), generator=g, dtype=torch.float64))
    return synth.su3_gram_schmidt(z).numpy()


def shift_index(dims, mu, h):
    """lexicographic index of x + h*mu for every site x."""
    c = coords(dims).copy()
    ext = [int(d) for d in dims]
    c[mu] = (c[mu] + h) % ext[mu]
    return c[0] + ext[0] * (c[1] + ext[1] * (c[2] + ext[2] * c[3]))


def gauge_rotate_links(dims, fat, lng, g):
    """F'_mu(x) = g(x) F_mu(x) g(x+mu)^dag ; K'_mu(x) = g(x) K_mu(x) g(x+3mu)^dag."""
    f2, l2 = np.empty_like(fat), np.empty_like(lng)
    for mu in range(4):
        g1 = g[shift_index(dims, mu, 1)].conj().transpose(0, 2, 1)
        g3 = g[shift_index(dims, mu, 3)].conj().transpose(0, 2, 1)
        f2[mu] = g @ fat[mu] @ g1
        l2[mu] = g @ lng[mu] @ g3
    return f2, l2


def gauge_rotate_field(dims, v, g, parity):
    """psi'(x) = g(x) psi(x) on a parity field v (N, Vh, 3)."""
    ev, od = parity_sites(dims)
    gs = g[ev if parity == 0 else od]
    return np.einsum("sab,nsb->nsa", gs, v)


def plane_wave(dims, n, colour_vec, parity=0):
    """exp(i p.x) v restricted to the sites of `parity`, p_mu = 2 pi n_mu / X_mu -> (1, Vh, 3)."""
    c = coords(dims)
    ev, od = parity_sites(dims)
    s = ev if parity == 0 else od
    phase = np.zeros(s.size)
    for mu in range(4):
        phase = phase + 2 * np.pi * n[mu] * c[mu, s] / int(dims[mu])
    return (np.exp(1j * phase)[:, None] * np.asarray(colour_vec, dtype=np.complex128)[None, :])[None]


def free_lambda(dims, n, mass, c1, c3):
    """4 m^2 + 4 sum_mu (c1 sin p_mu + c3 sin 3 p_mu)^2  (BASELINE.json north_star)."""
    lam = 4 * mass * mass
    for mu in range(4):
        p = 2 * np.pi * n[mu] / int(dims[mu])
        lam += 4 * (c1 * np.sin(p) + c3 * np.sin(3 * p)) ** 2
    return lam


def relerr_inf(a, b):
    """max |a - b| / max |b|  (U17)."""
    return float(np.abs(a - b).max() / np.abs(b).max())
