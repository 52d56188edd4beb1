"""GPU parity for blocks of 34..64 right-hand sides ("N <= 64", PAPER.md:324 blocks of 48
and 64): the multi-BLAS runs as two panels of N / 2 columns (one level of the paper's recursive tiling),
the stencil in chunks, the N x N algebra with two columns per lane.  Element by element against the oracle."""
import numpy as np
import pytest
import torch

import oracle
from tests import helpers as H

pytestmark = pytest.mark.gpu
TOL64, TOL32 = 1e-13, 1e-5


def _round32(a):
    return a.astype(np.complex64).astype(np.complex128)


@pytest.fixture(scope="module")
def lat():
    from paper_1710_09745_b200 import binding
    dims = (4, 6, 8, 10)
    fat, lng = H.np_links(dims, "random", seed=31)
    ctx = binding.Context(dims)
    ctx.load_links(torch.from_numpy(fat).cuda(), torch.from_numpy(lng).cuda(), also_f32=True)
    return dims, fat, lng, ctx


@pytest.mark.parametrize("N", [34, 40, 48, 64])
@pytest.mark.parametrize("hermitian", [False, True])
def test_gram_panels(lat, N, hermitian):
    dims, _, _, ctx = lat
    X = H.np_sources(dims, N, 3100 + N)
    Y = X if hermitian else H.np_sources(dims, N, 3200 + N)
    Xd = ctx.pack(torch.from_numpy(X).cuda())
    Yd = Xd if hermitian else ctx.pack(torch.from_numpy(Y).cuda())
    K = ctx.gram(N, Xd, Yd, hermitian=hermitian).cpu().numpy()
    want = oracle.gram(X, Y)
    assert np.abs(K - want).max() <= TOL64 * np.abs(want).max()
    if hermitian:
        assert np.abs(K - K.conj().T).max() == 0.0 and np.abs(np.diag(K).imag).max() == 0.0


@pytest.mark.parametrize("N", [34, 48, 64])
@pytest.mark.parametrize("tri", [0, 1, 2])
def test_block_update_panels(lat, N, tri):
    """Z = C + W a with a general / upper / lower triangular: entries on the zero side are poisoned -- never read"""
    dims, _, _, ctx = lat
    rng = np.random.default_rng(3300 + N + tri)
    a = (rng.normal(size=(N, N)) + 1j * rng.normal(size=(N, N))) * 0.3
    if tri == 1:
        a = np.triu(a)
    if tri == 2:
        a = np.tril(a)
    C, W = H.np_sources(dims, N, 3400 + N), H.np_sources(dims, N, 3500 + N)
    want = oracle.block_axpy(a, W, C)
    ap = a.copy()
    p = N // 2
    if tri == 1:
        ap[p:, :p] = np.nan      # the whole lower-left panel block is skipped
    if tri == 2:
        ap[:p, p:] = np.nan
    from paper_1710_09745_b200 import binding
    Cd, Wd = ctx.pack(torch.from_numpy(C).cuda()), ctx.pack(torch.from_numpy(W).cuda())
    Zd = ctx.empty_native(N)
    ctx.block_update(N, torch.from_numpy(ap).cuda(), Cd, Wd, Zd, tri=tri)
    got = ctx.unpack(Zd, N).cpu().numpy()
    assert np.abs(got - want).max() <= TOL64 * np.abs(want).max()
    # in place (Z = C), the way the solver calls it
    ctx.block_update(N, torch.from_numpy(ap).cuda(), Cd, Wd, Cd, tri=tri)
    got = ctx.unpack(Cd, N).cpu().numpy()
    assert np.abs(got - want).max() <= TOL64 * np.abs(want).max()


@pytest.mark.parametrize("N", [48, 64])
def test_block_update_panels_mixed_precision(lat, N):
    from paper_1710_09745_b200 import binding
    dims, _, _, ctx = lat
    rng = np.random.default_rng(3600 + N)
    a = (rng.normal(size=(N, N)) + 1j * rng.normal(size=(N, N))) * 0.3
    C, W = H.np_sources(dims, N, 3700 + N), _round32(H.np_sources(dims, N, 3800 + N))
    want = oracle.block_axpy(a, W, C)
    Cd = ctx.pack(torch.from_numpy(C).cuda())
    Wd = ctx.pack(torch.from_numpy(W).cuda(), prec=binding.F32)
    ctx.block_update(N, torch.from_numpy(a).cuda(), Cd, Wd, Cd, precZ=binding.F64, precW=binding.F32)
    got = ctx.unpack(Cd, N).cpu().numpy()
    assert np.abs(got - want).max() <= TOL64 * np.abs(want).max()


@pytest.mark.parametrize("N", [33, 48, 57, 64])
def test_small_matrix_kernel_large(lat, N):
    """Cholesky / triangular inverse / HPD inverse of the one-CTA kernel with two columns per lane (N > 32) and the fourth
    work matrix in global memory (N > 56), against the oracle (itself pinned to numpy.linalg, P11)"""
    _, _, _, ctx = lat
    rng = np.random.default_rng(3900 + N)
    A = rng.normal(size=(N + 5, N)) + 1j * rng.normal(size=(N + 5, N))
    Hm = A.conj().T @ A + 0.5 * np.eye(N)
    R, Ri, st = ctx.cholesky_upper(torch.from_numpy(Hm).cuda())
    assert st == 0
    Ro = oracle.cholesky_upper(Hm)
    assert np.abs(R.cpu().numpy() - Ro).max() <= 1e-12 * np.abs(Ro).max()
    Rio = oracle.upper_inverse(Ro)
    assert np.abs(Ri.cpu().numpy() - Rio).max() <= 1e-11 * np.abs(Rio).max()
    Gi, st = ctx.hpd_inverse(torch.from_numpy(Hm).cuda())
    assert st == 0
    Gio = oracle.hpd_inverse(Hm)
    assert np.abs(Gi.cpu().numpy() - Gio).max() <= 1e-10 * np.abs(Gio).max()


@pytest.mark.parametrize("N", [40, 64])
@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_dslash_and_apply_M_large_blocks(lat, N, prec):
    from paper_1710_09745_b200 import binding
    dims, fat, lng, ctx = lat
    v = H.np_sources(dims, N, 4000 + N)
    pr = binding.F64 if prec == "f64" else binding.F32
    if prec == "f32":
        v = _round32(v)
    got = ctx.apply_M_canonical(0.07, torch.from_numpy(v).cuda(), prec=pr).cpu().numpy()
    want = oracle.apply_M(dims, fat, lng, 0.07, v)
    tol = TOL64 if prec == "f64" else TOL32
    assert np.abs(got - want).max() <= tol * np.abs(want).max()


@pytest.fixture(scope="module")
def lat8():
    from paper_1710_09745_b200 import binding
    dims = (8, 8, 8, 8)
    fat, lng = H.np_links(dims, "perturbed", seed=41)
    ctx = binding.Context(dims)
    ctx.load_links(torch.from_numpy(fat).cuda(), torch.from_numpy(lng).cuda(), also_f32=True)
    return dims, fat, lng, ctx


@pytest.mark.parametrize("N", [48, 64])
def test_block_solve_large_blocks_vs_oracle(lat8, N):
    """blockCGrQ with 48 and 64 rhs on 8^4: true residuals by the oracle, solutions within 1e-8 of the
    oracle's, iterate after k iterations equal to the oracle's (the unfused path with panel launches)"""
    dims, fat, lng, ctx = lat8
    B = H.np_sources(dims, N, 4100 + N)
    Bd = torch.from_numpy(B).cuda()
    X, rr, st = ctx.solve_block(0.05, Bd, tol=1e-10)
    assert st["status"] == 0 and max(rr) <= 1e-10
    Xh = X.cpu().numpy()
    assert oracle.true_relres(dims, fat, lng, 0.05, B, Xh).max() <= 1e-10
    ro = oracle.block_cg(dims, fat, lng, 0.05, B, tol=1e-10)
    assert ro["status"] == 0 and abs(ro["iters"] - st["iters"]) <= 2
    assert np.abs(Xh - ro["X"]).max() <= 1e-8 * np.abs(ro["X"]).max()
    k = 3
    Xk, _, stk = ctx.solve_block(0.05, Bd, tol=1e-30, maxiter=k, raise_on=())
    rk = oracle.block_cg(dims, fat, lng, 0.05, B, tol=1e-30, maxiter=k)
    assert stk["iters"] == k and rk["iters"] == k
    assert np.abs(Xk.cpu().numpy() - rk["X"]).max() <= 1e-10 * np.abs(rk["X"]).max()


def test_block_solve_large_block_mixed(lat8):
    from paper_1710_09745_b200 import binding
    dims, fat, lng, ctx = lat8
    N = 48
    B = H.np_sources(dims, N, 4300)
    X, rr, st = ctx.solve_block(0.05, torch.from_numpy(B).cuda(), tol=1e-10, inner_prec=binding.F32, delta=0.1)
    assert st["status"] == 0 and st["reliable_updates"] >= 1
    assert oracle.true_relres(dims, fat, lng, 0.05, B, X.cpu().numpy()).max() <= 1e-10


@pytest.mark.parametrize("inner", ["f64", "f32"])
def test_solve_many_blocks_sloppy_and_fine(lat, inner):
    """bkr_solve_many (many rhs in blocks of N, sloppy sweep then fine sweep): 24 sources in blocks of 8
    against the oracle run block by block; the fine sweep starts from the sloppy solution, so it needs fewer iterations
    than a fine solve from zero"""
    from paper_1710_09745_b200 import binding
    dims, fat, lng, ctx = lat
    nrhs, N = 24, 8
    B = H.np_sources(dims, nrhs, 4500)
    kw = dict(inner_prec=binding.F32, delta=0.1) if inner == "f32" else {}
    X, rr, st = ctx.solve_many(0.1, torch.from_numpy(B).cuda(), N, tol_sloppy=5e-6, tol_fine=2e-9, **kw)
    Xh = X.cpu().numpy()
    assert len(st) == 3 and all(s[0]["status"] == 0 and s[1]["status"] == 0 for s in st)
    assert max(rr) <= 2e-9
    for b in range(3):
        Bb = B[b * N:(b + 1) * N]
        assert oracle.true_relres(dims, fat, lng, 0.1, Bb, Xh[b * N:(b + 1) * N]).max() <= 2e-9
        ro = oracle.block_cg(dims, fat, lng, 0.1, Bb, tol=2e-9)
        assert ro["status"] == 0
        assert np.abs(Xh[b * N:(b + 1) * N] - ro["X"]).max() <= 1e-7 * np.abs(ro["X"]).max()
        assert st[b][0]["iters"] > 0 and 0 < st[b][1]["iters"] < ro["iters"]
        assert st[b][0]["true_relres_max"] <= 5e-6
    # fine sweep only
    X2, rr2, st2 = ctx.solve_many(0.1, torch.from_numpy(B).cuda(), N, tol_sloppy=0.0, tol_fine=2e-9, **kw)
    assert all(s[0]["iters"] == 0 and s[1]["status"] == 0 for s in st2) and max(rr2) <= 2e-9
