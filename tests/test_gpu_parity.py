"""GPU parity tests: the CUDA path (through the C ABI, via the ctypes binding) against the fp64 CPU oracle,
element by element on the same seeded inputs.  Tolerances are BASELINE.json's north_star (U17):
max|y_gpu - y_oracle| / max|y_oracle| <= 1e-13 per fp64 operator application, <= 1e-5 in fp32 (fp32 result
against the fp64 oracle on the same fp32-rounded inputs).  Integer outputs (status codes, layouts) bit-exact.
"""
import numpy as np
import pytest
import torch

import oracle
from tests import helpers as H

pytestmark = pytest.mark.gpu

TOL64 = 1e-13
TOL32 = 1e-5
NS_ALL = [1, 2, 3, 4, 5, 7, 8, 12, 16, 24, 32]


def _ctx(dims, fat, lng, also_f32=True):
    from paper_1710_09745_b200 import binding
    ctx = binding.Context(dims)
    ctx.load_links(torch.from_numpy(fat).cuda(), torch.from_numpy(lng).cuda(), also_f32=also_f32)
    return ctx


def _round32(a):
    return a.astype(np.complex64).astype(np.complex128)


@pytest.fixture(scope="module")
def lat_asym():
    dims = (4, 6, 8, 10)
    fat, lng = H.np_links(dims, "random", seed=21)
    return dims, fat, lng, _ctx(dims, fat, lng)


@pytest.fixture(scope="module")
def lat4():
    dims = (4, 4, 4, 4)
    fat, lng = H.np_links(dims, "random", seed=11)
    return dims, fat, lng, _ctx(dims, fat, lng)


@pytest.fixture(scope="module")
def lat8():
    dims = (8, 8, 8, 8)
    fat, lng = H.np_links(dims, "perturbed", seed=31)
    return dims, fat, lng, _ctx(dims, fat, lng)


# ------------------------------------------------------------------ layouts (bit-exact)

@pytest.mark.parametrize("N", [1, 3, 8, 32])
def test_pack_unpack_roundtrip_bit_exact(lat_asym, N):
    from paper_1710_09745_b200 import binding
    dims, _, _, ctx = lat_asym
    v = torch.from_numpy(H.np_sources(dims, N, 5)).cuda()
    nat = ctx.pack(v)
    # native layout is [rhs][a][e] (include/bkr.h): check it directly, then the round trip
    want = v.permute(0, 2, 1).contiguous()
    assert torch.equal(torch.view_as_complex(nat.view(-1, 2)).view(N, 3, ctx.Vh), want)
    assert torch.equal(ctx.unpack(nat, N), v)
    nat32 = ctx.pack(v, binding.F32)
    assert torch.equal(torch.view_as_complex(nat32.view(-1, 2)).view(N, 3, ctx.Vh), want.to(torch.complex64))


# ------------------------------------------------------------------ operator

@pytest.mark.parametrize("N", NS_ALL)
@pytest.mark.parametrize("parity", [0, 1])
def test_dslash_fp64_asym(lat_asym, N, parity):
    dims, fat, lng, ctx = lat_asym
    v = H.np_sources(dims, N, 100 + N)
    got = ctx.dslash_canonical(parity, torch.from_numpy(v).cuda()).cpu().numpy()
    want = oracle.dslash(dims, fat, lng, parity, v)
    assert H.relerr_inf(got, want) <= TOL64


@pytest.mark.parametrize("N", [1, 4, 7, 16])
def test_dslash_fp64_extent4_wrap(lat4, N):
    """at extent 4, x+3 wraps onto x-1 (include/bkr.h): a different code path for the index arithmetic."""
    dims, fat, lng, ctx = lat4
    for parity in (0, 1):
        v = H.np_sources(dims, N, 200 + N)
        got = ctx.dslash_canonical(parity, torch.from_numpy(v).cuda()).cpu().numpy()
        assert H.relerr_inf(got, oracle.dslash(dims, fat, lng, parity, v)) <= TOL64


@pytest.mark.parametrize("N", NS_ALL)
def test_dslash_fp32(lat_asym, N):
    from paper_1710_09745_b200 import binding
    dims, fat, lng, ctx = lat_asym
    v = _round32(H.np_sources(dims, N, 300 + N))
    got = ctx.dslash_canonical(1, torch.from_numpy(v).cuda(), binding.F32).cpu().numpy()
    want = oracle.dslash(dims, _round32(fat), _round32(lng), 1, v)
    assert H.relerr_inf(got, want) <= TOL32


@pytest.mark.parametrize("N", [1, 2, 5, 8, 16, 32])
def test_apply_M_fp64(lat8, N):
    dims, fat, lng, ctx = lat8
    v = H.np_sources(dims, N, 400 + N)
    got = ctx.apply_M_canonical(0.05, torch.from_numpy(v).cuda()).cpu().numpy()
    want = oracle.apply_M(dims, fat, lng, 0.05, v)
    assert H.relerr_inf(got, want) <= TOL64


@pytest.mark.parametrize("N", [1, 6, 16])
def test_apply_M_fp32(lat8, N):
    from paper_1710_09745_b200 import binding
    dims, fat, lng, ctx = lat8
    v = _round32(H.np_sources(dims, N, 500 + N))
    got = ctx.apply_M_canonical(0.05, torch.from_numpy(v).cuda(), binding.F32).cpu().numpy()
    want = oracle.apply_M(dims, _round32(fat), _round32(lng), 0.05, v)
    assert H.relerr_inf(got, want) <= TOL32


def test_free_field_plane_wave_eigenvector_on_gpu():
    """pin P3 through the CUDA path at a size the dense check cannot reach: M psi_p = lambda(p) psi_p."""
    dims = (8, 4, 6, 12)
    c1, c3, m = 9.0 / 8.0, -1.0 / 24.0, 0.1
    fat, lng = H.np_links(dims, "free", seed=0, c1=c1, c3=c3)
    ctx = _ctx(dims, fat, lng, also_f32=False)
    for n in ((1, 0, 2, 5), (3, 1, 0, 7)):
        psi = H.plane_wave(dims, n, (1.0, 0.5j, -0.25))
        got = ctx.apply_M_canonical(m, torch.from_numpy(psi).cuda()).cpu().numpy()
        assert H.relerr_inf(got, H.free_lambda(dims, n, m, c1, c3) * psi) <= 1e-13


# ------------------------------------------------------------------ multi-BLAS

@pytest.mark.parametrize("N", NS_ALL)
@pytest.mark.parametrize("herm", [False, True])
def test_gram_fp64(lat_asym, N, herm):
    dims, _, _, ctx = lat_asym
    X = H.np_sources(dims, N, 600 + N)
    Y = X if herm else H.np_sources(dims, N, 700 + N)
    Xd = ctx.pack(torch.from_numpy(X).cuda())
    Yd = Xd if herm else ctx.pack(torch.from_numpy(Y).cuda())
    K = ctx.gram(N, Xd, Yd, hermitian=herm).cpu().numpy()
    want = oracle.gram(X, Y)
    assert np.abs(K - want).max() <= 1e-13 * np.abs(want).max()
    if herm:
        assert np.array_equal(K, K.conj().T) and np.all(K.diagonal().imag == 0)
    # P12: bit-identical on repetition
    assert torch.equal(ctx.gram(N, Xd, Yd, hermitian=herm).cpu(), torch.from_numpy(K))


@pytest.mark.parametrize("N", [1, 4, 7, 16, 32])
def test_gram_fp32_storage_fp64_accumulation(lat_asym, N):
    from paper_1710_09745_b200 import binding
    dims, _, _, ctx = lat_asym
    X, Y = _round32(H.np_sources(dims, N, 800 + N)), _round32(H.np_sources(dims, N, 900 + N))
    Xd = ctx.pack(torch.from_numpy(X).cuda(), binding.F32)
    Yd = ctx.pack(torch.from_numpy(Y).cuda(), binding.F32)
    K = ctx.gram(N, Xd, Yd, prec=binding.F32).cpu().numpy()
    want = oracle.gram(X, Y)
    assert np.abs(K - want).max() <= 1e-13 * np.abs(want).max()  # fp64 accumulation of exact fp32 inputs


@pytest.mark.parametrize("N", NS_ALL)
def test_block_axpy_fp64(lat_asym, N):
    dims, _, _, ctx = lat_asym
    X, Y = H.np_sources(dims, N, 1000 + N), H.np_sources(dims, N, 1100 + N)
    rng = np.random.default_rng(N)
    a = rng.standard_normal((N, N)) + 1j * rng.standard_normal((N, N))
    Xd, Yd = ctx.pack(torch.from_numpy(X).cuda()), ctx.pack(torch.from_numpy(Y).cuda())
    ctx.block_axpy(N, torch.from_numpy(a).cuda(), Xd, Yd)
    got = ctx.unpack(Yd, N).cpu().numpy()
    want = oracle.block_axpy(a, X, Y)
    assert H.relerr_inf(got, want) <= TOL64


@pytest.mark.parametrize("N", [1, 5, 16])
def test_block_axpy_fp32(lat_asym, N):
    from paper_1710_09745_b200 import binding
    dims, _, _, ctx = lat_asym
    X, Y = _round32(H.np_sources(dims, N, 1200 + N)), _round32(H.np_sources(dims, N, 1300 + N))
    rng = np.random.default_rng(N)
    a = _round32(rng.standard_normal((N, N)) + 1j * rng.standard_normal((N, N)))
    Xd, Yd = ctx.pack(torch.from_numpy(X).cuda(), binding.F32), ctx.pack(torch.from_numpy(Y).cuda(), binding.F32)
    ctx.block_axpy(N, torch.from_numpy(a).cuda(), Xd, Yd, prec=binding.F32)
    got = ctx.unpack(Yd, N, binding.F32).cpu().numpy()
    assert H.relerr_inf(got, oracle.block_axpy(a, X, Y)) <= TOL32


@pytest.mark.parametrize("N", [1, 3, 8, 13, 16, 24, 32])
def test_block_axpy_gram_fused_fp64(lat_asym, N):
    """fused update + aliased Hermitian Gram (Alg. 1 l.11 + Alg. 2 l.2) against the oracle's two separate operations"""
    dims, _, _, ctx = lat_asym
    X, Y = H.np_sources(dims, N, 1400 + N), H.np_sources(dims, N, 1500 + N)
    rng = np.random.default_rng(100 + N)
    a = rng.standard_normal((N, N)) + 1j * rng.standard_normal((N, N))
    Xd, Yd = ctx.pack(torch.from_numpy(X).cuda()), ctx.pack(torch.from_numpy(Y).cuda())
    K = ctx.block_axpy_gram(N, torch.from_numpy(a).cuda(), Xd, Yd).cpu().numpy()
    want = oracle.block_axpy(a, X, Y)
    assert H.relerr_inf(ctx.unpack(Yd, N).cpu().numpy(), want) <= TOL64
    wantK = oracle.gram(want, want)
    assert np.abs(K - wantK).max() <= 1e-13 * np.abs(wantK).max()
    assert np.array_equal(K, K.conj().T) and np.all(K.diagonal().imag == 0)
    # P12: bit-identical on repetition from the same inputs
    Yd2 = ctx.pack(torch.from_numpy(Y).cuda())
    assert torch.equal(ctx.block_axpy_gram(N, torch.from_numpy(a).cuda(), Xd, Yd2).cpu(), torch.from_numpy(K))


@pytest.mark.parametrize("N", [1, 4, 7, 13, 16, 24, 32])
def test_block_qpx_update_fp64(lat_asym, N):
    """fused Q / P / X update with triangular coefficients against three oracle block updates; the
    entries on the wrong side of Sinv / Sdag are poisoned to prove they are never read"""
    dims, _, _, ctx = lat_asym
    Q, P, X = (H.np_sources(dims, N, 1800 + 10 * k + N) for k in range(3))
    rng = np.random.default_rng(300 + N)
    full = lambda: rng.standard_normal((N, N)) + 1j * rng.standard_normal((N, N))
    Sinv, Sdag, Wm = np.triu(full()), np.tril(full()), full()
    poison = 1e30
    Sinv_d = torch.from_numpy(Sinv + poison * np.tril(np.ones((N, N)), -1) * _frag_mask(N, upper=True)).cuda()
    Sdag_d = torch.from_numpy(Sdag + poison * np.triu(np.ones((N, N)), 1) * _frag_mask(N, upper=False)).cuda()
    Qd, Pd, Xd = (ctx.pack(torch.from_numpy(v).cuda()) for v in (Q, P, X))
    Pn = torch.empty_like(Pd)
    ctx.block_qpx_update(N, Sinv_d, Sdag_d, torch.from_numpy(Wm).cuda(), Qd, Pd, Pn, Xd)
    Qn = oracle.block_axpy(Sinv, Q, np.zeros_like(Q))
    assert H.relerr_inf(ctx.unpack(Qd, N).cpu().numpy(), Qn) <= TOL64
    assert H.relerr_inf(ctx.unpack(Pn, N).cpu().numpy(), oracle.block_axpy(Sdag, P, Qn)) <= TOL64
    assert H.relerr_inf(ctx.unpack(Xd, N).cpu().numpy(), oracle.block_axpy(Wm, P, X)) <= TOL64
    # gating: do_x only leaves Q untouched
    Qd2, Xd2 = ctx.pack(torch.from_numpy(Q).cuda()), ctx.pack(torch.from_numpy(X).cuda())
    ctx.block_qpx_update(N, Sinv_d, Sdag_d, torch.from_numpy(Wm).cuda(), Qd2, Pd, Pn, Xd2, do_qp=False, do_x=True)
    assert torch.equal(Qd2, ctx.pack(torch.from_numpy(Q).cuda()))
    assert H.relerr_inf(ctx.unpack(Xd2, N).cpu().numpy(), oracle.block_axpy(Wm, P, X)) <= TOL64


def _frag_mask(N, upper):
    """1 where a whole 4 x 8 DMMA coefficient fragment lies strictly on the zero side of the triangle (those fragments
    are skipped); entries of fragments that straddle the diagonal are read and must be true zeros"""
    m = np.zeros((N, N))
    for i in range(N):
        for j in range(N):
            i0, j0 = 4 * (i // 4), 8 * (j // 8)
            if upper and i0 > j0 + 7:
                m[i, j] = 1.0
            if not upper and i0 + 3 < j0:
                m[i, j] = 1.0
    return m


@pytest.mark.parametrize("N", [4, 16])
def test_block_axpy_gram_fused_fp32(lat_asym, N):
    """fp32 blocks: K is the fp64-accumulated Gram matrix of the fp32-rounded result"""
    from paper_1710_09745_b200 import binding
    dims, _, _, ctx = lat_asym
    X, Y = _round32(H.np_sources(dims, N, 1600 + N)), _round32(H.np_sources(dims, N, 1700 + N))
    rng = np.random.default_rng(200 + N)
    a = _round32(rng.standard_normal((N, N)) + 1j * rng.standard_normal((N, N)))
    Xd, Yd = ctx.pack(torch.from_numpy(X).cuda(), binding.F32), ctx.pack(torch.from_numpy(Y).cuda(), binding.F32)
    K = ctx.block_axpy_gram(N, torch.from_numpy(a).cuda(), Xd, Yd, prec=binding.F32).cpu().numpy()
    got = ctx.unpack(Yd, N, binding.F32).cpu().numpy()
    assert H.relerr_inf(got, oracle.block_axpy(a, X, Y)) <= TOL32
    wantK = oracle.gram(got, got)  # of the stored (rounded) block: fp64 products of fp32 numbers are exact
    assert np.abs(K - wantK).max() <= 1e-13 * np.abs(wantK).max()


@pytest.mark.parametrize("N", [1, 2, 5, 8, 16, 32])
def test_small_matrix_kernel(lat4, N):
    """pin P11 through the CUDA path: Cholesky / triangular inverse / HPD inverse vs the oracle."""
    from paper_1710_09745_b200 import binding
    _, _, _, ctx = lat4
    rng = np.random.default_rng(50 + N)
    A = rng.standard_normal((3 * N + 2, N)) + 1j * rng.standard_normal((3 * N + 2, N))
    Hm = A.conj().T @ A
    R, Ri, st = ctx.cholesky_upper(torch.from_numpy(Hm).cuda())
    assert st == binding.OK
    R, Ri = R.cpu().numpy(), Ri.cpu().numpy()
    Ro = oracle.cholesky_upper(Hm)
    assert np.abs(R - Ro).max() <= 1e-12 * np.abs(Ro).max()
    assert np.all(np.tril(R, -1) == 0) and np.all(R.diagonal().imag == 0) and np.all(R.diagonal().real > 0)
    assert np.abs(Ri - oracle.upper_inverse(Ro)).max() <= 1e-11 * np.abs(Ri).max()
    Gi, st = ctx.hpd_inverse(torch.from_numpy(Hm).cuda())
    assert st == binding.OK
    Go = oracle.hpd_inverse(Hm)
    assert np.abs(Gi.cpu().numpy() - Go).max() <= 1e-11 * np.abs(Go).max()


def test_cholesky_breakdown_status(lat4):
    from paper_1710_09745_b200 import binding
    _, _, _, ctx = lat4
    Hm = np.ones((4, 4), dtype=np.complex128)  # rank 1
    _, _, st = ctx.cholesky_upper(torch.from_numpy(Hm).cuda())
    assert st == binding.EBREAKDOWN


def test_invalid_arguments(lat4):
    from paper_1710_09745_b200 import binding
    dims, _, _, ctx = lat4
    v = ctx.empty_native(4)
    with pytest.raises(binding.BkrError):
        ctx.dslash(0, 4, v, v)  # in-place not allowed
    with pytest.raises(binding.BkrError):
        ctx.dslash(2, 4, v, ctx.empty_native(4))
    with pytest.raises(binding.BkrError):
        ctx.dslash(0, 33, v, ctx.empty_native(4))
    c2 = binding.Context(dims)
    with pytest.raises(binding.BkrError) as ei:
        c2.dslash(0, 4, v, ctx.empty_native(4))
    assert ei.value.status == binding.ENOLINKS
