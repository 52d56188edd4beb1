"""GPU parity of the multi-BLAS template instances the solver and bench.py run but test_gpu_parity.py does not reach
through bkr_gram / bkr_block_axpy alone ("parity tests miss template instances the bench runs"):

  * Hermitian reduction of TWO DIFFERENT blocks, G = P^dag (M P) (Alg. 1 l.9): the
    gram_tma_kernel<HERM=1, ALIAS=0> instance at 1-4 column tiles (N = 8 .. 32);
  * streaming update with triangular coefficients at 4 column tiles (N = 28, 32: the unfused path of the solver beyond
    24 rhs) and the mixed-precision instances Z fp64 / W fp32, Z fp32 / W fp64, Z fp32 / W fp32;
  * the fused Q / P / X update with fp32 P, Q and fp64 X.
All against the oracle's plain loops (eq. 3 / eq. 4), element by element.
"""
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
    fat, lng = H.np_links(dims, "random", seed=21)
    ctx = binding.Context(dims)
    ctx.load_links(torch.from_numpy(fat).cuda(), torch.from_numpy(lng).cuda(), also_f32=True)
    return dims, fat, lng, ctx


def _frag_mask(N, upper):
    """1 where a whole 4 x 8 DMMA coefficient fragment lies strictly on the zero side of the triangle (skipped)"""
    m = np.zeros((N, N))
    for i in range(N):
        for j in range(N):
            i0, j0 = 4 * (i // 4), 8 * (j // 8)
            if upper and i0 > j0 + 7:
                m[i, j] = 1.0
            if not upper and i0 + 3 < j0:
                m[i, j] = 1.0
    return m


@pytest.mark.parametrize("N", [5, 8, 12, 16, 24, 32])
def test_gram_hermitian_two_blocks_general_Y(lat, N):
    """hermitian = 1 with X != Y: the kernel computes the tile pairs i <= j only and mirrors; for a general Y the upper
    triangle must equal the oracle's X^dag Y entry by entry, the lower one its conjugate, the diagonal real"""
    dims, _, _, ctx = lat
    X, Y = H.np_sources(dims, N, 2100 + N), H.np_sources(dims, N, 2200 + N)
    Xd, Yd = ctx.pack(torch.from_numpy(X).cuda()), ctx.pack(torch.from_numpy(Y).cuda())
    K = ctx.gram(N, Xd, Yd, hermitian=True).cpu().numpy()
    want = oracle.gram(X, Y)
    scale = np.abs(want).max()
    iu = np.triu_indices(N, 1)
    assert np.abs(K[iu] - want[iu]).max() <= TOL64 * scale
    assert np.abs(K.diagonal().real - want.diagonal().real).max() <= TOL64 * scale
    assert np.array_equal(K, K.conj().T) and np.all(K.diagonal().imag == 0)
    assert torch.equal(ctx.gram(N, Xd, Yd, hermitian=True).cpu(), torch.from_numpy(K))  # P12


@pytest.mark.parametrize("N", [8, 16, 32])
def test_gram_P_dag_MP_is_hermitian_and_matches_oracle(lat, N):
    """the instance as the solver uses it: Y = M X makes G = X^dag M X Hermitian positive definite (P2), so the whole
    mirrored matrix must match the oracle's full product"""
    dims, fat, lng, ctx = lat
    X = H.np_sources(dims, N, 2300 + N)
    Xd = ctx.pack(torch.from_numpy(X).cuda())
    MXd = ctx.apply_M(0.05, N, Xd, ctx.empty_native(N))
    K = ctx.gram(N, Xd, MXd, hermitian=True).cpu().numpy()
    want = oracle.gram(X, oracle.apply_M(dims, fat, lng, 0.05, X))
    assert np.abs(K - want).max() <= 1e-12 * np.abs(want).max()  # two rounded operator applications + the reduction
    assert np.linalg.eigvalsh(K).min() > 0


@pytest.mark.parametrize("N", [7, 16, 28, 32])
@pytest.mark.parametrize("tri", [1, 2])
def test_block_update_triangular_coefficients(lat, N, tri):
    """Z = C + W a with a upper (tri = 1: S^-1, C^-1) or lower (tri = 2: S^dag) triangular; the fragments on the zero side
    are poisoned to prove they are never read.  N = 28, 32: four column tiles, the solver's path beyond
    24 rhs; also the form without C (Q = R C^-1, Alg. 2 l.4)."""
    dims, _, _, ctx = lat
    W, C = H.np_sources(dims, N, 2400 + N), H.np_sources(dims, N, 2500 + N)
    rng = np.random.default_rng(400 + N + tri)
    full = rng.standard_normal((N, N)) + 1j * rng.standard_normal((N, N))
    a = np.triu(full) if tri == 1 else np.tril(full)
    zero_side = np.tril(np.ones((N, N)), -1) if tri == 1 else np.triu(np.ones((N, N)), 1)
    a_d = torch.from_numpy(a + 1e30 * zero_side * _frag_mask(N, upper=(tri == 1))).cuda()
    Wd, Cd = ctx.pack(torch.from_numpy(W).cuda()), ctx.pack(torch.from_numpy(C).cuda())
    Zd = ctx.block_update(N, a_d, Cd, Wd, ctx.empty_native(N), tri=tri)
    assert H.relerr_inf(ctx.unpack(Zd, N).cpu().numpy(), oracle.block_axpy(a, W, C)) <= TOL64
    Zd = ctx.block_update(N, a_d, None, Wd, ctx.empty_native(N), tri=tri)
    assert H.relerr_inf(ctx.unpack(Zd, N).cpu().numpy(), oracle.block_axpy(a, W, np.zeros_like(W))) <= TOL64
    ctx.block_update(N, a_d, Cd, Wd, Cd, tri=tri)  # in place: Z aliases C
    assert H.relerr_inf(ctx.unpack(Cd, N).cpu().numpy(), oracle.block_axpy(a, W, C)) <= TOL64


@pytest.mark.parametrize("N", [4, 16, 32])
@pytest.mark.parametrize("precs", ["64<-32", "32<-64", "32<-32"])
def test_block_update_mixed_precisions(lat, N, precs):
    """PAPER.md:260 (Y precision >= X precision) and Alg. 3 l.5 (Qhat = R C^-1 rounded to fp32 on store): products and
    sums in fp64 whatever the storage, so an fp64 Z carries no fp32 rounding beyond that of the stored W"""
    from paper_1710_09745_b200 import binding
    dims, _, _, ctx = lat
    pz, pw = {"64<-32": (binding.F64, binding.F32), "32<-64": (binding.F32, binding.F64), "32<-32": (binding.F32, binding.F32)}[precs]
    W, C = H.np_sources(dims, N, 2600 + N), H.np_sources(dims, N, 2700 + N)
    if pw == binding.F32:
        W = _round32(W)
    if pz == binding.F32:
        C = _round32(C)
    rng = np.random.default_rng(500 + N)
    a = rng.standard_normal((N, N)) + 1j * rng.standard_normal((N, N))
    Wd, Cd = ctx.pack(torch.from_numpy(W).cuda(), pw), ctx.pack(torch.from_numpy(C).cuda(), pz)
    Zd = ctx.block_update(N, torch.from_numpy(a).cuda(), Cd, Wd, ctx.empty_native(N, pz), precZ=pz, precW=pw)
    got = ctx.unpack(Zd, N, pz).cpu().numpy()
    want = oracle.block_axpy(a, W, C)
    assert H.relerr_inf(got, want) <= (TOL64 if pz == binding.F64 else TOL32)


@pytest.mark.parametrize("N", [4, 8, 16, 24])
def test_block_qpx_update_fp32_blocks_fp64_X(lat, N):
    """the fused Q / P / X update of the mixed solver: P, Q in fp32, X in fp64"""
    from paper_1710_09745_b200 import binding
    dims, _, _, ctx = lat
    Q, P = (_round32(H.np_sources(dims, N, 2800 + 10 * k + N)) for k in range(2))
    X = H.np_sources(dims, N, 2830 + N)
    rng = np.random.default_rng(600 + N)
    full = lambda: rng.standard_normal((N, N)) + 1j * rng.standard_normal((N, N))
    Sinv, Sdag, Wm = np.triu(full()), np.tril(full()), full()
    Qd, Pd = (ctx.pack(torch.from_numpy(v).cuda(), binding.F32) for v in (Q, P))
    Xd = ctx.pack(torch.from_numpy(X).cuda())
    Pn = torch.empty_like(Pd)
    ctx.block_qpx_update(N, *(torch.from_numpy(m).cuda() for m in (Sinv, Sdag, Wm)), Qd, Pd, Pn, Xd, prec=binding.F32)
    Qn = oracle.block_axpy(Sinv, Q, np.zeros_like(Q))
    got_Q = ctx.unpack(Qd, N, binding.F32).cpu().numpy()
    assert H.relerr_inf(got_Q, Qn) <= TOL32
    # P_new = Q_new + P S^dag is formed from the unrounded Q_new in the accumulators
    assert H.relerr_inf(ctx.unpack(Pn, N, binding.F32).cpu().numpy(), oracle.block_axpy(Sdag, P, Qn)) <= TOL32
    # X is fp64: only the fp32 rounding already present in the stored P enters -> fp64 accuracy against the oracle on that P
    assert H.relerr_inf(ctx.unpack(Xd, N).cpu().numpy(), oracle.block_axpy(Wm, P, X)) <= TOL64


@pytest.mark.parametrize("mask", [1, 2, 3, 4, 8, 15])
def test_ablation_switches_do_not_change_the_result(mask):
    """BKR_OPT_ABLATION (the arms of the paper's Fig. 4) changes which kernels run, not what they
    compute: same solution to 1e-8, true residual <= tol"""
    from paper_1710_09745_b200 import binding
    dims = (4, 4, 4, 8)
    fat, lng = H.np_links(dims, "random", seed=61)
    B = H.np_sources(dims, 6, seed=62)
    ctx = binding.Context(dims)
    ctx.load_links(torch.from_numpy(fat).cuda(), torch.from_numpy(lng).cuda(), also_f32=True)
    Bd = torch.from_numpy(B).cuda()
    X0, rr0, st0 = ctx.solve_block(0.1, Bd, tol=1e-10)
    ctx.set_option(binding.OPT_ABLATION, mask)
    X1, rr1, st1 = ctx.solve_block(0.1, Bd, tol=1e-10)
    assert st1["status"] == 0 and max(rr1) <= 1e-10 and abs(st1["iters"] - st0["iters"]) <= 2
    assert float((X1 - X0).abs().max() / X0.abs().max()) <= 1e-8
    assert st1["gpu_launches"] > st0["gpu_launches"]
    Xm, rrm, stm = ctx.solve_block(0.1, Bd, tol=1e-10, inner_prec=binding.F32, delta=0.1)
    assert stm["status"] == 0 and oracle.true_relres(dims, fat, lng, 0.1, B, Xm.cpu().numpy()).max() <= 1e-10
