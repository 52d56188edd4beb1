"""GPU solver parity: blockCGrQ / CG through the C ABI against the oracle's solves and the dense solve.
north_star: true relative residual <= 1e-10 and solutions within 1e-8 of the oracle's (U16: the
iterates of block CG are unique only up to rounding, so iteration counts may differ by a few; what is unique --
the converged solution -- is compared, and the rest is checked for validity)."""
import numpy as np
import pytest
import torch

import oracle
from tests import helpers as H

pytestmark = pytest.mark.gpu
TOL = 1e-10


def _ctx(dims, fat, lng, also_f32=True):
    from paper_1710_09745_b200 import binding
    ctx = binding.Context(dims)
    ctx.load_links(torch.from_numpy(fat).cuda(), torch.from_numpy(lng).cuda(), also_f32=also_f32)
    return ctx


def _soldiff(X, Xo):
    """max over rhs of ||x - x_o||_2 / ||x_o||_2 and the block inf-norm version (U16)."""
    per = [np.linalg.norm(X[i] - Xo[i]) / np.linalg.norm(Xo[i]) for i in range(X.shape[0])]
    return max(max(per), np.abs(X - Xo).max() / np.abs(Xo).max())


@pytest.fixture(scope="module")
def cfg1():
    """BASELINE.json config 1: 4^4, random SU(3), m = 0.1, N = 4."""
    dims = (4, 4, 4, 4)
    fat, lng = H.np_links(dims, "random", seed=11)
    B = H.np_sources(dims, 4, seed=12)
    return dims, fat, lng, B, _ctx(dims, fat, lng)


def test_config1_block_cg_vs_oracle_and_dense(cfg1):
    from paper_1710_09745_b200 import binding
    dims, fat, lng, B, ctx = cfg1
    X, rr, st = ctx.solve_block(0.1, torch.from_numpy(B).cuda(), tol=TOL)
    X = X.cpu().numpy()
    assert st["status"] == binding.OK and max(rr) <= TOL
    ro = oracle.block_cg(dims, fat, lng, 0.1, B, tol=TOL)
    assert ro["status"] == 0
    assert _soldiff(X, ro["X"]) <= 1e-8
    assert abs(st["iters"] - ro["iters"]) <= 3
    # the oracle's own true residual of the GPU's X (independent of the GPU's claim)
    assert oracle.true_relres(dims, fat, lng, 0.1, B, X).max() <= TOL
    # the definition: X* = M^-1 B from the dense matrix of tests/helpers.py
    _, _, M = H.dense_blocks(dims, fat, lng, 0.1)
    Xs = np.linalg.solve(M, B.reshape(4, -1).T).T.reshape(B.shape)
    assert _soldiff(X, Xs) <= 1e-8


def test_config1_cg_sequential_and_batched(cfg1):
    from paper_1710_09745_b200 import binding
    dims, fat, lng, B, ctx = cfg1
    Bd = torch.from_numpy(B).cuda()
    its_o = []
    Xo = np.empty_like(B)
    for j in range(4):
        Xo[j], it, rc, _ = oracle.cg(dims, fat, lng, 0.1, B[j], tol=TOL)
        assert rc == 0
        its_o.append(it)
    for batched in (False, True):
        X, its, rr, st = ctx.solve_cg(0.1, Bd, tol=TOL, batched=batched)
        assert st["status"] == binding.OK and max(rr) <= 1.5 * TOL
        assert _soldiff(X.cpu().numpy(), Xo) <= 1e-8
        assert max(abs(a - b) for a, b in zip(its, its_o)) <= 3


def test_block_N1_equals_cg(cfg1):
    """blockCGrQ with one rhs is CG."""
    dims, fat, lng, B, ctx = cfg1
    Bd = torch.from_numpy(B[:1]).cuda()
    Xb, _, sb = ctx.solve_block(0.1, Bd, tol=TOL)
    Xc, its, _, _ = ctx.solve_cg(0.1, Bd, tol=TOL)
    assert abs(sb["iters"] - its[0]) <= 3
    assert _soldiff(Xb.cpu().numpy(), Xc.cpu().numpy()) <= 1e-8


def test_free_field_finite_termination():
    """pin P9 through the CUDA path: 5 distinct eigenvalues on the free 4^4 field -> 5 iterations."""
    dims = (4, 4, 4, 4)
    fat, lng = H.np_links(dims, "free", seed=0, c1=9.0 / 8.0)
    ctx = _ctx(dims, fat, lng, also_f32=False)
    B = torch.from_numpy(H.np_sources(dims, 4, 77)).cuda()
    _, rr, st = ctx.solve_block(0.1, B, tol=TOL)
    assert st["iters"] <= 5 and max(rr) <= TOL
    _, its, rr, _ = ctx.solve_cg(0.1, B, tol=TOL, batched=True)
    assert max(its) <= 5 and max(rr) <= TOL


def test_initial_guess_is_honoured(cfg1):
    dims, fat, lng, B, ctx = cfg1
    Bd = torch.from_numpy(B).cuda()
    X, _, st0 = ctx.solve_block(0.1, Bd, tol=TOL)
    X2, rr, st = ctx.solve_block(0.1, Bd, X0=X, tol=TOL)
    assert st["iters"] <= 1 and max(rr) <= TOL
    X3, rr3, st3 = ctx.solve_block(0.1, Bd, X0=X * (1 + 1e-4), tol=TOL)
    assert 0 < st3["iters"] < st0["iters"] and max(rr3) <= TOL


def test_duplicate_rhs_reports_breakdown(cfg1):
    """U15: linearly dependent right-hand sides make R^dag R singular."""
    from paper_1710_09745_b200 import binding
    dims, fat, lng, B, ctx = cfg1
    B2 = B.copy()
    B2[3] = B2[0]
    _, _, st = ctx.solve_block(0.1, torch.from_numpy(B2).cuda(), tol=TOL)
    assert st["status"] == binding.EBREAKDOWN


def test_maxiter_reports_noconv(cfg1):
    from paper_1710_09745_b200 import binding
    dims, fat, lng, B, ctx = cfg1
    _, rr, st = ctx.solve_block(0.1, torch.from_numpy(B).cuda(), tol=TOL, maxiter=8)
    assert st["status"] == binding.ENOCONV and st["iters"] == 8 and max(rr) > TOL


@pytest.mark.parametrize("k", [1, 3, 9])
def test_iterate_after_k_iterations_matches_oracle(cfg1, k):
    """X after exactly k iterations (maxiter = k, not converged) equals the oracle's k-th iterate: the X update of
    Alg. 1 l.10 is deferred into the next iteration's P update on the GPU and must be flushed when the
    loop stops early -- a missing flush leaves X one iteration behind.  Iterates are basis independent (U16)."""
    import oracle
    from paper_1710_09745_b200 import binding
    dims, fat, lng, B, ctx = cfg1
    X, rr, st = ctx.solve_block(0.1, torch.from_numpy(B).cuda(), tol=TOL, maxiter=k)
    assert st["status"] == binding.ENOCONV and st["iters"] == k
    ro = oracle.block_cg(dims, fat, lng, 0.1, B, tol=TOL, maxiter=k)
    assert ro["iters"] == k
    assert _soldiff(X.cpu().numpy(), ro["X"]) <= 1e-10


def test_mixed_iterate_flushes_deferred_update(cfg1):
    """same check through the reliable-update path: Y += X must see the deferred update (Alg. 3)"""
    import oracle
    from paper_1710_09745_b200 import binding
    dims, fat, lng, B, ctx = cfg1
    X, rr, st = ctx.solve_block(0.1, torch.from_numpy(B).cuda(), tol=TOL, inner_prec=binding.F32, delta=0.1)
    assert st["status"] == 0 and st["reliable_updates"] >= 1 and max(rr) <= TOL
    tr = oracle.true_relres(dims, fat, lng, 0.1, B, X.cpu().numpy())
    assert tr.max() <= TOL


def test_host_buffer_entry_points(cfg1):
    from paper_1710_09745_b200 import binding
    dims, fat, lng, B, ctx = cfg1
    Bh = torch.from_numpy(B).pin_memory()
    Xh = torch.zeros_like(Bh).pin_memory()
    rr, st = ctx.solve_block_host(0.1, Bh, Xh, tol=TOL)
    assert st["status"] == binding.OK and max(rr) <= TOL
    assert oracle.true_relres(dims, fat, lng, 0.1, B, Xh.numpy()).max() <= TOL
    Xh.zero_()
    its, rr, st = ctx.solve_cg_host(0.1, Bh, Xh, tol=TOL, batched=True)
    assert st["status"] == binding.OK
    assert oracle.true_relres(dims, fat, lng, 0.1, B, Xh.numpy()).max() <= 1.5 * TOL


def test_mixed_precision_block_cg(cfg1):
    """Algorithm 3: fp32 inner iteration + fp64 reliable updates reaches the fp64 tolerance."""
    from paper_1710_09745_b200 import binding
    dims, fat, lng, B, ctx = cfg1
    X, rr, st = ctx.solve_block(0.1, torch.from_numpy(B).cuda(), tol=TOL, inner_prec=binding.F32, delta=0.1)
    assert st["status"] == binding.OK and st["reliable_updates"] >= 3
    assert oracle.true_relres(dims, fat, lng, 0.1, B, X.cpu().numpy()).max() <= TOL
    ro = oracle.block_cg(dims, fat, lng, 0.1, B, tol=TOL)
    assert _soldiff(X.cpu().numpy(), ro["X"]) <= 1e-8
    assert st["iters"] <= 2 * ro["iters"]


@pytest.fixture(scope="module")
def cfg2():
    """BASELINE.json config 2: 16^4, proj_SU3(1 + 0.3 G), m = 0.05, N = 8."""
    dims = (16, 16, 16, 16)
    fat, lng = H.np_links(dims, "perturbed", seed=2)
    B = H.np_sources(dims, 8, seed=3)
    return dims, fat, lng, B, _ctx(dims, fat, lng)


def test_config2_block_cg_vs_oracle(cfg2):
    from paper_1710_09745_b200 import binding
    dims, fat, lng, B, ctx = cfg2
    X, rr, st = ctx.solve_block(0.05, torch.from_numpy(B).cuda(), tol=TOL)
    X = X.cpu().numpy()
    assert st["status"] == binding.OK and max(rr) <= TOL
    ro = oracle.block_cg(dims, fat, lng, 0.05, B, tol=TOL)
    assert ro["status"] == 0
    assert _soldiff(X, ro["X"]) <= 1e-8
    assert abs(st["iters"] - ro["iters"]) <= max(3, ro["iters"] // 50)
    assert oracle.true_relres(dims, fat, lng, 0.05, B, X).max() <= TOL


def test_config2_cg_vs_block(cfg2):
    from paper_1710_09745_b200 import binding
    dims, fat, lng, B, ctx = cfg2
    Bd = torch.from_numpy(B).cuda()
    Xb, _, sb = ctx.solve_block(0.05, Bd, tol=TOL)
    Xc, its, rr, sc = ctx.solve_cg(0.05, Bd, tol=TOL, batched=True)
    assert sc["status"] == binding.OK
    assert _soldiff(Xc.cpu().numpy(), Xb.cpu().numpy()) <= 1e-8
    assert sb["iters"] <= max(its)  # a block of 8 never needs more applications of M than CG
    x0, it0, rc, _ = oracle.cg(dims, fat, lng, 0.05, B[0], tol=TOL)
    assert rc == 0 and abs(it0 - its[0]) <= max(3, it0 // 50)


def test_config2_mixed_precision(cfg2):
    from paper_1710_09745_b200 import binding
    dims, fat, lng, B, ctx = cfg2
    X, rr, st = ctx.solve_block(0.05, torch.from_numpy(B).cuda(), tol=TOL, inner_prec=binding.F32, delta=0.1)
    assert st["status"] == binding.OK and st["reliable_updates"] >= 3
    assert oracle.true_relres(dims, fat, lng, 0.05, B, X.cpu().numpy()).max() <= TOL


# ------------------------------------------------------------------ blocks of more than 16 rhs (host control flow of solver.cu)

@pytest.fixture(scope="module")
def lat8():
    dims = (8, 8, 8, 8)
    fat, lng = H.np_links(dims, "perturbed", seed=71)
    return dims, fat, lng, _ctx(dims, fat, lng)


@pytest.mark.parametrize("N", [20, 24, 28, 32])
def test_large_block_solve_vs_oracle(lat8, N):
    """N = 17..24: fused Q/P/X update without Gram fusion; N > 24: the unfused path with per-iteration Q/Q2 and P/P2
    pointer swaps and tri = 1/2 block updates.  Solution, true residual and iteration count against
    the oracle's blockCGrQ; the k-th iterate (maxiter = k) must match too."""
    from paper_1710_09745_b200 import binding
    dims, fat, lng, ctx = lat8
    B = H.np_sources(dims, N, seed=72 + N)
    Bd = torch.from_numpy(B).cuda()
    X, rr, st = ctx.solve_block(0.05, Bd, tol=TOL)
    assert st["status"] == binding.OK and max(rr) <= TOL
    ro = oracle.block_cg(dims, fat, lng, 0.05, B, tol=TOL)
    assert ro["status"] == 0
    assert _soldiff(X.cpu().numpy(), ro["X"]) <= 1e-8
    assert abs(st["iters"] - ro["iters"]) <= 3
    assert oracle.true_relres(dims, fat, lng, 0.05, B, X.cpu().numpy()).max() <= TOL
    for k in (1, 4):
        Xk, _, stk = ctx.solve_block(0.05, Bd, tol=TOL, maxiter=k)
        assert stk["iters"] == k
        assert _soldiff(Xk.cpu().numpy(), oracle.block_cg(dims, fat, lng, 0.05, B, tol=TOL, maxiter=k)["X"]) <= 1e-10


@pytest.mark.parametrize("N", [24, 32])
def test_large_block_mixed_precision(lat8, N):
    from paper_1710_09745_b200 import binding
    dims, fat, lng, ctx = lat8
    B = H.np_sources(dims, N, seed=82 + N)
    X, rr, st = ctx.solve_block(0.05, torch.from_numpy(B).cuda(), tol=TOL, inner_prec=binding.F32, delta=0.1)
    assert st["status"] == binding.OK and st["reliable_updates"] >= 3
    assert oracle.true_relres(dims, fat, lng, 0.05, B, X.cpu().numpy()).max() <= TOL
    ro = oracle.block_cg(dims, fat, lng, 0.05, B, tol=TOL)
    assert _soldiff(X.cpu().numpy(), ro["X"]) <= 1e-8


def test_duplicate_rhs_reports_breakdown_mixed(cfg1):
    """the same negative case with the fp32 inner solver: the rank deficit is caught by the fp64 QR of the initial
    residual (Alg. 1 l.4 runs in fp64 also in the mixed solver), before any fp32 Gram matrix is factored"""
    from paper_1710_09745_b200 import binding
    dims, fat, lng, B, ctx = cfg1
    B2 = B.copy()
    B2[3] = B2[0]
    _, _, st = ctx.solve_block(0.1, torch.from_numpy(B2).cuda(), tol=TOL, inner_prec=binding.F32, delta=0.1)
    assert st["status"] == binding.EBREAKDOWN


@pytest.mark.parametrize("inner", ["f64", "f32"])
def test_nearly_dependent_rhs_two_pass_qr(cfg1, inner):
    """SURVEY.md NEXT-2 (refs [43, 44]): two sources equal to 1e-7 make the Gram matrix of the initial
    residual lose 14 digits; one Cholesky-QR pass breaks down (round 1 returned BKR_EBREAKDOWN), the two-pass QR
    orthonormalises the block and the solve converges to what the oracle's two-pass solver and the dense solve give."""
    from paper_1710_09745_b200 import binding
    dims, fat, lng, B, ctx = cfg1
    Bd = B.copy()
    Bd[3] = Bd[1] + 1e-7 * Bd[3]
    kw = dict(inner_prec=binding.F32, delta=0.1) if inner == "f32" else {}
    X, rr, st = ctx.solve_block(0.1, torch.from_numpy(Bd).cuda(), tol=1e-11, **kw)
    assert st["status"] == 0 and st["reorthonormalisations"] >= 1, st
    Xh = X.cpu().numpy()
    assert oracle.true_relres(dims, fat, lng, 0.1, Bd, Xh).max() <= TOL
    ro = oracle.block_cg(dims, fat, lng, 0.1, Bd, tol=1e-11, reorth=True)
    assert ro["status"] == 0
    assert _soldiff(Xh, ro["X"]) <= 1e-8
    _, _, M = H.dense_blocks(dims, fat, lng, 0.1)
    Xs = np.linalg.solve(M, Bd.reshape(4, -1).T).T.reshape(Bd.shape)
    assert _soldiff(Xh, Xs) <= 1e-8
    # a well conditioned block never takes the second pass
    _, _, st0 = ctx.solve_block(0.1, torch.from_numpy(B).cuda(), tol=TOL, **kw)
    assert st0["status"] == 0 and st0["reorthonormalisations"] == 0
