"""Pins of the oracle against what the paper and the mathematics fix (CPU only).

Each test names the pin of DESIGN.md section 3 it implements.  None of them compares the oracle with
itself: expected values come from closed forms, from dense matrices assembled independently in
tests/helpers.py, from numpy.linalg, or from invariants.
"""
import os

import numpy as np
import pytest

import oracle
from tests import helpers as H

D4 = (4, 4, 4, 4)
DASYM = (4, 6, 8, 10)


@pytest.fixture(scope="module")
def cfg1():
    fat, lng = H.np_links(D4, "random", seed=11)
    return fat, lng, H.np_sources(D4, 4, seed=12)


def inner(a, b):
    return np.vdot(a.ravel(), b.ravel())


# ---------------------------------------------------------------- operator

def test_P1_D_anti_hermitian():
    fat, lng = H.np_links(DASYM, "random", seed=1)
    psi_e, phi_o = H.np_sources(DASYM, 2, 3), H.np_sources(DASYM, 2, 4)
    lhs = inner(phi_o, oracle.dslash(DASYM, fat, lng, 1, psi_e))
    rhs = -np.conj(inner(psi_e, oracle.dslash(DASYM, fat, lng, 0, phi_o)))
    assert abs(lhs - rhs) <= 1e-13 * abs(lhs)


def test_P2_M_hermitian_positive_definite():
    fat, lng = H.np_links(DASYM, "perturbed", seed=2)
    m = 0.05
    psi, phi = H.np_sources(DASYM, 1, 5), H.np_sources(DASYM, 1, 6)
    Mpsi, Mphi = oracle.apply_M(DASYM, fat, lng, m, psi), oracle.apply_M(DASYM, fat, lng, m, phi)
    a, b = inner(phi, Mpsi), np.conj(inner(psi, Mphi))
    assert abs(a - b) <= 1e-13 * abs(a)
    q = inner(psi, Mpsi)
    want = 4 * m * m * np.linalg.norm(psi) ** 2 + np.linalg.norm(oracle.dslash(DASYM, fat, lng, 1, psi)) ** 2
    assert abs(q.imag) <= 1e-13 * abs(q) and abs(q.real - want) <= 1e-13 * want


def _golden_spectrum():
    path = os.path.join(os.path.dirname(__file__), "golden", "free_field_4x4x4x4_spectrum.txt")
    rows = [l.split() for l in open(path) if l.strip() and not l.startswith("#")]
    return np.concatenate([np.full(int(r[2]), float(r[1])) for r in rows])


def _dense_from_oracle(dims, fat, lng, mass):
    L = H.synth.volume(dims) // 2 * 3
    M = np.empty((L, L), dtype=np.complex128)
    eye = np.eye(L, dtype=np.complex128).reshape(L, L // 3, 3)
    for j0 in range(0, L, 64):
        M[:, j0:j0 + 64] = oracle.apply_M(dims, fat, lng, mass, eye[j0:j0 + 64]).reshape(-1, L).T
    return M


def test_P3_free_field_spectrum_worked_example():
    fat, lng = H.np_links(D4, "free", seed=0, c1=9.0 / 8.0)
    M = _dense_from_oracle(D4, fat, lng, 0.1)
    ev = np.sort(np.linalg.eigvalsh(0.5 * (M + M.conj().T)))
    assert np.abs(M - M.conj().T).max() < 1e-13
    assert np.abs(ev - np.sort(_golden_spectrum())).max() < 1e-12


@pytest.mark.parametrize("n", [(1, 0, 0, 0), (0, 2, 0, 0), (1, 2, 3, 4), (3, 5, 1, 7), (0, 0, 0, 3)])
def test_P3_free_field_plane_waves(n):
    c1, m = 9.0 / 8.0, 0.07
    fat, lng = H.np_links(DASYM, "free", seed=0, c1=c1)
    psi = H.plane_wave(DASYM, n, [0.3 - 0.2j, 1.0, -0.5j])
    out = oracle.apply_M(DASYM, fat, lng, m, psi)
    lam = H.free_lambda(DASYM, n, m, c1, H.synth.C3)
    assert H.relerr_inf(out, lam * psi) < 1e-13


def test_P4_gauge_covariance_random_links():
    fat, lng = H.np_links(DASYM, "random", seed=7)
    g = H.random_su3_field(DASYM, 8)
    f2, l2 = H.gauge_rotate_links(DASYM, fat, lng, g)
    psi = H.np_sources(DASYM, 2, 9)
    lhs = oracle.dslash(DASYM, f2, l2, 1, H.gauge_rotate_field(DASYM, psi, g, 0))
    rhs = H.gauge_rotate_field(DASYM, oracle.dslash(DASYM, fat, lng, 1, psi), g, 1)
    assert H.relerr_inf(lhs, rhs) < 1e-13


def test_P4_gauge_rotated_free_field_has_closed_form_eigenvectors():
    c1, m, n = 9.0 / 8.0, 0.1, (1, 2, 5, 3)
    fat, lng = H.np_links(DASYM, "free", seed=0, c1=c1)
    g = H.random_su3_field(DASYM, 21)
    f2, l2 = H.gauge_rotate_links(DASYM, fat, lng, g)
    psi = H.gauge_rotate_field(DASYM, H.plane_wave(DASYM, n, [1.0, 0.5j, -0.25]), g, 0)
    out = oracle.apply_M(DASYM, f2, l2, m, psi)
    assert H.relerr_inf(out, H.free_lambda(DASYM, n, m, c1, H.synth.C3) * psi) < 1e-13


def test_P5_dense_brute_force_operator(cfg1):
    fat, lng, B = cfg1
    Doe, Deo, M = H.dense_blocks(D4, fat, lng, 0.1)
    assert np.abs(Doe + Deo.conj().T).max() == 0.0  # D anti-Hermitian exactly (P1, dense)
    v = B.reshape(4, -1)
    assert H.relerr_inf(oracle.dslash(D4, fat, lng, 1, B).reshape(4, -1), v @ Doe.T) < 1e-14
    assert H.relerr_inf(oracle.dslash(D4, fat, lng, 0, B).reshape(4, -1), v @ Deo.T) < 1e-14
    assert H.relerr_inf(oracle.apply_M(D4, fat, lng, 0.1, B).reshape(4, -1), v @ M.T) < 1e-14
    ev = np.linalg.eigvalsh(M)
    assert ev.min() >= 0.04 - 1e-12 and ev.max() < 40.0


def test_dslash_sites_matches_full(cfg1):
    fat, lng, B = cfg1
    e = np.array([0, 5, 17, 127, 64])
    full = oracle.dslash(D4, fat, lng, 1, B)
    assert np.array_equal(oracle.dslash_sites(D4, fat, lng, 1, B, e), full[:, e, :])


# ---------------------------------------------------------------- block BLAS and small matrices

def test_P10_gram_and_block_axpy_vs_numpy():
    rng = np.random.default_rng(3)
    N, L = 5, 3 * 77
    X = rng.normal(size=(N, L)) + 1j * rng.normal(size=(N, L))
    Y = rng.normal(size=(N, L)) + 1j * rng.normal(size=(N, L))
    a = rng.normal(size=(N, N)) + 1j * rng.normal(size=(N, N))
    assert H.relerr_inf(oracle.gram(X, Y), X.conj() @ Y.T) < 1e-14
    K = oracle.gram(X, X)
    assert np.abs(K - K.conj().T).max() < 1e-13 and np.allclose(np.diag(K).real, (abs(X) ** 2).sum(1))
    assert H.relerr_inf(oracle.block_axpy(a, X, Y), Y + a.T @ X) < 1e-14


@pytest.mark.parametrize("N", [1, 2, 7, 16, 32])
def test_P11_small_matrices_vs_numpy_linalg(N):
    rng = np.random.default_rng(N)
    A = rng.normal(size=(N + 3, N)) + 1j * rng.normal(size=(N + 3, N))
    Hm = A.conj().T @ A + 0.5 * np.eye(N)
    R = oracle.cholesky_upper(Hm)
    assert np.allclose(np.tril(R, -1), 0) and (np.diag(R).real > 0).all() and np.allclose(np.diag(R).imag, 0)
    assert H.relerr_inf(R, np.linalg.cholesky(Hm).conj().T) < 1e-12
    assert H.relerr_inf(oracle.upper_inverse(R), np.linalg.inv(R)) < 1e-12
    assert H.relerr_inf(oracle.hpd_inverse(Hm), np.linalg.inv(Hm)) < 1e-12


def test_P7_thin_qr_identities():
    rng = np.random.default_rng(5)
    N, L = 6, 3 * 50
    Z = rng.normal(size=(N, L)) + 1j * rng.normal(size=(N, L))
    Q, R = oracle.thin_qr(Z)
    assert np.abs(Q.conj() @ Q.T - np.eye(N)).max() < 1e-13
    assert H.relerr_inf(R.T @ Q, Z) < 1e-14           # Z = Q R, blocks stored (N, L)
    assert np.allclose(np.tril(R, -1), 0) and (np.diag(R).real > 0).all()
    Qn, Rn = np.linalg.qr(Z.T)                        # library thin QR, fix the phase convention
    ph = np.diag(Rn) / abs(np.diag(Rn))
    assert H.relerr_inf(R, (Rn / ph[:, None])) < 1e-12


def test_P7b_two_pass_qr_on_nearly_dependent_columns():
    """orc_thin_qr2 (refs [43, 44] of PAPER.md:184-186; U24): on a well conditioned block it is Algorithm 2 up
    to rounding; with two columns equal to 1e-7 (kappa(Z) ~ 1e7, kappa(Z^dag Z) ~ 1e14) it still returns an orthonormal
    Q and the R of a library QR, where one pass leaves Q^dag Q off by ~1e-3 or breaks down; a block of rank N - 1 is
    reported as a breakdown."""
    rng = np.random.default_rng(15)
    N, L = 6, 3 * 64
    Z = rng.normal(size=(N, L)) + 1j * rng.normal(size=(N, L))
    Q1, R1 = oracle.thin_qr(Z)
    Q2, R2 = oracle.thin_qr(Z, two_pass=True)
    assert H.relerr_inf(R2, R1) < 1e-13 and H.relerr_inf(Q2, Q1) < 1e-13
    Zb = Z.copy()
    Zb[4] = Zb[1] + 1e-7 * Zb[4]
    Q, R = oracle.thin_qr(Zb, two_pass=True)
    assert np.abs(Q.conj() @ Q.T - np.eye(N)).max() < 1e-12
    assert H.relerr_inf(R.T @ Q, Zb) < 1e-13
    assert np.allclose(np.tril(R, -1), 0) and (np.diag(R).real > 0).all()
    Qn, Rn = np.linalg.qr(Zb.T)                        # Householder QR of the library: backward stable for any kappa
    ph = np.diag(Rn) / abs(np.diag(Rn))
    Rl = Rn / ph[:, None]
    assert np.abs(R - Rl).max() / np.abs(Rl).max() < 1e-9    # forward error of R ~ kappa(Z) u
    assert abs(R[4, 4] - Rl[4, 4]) / abs(Rl[4, 4]) < 1e-3   # the tiny pivot itself, to the digits kappa leaves
    try:                                               # one pass: broken down, or visibly not orthonormal
        Qp, _ = oracle.thin_qr(Zb)
        assert np.abs(Qp.conj() @ Qp.T - np.eye(N)).max() > 1e-6
    except ArithmeticError:
        pass
    Zc = Z.copy()
    Zc[4] = Zc[1]
    with pytest.raises(ArithmeticError):
        oracle.thin_qr(Zc, two_pass=True)


# ---------------------------------------------------------------- solvers

def test_P5_solutions_vs_dense_solve(cfg1):
    fat, lng, B = cfg1
    _, _, M = H.dense_blocks(D4, fat, lng, 0.1)
    Xstar = np.linalg.solve(M, B.reshape(4, -1).T).T.reshape(B.shape)
    res = oracle.block_cg(D4, fat, lng, 0.1, B, tol=1e-10)
    assert res["status"] == 0
    assert H.relerr_inf(res["X"], Xstar) < 1e-8
    for j in range(4):
        x, it, rc, _ = oracle.cg(D4, fat, lng, 0.1, B[j], tol=1e-10)
        assert rc == 0 and H.relerr_inf(x, Xstar[j]) < 1e-8
    assert oracle.true_relres(D4, fat, lng, 0.1, B, res["X"]).max() < 2e-10
    # block CG needs fewer applications of M per rhs than CG
    assert res["iters"] < it


def test_P6_block_cg_N1_reduces_to_cg(cfg1):
    fat, lng, B = cfg1
    _, it, rc, hist = oracle.cg(D4, fat, lng, 0.1, B[0], tol=1e-10)
    res = oracle.block_cg(D4, fat, lng, 0.1, B[:1], tol=1e-10)
    assert rc == 0 and res["status"] == 0 and abs(res["iters"] - it) <= 2
    n = 40
    assert np.abs(res["hist"][:n] / hist[:n] - 1).max() < 1e-9


def test_P8_iterated_residual_equals_true_residual(cfg1):
    fat, lng, B = cfg1
    for maxiter in (7, 30):
        res = oracle.block_cg(D4, fat, lng, 0.1, B, tol=1e-30, maxiter=maxiter, ntrace=maxiter)
        assert res["status"] == -6 and res["iters"] == maxiter
        true = oracle.true_relres(D4, fat, lng, 0.1, B, res["X"])
        C = res["C"][-1]
        bn = np.linalg.norm(B.reshape(4, -1), axis=1)
        it_res = np.linalg.norm(C, axis=0) / bn            # column norms of C (U11)
        assert np.abs(it_res / true - 1).max() < 1e-6
        assert np.allclose(np.tril(C, -1), 0)
        G = res["G"][-1]
        assert np.abs(G - G.conj().T).max() == 0 and np.linalg.eigvalsh(G).min() > 0


def test_P9_finite_termination_free_field():
    fat, lng = H.np_links(D4, "free", seed=0, c1=9.0 / 8.0)
    B = H.np_sources(D4, 4, 31)
    for j in range(4):
        _, it, rc, _ = oracle.cg(D4, fat, lng, 0.1, B[j], tol=1e-10)
        assert rc == 0 and it == 5
    res = oracle.block_cg(D4, fat, lng, 0.1, B, tol=1e-10)
    assert res["status"] == 0 and res["iters"] <= 5


def test_initial_guess_is_honoured(cfg1):
    fat, lng, B = cfg1
    res = oracle.block_cg(D4, fat, lng, 0.1, B, tol=1e-10)
    again = oracle.block_cg(D4, fat, lng, 0.1, B, X0=res["X"], tol=1e-9)
    assert again["status"] == 0 and again["iters"] == 0


def test_U15_breakdown_on_rank_deficient_block(cfg1):
    # a zero column makes R^dag R exactly singular: the Cholesky pivot is exactly 0.
    # (Exactly duplicated columns give a pivot of +-1e-16 in floating point, either sign: not a test.)
    fat, lng, B = cfg1
    B2 = B.copy()
    B2[2] = 0
    assert oracle.block_cg(D4, fat, lng, 0.1, B2, tol=1e-10)["status"] == -5
    with pytest.raises(ArithmeticError):
        oracle.cholesky_upper(np.array([[1.0, 2.0], [2.0, 1.0]], dtype=complex))


def test_mixed_precision_reliable_updates_reach_true_tolerance(cfg1):
    fat, lng, B = cfg1
    pure = oracle.block_cg(D4, fat, lng, 0.1, B, tol=1e-10)
    mix = oracle.block_cg(D4, fat, lng, 0.1, B, tol=1e-10, mixed=True, delta=0.1)
    assert mix["status"] == 0 and mix["reliable_updates"] >= 5
    assert oracle.true_relres(D4, fat, lng, 0.1, B, mix["X"]).max() <= 1e-10
    assert mix["iters"] <= 2 * pure["iters"]
    assert H.relerr_inf(mix["X"], pure["X"]) < 1e-8


def test_U13_fp32_storage_stalls_true_residual_without_updates(cfg1):
    """The oracle's fp32 emulation (round_f32 on P, Q, MP and the inner links, U13) must bite: with the delta trigger
    switched off (delta = 1e-30) the first reliable update only happens when the ITERATED residual reports tol, and the
    true residual that update computes is stuck near fp32 precision (SURVEY U13 probe: ~1e-7 .. 1e-6), orders of
    magnitude above the 1e-10 the iteration claims; the solve then stalls there (the search space was not preserved).
    With round_f32 a no-op the jump would not exist and that one update would end the solve.  The same solve with
    delta = 0.1 reaches the true 1e-10."""
    fat, lng, B = cfg1
    tol = 1e-10
    lazy = oracle.block_cg(D4, fat, lng, 0.1, B, tol=tol, mixed=True, delta=1e-30, maxiter=400)
    hist = lazy["hist"]
    first = next(i for i in range(1, len(hist)) if hist[i] > 20 * hist[i - 1])  # the update replaces r by the true value
    assert hist[first - 1] < 1e-8 and hist[first - 1] > tol * 0.01  # the iteration had (nearly) reported convergence ...
    assert 1e-9 < hist[first] < 1e-5                                 # ... while the true residual sat at fp32 level
    assert lazy["status"] == -6 and lazy["reliable_updates"] == 1 and hist[-1] > 1e-8  # and it never recovers
    mix = oracle.block_cg(D4, fat, lng, 0.1, B, tol=tol, mixed=True, delta=0.1)
    assert mix["status"] == 0 and oracle.true_relres(D4, fat, lng, 0.1, B, mix["X"]).max() <= tol


def test_P8_Qold_dag_P_is_identity_after_line8(cfg1):
    """(Q_old)^dag P = 1 right after Alg. 1 l.8 -- the new residual block is orthogonal to the previous
    search directions -- in pure fp64 and across block reliable updates (S = C_new C_prev^-1, U12, is what keeps it)."""
    fat, lng, B = cfg1
    N = B.shape[0]
    pure = oracle.block_cg(D4, fat, lng, 0.1, B, tol=1e-10, ntrace=40)
    for k in range(40):
        assert np.abs(pure["QP"][k] - np.eye(N)).max() <= 1e-9, k
    mix = oracle.block_cg(D4, fat, lng, 0.1, B, tol=1e-10, mixed=True, delta=0.1, ntrace=60)
    assert mix["reliable_updates"] >= 3
    for k in range(60):
        assert np.abs(mix["QP"][k] - np.eye(N)).max() <= 2e-5, k  # fp32 storage of P and Q


def test_reorth_solver_matches_plain_solver_and_survives_dependent_rhs(cfg1):
    """block CG with two-pass QR (oracle.block_cg(reorth=True)): same solutions and iteration count as Algorithm 1 on a
    well conditioned block; on a block with two sources equal to 1e-7 it converges to the dense solutions (P5's
    definition of X*), where the plain solver breaks down or stalls."""
    fat, lng, B = cfg1
    a = oracle.block_cg(D4, fat, lng, 0.1, B, tol=1e-10)
    b = oracle.block_cg(D4, fat, lng, 0.1, B, tol=1e-10, reorth=True)
    assert a["status"] == 0 and b["status"] == 0 and abs(a["iters"] - b["iters"]) <= 1
    assert H.relerr_inf(b["X"], a["X"]) < 1e-9
    Bd = B.copy()
    Bd[3] = Bd[1] + 1e-7 * Bd[3]
    r = oracle.block_cg(D4, fat, lng, 0.1, Bd, tol=1e-11, reorth=True)
    assert r["status"] == 0
    assert oracle.true_relres(D4, fat, lng, 0.1, Bd, r["X"]).max() <= 1e-10
    _, _, M = H.dense_blocks(D4, fat, lng, 0.1)
    Xs = np.linalg.solve(M, Bd.reshape(4, -1).T).T.reshape(Bd.shape)
    assert H.relerr_inf(r["X"], Xs) < 1e-8
