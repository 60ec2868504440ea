"""Pins of the CPU oracle (oracle/pca_oracle.cpp) against what the paper and the mathematics fix.

Nothing here compares the oracle with itself or with the CUDA path: expected values are hand
derivations (tests/golden/*.json, cited), closed forms, invariants the paper states (eq. 4,
orthogonality, "full SVD for K = N"), library routines (numpy SVD / eigh / mean) and brute
force (cyclic Jacobi on X^T X).  All run on CPU (`-m "not gpu"`).
"""
import json
import math
import os

import numpy as np
import pytest

from paper_0811_1081_b200 import inputs

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def _abs_cos(a, b):
    return abs(float(a @ b)) / (np.linalg.norm(a) * np.linalg.norm(b))


# ----------------------------------------------------------------------------- worked examples
def test_golden_worked_3x2_nipals(oracle_mod):
    g = json.load(open(os.path.join(GOLD, "worked_3x2.json")))
    X = np.array(g["X_rows"], dtype=np.float64)
    r = oracle_mod.pca(X, g["K"], g["eps"], g["max_iter"], oracle_mod.ALGO_NIPALS)
    assert list(r.iters) == g["iters"]
    lam = math.sqrt(g["lambda_sq_num"] / g["lambda_sq_den"])
    nrm = math.sqrt(g["norm_sq"])
    assert abs(r.lam[0] - lam) <= 1e-14 * lam
    np.testing.assert_allclose(r.P[:, 0], np.array(g["p_int"]) / nrm, rtol=1e-14, atol=0)
    np.testing.assert_allclose(r.T[:, 0], np.array(g["t_int"]) / nrm, rtol=1e-14, atol=0)
    R = X - np.outer(g["t_int"], g["p_int"]) / g["norm_sq"]          # eq. (3)
    np.testing.assert_allclose(r.R, R, rtol=0, atol=1e-14)
    # one pass only (max_iter = 1) returns the pass-1 lambda: pins "lambda' is taken every pass"
    r1 = oracle_mod.pca(X, 1, 1.0, 1, oracle_mod.ALGO_NIPALS)
    assert list(r1.iters) == [1]
    lam1 = math.sqrt(g["lambda_pass1_sq_num"] / g["lambda_pass1_sq_den"])
    assert abs(r1.lam[0] - lam1) <= 1e-14 * lam1


@pytest.mark.parametrize("algo", [0, 1])
def test_golden_diag_2x2(oracle_mod, algo):
    g = json.load(open(os.path.join(GOLD, "diag_2x2.json")))
    X = np.array(g["X_rows"], dtype=np.float64)
    r = oracle_mod.pca(X, g["K"], g["eps"], g["max_iter"], algo)
    assert list(r.iters) == g["iters"]
    np.testing.assert_array_equal(r.lam, np.array(g["lambda"], dtype=np.float64))
    np.testing.assert_array_equal(r.T, np.array(g["T_rows"], dtype=np.float64))
    np.testing.assert_array_equal(r.P, np.array(g["P_rows"], dtype=np.float64))
    np.testing.assert_array_equal(r.R, np.array(g["R_rows"], dtype=np.float64))


# ----------------------------------------------------------------------------- P1 prescribed spectrum
@pytest.mark.parametrize("algo", [0, 1])
def test_prescribed_spectrum_noise_free(oracle_mod, algo):
    """X = U diag(s) V^T exactly (no noise): lambda_k = s_k, P = +-V, T = +-s_k U."""
    cfg = inputs.scaled(inputs.config(0), 256, 64, K=8, noise=0.0)
    pr = inputs.generate(cfg, keep_factors=True)
    # use the float64 product, not the float32 cast, so the pin is at double precision
    U, V, s = pr.truth["U"], pr.truth["V"], pr.truth["s"]
    X = oracle_mod.center((U * s[None, :]) @ V.T)
    r = oracle_mod.pca(X, 8, 1e-14, 10000, algo)
    assert np.all(r.iters < 10000) and np.all(r.iters >= 2)
    np.testing.assert_allclose(r.lam, s[:8], rtol=1e-11)
    for k in range(8):
        assert _abs_cos(r.P[:, k], V[:, k]) >= 1 - 1e-11
        assert _abs_cos(r.T[:, k], U[:, k]) >= 1 - 1e-11
        assert abs(np.linalg.norm(r.T[:, k]) - r.lam[k]) <= 1e-12 * r.lam[k]
        assert abs(np.linalg.norm(r.P[:, k]) - 1.0) <= 1e-14
        # joint sign: T[:,k] P[:,k]^T is the rank-1 term s_k U_k V_k^T
        sg = np.sign(r.P[:, k] @ V[:, k])
        # lambda stagnates quadratically faster than the vector converges (Rayleigh quotient), so a
        # 1e-14 stagnation test leaves an O(1e-7) angle: elementwise agreement is ~1e-7, not 1e-14
        np.testing.assert_allclose(sg * r.T[:, k], s[k] * U[:, k], atol=2e-6)


# ----------------------------------------------------------------------------- P2 Jacobi, P3 SVD
def test_jacobi_matches_library_eigh(oracle_mod):
    rng = np.random.default_rng(5)
    A = rng.standard_normal((40, 40))
    A = A + A.T
    w, V, sweeps = oracle_mod.jacobi_eigh(A)
    assert 1 <= sweeps < 60
    wl = np.linalg.eigvalsh(A)
    np.testing.assert_allclose(np.sort(w), wl, rtol=0, atol=1e-12 * np.abs(wl).max())
    np.testing.assert_allclose(V.T @ V, np.eye(40), atol=1e-13)
    np.testing.assert_allclose(A @ V, V * w[None, :], atol=1e-12 * np.abs(wl).max())


@pytest.mark.parametrize("algo", [0, 1])
def test_cfg1_against_jacobi_and_svd(oracle_mod, algo):
    """Config 1: converged values are the eigen-pairs of X^T X (brute force) / the SVD (library)."""
    cfg = inputs.config(0)
    X = oracle_mod.center(inputs.generate(cfg).X)
    r = oracle_mod.pca(X, cfg.K, cfg.eps, cfg.max_iter, algo)
    w, Vec, _ = oracle_mod.jacobi_eigh(X.T @ X)
    order = np.argsort(-w)
    sv = np.linalg.svd(X, compute_uv=False)
    for k in range(cfg.K):
        # "maximum error eps for eigenvalues": eps = 1e-7 relative stagnation test
        assert abs(r.lam[k] ** 2 / w[order[k]] - 1) <= 5e-6
        assert abs(r.lam[k] / sv[k] - 1) <= 5e-6
        assert _abs_cos(r.P[:, k], Vec[:, order[k]]) >= 1 - 1e-5


def test_scaled_cfg2_against_svd(oracle_mod):
    cfg = inputs.scaled(inputs.config(1), 512, 128, K=16)
    X = oracle_mod.center(inputs.generate(cfg).X)
    r = oracle_mod.pca(X, cfg.K, cfg.eps, cfg.max_iter, oracle_mod.ALGO_GS)
    Us, sv, Vt = np.linalg.svd(X, full_matrices=False)
    np.testing.assert_allclose(r.lam, sv[:cfg.K], rtol=5e-6)
    for k in range(cfg.K):
        assert _abs_cos(r.P[:, k], Vt[k]) >= 1 - 1e-4
        assert _abs_cos(r.T[:, k], Us[:, k]) >= 1 - 1e-4


def test_K1_is_top_singular_triplet(oracle_mod):
    rng = np.random.default_rng(11)
    X = oracle_mod.center(rng.standard_normal((200, 30)) * np.linspace(3, 1, 30)[None, :])
    Us, sv, Vt = np.linalg.svd(X, full_matrices=False)
    for algo in (0, 1):
        r = oracle_mod.pca(X, 1, 1e-13, 100000, algo)
        assert abs(r.lam[0] / sv[0] - 1) <= 1e-9
        assert _abs_cos(r.P[:, 0], Vt[0]) >= 1 - 1e-9
        assert _abs_cos(r.T[:, 0], Us[:, 0]) >= 1 - 1e-9


# ----------------------------------------------------------------------------- P4, P5 identities
@pytest.mark.parametrize("algo", [0, 1])
@pytest.mark.parametrize("eps", [1e-3, 1e-9])
def test_energy_and_decomposition_identities(oracle_mod, algo, eps):
    """eq. (4) X = T_K P_K^T + R elementwise, and ||R||_F^2 = ||X||_F^2 - sum lambda_k^2, any eps."""
    cfg = inputs.scaled(inputs.config(2), 300, 80, K=12)
    X = oracle_mod.center(inputs.generate(cfg).X)
    r = oracle_mod.pca(X, cfg.K, eps, 10000, algo)
    np.testing.assert_allclose(r.T @ r.P.T + r.R, X, rtol=0, atol=1e-11 * np.abs(X).max())
    e_x, e_r = np.sum(X * X), np.sum(r.R * r.R)
    assert abs(e_x - np.sum(r.lam ** 2) - e_r) <= 1e-12 * e_x
    for k in range(cfg.K):
        assert abs(np.linalg.norm(r.T[:, k]) - r.lam[k]) <= 1e-12 * r.lam[k]


# ----------------------------------------------------------------------------- P6 orthogonality
def test_gs_orthogonality_and_nipals_loss(oracle_mod):
    """GS-PCA: loads AND scores orthogonal; NIPALS scores are not."""
    cfg = inputs.config(0)
    X = oracle_mod.center(inputs.generate(cfg).X)
    g = oracle_mod.pca(X, cfg.K, cfg.eps, cfg.max_iter, oracle_mod.ALGO_GS)
    n = oracle_mod.pca(X, cfg.K, cfg.eps, cfg.max_iter, oracle_mod.ALGO_NIPALS)
    I = np.eye(cfg.K)

    def offdiag(T):
        Vn = T / np.linalg.norm(T, axis=0, keepdims=True)
        return np.max(np.abs(Vn.T @ Vn - I))

    assert np.max(np.abs(g.P.T @ g.P - I)) <= 1e-12
    assert offdiag(g.T) <= 1e-12
    assert offdiag(n.T) > 1e-8          # early stopping leaves NIPALS scores visibly non-orthogonal
    assert offdiag(n.T) > 1e3 * offdiag(g.T)


def test_gs_orthogonality_collinear(oracle_mod):
    cfg = inputs.scaled(inputs.config(2), 400, 96, K=24)        # X = A B + noise, rank-16 signal
    X = oracle_mod.center(inputs.generate(cfg).X)
    g = oracle_mod.pca(X, cfg.K, cfg.eps, cfg.max_iter, oracle_mod.ALGO_GS)
    I = np.eye(cfg.K)
    Vn = g.T / g.lam[None, :]
    assert np.max(np.abs(g.P.T @ g.P - I)) <= 1e-12
    assert np.max(np.abs(Vn.T @ Vn - I)) <= 1e-12


# ----------------------------------------------------------------------------- P7 K = N
def test_full_decomposition_K_equals_N(oracle_mod):
    """K = N: 'full SVD ... with a maximum error eps for eigenvalues'."""
    cfg = inputs.scaled(inputs.config(4), 256, 32, K=32)
    X = oracle_mod.center(inputs.generate(cfg).X)
    r = oracle_mod.pca(X, 32, 1e-10, 100000, oracle_mod.ALGO_GS)
    sv = np.linalg.svd(X, compute_uv=False)
    np.testing.assert_allclose(np.sort(r.lam)[::-1], sv, rtol=1e-6)
    assert np.linalg.norm(X - r.T @ r.P.T) <= 1e-3 * np.linalg.norm(X)
    assert np.max(np.abs(r.P.T @ r.P - np.eye(32))) <= 1e-12
    assert np.max(np.abs(r.P @ r.P.T - np.eye(32))) <= 1e-12      # square orthogonal


# ----------------------------------------------------------------------------- P8 control flow
def test_eps_zero_runs_exactly_max_iter(oracle_mod):
    rng = np.random.default_rng(3)
    X = rng.standard_normal((50, 10))
    for algo in (0, 1):
        r = oracle_mod.pca(X, 3, 0.0, 17, algo)       # strict '<' never fires with eps = 0
        assert list(r.iters) == [17, 17, 17]


def test_eps_one_stops_at_second_pass(oracle_mod):
    """lambda starts at 0 and the test is strict: pass 1 cannot fire, pass 2 does."""
    rng = np.random.default_rng(4)
    X = rng.standard_normal((50, 10))
    for algo in (0, 1):
        r = oracle_mod.pca(X, 3, 1.0, 100, algo)
        assert list(r.iters) == [2, 2, 2]


def test_rank_one_converges_in_two_passes(oracle_mod):
    rng = np.random.default_rng(6)
    a, b = rng.standard_normal(64), rng.standard_normal(12)
    X = np.outer(a, b)
    for algo in (0, 1):
        r = oracle_mod.pca(X, 1, 1e-12, 100, algo)
        assert r.iters[0] == 2
        assert abs(r.lam[0] - np.linalg.norm(a) * np.linalg.norm(b)) <= 1e-12 * r.lam[0]
        assert _abs_cos(r.P[:, 0], b) >= 1 - 1e-14


def test_gs_first_component_equals_nipals(oracle_mod):
    """For k = 0 no projection is applied; GS-PCA only rescales t each pass."""
    cfg = inputs.config(0)
    X = oracle_mod.center(inputs.generate(cfg).X)
    g = oracle_mod.pca(X, 1, cfg.eps, cfg.max_iter, oracle_mod.ALGO_GS)
    n = oracle_mod.pca(X, 1, cfg.eps, cfg.max_iter, oracle_mod.ALGO_NIPALS)
    assert g.iters[0] == n.iters[0]
    assert abs(g.lam[0] - n.lam[0]) <= 1e-13 * n.lam[0]
    np.testing.assert_allclose(g.P, n.P, atol=1e-13)
    np.testing.assert_allclose(g.T, n.T, atol=1e-12)


def test_degenerate_zero_column_and_zero_matrix(oracle_mod):
    rng = np.random.default_rng(8)
    X = rng.standard_normal((30, 6))
    X[:, 1] = 0.0                                   # start column of component 1 is exactly zero
    for algo in (0, 1):
        r = oracle_mod.pca(X, 3, 1e-9, 1000, algo)
        assert r.iters[1] == 0 and r.lam[1] == 0.0
        assert not r.T[:, 1].any() and not r.P[:, 1].any()
        assert r.iters[0] >= 2 and r.iters[2] >= 2
        np.testing.assert_allclose(r.T @ r.P.T + r.R, X, atol=1e-12)
        z = oracle_mod.pca(np.zeros((5, 3)), 2, 1e-7, 10, algo)
        assert list(z.iters) == [0, 0] and not z.lam.any() and not z.R.any()


def test_invalid_arguments(oracle_mod):
    X = np.ones((4, 3))
    for bad in (dict(K=0), dict(K=4), dict(eps=-1.0), dict(max_iter=0), dict(algo=2)):
        kw = dict(K=2, eps=1e-7, max_iter=10, algo=0)
        kw.update(bad)
        with pytest.raises(ValueError):
            oracle_mod.pca(X, **kw)


# ----------------------------------------------------------------------------- centring
def test_center_matches_library_mean(oracle_mod):
    rng = np.random.default_rng(9)
    X = rng.standard_normal((123, 17)) + 100.0 * rng.standard_normal(17)[None, :]
    Xc = oracle_mod.center(X)
    np.testing.assert_allclose(Xc, X - X.mean(axis=0, keepdims=True), atol=1e-12)
    assert np.max(np.abs(Xc.sum(axis=0))) <= 1e-10
    # literal eq. (1): the mean COLUMN is removed, so every ROW sums to zero and rank drops by one
    Xe = oracle_mod.center_eq1(X)
    np.testing.assert_allclose(Xe, X - X.mean(axis=1, keepdims=True), atol=1e-12)
    assert np.linalg.matrix_rank(Xe) == 16


# ----------------------------------------------------------------------------- determinism
def test_thread_count_independence(oracle_mod):
    cfg = inputs.scaled(inputs.config(1), 700, 96, K=6)
    X = oracle_mod.center(inputs.generate(cfg).X)
    n0 = oracle_mod.num_threads()
    try:
        oracle_mod.set_num_threads(1)
        a = oracle_mod.pca(X, cfg.K, cfg.eps, cfg.max_iter, oracle_mod.ALGO_GS)
        oracle_mod.set_num_threads(max(2, n0))
        b = oracle_mod.pca(X, cfg.K, cfg.eps, cfg.max_iter, oracle_mod.ALGO_GS)
    finally:
        oracle_mod.set_num_threads(n0)
    assert np.array_equal(a.iters, b.iters)
    assert np.array_equal(a.lam, b.lam) and np.array_equal(a.T, b.T) and np.array_equal(a.P, b.P)


def test_absolute_test_mode_worked_example(oracle_mod):
    """The text's absolute test |lambda' - lambda| <= eps (reading C3, non-default mode):
    hand-derived first-pass values of the 3 x 2 example (lambda starts at 0, so eps >= lambda'_1 stops on pass 1)."""
    g = json.load(open(os.path.join(GOLD, "worked_3x2.json")))
    a = g["absolute_test"]
    X = np.asfortranarray(np.array(g["X_rows"], dtype=np.float64))
    r = oracle_mod.pca(X, 1, a["eps"], g["max_iter"], oracle_mod.ALGO_NIPALS, test_mode=1)
    nrm = np.sqrt(a["norm_sq"])
    assert r.iters.tolist() == a["iters"]
    np.testing.assert_allclose(r.lam[0] ** 2, a["lambda_sq_num"] / a["lambda_sq_den"], rtol=1e-14)
    np.testing.assert_allclose(r.P[:, 0], np.array(a["p_int"]) / nrm, rtol=1e-14)
    np.testing.assert_allclose(r.T[:, 0], np.array(a["t_int"]) / nrm, rtol=1e-14)
    # the same eps under the listings' relative test runs on (strict test cannot fire on pass 1, reading C8)
    r0 = oracle_mod.pca(X, 1, 1.0, g["max_iter"], oracle_mod.ALGO_NIPALS, test_mode=0)
    assert r0.iters.tolist() == g["iters"]


def test_absolute_and_relative_tests_agree_when_tight(oracle_mod):
    """eps_abs = eps_rel * lambda makes the two tests the same decision up to the <= / < boundary: same passes +- 1,
    same lambda to the convergence error (the choice changes iteration counts, not results)."""
    cfg = inputs.config(0)
    pr = inputs.generate(cfg)
    Xc = oracle_mod.center(pr.X)
    rel = oracle_mod.pca(Xc, 3, 1e-9, 10000, oracle_mod.ALGO_GS, want_residual=False)
    for k in range(3):
        ab = oracle_mod.pca(Xc, k + 1, 1e-9 * rel.lam[k], 10000, oracle_mod.ALGO_GS, want_residual=False, test_mode=1)
        assert abs(int(ab.iters[k]) - int(rel.iters[k])) <= 1
        np.testing.assert_allclose(ab.lam[k], rel.lam[k], rtol=1e-8)


# ----------------------------------------------------------------------------- round-2 pins
def test_golden_worked_gs_3x3_one_pass(oracle_mod):
    """Hand-derived GS-PCA example (tests/golden/worked_gs_3x3.json): K = 2, max_iter = 1.  Component 1 depends on the start vector
    being column 1 of the DEFLATED residual and on a non-zero scores-side coefficient B (:1030-1031)."""
    g = json.load(open(os.path.join(GOLD, "worked_gs_3x3.json")))
    X = np.array(g["X_rows"], dtype=np.float64)
    r = oracle_mod.pca(X, g["K"], g["eps"], g["max_iter"], oracle_mod.ALGO_GS)
    assert list(r.iters) == g["iters"]
    for k in range(2):
        num, den = g["lambda_sq"][k]
        np.testing.assert_allclose(r.lam[k] ** 2, num / den, rtol=1e-14)
        np.testing.assert_allclose(r.P[:, k], np.array(g["P_int"][k]) / math.sqrt(g["P_norm_sq"][k]), rtol=0, atol=1e-15)
        np.testing.assert_allclose(r.T[:, k], np.array(g["T_int"][k]) / math.sqrt(g["T_den_sq"][k]), rtol=0, atol=2e-15)
    np.testing.assert_allclose(r.R, np.array(g["R_num"], dtype=np.float64) / np.array(g["R_den"], dtype=np.float64), rtol=0, atol=2e-15)
    # what the two plausible mistakes would have produced instead (same derivation): far outside the tolerance above
    num, den = g["mutants"]["no_scores_projection_lambda1_sq"]
    assert abs(r.lam[1] ** 2 - num / den) > 1e-1


@pytest.mark.parametrize("seed", [0, 1, 2])
def test_gs_loads_projection_is_needed_after_one_pass(oracle_mod, seed):
    """The loads-side Gram-Schmidt step A = P_(k)^T p, p -= P_(k) A.  After >= 2 passes R^T t is
    orthogonal to the previous loadings to rounding anyway, so only an EARLY-STOPPED run sees the step: with max_iter = 1 the
    deflation leaves R p_1 = V_(1) B != 0, the raw loads of component 2 have a component along p_1 of order 1e-2, and the claim
    'orthogonal loads' holds only because of this step (a dropped step, a wrong sign or k-1 columns all
    give max|P^T P - I| ~ 1e-2)."""
    rng = np.random.default_rng(100 + seed)
    X = rng.standard_normal((6, 4))
    r = oracle_mod.pca(X, 3, 1e-7, 1, oracle_mod.ALGO_GS)
    assert list(r.iters) == [1, 1, 1]
    assert np.max(np.abs(r.P.T @ r.P - np.eye(3))) <= 1e-12
    Vn = r.T / r.lam[None, :]
    assert np.max(np.abs(Vn.T @ Vn - np.eye(3))) <= 1e-12
    # the raw loads of component 2 are NOT orthogonal to p_1: recompute them from the returned quantities
    # (R_2 = X - T_(2) P_(2)^T by eq. (4); start vector = column 2 of R_2)
    R2 = X - r.T[:, :2] @ r.P[:, :2].T
    p_raw = R2.T @ R2[:, 2]
    assert abs(r.P[:, 1] @ p_raw) / np.linalg.norm(p_raw) > 1e-4
    # eq. (4) still holds elementwise
    np.testing.assert_allclose(r.T @ r.P.T + r.R, X, rtol=0, atol=1e-13)


def test_relative_test_scales_eps_with_the_newest_lambda(oracle_mod):
    """`fabs(a-b) < er*b` with b the NEWEST lambda': on the 3 x 2 example lambda = 0 before pass 1, so
    with eps = 2 the test |0 - lambda'| = lambda' < 2 lambda' fires on pass 1.  Scaling with the OLD lambda (= 0) could not."""
    g = json.load(open(os.path.join(GOLD, "worked_3x2.json")))
    X = np.array(g["X_rows"], dtype=np.float64)
    for algo in (oracle_mod.ALGO_NIPALS, oracle_mod.ALGO_GS):
        r = oracle_mod.pca(X, 1, 2.0, g["max_iter"], algo)
        assert list(r.iters) == [1]
        np.testing.assert_allclose(r.lam[0] ** 2, g["lambda_pass1_sq_num"] / g["lambda_pass1_sq_den"], rtol=1e-14)


def test_start_vector_is_the_deflated_column_numeric(oracle_mod):
    """Reading C6 on a random matrix with max_iter = 1: the loadings of component 1 are
    R_1^T R_1[:,1] normalised (R_1 = X - t_0 p_0^T, eq. 3), NOT R_1^T X[:,1]."""
    rng = np.random.default_rng(21)
    X = rng.standard_normal((7, 5))
    r = oracle_mod.pca(X, 2, 1e-7, 1, oracle_mod.ALGO_NIPALS)
    R1 = X - np.outer(r.T[:, 0], r.P[:, 0])
    p_good = R1.T @ R1[:, 1]
    p_bad = R1.T @ X[:, 1]
    np.testing.assert_allclose(r.P[:, 1], p_good / np.linalg.norm(p_good), rtol=0, atol=1e-14)
    assert np.max(np.abs(r.P[:, 1] - p_bad / np.linalg.norm(p_bad))) > 1e-3


def test_separation_threshold_measurement(oracle_mod):
    """DESIGN.md reading P9 (why single-vector parity is asserted only above a 2 % eigenvalue gap), as a measurement: the method
    stops when lambda stagnates, so even the float64 oracle's loading vector is off the true singular vector
    (LAPACK SVD) by about 0.15 eps / gap^2.  On the scaled config 3 (16 signal values with gaps of 0.5 ... 3.3 %), eps = 1e-7:
    every component with a gap >= 2 % is within 5e-5 (half the north_star tolerance), components with 1 % <= gap < 1.5 % already
    reach 1e-4 -- the tolerance itself -- so a 1 % separation rule would compare vectors that are not unique at that tolerance."""
    cfg = inputs.scaled(inputs.config(2), 2048, 512, K=16)
    X = oracle_mod.center(inputs.generate(cfg).X)
    r = oracle_mod.pca(X, 17, 1e-7, 10000, oracle_mod.ALGO_GS, want_residual=False)
    _, s, Vt = np.linalg.svd(X, full_matrices=False)
    gap = np.array([min(abs(s[k] - s[j]) for j in range(17) if j != k) / s[k] for k in range(16)])
    defect = np.array([1.0 - _abs_cos(r.P[:, k], Vt[k]) for k in range(16)])
    assert np.all(defect[gap >= 0.02] <= 5e-5), (gap, defect)
    assert np.all(defect <= 0.6e-7 / gap ** 2), (gap, defect)               # 1 - cos <~ 0.15 eps / gap^2, with a factor 4 of slack
    narrow = (gap >= 0.01) & (gap < 0.015)
    assert narrow.any() and defect[narrow].max() >= 1e-4, (gap, defect)


def test_cgs2_mode_is_the_identity_in_double(oracle_mod):
    """gs_passes = 2 (CGS2, "applying it iteratively"): in exact arithmetic the second projection removes
    nothing, so in float64 the results agree with the listings' single projection to rounding and orthogonality is not
    worse -- for converged runs and for early-stopped ones (max_iter = 1), where the first projection is doing real work.
    (The second projection itself is visible only at the rounding level: this idempotence is its pin.)"""
    cfg = inputs.scaled(inputs.config(2), 300, 80, K=12)
    X = oracle_mod.center(inputs.generate(cfg).X)
    for max_iter in (10000, 1):
        a = oracle_mod.pca(X, cfg.K, 1e-9, max_iter, oracle_mod.ALGO_GS, gs_passes=1)
        b = oracle_mod.pca(X, cfg.K, 1e-9, max_iter, oracle_mod.ALGO_GS, gs_passes=2)
        assert np.array_equal(a.iters, b.iters)
        np.testing.assert_allclose(b.lam, a.lam, rtol=1e-12)
        np.testing.assert_allclose(b.P, a.P, rtol=0, atol=1e-11)
        I = np.eye(cfg.K)
        assert np.max(np.abs(b.P.T @ b.P - I)) <= max(np.max(np.abs(a.P.T @ a.P - I)), 1e-15) * 1.5
        Vn = b.T / b.lam[None, :]
        assert np.max(np.abs(Vn.T @ Vn - I)) <= 1e-12
    n1 = oracle_mod.pca(X, 4, 1e-9, 100, oracle_mod.ALGO_NIPALS, gs_passes=1)      # ignored by NIPALS-PCA
    n2 = oracle_mod.pca(X, 4, 1e-9, 100, oracle_mod.ALGO_NIPALS, gs_passes=2)
    assert np.array_equal(n1.T, n2.T) and np.array_equal(n1.P, n2.P)
    with pytest.raises(ValueError):
        oracle_mod.pca(X, 2, 1e-9, 10, oracle_mod.ALGO_GS, gs_passes=3)
