"""Parity metrics between a result of the CUDA path and a result of the CPU oracle (test helper).

No method arithmetic lives here: only comparisons (cosines, relative differences, Gram
matrices) in float64 numpy.  Tolerances are BASELINE.json's north_star values:
    separated components :  |lambda_gpu - lambda_or| / lambda_or <= 1e-4
                            |cos(P_gpu, P_or)|, |cos(T_gpu, T_or)| >= 1 - 1e-4, joint sign
    GS-PCA               :  max |P^T P - I| <= 1e-5
"separated" is decided from the ORACLE's lambdas only (reading P9):
component k is separated when every other stored oracle lambda differs from lambda_k by at
least 2 % of lambda_k.  Why 2 %: the method stops early, so even the float64 oracle's vector is
off the true singular vector by 1 - cos ~= 0.15 * eps / gap^2 (measured oracle-vs-SVD on the
scaled config 3: 1.1e-4 at a 1.2 % gap, 2.7e-5 at 2.9 %, 8e-6 at 3.3 %, eps = 1e-7); which
early-stopped vector comes out depends on the pass at which the stagnation test fires, and that
legitimately differs between float32 and float64 (reading C4).  Below a 2 % gap this ambiguity
alone reaches the 1e-4 tolerance, so single vectors are not a unique result there.
Non-separated components have no unique early-stopped vector (several results are correct);
for them the tests check what is unique: invariants, cluster energy, spanned subspace.
"""
from __future__ import annotations

import numpy as np

TOL_LAMBDA = 1e-4
TOL_COS = 1e-4
TOL_ORTHO_P = 1e-5
SEPARATION = 2e-2


def f64(a):
    return np.asarray(a, dtype=np.float64)


def separated_mask(lam_oracle: np.ndarray, count: int) -> np.ndarray:
    """mask[k] (k < count): min_{j != k} |lam_j - lam_k| >= SEPARATION * lam_k over ALL given lambdas."""
    lam = f64(lam_oracle)
    out = np.zeros(count, dtype=bool)
    for k in range(count):
        if lam[k] <= 0:
            continue
        others = np.delete(lam, k)
        out[k] = others.size == 0 or np.min(np.abs(others - lam[k])) >= SEPARATION * lam[k]
    return out


def signed_cos(a, b) -> float:
    a, b = f64(a), f64(b)
    na, nb = np.linalg.norm(a), np.linalg.norm(b)
    if na == 0 or nb == 0:
        return 0.0
    return float(a @ b) / (na * nb)


def ortho_defect(Q, unit: bool = True) -> float:
    """max |Q^T Q - I| (columns normalised first unless they are meant to be unit already)."""
    Q = f64(Q)
    if not unit:
        nrm = np.linalg.norm(Q, axis=0)
        nrm[nrm == 0] = 1.0
        Q = Q / nrm
    G = Q.T @ Q
    return float(np.max(np.abs(G - np.eye(G.shape[0]))))


def component_metrics(got_P, got_T, got_lam, ref_P, ref_T, ref_lam, count: int):
    """Per-component relative lambda error, signed cosines of loadings and scores."""
    rel = np.zeros(count)
    cp = np.zeros(count)
    ct = np.zeros(count)
    for k in range(count):
        rel[k] = abs(float(got_lam[k]) - float(ref_lam[k])) / float(ref_lam[k]) if ref_lam[k] > 0 else abs(float(got_lam[k]))
        cp[k] = signed_cos(got_P[:, k], ref_P[:, k])
        ct[k] = signed_cos(got_T[:, k], ref_T[:, k])
    return rel, cp, ct


def assert_separated_parity(got_P, got_T, got_lam, ref_P, ref_T, ref_lam, mask, what=""):
    count = len(mask)
    rel, cp, ct = component_metrics(got_P, got_T, got_lam, ref_P, ref_T, ref_lam, count)
    for k in range(count):
        if not mask[k]:
            continue
        assert rel[k] <= TOL_LAMBDA, f"{what} lambda[{k}] rel err {rel[k]:.3e}"
        assert abs(cp[k]) >= 1.0 - TOL_COS, f"{what} P[:, {k}] |cos| = {abs(cp[k]):.8f}"
        assert abs(ct[k]) >= 1.0 - TOL_COS, f"{what} T[:, {k}] |cos| = {abs(ct[k]):.8f}"
        assert np.sign(cp[k]) == np.sign(ct[k]), f"{what} joint sign of (T, P)[:, {k}] differs from the oracle"
    return rel, cp, ct


def subspace_cos_min(A, B) -> float:
    """Smallest cosine of the principal angles between span(A) and span(B) (same column count)."""
    Qa, _ = np.linalg.qr(f64(A))
    Qb, _ = np.linalg.qr(f64(B))
    s = np.linalg.svd(Qa.T @ Qb, compute_uv=False)
    return float(np.min(s))
