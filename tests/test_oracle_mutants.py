"""Mutation test of the oracle's pins (`-m "not gpu"`).

Each mutant is oracle/pca_oracle.cpp with ONE plausible mistake typed in (a dropped term, a wrong sign or index, the wrong
operand: the list VERDICT r1 used, plus a few more), compiled to a scratch library; tests/test_oracle_pins.py is then run
against it in a subprocess (PCA_ORACLE_LIB).  A mutant that survives all pins would mean that part of the oracle is
"parity unpinned".  Nothing here touches the CUDA path."""
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SRC = os.path.join(ROOT, "oracle", "pca_oracle.cpp")

# (name, old, new, which occurrence of `old` (0-based))
MUTANTS = [
    ("gs_loads_sign", "p[n] -= pi[n] * a;", "p[n] += pi[n] * a;", 0),
    ("gs_loads_dropped", "gemv_t(P, N, k, p, coef.data());", "for (int i = 0; i < k; ++i) coef[i] = 0.0;", 0),   # :71,:1025
    ("gs_loads_k_minus_1", "for (int i = 0; i < k; ++i) {", "for (int i = 0; i < k - 1; ++i) {", 0),       # :72 (first loop = loads)
    ("gs_scores_sign", "t[m] -= vi[m] * b;", "t[m] += vi[m] * b;", 0),                                    # :79,:1031
    ("gs_scores_dropped", "gemv_t(T, M, k, t, coef.data());", "for (int i = 0; i < k; ++i) coef[i] = 0.0;", 0),  # :78,:1030
    ("gs_scores_k_minus_1", "for (int i = 0; i < k; ++i) {", "for (int i = 0; i < k - 1; ++i) {", 1),      # :79 (second loop = scores)
    ("start_vector_undeflated", "t[m] = R[id(m, k, M)];", "t[m] = X[id(m, k, M)];", 0),                  # :556,:1017 (C6)
    ("eps_scaled_by_old_lambda", "std::fabs(lam - lam_new) < eps * lam_new", "std::fabs(lam - lam_new) < eps * lam", 0),  # :566
    ("test_not_strict", "std::fabs(lam - lam_new) < eps * lam_new", "std::fabs(lam - lam_new) <= eps * lam_new", 0),       # :566
    ("gs_deflation_without_lambda", "ger(R, M, N, gs ? -lam_new : -1.0, t, p);", "ger(R, M, N, -1.0, t, p);", 0),          # :1036
    ("deflation_sign", "ger(R, M, N, gs ? -lam_new : -1.0, t, p);", "ger(R, M, N, gs ? lam_new : 1.0, t, p);", 0),          # eq. 3
    ("loads_not_normalised", "for (int64_t n = 0; n < N; ++n) p[n] /= pn;", ";", 0),                      # :563,:1027
    ("gs_scores_not_normalised", "for (int64_t m = 0; m < M; ++m) t[m] /= lam_new;", ";", 0),              # :83,:1033
    ("epilogue_dropped", "for (int64_t m = 0; m < M; ++m) T[id(m, k, M)] *= lambda[k];", ";", 0),          # :87,:1037
    ("lambda_not_updated", "lam = lam_new;                                                 // PAPER.md:567,:1035", ";", 0),
    ("centre_divides_by_N", "const double mu = s / (double)M;", "const double mu = s / (double)N;", 0),  # :21 (C1)
    ("loads_use_untransposed_panel_count", "gemv_t(P, N, k, p, coef.data());", "gemv_t(P, N, k > 1 ? 1 : k, p, coef.data());", 0),
]


def _mutate(text, old, new, occurrence):
    pos = -1
    for _ in range(occurrence + 1):
        pos = text.find(old, pos + 1)
        assert pos >= 0, f"mutation site not found: {old!r} (#{occurrence}) -- update MUTANTS after editing the oracle"
    return text[:pos] + new + text[pos + len(old):]


@pytest.mark.parametrize("name,old,new,occ", MUTANTS, ids=[m[0] for m in MUTANTS])
def test_every_mutant_is_killed_by_a_pin(tmp_path, name, old, new, occ):
    src = tmp_path / f"{name}.cpp"
    lib = tmp_path / f"lib{name}.so"
    src.write_text(_mutate(open(SRC).read(), old, new, occ))
    subprocess.run(["g++", "-O1", "-std=c++17", "-fopenmp", "-fPIC", "-shared", "-ffp-contract=off", "-o", str(lib), str(src)],
                   check=True)
    env = dict(os.environ, PCA_ORACLE_LIB=str(lib), OMP_NUM_THREADS="2")
    r = subprocess.run([sys.executable, "-m", "pytest", os.path.join(ROOT, "tests", "test_oracle_pins.py"), "-x", "-q",
                        "-p", "no:cacheprovider", "-k", "not separation_threshold"],
                       capture_output=True, text=True, cwd=ROOT, env=env, timeout=600)
    assert r.returncode == 1, f"mutant {name} SURVIVED the pins:\n{r.stdout[-1500:]}"
    assert " failed" in r.stdout, r.stdout[-1500:]


def test_unmutated_oracle_passes_the_same_selection(tmp_path):
    """Control: the same subprocess command on the real source is green (so a red mutant run means a pin fired)."""
    lib = tmp_path / "libcontrol.so"
    subprocess.run(["g++", "-O1", "-std=c++17", "-fopenmp", "-fPIC", "-shared", "-ffp-contract=off", "-o", str(lib), SRC], check=True)
    env = dict(os.environ, PCA_ORACLE_LIB=str(lib), OMP_NUM_THREADS="2")
    r = subprocess.run([sys.executable, "-m", "pytest", os.path.join(ROOT, "tests", "test_oracle_pins.py"), "-x", "-q",
                        "-p", "no:cacheprovider", "-k", "not separation_threshold"],
                       capture_output=True, text=True, cwd=ROOT, env=env, timeout=600)
    assert r.returncode == 0, r.stdout[-1500:]
