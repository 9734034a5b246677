"""Pins for the CPU oracle (run with -m "not gpu").

The oracle is checked against things OTHER than itself: LAPACK's
eigendecomposition, first-order perturbation theory, finite differences,
algebraic invariants of a projector, exact closed forms on tiny matrices
(tests/golden/closed_forms.txt) and exact rational arithmetic.  Each pin is
chosen so that a plausible slip (dropped term, wrong sign / branch, transposed
operand, wrong bound, spin factor 2) fails at least one of them.
"""
import os
from fractions import Fraction

import numpy as np
import pytest

import oracle
from paper_2107_02737_b200 import inputs

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "closed_forms.txt")


def _golden():
    out = {}
    with open(GOLDEN) as f:
        for line in f:
            line = line.split("#", 1)[0].strip()
            if not line or "=" not in line:
                continue
            k, v = (s.strip() for s in line.split("=", 1))
            out[k] = v
    return out


def _vec(s):
    return np.array([float(x) for x in s.split()])


G = _golden()


@pytest.fixture(scope="module")
def cfg1():
    return inputs.make_problem(inputs.CONFIGS[1])


@pytest.fixture(scope="module")
def cfg2():
    p = inputs.make_problem(inputs.CONFIGS[2])
    p["sp2"] = oracle.sp2_density(p["H"], p["n_occ"], H1=p["H1"])
    return p


# ----------------------------------------------------------------- bounds (a1)
def test_gershgorin_textbook_and_diagonal():
    H = _vec(G["C.H"]).reshape(3, 3)
    lo, hi = oracle.gershgorin_bounds(H)
    assert (lo, hi) == (float(G["C.eps_min"]), float(G["C.eps_max"]))
    d = np.array([-2.0, -1.0, 1.0, 2.0])
    assert oracle.gershgorin_bounds(np.diag(d)) == (-2.0, 2.0)   # exact for diagonal H


def test_gershgorin_encloses_spectrum_and_uses_offdiag_abs():
    rng = np.random.default_rng(1)
    A = rng.standard_normal((40, 40))
    H = A + A.T
    lo, hi = oracle.gershgorin_bounds(H)
    w = np.linalg.eigvalsh(H)
    assert lo <= w[0] and w[-1] <= hi
    # brute force, element loops (catches a missing abs() or an included diagonal)
    lo2 = min(H[i, i] - sum(abs(H[i, j]) for j in range(40) if j != i) for i in range(40))
    hi2 = max(H[i, i] + sum(abs(H[i, j]) for j in range(40) if j != i) for i in range(40))
    assert lo == pytest.approx(lo2, rel=1e-14) and hi == pytest.approx(hi2, rel=1e-14)


def test_rescale_reverses_spectrum_into_unit_interval(cfg1):
    H = cfg1["H"]
    lo, hi = oracle.gershgorin_bounds(H)
    X0 = oracle.rescale_to_unit_interval(H, lo, hi)
    w = np.linalg.eigvalsh(H)
    x = np.linalg.eigvalsh(X0)
    assert x[0] >= 0.0 and x[-1] <= 1.0
    # lowest H eigenvalue -> closest to 1, highest -> closest to 0
    np.testing.assert_allclose(x[::-1], (hi - w) / (hi - lo), atol=1e-13)
    with pytest.raises(ValueError):
        oracle.rescale_to_unit_interval(np.eye(3), 1.0, 1.0)


# ------------------------------------------------------- closed forms (golden)
def test_case_A_diagonal_hand_example():
    H = np.diag(_vec(G["A.diag_H"]))
    r = oracle.sp2_density(H, int(G["A.n_occ"]))
    assert (r["eps_min"], r["eps_max"]) == (float(G["A.eps_min"]), float(G["A.eps_max"]))
    np.testing.assert_allclose(np.diag(r["D"]), _vec(G["A.D_diag"]), atol=1e-13)
    assert np.abs(r["D"] - np.diag(np.diag(r["D"]))).max() == 0.0
    assert r["tr_dh"] == pytest.approx(float(G["A.tr_DH"]), abs=1e-12)
    assert r["signs"].startswith(G["A.signs_prefix"])            # tie at n=0 -> '-'
    np.testing.assert_array_equal(r["tr_x"][:3], _vec(G["A.tr_X"]))   # exact dyadics
    t2 = [r["tr_x"][k] - r["e"][k] for k in range(2)]
    np.testing.assert_array_equal(t2, _vec(G["A.tr_X2"]))


def test_case_A_against_exact_rational_arithmetic():
    """Every trace of the float64 loop equals the exact rational value while
    the dyadic numbers still fit in 53 bits (first 4 layers)."""
    H = np.diag(_vec(G["A.diag_H"]))
    r = oracle.sp2_density(H, 2)
    x = [Fraction(2 - int(v), 4) for v in _vec(G["A.diag_H"])]
    for n in range(4):
        t = sum(x)
        t2 = sum(v * v for v in x)
        assert Fraction(r["tr_x"][n]) == t
        plus = abs(t2 - 2) < abs(2 * t - t2 - 2)
        assert r["signs"][n] == ("+" if plus else "-")
        x = [v * v if plus else 2 * v - v * v for v in x]


def test_case_B_2x2_converged_on_entry_and_response():
    H = _vec(G["B.H"]).reshape(2, 2)
    H1 = _vec(G["B.H1"]).reshape(2, 2)
    r = oracle.sp2_density(H, 1, H1=H1)
    assert (r["eps_min"], r["eps_max"]) == (-1.0, 1.0)
    np.testing.assert_allclose(r["D"], _vec(G["B.D"]).reshape(2, 2), atol=1e-15)
    np.testing.assert_allclose(r["D1"], _vec(G["B.D1"]).reshape(2, 2), atol=1e-15)
    assert r["tr_dh"] == pytest.approx(float(G["B.tr_DH"]))
    assert r["layers"] == 0 and r["stop"] == "idempotent"
    # the independent routes agree with the hand value too
    D, _ = oracle.density_eigh(H, 1)
    np.testing.assert_allclose(D, _vec(G["B.D"]).reshape(2, 2), atol=1e-15)
    Q = np.array([[1.0, 1.0], [-1.0, 1.0]]) / np.sqrt(2.0)
    D1 = oracle.response_closed_form(Q, np.array([-1.0, 1.0]), 1, H1)
    np.testing.assert_allclose(D1, _vec(G["B.D1"]).reshape(2, 2), atol=1e-15)


# ---------------------------------------------- definition vs algorithm (O-1/O-2)
def test_config1_sp2_equals_eigh_projector(cfg1):
    H, n_occ = cfg1["H"], cfg1["n_occ"]
    r = oracle.sp2_density(H, n_occ)
    D_eig, w = oracle.density_eigh(H, n_occ)
    assert np.abs(r["D"] - D_eig).max() < 1e-12
    D_gen = oracle.density_from_eigenpairs(cfg1["Q"], cfg1["lam"], n_occ)
    assert np.abs(D_eig - D_gen).max() < 1e-12
    assert r["stop"] == "floor" and 13 <= r["layers"] <= 40
    # band energy: sum of the lowest eigenvalues (closed form of the generator)
    assert r["tr_dh"] == pytest.approx(inputs.band_energy_closed_form(cfg1["lam"], n_occ), rel=1e-12)
    assert r["tr_dh"] == pytest.approx(w[:n_occ].sum(), rel=1e-12)


def test_projector_invariants(cfg1):
    H, n_occ = cfg1["H"], cfg1["n_occ"]
    D = oracle.sp2_density(H, n_occ)["D"]
    assert abs(np.trace(D) - n_occ) < 1e-10                       # no spin factor (Eq. 17)
    assert np.linalg.norm(D @ D - D) < 1e-11                      # idempotent
    assert np.linalg.norm(H @ D - D @ H) < 1e-11                  # same eigenvectors as H
    assert np.abs(D - D.T).max() < 1e-13
    assert np.linalg.matrix_rank(D, tol=1e-8) == n_occ


def test_particle_hole_symmetry(cfg1):
    H, n_occ, N = cfg1["H"], cfg1["n_occ"], cfg1["n"]
    D = oracle.sp2_density(H, n_occ)["D"]
    Dm = oracle.sp2_density(-H, N - n_occ)["D"]
    assert np.abs(Dm - (np.eye(N) - D)).max() < 1e-12


def test_uneven_occupation_and_sampled_entries():
    cfg = inputs.scaled_config(inputs.CONFIGS[3], 96)             # n_occ/N = 2/3
    cfg = inputs.Sp2Config(cfg.name, 3, 96, 64, cfg.occ, cfg.unocc, "f64", False)
    p = inputs.make_problem(cfg)
    r = oracle.sp2_density(p["H"], 64)
    D_eig, _ = oracle.density_eigh(p["H"], 64)
    assert np.abs(r["D"] - D_eig).max() < 1e-12
    rows = np.array([0, 5, 95, 17])
    cols = np.array([0, 77, 95, 3])
    np.testing.assert_allclose(oracle.density_from_eigenpairs(p["Q"], p["lam"], 64, rows, cols),
                               D_eig[rows, cols], atol=1e-13)


def test_trivial_occupations(cfg1):
    H, N = cfg1["H"], cfg1["n"]
    assert np.array_equal(oracle.sp2_density(H, 0)["D"], np.zeros((N, N)))
    r = oracle.sp2_density(H, N)
    assert np.array_equal(r["D"], np.eye(N)) and r["tr_dh"] == pytest.approx(np.trace(H))
    with pytest.raises(ValueError):
        oracle.sp2_density(H, N + 1)
    with pytest.raises(ValueError):
        oracle.sp2_density(H + np.triu(np.ones((N, N)), 1), 3)    # not symmetric


def test_user_bounds_give_same_projector_fewer_layers(cfg1):
    H, n_occ = cfg1["H"], cfg1["n_occ"]
    w = np.linalg.eigvalsh(H)
    r_g = oracle.sp2_density(H, n_occ)
    r_t = oracle.sp2_density(H, n_occ, bounds=(w[0], w[-1]))
    assert np.abs(r_g["D"] - r_t["D"]).max() < 1e-12
    assert r_t["layers"] < r_g["layers"]


def test_tol_stop_rule(cfg1):
    H, n_occ = cfg1["H"], cfg1["n_occ"]
    r = oracle.sp2_density(H, n_occ, tol=1e-3)
    assert r["stop"] == "tol" and 0.0 <= r["e"][-1] <= 1e-3
    full = oracle.sp2_density(H, n_occ)
    assert r["layers"] < full["layers"]
    assert np.abs(r["D"] - full["D"]).max() < 1e-2
    r3 = oracle.sp2_density(H, n_occ, max_layers=5)
    assert r3["stop"] == "max_layers" and r3["layers"] == 5


# ----------------------------------------------------- spectrum-only simulator
def test_spectrum_simulator_matches_matrix_loop(cfg1):
    H, n_occ = cfg1["H"], cfg1["n_occ"]
    r = oracle.sp2_density(H, n_occ)
    w = np.linalg.eigvalsh(H)
    s = oracle.sp2_spectrum_simulator(w, n_occ, r["eps_min"], r["eps_max"])
    k = min(len(s["signs"]), len(r["signs"])) - 3                 # last layers are noise-driven
    assert s["signs"][:k] == r["signs"][:k]
    np.testing.assert_allclose(s["tr_x"][:k], r["tr_x"][:k], rtol=0, atol=1e-9)
    assert abs(s["layers"] - r["layers"]) <= 3
    occ = np.sort(s["x"])[::-1]
    np.testing.assert_allclose(occ[:n_occ], 1.0, atol=1e-12)
    np.testing.assert_allclose(occ[n_occ:], 0.0, atol=1e-12)


def test_diagonal_matrix_is_the_scalar_map():
    lam = np.array([-1.3, -0.2, 0.05, 0.4, 0.9, 1.7])
    r = oracle.sp2_density(np.diag(lam), 3)
    s = oracle.sp2_spectrum_simulator(lam, 3, r["eps_min"], r["eps_max"])
    assert s["signs"] == r["signs"] and s["layers"] == r["layers"]
    np.testing.assert_allclose(np.diag(r["D"]), s["x"], atol=0)
    np.testing.assert_allclose(np.diag(r["D"]), [1, 1, 1, 0, 0, 0], atol=1e-12)


def test_layer_count_estimates_for_big_configs():
    """Configs 4/5 at full size via the O(N L) simulator with Gershgorin-like
    bounds ~ +-sqrt(2/pi) sqrt(N <lam^2>): BASELINE.json expects ~35-45 layers."""
    for k in (4, 5):
        cfg = inputs.CONFIGS[k]
        rng = np.random.default_rng(0)
        lam = np.concatenate([rng.uniform(*cfg.occ, cfg.n_occ), rng.uniform(*cfg.unocc, cfg.n - cfg.n_occ)])
        half = np.sqrt(2 / np.pi) * np.sqrt(cfg.n * np.mean(lam ** 2))
        s = oracle.sp2_spectrum_simulator(lam, cfg.n_occ, -half, half)
        assert 30 <= s["layers"] <= 50 and s["stop"] == "floor"


# ------------------------------------------------------------- response (O-3)
def test_response_recursion_vs_perturbation_theory_vs_finite_difference(cfg2):
    H, H1, n_occ = cfg2["H"], cfg2["H1"], cfg2["n_occ"]
    r = cfg2["sp2"]
    D_eig, w = oracle.density_eigh(H, n_occ)
    assert np.abs(r["D"] - D_eig).max() < 1e-12
    D1_pt = oracle.response_closed_form(cfg2["Q"], cfg2["lam"], n_occ, H1)
    scale = np.abs(D1_pt).max()
    assert np.abs(r["D1"] - D1_pt).max() < 1e-10 * scale
    D1_fd = oracle.response_finite_difference(H, H1, n_occ, eps=1e-5)
    assert np.abs(D1_fd - D1_pt).max() < 1e-6 * scale
    assert r["tr_dh"] == pytest.approx(w[:n_occ].sum(), rel=1e-12)


def test_response_invariants(cfg2):
    D, D1 = cfg2["sp2"]["D"], cfg2["sp2"]["D1"]
    s = np.abs(D1).max()
    assert abs(np.trace(D1)) < 1e-10 * s * len(D)                # particle number conserved
    assert np.abs(D1 - D1.T).max() < 1e-13 * s
    assert np.abs(D @ D1 + D1 @ D - D1).max() < 1e-10 * s        # derivative of D^2 = D
    assert np.abs(D @ D1 @ D).max() < 1e-10 * s                  # no occ-occ block


def test_response_is_linear_and_sign_sensitive(cfg2):
    """A transposed/dropped term in X Z + Z X or a wrong branch sign breaks this
    on a small non-commuting case (H1 does not commute with H)."""
    cfg = inputs.Sp2Config("t", 2, 48, 20, (-1.5, -0.25), (0.25, 1.5), "f64", True)
    p = inputs.make_problem(cfg)
    r = oracle.sp2_density(p["H"], 20, H1=p["H1"])
    D1_pt = oracle.response_closed_form(p["Q"], p["lam"], 20, p["H1"])
    assert np.abs(r["D1"] - D1_pt).max() < 1e-11 * np.abs(D1_pt).max()
    r2 = oracle.sp2_density(p["H"], 20, H1=-3.0 * p["H1"])
    np.testing.assert_allclose(r2["D1"], -3.0 * r["D1"], atol=1e-12)
    assert np.abs(p["H"] @ p["H1"] - p["H1"] @ p["H"]).max() > 1e-3


def test_sampled_response_entries_match_the_full_closed_form():
    cfg = inputs.Sp2Config("t", 2, 60, 22, (-1.5, -0.25), (0.25, 1.5), "f64", True)
    p = inputs.make_problem(cfg)
    full = oracle.response_closed_form(p["Q"], p["lam"], 22, p["H1"])
    rows = np.array([0, 3, 59, 17, 40, 40])
    cols = np.array([0, 51, 59, 3, 7, 40])
    got = oracle.response_closed_form_sampled(p["Q"], p["lam"], 22, p["H1"], rows, cols)
    np.testing.assert_allclose(got, full[rows, cols], rtol=0, atol=1e-13 * np.abs(full).max())
    # and against the finite difference of the definition (independent of both closed forms)
    fd = oracle.response_finite_difference(p["H"], p["H1"], 22, eps=1e-5)
    np.testing.assert_allclose(got, fd[rows, cols], rtol=0, atol=1e-6 * np.abs(full).max())


def test_structured_chain_tight_bounds_paper_like_layer_count():
    """Sparse tight-binding chain with TIGHT Gershgorin bounds: closed-form spectrum, and the layer
    count drops to the paper's range ("between 14 and 16 deep layers") instead of the
    35-45 of the dense random-Q configs."""
    n = 512
    H, lam = inputs.ssh_chain(n, 1.0, 0.6)
    w = np.linalg.eigvalsh(H)
    np.testing.assert_allclose(w, lam, atol=1e-12)                  # generator's closed form
    lo, hi = oracle.gershgorin_bounds(H)
    assert (lo, hi) == (-1.6, 1.6) and abs(w[0] - lo) < 1e-12       # tight
    r = oracle.sp2_density(H, n // 2)
    D_eig, _ = oracle.density_eigh(H, n // 2)
    assert np.abs(r["D"] - D_eig).max() < 1e-12
    assert 10 <= r["layers"] <= 18
    assert r["tr_dh"] == pytest.approx(lam[: n // 2].sum(), rel=1e-12)


def test_refinement_layers_purify_eigenvalues_and_keep_eigenvectors(cfg1):
    """PAPER.md:170 refinement: two more layers act on the eigenvalues only.  Start from the exact projector with
    its eigenvalues perturbed by +-1e-4: the scalar maps x^2 / 2x - x^2 predict every refined eigenvalue, the
    eigenvectors do not move, the exact projector is a fixed point, and two layers square the error twice."""
    Q, lam, n_occ, n = cfg1["Q"], cfg1["lam"], cfg1["n_occ"], cfg1["n"]
    rng = np.random.default_rng(11)
    occ = (np.argsort(np.argsort(lam)) < n_occ).astype(float)
    x0 = occ + 1e-4 * rng.uniform(-1, 1, n)
    X0 = (Q * x0) @ Q.T
    X0 = 0.5 * (X0 + X0.T)
    Xr, signs = oracle.sp2_refine_layers(X0, n_occ, layers=2)
    x = x0.copy()
    for sg in signs:                                   # the same branches on the scalar spectrum
        x = x * x if sg == "+" else 2 * x - x * x
    np.testing.assert_allclose(np.sort(np.linalg.eigvalsh(Xr)), np.sort(x), atol=1e-13)
    assert signs in ("+-", "-+")                       # near idempotency the branches alternate
    assert np.abs(x - occ).max() < 5e-8 and np.abs(x - occ).max() > 1e-10       # ~ (2 * 1e-4)^2
    P = (Q * occ) @ Q.T
    assert np.abs(Xr - P).max() < 1e-7 and np.linalg.norm(Xr @ P - P @ Xr) < 1e-12   # same eigenvectors
    Pr, _ = oracle.sp2_refine_layers(P, n_occ, layers=2)
    assert np.abs(Pr - P).max() < 1e-13                # the projector is a fixed point


def test_congruence_against_the_generalised_eigenproblem():
    """with Z^T S Z = I, the orthogonalised problem has the spectrum of the generalised problem
    H c = eps S c, and D = Z D_orth Z^T is the S-metric projector: D S D = D, tr(D S) = N_occ (scipy's generalised
    eigensolver is the independent reference)."""
    import scipy.linalg

    q = inputs.overlap_problem(60, 25)
    H, S, Z, n_occ = q["H"], q["S"], q["Z"], q["n_occ"]
    np.testing.assert_allclose(oracle.congruence(Z, S), np.eye(60), atol=1e-12)         # Z^T S Z = I
    Horth = oracle.congruence(Z, H)
    eps, Cg = scipy.linalg.eigh(H, S)
    np.testing.assert_allclose(np.linalg.eigvalsh(Horth), eps, atol=1e-11)
    np.testing.assert_allclose(np.sort(eps), np.sort(q["lam"]), atol=1e-11)             # the generator's spectrum
    Dorth, _ = oracle.density_eigh(Horth, n_occ)
    D = oracle.congruence(Z, Dorth, transpose_first=False)
    np.testing.assert_allclose(D, Cg[:, :n_occ] @ Cg[:, :n_occ].T, atol=1e-11)          # S-normalised eigenvectors
    assert np.abs(D @ S @ D - D).max() < 1e-11 and abs(np.trace(D @ S) - n_occ) < 1e-11
    # a non-symmetric Z tells Z^T X Z from Z X Z^T
    rng = np.random.default_rng(2)
    Zg = rng.standard_normal((5, 5)); X = rng.standard_normal((5, 5)); X = X + X.T
    a = oracle.congruence(Zg, X, True); b = oracle.congruence(Zg, X, False)
    assert a[1, 2] == pytest.approx(sum(Zg[k, 1] * X[k, l] * Zg[l, 2] for k in range(5) for l in range(5)))
    assert b[1, 2] == pytest.approx(sum(Zg[1, k] * X[k, l] * Zg[2, l] for k in range(5) for l in range(5)))


def test_lanczos_bounds_enclose_the_spectrum_and_are_tighter(cfg1):
    """The Lanczos interval must contain every eigenvalue (LAPACK is the reference) on dense, sparse and diagonal
    matrices, never be wider than Gershgorin, be far tighter for the dense random-Q configs, and give the SAME
    projector in fewer layers."""
    mats = [cfg1["H"], inputs.ssh_chain(200, 1.0, 0.6, onsite=0.3)[0], np.diag(np.linspace(-3.0, 5.0, 50)),
            inputs.make_problem(inputs.scaled_config(inputs.CONFIGS[3], 150))["H"].astype(np.float64)]
    for H in mats:
        w = np.linalg.eigvalsh(H)
        g_lo, g_hi = oracle.gershgorin_bounds(H)
        for k in (4, 12, 24):
            lo, hi = oracle.lanczos_bounds(H, k)
            assert lo <= w[0] + 1e-12 and hi >= w[-1] - 1e-12
            assert lo >= g_lo - 1e-12 and hi <= g_hi + 1e-12
    H, n_occ = cfg1["H"], cfg1["n_occ"]
    lo, hi = oracle.lanczos_bounds(H, 12)
    g_lo, g_hi = oracle.gershgorin_bounds(H)
    assert (hi - lo) < 0.35 * (g_hi - g_lo)
    r_g = oracle.sp2_density(H, n_occ)
    r_l = oracle.sp2_density(H, n_occ, bounds=(lo, hi))
    assert np.abs(r_g["D"] - r_l["D"]).max() < 1e-12 and r_l["layers"] <= r_g["layers"] - 3


def test_power_trace_bounds_are_a_rigorous_enclosure(cfg1):
    """power_trace_bounds: [mu - r, mu + r] with r = (tr A^(2^(s+1)))^(1/2^(s+1)) must (i) enclose the LAPACK spectrum
    on EVERY matrix, including the ones built against the Lanczos start vector, (ii) be sandwiched between the true
    radius rho and N^(1/2^(s+1)) rho, (iii) tighten monotonically with s, (iv) reproduce the closed form on a diagonal
    matrix, (v) never leave the Gershgorin interval, and (vi) give the same projector in fewer layers."""
    n = 300
    v0 = np.cos(0.7 * np.arange(n) + 0.3)
    mats = [cfg1["H"], inputs.ssh_chain(200, 1.0, 0.6, onsite=0.3)[0], np.diag(np.linspace(-3.0, 5.0, 50)),
            inputs.make_problem(inputs.scaled_config(inputs.CONFIGS[3], 150))["H"].astype(np.float64),
            inputs.hidden_eigenvector_problem(n, 40, -3.0, v0)[0], inputs.hidden_eigenvector_problem(n, 150, 3.0, v0)[0],
            np.array([[2.0]]), 1e6 * cfg1["H"], 1e-6 * cfg1["H"] + 7.0 * np.eye(cfg1["H"].shape[0])]
    for H in mats:
        w = np.linalg.eigvalsh(H)
        N = H.shape[0]
        mu = np.trace(H) / N
        rho = np.abs(w - mu).max()
        g_lo, g_hi = oracle.gershgorin_bounds(H)
        prev = None
        for s in (0, 1, 2, 3, 4, 6):
            lo, hi = oracle.power_trace_bounds(H, s)
            tol = 1e-12 * max(1.0, np.abs(w).max())
            assert lo <= w[0] + tol and hi >= w[-1] - tol, (N, s)                     # (i) enclosure, always
            assert lo >= g_lo - tol and hi <= g_hi + tol                              # (v)
            r_raw = rho * (np.sum((np.abs(w - mu) / rho) ** (2 ** (s + 1)))) ** (1.0 / 2 ** (s + 1)) if rho > 0 else 0.0   # the definition, from the eigenvalues
            assert rho * (1 - 1e-12) <= r_raw <= N ** (1.0 / 2 ** (s + 1)) * rho * (1 + 1e-12)   # (ii)
            if mu - r_raw >= g_lo and mu + r_raw <= g_hi:                              # not clipped by the discs: the formula itself
                assert lo == pytest.approx(mu - r_raw, rel=1e-9, abs=1e-9 * rho) and hi == pytest.approx(mu + r_raw, rel=1e-9, abs=1e-9 * rho)
            if prev is not None:
                assert hi - lo <= prev * (1 + 1e-12)                                   # (iii)
            prev = hi - lo
    d = np.array([-2.0, 0.5, 1.5, 4.0])                                               # (iv) mu = 1, a = (-3, -.5, .5, 3)
    lo, hi = oracle.power_trace_bounds(np.diag(d), 1)
    r = (2 * 3.0 ** 4 + 2 * 0.5 ** 4) ** 0.25
    assert (lo, hi) == (pytest.approx(max(-2.0, 1 - r)), pytest.approx(min(4.0, 1 + r)))
    H, n_occ = cfg1["H"], cfg1["n_occ"]                                               # (vi)
    lo, hi = oracle.power_trace_bounds(H, 4)
    g_lo, g_hi = oracle.gershgorin_bounds(H)
    assert (hi - lo) < 0.35 * (g_hi - g_lo)
    r_g = oracle.sp2_density(H, n_occ)
    r_p = oracle.sp2_density(H, n_occ, bounds=(lo, hi))
    assert np.abs(r_g["D"] - r_p["D"]).max() < 1e-12 and r_p["layers"] <= r_g["layers"] - 3
    # where Lanczos misses the hidden outlier and ruins the solve, this bound does not
    Hh, _ = inputs.hidden_eigenvector_problem(n, 40, -3.0, v0)
    D_eig, _ = oracle.density_eigh(Hh, 40)
    r_h = oracle.sp2_density(Hh, 40, bounds=oracle.power_trace_bounds(Hh, 4))
    assert np.abs(r_h["D"] - D_eig).max() < 1e-11


def test_converged_flag_is_bookkeeping_only(cfg1):
    """`converged` = a stop rule other than the cap fired AND the occupation is the requested one."""
    r = oracle.sp2_density(cfg1["H"], cfg1["n_occ"])
    assert r["converged"] and r["stop"] in ("floor", "idempotent") and abs(r["tr_d"] - cfg1["n_occ"]) < 1e-9
    r5 = oracle.sp2_density(cfg1["H"], cfg1["n_occ"], max_layers=5)
    assert not r5["converged"] and r5["stop"] == "max_layers"
    # a degenerate level at the Fermi energy that N_occ splits: fractional occupation, never a converged projector
    lam = np.array([-1.0, -0.5, 0.0, 0.0, 0.7, 1.2])
    rng = np.random.default_rng(3)
    Q, _ = np.linalg.qr(rng.standard_normal((6, 6)))
    H = (Q * lam) @ Q.T
    rd = oracle.sp2_density(0.5 * (H + H.T), 3)
    assert not rd["converged"]


def test_lanczos_bounds_are_a_heuristic_not_an_enclosure():
    """The other side of the pin above: the Lanczos interval is NOT rigorous.  With an extreme eigenvector exactly
    orthogonal to the start vector v_i = cos(0.7 i + 0.3), the Krylov space never contains it, the interval misses the
    outlier eigenvalue by more than the whole remaining spectrum, and the SP2 loop run with those bounds maps that
    eigenvalue outside [0, 1] and returns garbage -- which is why the GPU path guards every solve
    (SP2_ERR_BOUNDS) and falls back to the Gershgorin discs (tests/test_gpu_lanczos.py)."""
    n = 300
    v0 = np.cos(0.7 * np.arange(n) + 0.3)
    for n_occ, hidden in ((40, -3.0), (150, 3.0)):
        H, lam = inputs.hidden_eigenvector_problem(n, n_occ, hidden, v0)
        w = np.linalg.eigvalsh(H)
        assert w[0 if hidden < 0 else -1] == pytest.approx(hidden, abs=1e-12)
        lo, hi = oracle.lanczos_bounds(H, 12)
        if hidden < 0:
            assert lo > w[0] + 1.0 and hi >= w[-1]                    # misses the lowest eigenvalue by > 1
        else:
            assert hi < w[-1] - 1.0 and lo <= w[0]                    # misses the highest eigenvalue by > 1
        g_lo, g_hi = oracle.gershgorin_bounds(H)
        assert g_lo <= w[0] and g_hi >= w[-1]                         # the discs are rigorous
        D_eig, _ = oracle.density_eigh(H, n_occ)
        bad = oracle.sp2_density(H, n_occ, bounds=(lo, hi), max_layers=60)
        assert min(bad["e"]) < -1.0                                   # tr X - tr X^2 < 0: an eigenvalue left [0, 1]
        assert not np.abs(bad["D"] - D_eig).max() < 1.0
        good = oracle.sp2_density(H, n_occ)
        assert np.abs(good["D"] - D_eig).max() < 1e-11


def test_batched_response_vs_perturbation_theory_and_linearity():
    """NEXT-4: every D1_b of the one-stack loop equals first-order perturbation theory for its own H1_b (an
    index mix-up between the Z_b, a dropped factor or a shared update fails this), and the map H1 -> D1 is linear."""
    cfg = inputs.Sp2Config("t", 2, 56, 21, (-1.5, -0.25), (0.25, 1.5), "f64", False)
    p = inputs.make_problem(cfg)
    H1s = inputs.perturbations(56, 3, seed=5)
    r = oracle.sp2_response_batch(p["H"], 21, H1s)
    D_eig, w = oracle.density_eigh(p["H"], 21)
    assert np.abs(r["D"] - D_eig).max() < 1e-12
    assert r["tr_dh"] == pytest.approx(w[:21].sum(), rel=1e-12)
    for b, H1 in enumerate(H1s):
        pt = oracle.response_closed_form(p["Q"], p["lam"], 21, H1)
        assert np.abs(r["D1"][b] - pt).max() < 1e-11 * np.abs(pt).max()
        assert abs(r["tr_d1"][b]) < 1e-10 * np.abs(pt).max() * 56
    mix = 2.0 * H1s[0] - 30.0 * H1s[1] + 500.0 * H1s[2]
    rm = oracle.sp2_response_batch(p["H"], 21, [mix])
    want = 2.0 * r["D1"][0] - 30.0 * r["D1"][1] + 500.0 * r["D1"][2]
    np.testing.assert_allclose(rm["D1"][0], want, rtol=0, atol=1e-11 * np.abs(want).max())
    # trivial occupations and the empty batch
    assert oracle.sp2_response_batch(p["H"], 0, H1s)["D1"][2].max() == 0.0
    r0 = oracle.sp2_response_batch(p["H"], 21, [])
    assert r0["D1"] == [] and r0["signs"] == r["signs"]
