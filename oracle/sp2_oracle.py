"""Plain, slow, float64 CPU oracle of the DNN-SP2 density-matrix solver.

TEST INFRASTRUCTURE ONLY (see ``oracle/__init__.py``).  NumPy float64, full
products with ``@``; no symmetry exploitation, no operand splitting, no shifted
iterate, no blocking, no fusion -- so that every line can be checked against
the paper by eye.  Citations are ``PAPER.md:<line>`` (= /root/reference/PAPER.md
at build time; the file is not needed at run time).

What the method computes (Eq. 17-18): the density matrix
``D = theta(mu*I - H)``, i.e. the orthogonal projector onto the ``n_occ``
lowest eigenvectors of the symmetric (orthogonalised) Hamiltonian ``H``.
SP2 (Eq. 19, Fig. 1) is an iteration that converges to that
projector, so the oracle has two independent parts that must agree:

* the definition written out  -> ``density_eigh`` / ``density_from_eigenpairs``
* the algorithm step by step  -> ``sp2_density``

plus, for the first-order response ``D1`` that rides the same layers
(BASELINE.json north_star; the recursion itself is not printed in the paper,
PAPER.md:231 only names the Krylov kernel that consumes it):

* first-order perturbation theory  -> ``response_closed_form``
* central finite difference        -> ``response_finite_difference``

and, for the rows SURVEY 8(f) marks "next":

* float64 refinement layers          -> ``sp2_refine_layers``
* congruence transforms of PAPER.md:137             -> ``congruence``
* Lanczos spectral bounds (tighter than Gershgorin) -> ``lanczos_bounds``
* rigorous bounds from the trace of a matrix power  -> ``power_trace_bounds``
* several perturbations on one stack of layers      -> ``sp2_response_batch``

Pin status: every function here is pinned by ``tests/test_oracle_pins.py``
(eigendecomposition, closed forms, invariants, textbook special cases,
brute force on tiny inputs, the generalised eigenproblem for the congruence,
LAPACK spectra for the Lanczos enclosure, scalar eigenvalue maps for the
refinement, perturbation theory and linearity for the batched response).
Nothing is "parity unpinned".

Readings where the paper is silent (full list with reasons in DESIGN.md):
  R1  spectral bounds  = Gershgorin discs                     (PAPER.md:145 silent)
  R2  W0 = -I/Delta, B0 = eps_max*I/Delta
  R3  sign rule: take the branch whose trace is closer to n_occ, ties -> '-'
  R4  stop rule: see ``sp2_stop``
  R5  response recursion: product rule on every layer, zeroth-order signs,
      Z0 = -H1/Delta with the bounds of H held fixed
  R6  tr(DH) = sum_ij D_ij H_ij with the caller's unscaled H
  R7  no spin factor: eigenvalues of D are 0/1, tr D = n_occ   (Eq. 17)
"""
from __future__ import annotations

import numpy as np

__all__ = [
    "gershgorin_bounds",
    "lanczos_bounds",
    "power_trace_bounds",
    "rescale_to_unit_interval",
    "sp2_stop",
    "sp2_density",
    "sp2_response_batch",
    "sp2_refine_layers",
    "congruence",
    "density_eigh",
    "density_from_eigenpairs",
    "response_closed_form",
    "response_closed_form_sampled",
    "response_finite_difference",
    "sp2_spectrum_simulator",
]


def _as_f64_symmetric(H, name="H"):
    H = np.asarray(H, dtype=np.float64)
    if H.ndim != 2 or H.shape[0] != H.shape[1]:
        raise ValueError(f"{name} must be a square matrix")
    if not np.all(np.isfinite(H)):
        raise ValueError(f"{name} has non-finite entries")
    scale = np.abs(H).max() if H.size else 0.0
    if H.size and np.abs(H - H.T).max() > 1e-12 * max(scale, 1e-300):
        raise ValueError(f"{name} is not symmetric")
    return H


def gershgorin_bounds(H):
    """Enclosing interval of the spectrum of symmetric ``H`` from Gershgorin discs.

    r_i = sum_{j != i} |H_ij|;  eps_min = min_i(H_ii - r_i);  eps_max = max_i(H_ii + r_i).

    PAPER.md:145 only says that W0, B0 "linearly transform the eigenvalue
    spectrum of H to the interval [0, 1]"; how the spectral bounds are obtained
    is not stated.  Reading R1 (BASELINE.json north_star): Gershgorin row sums.
    """
    H = np.asarray(H, dtype=np.float64)
    d = np.diag(H)
    r = np.abs(H).sum(axis=1) - np.abs(d)
    return float((d - r).min()), float((d + r).max())


def lanczos_bounds(H, steps=12):
    """Tighter spectral bounds than Gershgorin (the paper leaves accelerated variants that need
    spectral estimates aside): ``steps`` iterations of the Lanczos process on H from the fixed start
    vector v_i = cos(0.7 i + 0.3); with T_k the tridiagonal matrix of the alphas and betas and beta_k the norm of
    the last residual, returns (theta_min - beta_k, theta_max + beta_k) intersected with the Gershgorin interval.
    The extreme Ritz values lie inside the spectrum; widening by the residual norm is the usual "safe" bound, but it
    is a HEURISTIC, not an enclosure: an extreme eigenvector orthogonal to the start vector is never seen
    (pinned both ways: enclosure on ordinary matrices, a miss by > 1 on the adversarial one)."""
    H = np.asarray(H, dtype=np.float64)
    n = H.shape[0]
    k = max(1, min(steps, n - 1))
    v = np.cos(0.7 * np.arange(n) + 0.3)
    v /= np.linalg.norm(v)
    v_prev = np.zeros(n)
    alpha, beta = [], [0.0]
    for j in range(k):
        w = H @ v
        a = float(w @ v)
        w = w - a * v - beta[j] * v_prev
        b = float(np.linalg.norm(w))
        alpha.append(a)
        beta.append(b)
        v_prev, v = v, (w / b if b > 0.0 else w)
    T = np.diag(alpha) + np.diag(beta[1:k], 1) + np.diag(beta[1:k], -1)
    theta = np.linalg.eigvalsh(T)
    g_lo, g_hi = gershgorin_bounds(H)
    return max(g_lo, float(theta[0] - beta[k])), min(g_hi, float(theta[-1] + beta[k]))


def power_trace_bounds(H, squarings=4):
    """RIGOROUS spectral bounds tighter than Gershgorin ("a few Lanczos or power iterations
    instead of Gershgorin"), from the trace of a matrix power.  With mu = tr H / N and A = H - mu I (symmetric,
    eigenvalues a_i = lambda_i - mu), every even power has a trace of non-negative terms, so for p = 2^(s+1)

        max_i |a_i|^p  <=  sum_i a_i^p  =  tr A^p  =  || A^(2^s) ||_F^2        (A^(2^s) symmetric)

    and therefore  |lambda_i - mu| <= r := ||A^(2^s)||_F^(1 / 2^s)  for EVERY eigenvalue: [mu - r, mu + r] encloses the
    spectrum whatever the eigenvectors are (no start vector, unlike ``lanczos_bounds``), and r <= N^(1/2^(s+1)) rho(A)
    overshoots the true radius by at most that factor (8192^(1/32) = 1.33 for s = 4).  A^(2^s) takes s = ``squarings``
    matrix squarings.  The iterate is renormalised by its Frobenius norm after every squaring (a scalar, tracked in
    log form) so that no power over- or underflows.  Returns the interval intersected with the Gershgorin discs.
    """
    H = np.asarray(H, dtype=np.float64)
    n = H.shape[0]
    mu = float(np.trace(H)) / n
    B = H - mu * np.eye(n)
    log_scale = 0.0                                  # A^(2^k) = exp(log_scale) * B
    for _ in range(squarings):
        nrm = float(np.linalg.norm(B))
        if nrm == 0.0:
            break
        B = B / nrm
        log_scale += np.log(nrm)
        B = B @ B
        log_scale *= 2.0
    nrm = float(np.linalg.norm(B))                   # ||A^(2^s)||_F = exp(log_scale) * nrm
    r = 0.0 if nrm == 0.0 else float(np.exp((log_scale + np.log(nrm)) / 2.0 ** squarings))
    g_lo, g_hi = gershgorin_bounds(H)
    return max(g_lo, mu - r), min(g_hi, mu + r)


def rescale_to_unit_interval(H, eps_min, eps_max):
    """Input layer X0 = W0*H + B0 with W0 = -I/Delta, B0 = eps_max*I/Delta.

    PAPER.md:145: "The initial weight and bias values, W0 and B0, are chosen to
    linearly transform the eigenvalue spectrum of H to the interval [0, 1] in
    reverse order, i.e. with the lowest lying eigenvalues closer to 1 and the
    highest closer to 0."  The only affine map sending eps_max -> 0 and
    eps_min -> 1 is X0 = (eps_max*I - H)/(eps_max - eps_min)   (reading R2).
    """
    H = np.asarray(H, dtype=np.float64)
    delta = eps_max - eps_min
    if not delta > 0.0:
        raise ValueError("degenerate spectral bounds (eps_max == eps_min)")
    return (eps_max * np.eye(H.shape[0]) - H) / delta


def sp2_stop(n, e_hist, sign_hist, tr_x, n_occ, tol, max_layers):
    """Stop test evaluated at the top of layer ``n`` (before its sign is chosen).

    ``e_hist[k] = tr X_k - tr X_k^2`` for k = 0..n is the idempotency estimate
    "from traces of intermediate matrices"; ``sign_hist[k]`` for
    k = 0..n-1 are the branches already applied.  PAPER.md:151 only says the
    layers are "repeated until all eigenvalues of the output matrix are
    sufficiently close to 1 or 0".  Reading R4, returns a reason string or None:

    (i)    tol > 0:  0 <= e_n <= tol  and |tr X_n - n_occ| < 0.5
    (ii)   parameter-free: n >= 3, the last two branches alternated
           (sigma_{n-1} != sigma_{n-2}), e_{n-2} < 1, and
           (e_n <= 0  or  e_n > 4.5 * e_{n-2}^2).
           In exact arithmetic an alternating +/- pair maps an eigenvalue error
           d to <= 4 d^2, so e_n <= 4 e_{n-2}^2 until rounding noise dominates;
           4.5 is slack.  This is "until |tr X - n_occ| and the idempotency
           error stop decreasing" (BASELINE.json config 1).
    (ii-b) e_n <= 0 with |tr X_n - n_occ| < 0.5 at any n (X_0 already idempotent)
    (iii)  n == max_layers  -> "max_layers" (not converged)
    """
    e_n = e_hist[n]
    near = abs(tr_x - n_occ) < 0.5
    if tol > 0.0 and 0.0 <= e_n <= tol and near:
        return "tol"
    if n >= 3 and sign_hist[n - 1] != sign_hist[n - 2] and e_hist[n - 2] < 1.0:
        if e_n <= 0.0 or e_n > 4.5 * e_hist[n - 2] ** 2:
            return "floor"
    if e_n <= 0.0 and near:
        return "idempotent"
    if n >= max_layers:
        return "max_layers"
    return None


def sp2_density(H, n_occ, H1=None, tol=0.0, max_layers=100, bounds=None):
    """The DNN-SP2 recursion, one plain loop (Eq. 19, Fig. 1).

    Each layer applies the activation f(X) = X^2 and then
    S_n = W_n X_n + B_n with W_n = +-I, B_n = (1 - W_n) S_{n-1}, i.e.
    "either S_n = S_{n-1}^2 or S_n = 2 S_{n-1} - S_{n-1}^2" (Fig. 1 caption,
    PAPER.md:149; the superscript "-2" there is an extraction artefact of "2").
    The signs are "selected such that the density matrix converges to the
    correct occupation"; reading R3: pick the branch whose trace
    is closer to n_occ, '+' (X^2) iff |tr X^2 - n_occ| < |2 tr X - tr X^2 - n_occ|,
    ties to '-' (2X - X^2).

    With ``H1`` given, the first-order response rides the same layers
    (reading R5): Z0 = -H1/Delta and, by the product rule with the SAME sign,
        '+':  Z <- X Z + Z X            '-':  Z <- 2 Z - (X Z + Z X).

    Returns a dict with D, D1 (or None), layers, signs (str of '+'/'-'),
    tr_x[n], e[n] (per evaluated layer), stop (reason), converged, eps_min, eps_max,
    tr_d, tr_dh (= sum_ij D_ij H_ij, reading R6), tr_d1.
    """
    H = _as_f64_symmetric(H, "H")
    N = H.shape[0]
    if not 0 <= n_occ <= N:
        raise ValueError("n_occ out of range")
    Z = None
    if H1 is not None:
        H1 = _as_f64_symmetric(H1, "H1")
        if H1.shape != H.shape:
            raise ValueError("H1 shape mismatch")

    eps_min, eps_max = gershgorin_bounds(H) if bounds is None else map(float, bounds)

    # Trivial occupations answered from the definition: projector onto no / all states.
    if n_occ == 0 or n_occ == N:
        D = np.zeros((N, N)) if n_occ == 0 else np.eye(N)
        D1 = None if H1 is None else np.zeros((N, N))
        return dict(D=D, D1=D1, layers=0, signs="", tr_x=[], e=[], stop="trivial",
                    eps_min=eps_min, eps_max=eps_max, tr_d=float(n_occ),
                    tr_dh=float(np.sum(D * H)), tr_d1=0.0 if H1 is not None else None)

    delta = eps_max - eps_min
    X = rescale_to_unit_interval(H, eps_min, eps_max)
    if H1 is not None:
        Z = -H1 / delta                                          # derivative of the line above (R5)

    tr_hist, e_hist, signs = [], [], []
    n = 0
    while True:
        X2 = X @ X                                               # f(X) = X^2
        t = float(np.trace(X))
        t2 = float(np.trace(X2))
        tr_hist.append(t)
        e_hist.append(t - t2)
        stop = sp2_stop(n, e_hist, signs, t, n_occ, tol, max_layers)
        if stop is not None:
            break
        plus = abs(t2 - n_occ) < abs(2.0 * t - t2 - n_occ)       # R3, ties -> '-'
        if Z is not None:
            W = X @ Z + Z @ X
        if plus:                                                 # S_n = S_{n-1}^2
            X = X2
            if Z is not None:
                Z = W
        else:                                                    # S_n = 2 S_{n-1} - S_{n-1}^2
            X = 2.0 * X - X2
            if Z is not None:
                Z = 2.0 * Z - W
        signs.append("+" if plus else "-")
        n += 1

    # converged: stopped by a rule other than the layer cap AND at the requested occupation (the floor rule can fire
    # at a fractional occupation when a degenerate level sits at the Fermi energy); bookkeeping only, no arithmetic
    converged = stop != "max_layers" and abs(float(np.trace(X)) - n_occ) < 0.5
    return dict(D=X, D1=Z, layers=n, signs="".join(signs), tr_x=tr_hist, e=e_hist, stop=stop, converged=converged,
                eps_min=eps_min, eps_max=eps_max, tr_d=float(np.trace(X)),
                tr_dh=float(np.sum(X * H)),
                tr_d1=None if Z is None else float(np.trace(Z)))


def sp2_response_batch(H, n_occ, H1s, tol=0.0, max_layers=100, bounds=None):
    """Several perturbations H1_b of the same H carried through ONE stack of layers (the
    "preconditioned Krylov subspace approximation" of the kernel, asks for the response of the same
    Hamiltonian to several perturbations per MD step).  Same loop as ``sp2_density``; reading R5 applied to every
    Z_b = dX/d(lambda_b) with the zeroth-order signs:
        Z_b0 = -H1_b/Delta;    '+':  Z_b <- X Z_b + Z_b X;    '-':  Z_b <- 2 Z_b - (X Z_b + Z_b X).
    The first-order terms do not couple, so D1_b is the response ``sp2_density(H, n_occ, H1=H1_b)`` would return.

    Returns a dict with D, D1 (list), layers, signs, stop, eps_min, eps_max, tr_d, tr_dh, tr_d1 (list).
    """
    H = _as_f64_symmetric(H, "H")
    N = H.shape[0]
    if not 0 <= n_occ <= N:
        raise ValueError("n_occ out of range")
    H1s = [_as_f64_symmetric(H1, "H1") for H1 in H1s]
    for H1 in H1s:
        if H1.shape != H.shape:
            raise ValueError("H1 shape mismatch")
    eps_min, eps_max = gershgorin_bounds(H) if bounds is None else map(float, bounds)
    if n_occ == 0 or n_occ == N:
        D = np.zeros((N, N)) if n_occ == 0 else np.eye(N)
        return dict(D=D, D1=[np.zeros((N, N)) for _ in H1s], layers=0, signs="", stop="trivial", eps_min=eps_min,
                    eps_max=eps_max, tr_d=float(n_occ), tr_dh=float(np.sum(D * H)), tr_d1=[0.0 for _ in H1s])
    delta = eps_max - eps_min
    X = rescale_to_unit_interval(H, eps_min, eps_max)
    Zs = [-H1 / delta for H1 in H1s]                             # R5
    e_hist, signs = [], []
    n = 0
    while True:
        X2 = X @ X                                               # f(X) = X^2
        t = float(np.trace(X))
        t2 = float(np.trace(X2))
        e_hist.append(t - t2)
        stop = sp2_stop(n, e_hist, signs, t, n_occ, tol, max_layers)
        if stop is not None:
            break
        plus = abs(t2 - n_occ) < abs(2.0 * t - t2 - n_occ)       # R3, ties -> '-'
        Ws = [X @ Z + Z @ X for Z in Zs]
        if plus:                                                 # S_n = S_{n-1}^2
            X = X2
            Zs = Ws
        else:                                                    # S_n = 2 S_{n-1} - S_{n-1}^2
            X = 2.0 * X - X2
            Zs = [2.0 * Z - W for Z, W in zip(Zs, Ws)]
        signs.append("+" if plus else "-")
        n += 1
    return dict(D=X, D1=Zs, layers=n, signs="".join(signs), stop=stop, eps_min=eps_min, eps_max=eps_max,
                tr_d=float(np.trace(X)), tr_dh=float(np.sum(X * H)), tr_d1=[float(np.trace(Z)) for Z in Zs])


def sp2_refine_layers(X, n_occ, layers=2):
    """Refinement step of PAPER.md:170: "two extra layers in Eq. (19), with a higher-order double-precision
    (64 bit) representation of X in the activation function ... where the eigenvalues are purified to be closer
    to exactly 1 and 0".  ``X`` is an (approximately idempotent) iterate; ``layers`` more SP2 layers
    X <- X^2 or 2X - X^2 are applied in float64 with the same trace rule as ``sp2_density`` (reading R3).
    Returns (X_refined, signs)."""
    X = np.array(X, dtype=np.float64)
    signs = []
    for _ in range(layers):
        X2 = X @ X
        t, t2 = float(np.trace(X)), float(np.trace(X2))
        plus = abs(t2 - n_occ) < abs(2.0 * t - t2 - n_occ)
        X = X2 if plus else 2.0 * X - X2
        signs.append("+" if plus else "-")
    return X, "".join(signs)


def congruence(Z, X, transpose_first=True):
    """The transforms either side of the solver in a non-orthogonal basis: "H_orth = Z^T H Z, where
    Z is the inverse factor of the overlap matrix, S, determined by the relation Z^T S Z = I", and back,
    "D = Z D_orth Z^T".  transpose_first: Z^T X Z, else Z X Z^T."""
    Z = np.asarray(Z, dtype=np.float64)
    X = np.asarray(X, dtype=np.float64)
    return Z.T @ X @ Z if transpose_first else Z @ X @ Z.T


def density_eigh(H, n_occ):
    """The definition written out (Eq. 17-18).

    D_ij = sum_k f_k c_i^(k) c_j^(k) with f_k = 1 for the n_occ lowest
    eigenvalues (below the chemical potential mu) and 0 above: the projector
    V_occ V_occ^T from a full symmetric eigendecomposition (LAPACK via NumPy).
    Returns (D, eigenvalues).
    """
    H = _as_f64_symmetric(H, "H")
    w, V = np.linalg.eigh(H)
    N = H.shape[0]
    if 0 < n_occ < N and not w[n_occ - 1] < w[n_occ]:
        raise ValueError("no gap at the chemical potential")
    Vo = V[:, :n_occ]
    return Vo @ Vo.T, w


def density_from_eigenpairs(Q, lam, n_occ, rows=None, cols=None):
    """Eq. 17 evaluated from KNOWN eigenpairs, no eigensolve.

    ``Q`` orthogonal (columns = eigenvectors), ``lam`` the eigenvalue of each
    column.  The occupied columns are the n_occ smallest ``lam``.  With
    ``rows``/``cols`` index arrays, only D[rows[k], cols[k]] is returned
    (element by element: usable at any N for sampled parity checks).
    """
    Q = np.asarray(Q, dtype=np.float64)
    lam = np.asarray(lam, dtype=np.float64)
    occ = np.argsort(lam, kind="stable")[:n_occ]
    Qo = Q[:, occ]
    if rows is None:
        return Qo @ Qo.T
    rows = np.asarray(rows)
    cols = np.asarray(cols)
    return np.einsum("kp,kp->k", Qo[rows, :], Qo[cols, :])


def response_closed_form(Q, lam, n_occ, H1):
    """First-order change of the projector under H -> H + eps*H1 (non-degenerate
    first-order perturbation theory; independent of the SP2 recursion):

        D1 = Q M Q^T,   M_ia = M_ai = (Q^T H1 Q)_ia / (lam_i - lam_a)
        for i occupied, a unoccupied; M = 0 on the occ-occ and unocc-unocc blocks.
    """
    Q = np.asarray(Q, dtype=np.float64)
    lam = np.asarray(lam, dtype=np.float64)
    H1 = np.asarray(H1, dtype=np.float64)
    order = np.argsort(lam, kind="stable")
    occ, un = order[:n_occ], order[n_occ:]
    G = Q.T @ H1 @ Q
    M = np.zeros_like(G)
    blk = G[np.ix_(occ, un)] / (lam[occ][:, None] - lam[un][None, :])
    M[np.ix_(occ, un)] = blk
    M[np.ix_(un, occ)] = blk.T
    return Q @ M @ Q.T


def response_closed_form_sampled(Q, lam, n_occ, H1, rows, cols):
    """Entries D1[rows[k], cols[k]] of ``response_closed_form`` without forming the N x N result
    (sampled parity checks at full size).  Same formula: with C_o / C_u the occupied / unoccupied
    eigenvector blocks and B = (C_o^T H1 C_u) / (lam_o - lam_u),
        D1 = C_o B C_u^T + C_u B^T C_o^T,
    so  D1_ij = sum_{o,u} B_ou (C_o[i,o] C_u[j,u] + C_u[i,u] C_o[j,o]).
    """
    Q = np.asarray(Q, dtype=np.float64)
    lam = np.asarray(lam, dtype=np.float64)
    H1 = np.asarray(H1, dtype=np.float64)
    order = np.argsort(lam, kind="stable")
    occ, un = order[:n_occ], order[n_occ:]
    Co, Cu = Q[:, occ], Q[:, un]
    B = (Co.T @ H1 @ Cu) / (lam[occ][:, None] - lam[un][None, :])
    rows = np.asarray(rows)
    cols = np.asarray(cols)
    left = Co[rows, :] @ B                   # (k, n_un)
    right = Co[cols, :] @ B
    return np.einsum("ku,ku->k", left, Cu[cols, :]) + np.einsum("ku,ku->k", right, Cu[rows, :])


def response_finite_difference(H, H1, n_occ, eps=1e-5):
    """(D(H + eps*H1) - D(H - eps*H1)) / (2 eps) with D from ``density_eigh``
    (BASELINE.json north_star: "a finite-difference D1")."""
    H = np.asarray(H, dtype=np.float64)
    H1 = np.asarray(H1, dtype=np.float64)
    Dp, _ = density_eigh(H + eps * H1, n_occ)
    Dm, _ = density_eigh(H - eps * H1, n_occ)
    return (Dp - Dm) / (2.0 * eps)


def sp2_spectrum_simulator(lam, n_occ, eps_min, eps_max, tol=0.0, max_layers=100):
    """SP2 acts on every eigenvalue independently (the activation
    functions are "matrix square functions acting on the eigenvalue spectrum"),
    so the scalar maps x -> x^2 / 2x - x^2 on x_0 = (eps_max - lam)/Delta,
    with traces as plain sums, reproduce layer count, sign string, tr X_n and
    e_n of the matrix loop in O(N L).  Returns the same keys as ``sp2_density``
    minus the matrices, plus ``x`` (final occupations).
    """
    x = (eps_max - np.asarray(lam, dtype=np.float64)) / (eps_max - eps_min)
    tr_hist, e_hist, signs = [], [], []
    n = 0
    while True:
        x2 = x * x
        t, t2 = float(x.sum()), float(x2.sum())
        tr_hist.append(t)
        e_hist.append(t - t2)
        stop = sp2_stop(n, e_hist, signs, t, n_occ, tol, max_layers)
        if stop is not None:
            break
        plus = abs(t2 - n_occ) < abs(2.0 * t - t2 - n_occ)
        x = x2 if plus else 2.0 * x - x2
        signs.append("+" if plus else "-")
        n += 1
    return dict(x=x, layers=n, signs="".join(signs), tr_x=tr_hist, e=e_hist, stop=stop)
