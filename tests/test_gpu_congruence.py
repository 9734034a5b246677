"""GPU parity of sp2_congruence against the oracle's float64 products, and the
whole non-orthogonal pipeline H, S -> H_orth -> D_orth -> D against the generalised-eigenproblem projector."""
import numpy as np
import pytest

from paper_2107_02737_b200 import inputs

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("n, cta_group", [(200, 1), (520, 1), (520, 2), (1100, 0)])
@pytest.mark.parametrize("transpose_first", [True, False])
def test_congruence_matches_float64_products(torch_cuda, sp2, n, cta_group, transpose_first):
    import oracle

    torch = torch_cuda
    rng = np.random.default_rng(n)
    Z = rng.standard_normal((n, n)) / np.sqrt(n) + np.eye(n)            # general, non-symmetric
    X = rng.standard_normal((n, n)); X = 0.5 * (X + X.T)
    ref = oracle.congruence(Z, X, transpose_first)
    h = sp2.Sp2Handle(n, response=True)
    h.set_options(cta_group=cta_group)
    C = h.congruence(torch.from_numpy(Z).cuda(), torch.from_numpy(X).cuda(), transpose_first=transpose_first)
    # operands carry 22 bits, two chained products: a few 2^-22 of the row/column norms involved
    tol = 16 * 2.0 ** -22 * np.abs(ref).max()
    assert np.abs(C.cpu().numpy() - ref).max() <= tol
    # f32 in / f32 out, a pitch larger than N, and values far from 1 (plane exponents)
    Zs = torch.zeros(n, n + 8, dtype=torch.float32, device="cuda"); Zs[:, :n] = torch.from_numpy(Z).float().cuda() * 1e3
    Xs = torch.zeros(n, n + 8, dtype=torch.float32, device="cuda"); Xs[:, :n] = torch.from_numpy(X).float().cuda() * 1e-4
    ref32 = oracle.congruence(Zs[:, :n].double().cpu().numpy(), Xs[:, :n].double().cpu().numpy(), transpose_first)
    C32 = h.congruence(Zs[:, :n], Xs[:, :n], transpose_first=transpose_first)
    assert C32.dtype == torch.float32
    assert np.abs(C32.double().cpu().numpy() - ref32).max() <= 16 * 2.0 ** -22 * np.abs(ref32).max() + 2.0 ** -23 * np.abs(ref32).max()
    h.close()


def test_nonorthogonal_pipeline(torch_cuda, sp2):
    """H, S -> Z (host, Loewdin) -> H_orth = Z^T H Z (GPU) -> D_orth (GPU SP2) -> D = Z D_orth Z^T (GPU)."""
    import oracle
    import scipy.linalg

    torch = torch_cuda
    q = inputs.overlap_problem(640, 300)
    n, n_occ = q["n"], q["n_occ"]
    H, S, Z = (torch.from_numpy(q[k]).cuda() for k in ("H", "S", "Z"))
    h = sp2.Sp2Handle(n, response=True)
    Horth = h.congruence(Z, H, transpose_first=True)
    Dorth, r = h.density(Horth, n_occ)
    D = h.congruence(Z, Dorth, transpose_first=False)
    h.close()
    eps, Cg = scipy.linalg.eigh(q["H"], q["S"])
    D_ref = Cg[:, :n_occ] @ Cg[:, :n_occ].T
    assert r["status"] == 0
    assert np.abs(D.cpu().numpy() - D_ref).max() <= 1e-4
    assert abs(float((D * S).sum()) - n_occ) <= 1e-3                       # tr(D S) = N_occ
    assert abs(r["tr_dh"] - eps[:n_occ].sum()) <= 1e-5 * abs(eps[:n_occ].sum())   # tr(D_orth H_orth) = band energy
    assert np.abs(Horth.cpu().numpy() - oracle.congruence(q["Z"], q["H"])).max() <= 16 * 2.0 ** -22


def test_congruence_errors(torch_cuda, sp2):
    torch = torch_cuda
    X = torch.eye(64, dtype=torch.float64, device="cuda")
    h = sp2.Sp2Handle(64)                       # no second plane set
    with pytest.raises(sp2.Sp2Error) as ei:
        h.congruence(X, X)
    assert ei.value.status == sp2.SP2_ERR_WORKSPACE
    h.close()
    h = sp2.Sp2Handle(64, response=True)
    Xn = X.clone(); Xn[3, 4] = float("nan")
    with pytest.raises(sp2.Sp2Error) as ei:
        h.congruence(X, Xn)
    assert ei.value.status == sp2.SP2_ERR_NONFINITE
    C = h.congruence(2.0 * X, X)                # still usable: (2I)^T I (2I) = 4I
    assert torch.allclose(C, 4.0 * X, atol=1e-6)
    h.close()
