"""GPU parity at BASELINE.json's full sizes (configs 3, 4, 5), in the launch configuration bench.py
times.  The float64 SP2 loop of the oracle would take minutes to hours here, so D is compared with
the oracle's DEFINITION evaluated from the generator's eigenpairs (oracle.density_from_eigenpairs,
Eq. 17: exact projector, sampled element by element) and D1 with the sampled closed form of
first-order perturbation theory; plus properties that hold at any size (trace, band energy,
bit-symmetry) and float64 idempotency / commutator / response identities evaluated with torch on the
GPU as a labelled CROSS-CHECK (torch is the harness here, never the library).
"""
import numpy as np
import pytest

from paper_2107_02737_b200 import inputs

pytestmark = pytest.mark.gpu

TOL_D, TOL_TR, TOL_E, TOL_D1 = 1e-4, 1e-3, 1e-5, 1e-3


def _samples(n, k=4000, seed=7):
    rng = np.random.default_rng(seed)
    rows = np.concatenate([rng.integers(0, n, k), np.arange(0, n, max(1, n // 512)), [0, n - 1, n - 1]])
    cols = np.concatenate([rng.integers(0, n, k), np.arange(0, n, max(1, n // 512)), [n - 1, 0, n - 1]])
    return rows, cols


def _gather(torch, M, rows, cols):
    return M[torch.from_numpy(rows).cuda(), torch.from_numpy(cols).cuda()].double().cpu().numpy()


def _crosscheck_projector(torch, D, H, n_occ):
    """float64 invariants on the GPU (cross-check, not the oracle): idempotency and [H, D] = 0."""
    D64, H64 = D.double(), H.double()
    idem = float(torch.linalg.norm(D64 @ D64 - D64)) / n_occ ** 0.5
    comm = float(torch.linalg.norm(H64 @ D64 - D64 @ H64)) / float(torch.linalg.norm(H64))
    return idem, comm


def test_config3_waterbox_n6000_f32(torch_cuda, sp2):
    import oracle

    torch = torch_cuda
    p = inputs.make_problem(inputs.CONFIGS[3], device="cuda")
    n, n_occ = p["n"], p["n_occ"]
    assert (n, n_occ, p["H"].dtype) == (6000, 4000, np.float32)
    H = torch.from_numpy(p["H"]).cuda()
    h = sp2.Sp2Handle(n)
    D, r = h.density(H, n_occ)
    h.close()
    rows, cols = _samples(n)
    De = oracle.density_from_eigenpairs(p["Q"], p["lam"], n_occ, rows, cols)
    assert r["status"] == 0 and 25 <= r["layers"] <= 50
    assert np.abs(_gather(torch, D, rows, cols) - De).max() <= TOL_D
    assert abs(r["tr_d"] - n_occ) <= TOL_TR
    E = inputs.band_energy_closed_form(p["lam"], n_occ)
    assert abs(r["tr_dh"] - E) <= TOL_E * abs(E)
    assert bool(torch.equal(D, D.T))
    idem, comm = _crosscheck_projector(torch, D, H, n_occ)
    assert idem < 1e-4 and comm < 1e-5


def test_config4_smallgap_n8192_response(torch_cuda, sp2):
    import oracle

    torch = torch_cuda
    p = inputs.make_problem(inputs.CONFIGS[4], device="cuda")
    n, n_occ = p["n"], p["n_occ"]
    assert (n, n_occ) == (8192, 4096)
    H = torch.from_numpy(p["H"]).cuda()
    H1 = torch.from_numpy(p["H1"]).cuda()
    h = sp2.Sp2Handle(n, response=True)
    D, D1, r = h.response(H, H1, n_occ)
    h.close()
    rows, cols = _samples(n)
    De = oracle.density_from_eigenpairs(p["Q"], p["lam"], n_occ, rows, cols)
    D1e = oracle.response_closed_form_sampled(p["Q"], p["lam"], n_occ, p["H1"], rows, cols)
    scale1 = np.abs(D1e).max()
    assert r["status"] == 0 and 35 <= r["layers"] <= 52                     # BASELINE.json: ~35-45 layers
    assert np.abs(_gather(torch, D, rows, cols) - De).max() <= TOL_D
    assert np.abs(_gather(torch, D1, rows, cols) - D1e).max() <= TOL_D1 * scale1
    assert abs(r["tr_d"] - n_occ) <= TOL_TR
    E = inputs.band_energy_closed_form(p["lam"], n_occ)
    assert abs(r["tr_dh"] - E) <= TOL_E * abs(E)
    assert bool(torch.equal(D, D.T)) and bool(torch.equal(D1, D1.T))
    assert abs(r["tr_d1"]) <= 1e-3 * scale1 * n ** 0.5
    idem, comm = _crosscheck_projector(torch, D, H, n_occ)
    assert idem < 1e-4 and comm < 1e-5
    # derivative of D^2 = D (cross-check in float64 on the GPU): D D1 + D1 D = D1
    resid = float((D @ D1 + D1 @ D - D1).abs().max())
    assert resid <= TOL_D1 * scale1


def test_config5_all_50_steps_n16384(torch_cuda, sp2):
    """The whole 50-step sweep of config 5 at full size through sp2_sequence_* (one host synchronisation, at the end):
    status, trace and band-energy law for EVERY step from the per-step results; bit-symmetry, idempotency and commutator
    (float64 on the GPU, cross-check) on the steps whose D is kept (0, 25, 49; the others share one output buffer);
    t = 0 against the exact projector.  The oracle comparison for t > 0 is test_config5_shape_n4096_steps_against_oracle."""
    import oracle

    torch = torch_cuda
    p = inputs.make_problem(inputs.CONFIGS[5], device="cuda", want_p=True)
    n, n_occ, n_steps = p["n"], p["n_occ"], inputs.CONFIGS[5].n_steps
    assert n_steps == 50
    H0 = torch.from_numpy(p["H"]).cuda()
    P = torch.from_numpy(p["P"]).cuda()
    keep = {0: torch.empty_like(H0), 25: torch.empty_like(H0), 49: torch.empty_like(H0)}
    scratch_D = torch.empty_like(H0)
    Ht = torch.empty_like(H0)
    h = sp2.Sp2Handle(n)
    h.density(H0, n_occ, out=scratch_D)                      # warm-up: gives the sequence its layer-count hint
    h.sequence_begin(n, n_occ, n_steps_hint=n_steps)
    for t in range(n_steps):
        torch.add(H0, P, alpha=1e-3 * t, out=Ht)             # stream-ordered: the previous step has read Ht by then
        h.sequence_step(Ht, keep.get(t, scratch_D))
    res = h.sequence_end()
    h.close()
    assert len(res) == n_steps and [r["status"] for r in res] == [0] * n_steps
    E0 = inputs.band_energy_closed_form(p["lam"], n_occ)
    assert abs(res[0]["tr_dh"] - E0) <= TOL_E * abs(E0)
    d1 = 1e-3 * float((keep[0].double() * P.double()).sum())   # first-order slope dE/dt = eps tr(D_0 P)
    # E(t) = E_0 + t d1 - c t^2 + O(t^3), c > 0: second-order perturbation theory lowers the occupied sum, so every
    # step lies below the first-order line and the drop follows one t^2 law along the whole sweep
    curv = {t: (t * d1 - (res[t]["tr_dh"] - res[0]["tr_dh"])) / t ** 2 for t in range(5, n_steps)}
    for t, r in enumerate(res):
        assert 30 <= r["layers"] <= 50 and abs(r["tr_d"] - n_occ) <= TOL_TR, t
    for t, c in curv.items():
        assert c > 0 and 0.6 * curv[49] <= c <= 1.6 * curv[49], (t, c, curv[49])
    rows, cols = _samples(n, k=2000)
    De = oracle.density_from_eigenpairs(p["Q"], p["lam"], n_occ, rows, cols)
    assert np.abs(_gather(torch, keep[0], rows, cols) - De).max() <= TOL_D
    for t, D in keep.items():
        assert bool(torch.equal(D, D.T)), t
        idem, comm = _crosscheck_projector(torch, D, torch.add(H0, P, alpha=1e-3 * t), n_occ)
        assert idem < 1e-4 and comm < 1e-5, t


def test_config5_shape_n4096_steps_against_oracle(torch_cuda, sp2):
    """Config 5's recipe at N = 4096 (f32, gap 0.2, H_t = H_0 + t 1e-3 P): all 50 steps through the sequence call, every
    step's status and trace, and steps 0, 12, 25, 37, 49 element by element against the oracle's DEFINITION
    (oracle.density_eigh of the same H_t in float64: a full eigendecomposition per compared step)."""
    import oracle

    torch = torch_cuda
    n = 4096
    p = inputs.make_problem(inputs.scaled_config(inputs.CONFIGS[5], n), device="cuda", want_p=True)
    n_occ = p["n_occ"]
    H0 = torch.from_numpy(p["H"]).cuda()
    P = torch.from_numpy(p["P"]).cuda()
    Hs = [torch.add(H0, P, alpha=1e-3 * t) for t in range(50)]
    Ds = [torch.empty_like(H0) for _ in range(50)]
    h = sp2.Sp2Handle(n)
    h.sequence_begin(n, n_occ, n_steps_hint=50)
    for a, b in zip(Hs, Ds):
        h.sequence_step(a, b)
    res = h.sequence_end()
    h.close()
    assert [r["status"] for r in res] == [0] * 50
    for t, r in enumerate(res):
        assert abs(r["tr_d"] - n_occ) <= TOL_TR, t
    for t in (0, 12, 25, 37, 49):
        H64 = Hs[t].double().cpu().numpy()
        H64 = 0.5 * (H64 + H64.T)
        De, w = oracle.density_eigh(H64, n_occ)
        assert np.abs(Ds[t].double().cpu().numpy() - De).max() <= TOL_D, t
        E = float(w[:n_occ].sum())
        assert abs(res[t]["tr_dh"] - E) <= TOL_E * abs(E), t


def test_maximum_size_n32768_f32(torch_cuda, sp2):
    """SP2_MAX_N: the largest supported dimension (planes of 2 GiB each, 2^30 elements; seg_kb = 2 above N = 16384).
    Same recipe as config 5, scaled."""
    import oracle

    torch = torch_cuda
    n = sp2_max_n = 32768
    p = inputs.make_problem(inputs.scaled_config(inputs.CONFIGS[5], n), device="cuda")
    n_occ = p["n_occ"]
    H = torch.from_numpy(p["H"]).cuda()
    h = sp2.Sp2Handle(sp2_max_n)
    D, r = h.density(H, n_occ)
    h.close()
    rows, cols = _samples(n, k=2000)
    De = oracle.density_from_eigenpairs(p["Q"], p["lam"], n_occ, rows, cols)
    assert r["status"] == 0 and 30 <= r["layers"] <= 55
    assert np.abs(_gather(torch, D, rows, cols) - De).max() <= TOL_D
    assert abs(r["tr_d"] - n_occ) <= TOL_TR
    E = inputs.band_energy_closed_form(p["lam"], n_occ)
    assert abs(r["tr_dh"] - E) <= TOL_E * abs(E)
    assert bool(torch.equal(D, D.T))
    with pytest.raises(sp2.Sp2Error):
        sp2.Sp2Handle(sp2_max_n + 1)
