"""GPU parity of the optional Lanczos spectral bounds: the bounds against the oracle's plain
float64 Lanczos process, and D / D1 against the oracle run with those bounds (fewer layers, same projector)."""
import numpy as np
import pytest

from paper_2107_02737_b200 import inputs

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("n, base, response, steps", [(300, 2, True, 12), (520, 3, False, 8), (1024, 4, True, 16)])
def test_lanczos_bounds_and_density(torch_cuda, sp2, n, base, response, steps):
    import oracle

    torch = torch_cuda
    p = inputs.make_problem(inputs.scaled_config(inputs.CONFIGS[base], n), want_h1=response)
    n_occ = p["n_occ"]
    H64 = p["H"].astype(np.float64)
    lo, hi = oracle.lanczos_bounds(H64, steps)
    ref = oracle.sp2_density(H64, n_occ, H1=p["H1"].astype(np.float64) if response else None, bounds=(lo, hi))
    ref_g = oracle.sp2_density(H64, n_occ)
    h = sp2.Sp2Handle(n, response=response)
    h.set_options(lanczos_steps=steps)
    H = torch.from_numpy(p["H"]).cuda()
    if response:
        D, D1, r = h.response(H, torch.from_numpy(p["H1"]).cuda(), n_occ)
        assert np.abs(D1.cpu().numpy().astype(np.float64) - ref["D1"]).max() <= 1e-3 * np.abs(ref["D1"]).max()
    else:
        D, r = h.density(H, n_occ)
    h.close()
    assert r["status"] == 0
    width = hi - lo
    assert abs(r["eps_min"] - lo) <= 1e-6 * width and abs(r["eps_max"] - hi) <= 1e-6 * width
    w = np.linalg.eigvalsh(H64)
    assert r["eps_min"] <= w[0] and r["eps_max"] >= w[-1]                  # still an enclosure
    assert np.abs(D.cpu().numpy().astype(np.float64) - ref["D"]).max() <= 1e-4
    assert abs(r["tr_d"] - n_occ) <= 1e-3 and abs(r["tr_dh"] - ref["tr_dh"]) <= 1e-5 * abs(ref["tr_dh"])
    assert abs(r["layers"] - ref["layers"]) <= 6 and r["layers"] <= ref_g["layers"] - 3   # fewer layers than Gershgorin


def test_lanczos_is_ignored_with_user_bounds_and_sparse_tight_case(torch_cuda, sp2):
    torch = torch_cuda
    Hn, lam = inputs.ssh_chain(512, 1.0, 0.6)
    h = sp2.Sp2Handle(512)
    H = torch.from_numpy(Hn).cuda()
    D0, r0 = h.density(H, 256)
    h.set_options(lanczos_steps=12)
    D1, r1 = h.density(H, 256)                      # Gershgorin is already tight here: the intersection keeps it
    assert r1["eps_min"] >= r0["eps_min"] and r1["eps_max"] <= r0["eps_max"] and abs(r1["layers"] - r0["layers"]) <= 2
    assert float((D1 - D0).abs().max()) <= 1e-5
    h.set_options(lanczos_steps=12, user_bounds=(-2.0, 2.0))
    D2, r2 = h.density(H, 256)
    assert (r2["eps_min"], r2["eps_max"]) == (-2.0, 2.0)
    h.close()


@pytest.mark.parametrize("n_occ, hidden", [(40, -3.0), (150, 3.0)])
def test_lanczos_bounds_that_miss_an_eigenvalue_fall_back_to_gershgorin(torch_cuda, sp2, n_occ, hidden):
    """Adversarial input: an outlier eigenvalue whose eigenvector is orthogonal to the Lanczos start vector, so the
    Lanczos interval misses it by > 1 (tests/test_oracle_pins.py shows the oracle's own Lanczos bounds do too and that SP2
    with them returns garbage).  The device guard must see an eigenvalue of X leave [0, 1] (SP2_ERR_BOUNDS inside the
    call) and the blocking call must re-run with the Gershgorin discs: right answer, flagged."""
    import oracle

    torch = torch_cuda
    n = 300
    H, lam = inputs.hidden_eigenvector_problem(n, n_occ, hidden, np.cos(0.7 * np.arange(n) + 0.3))
    ref = oracle.sp2_density(H, n_occ)
    lo, hi = oracle.lanczos_bounds(H, 12)
    assert (lo > -2.0) if hidden < 0 else (hi < 2.0)
    h = sp2.Sp2Handle(n)
    h.set_options(lanczos_steps=12)
    D, r = h.density(torch.from_numpy(H).cuda(), n_occ)
    assert r["status"] == 0 and r["bounds_fallback"] == 1
    assert r["eps_min"] == pytest.approx(ref["eps_min"], rel=1e-12) and r["eps_max"] == pytest.approx(ref["eps_max"], rel=1e-12)
    assert np.abs(D.cpu().numpy() - ref["D"]).max() <= 1e-4
    assert abs(r["tr_d"] - n_occ) <= 1e-3 and abs(r["tr_dh"] - ref["tr_dh"]) <= 1e-5 * abs(ref["tr_dh"])
    # the same matrix with wrong USER bounds is the caller's error: reported, not repaired
    h.set_options(lanczos_steps=0, user_bounds=(lo, hi))
    with pytest.raises(sp2.Sp2Error) as ei:
        h.density(torch.from_numpy(H).cuda(), n_occ)
    assert ei.value.status == sp2.SP2_ERR_BOUNDS
    # and in a sequence step (no host round trip, so no re-run) the step reports SP2_ERR_BOUNDS
    h.set_options(lanczos_steps=12, user_bounds=None)
    h.sequence_begin(n, n_occ, n_steps_hint=1)
    Dt = torch.empty(n, n, dtype=torch.float64, device="cuda")
    h.sequence_step(torch.from_numpy(H).cuda(), Dt)
    with pytest.raises(sp2.Sp2Error) as ei:
        h.sequence_end()
    assert ei.value.status == sp2.SP2_ERR_BOUNDS
    h.close()
