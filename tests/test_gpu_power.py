"""GPU parity of the rigorous power-trace spectral bounds (sp2_options_t.power_squarings): the
interval against the oracle's definition (plain float64 matrix powers), enclosure of the LAPACK spectrum -- also on the
matrices built against the Lanczos start vector -- and D / D1 against the oracle run with the oracle's interval."""
import numpy as np
import pytest

from paper_2107_02737_b200 import inputs

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("n, base, response, s, opts", [
    (77, 1, False, 3, {}),                          # one CTA, shared-memory stack (unfused prologue)
    (300, 2, True, 4, {}),                          # persistent kernel, power phase on its own density-only work lists
    (520, 3, False, 2, dict(cta_group=2)),          # f32 input, 2/3 filling, CTA pairs
    (1100, 4, True, 4, dict(persistent=2)),         # one launch per layer, split-k tails
])
def test_power_trace_bounds_and_density(torch_cuda, sp2, n, base, response, s, opts):
    import oracle

    torch = torch_cuda
    p = inputs.make_problem(inputs.scaled_config(inputs.CONFIGS[base], n), want_h1=response)
    n_occ = p["n_occ"]
    H64 = p["H"].astype(np.float64)
    lo, hi = oracle.power_trace_bounds(H64, s)
    ref = oracle.sp2_density(H64, n_occ, H1=p["H1"].astype(np.float64) if response else None, bounds=(lo, hi))
    ref_g = oracle.sp2_density(H64, n_occ)
    h = sp2.Sp2Handle(n, response=response)
    h.set_options(power_squarings=s, **opts)
    H = torch.from_numpy(p["H"]).cuda()
    if response:
        D, D1, r = h.response(H, torch.from_numpy(p["H1"]).cuda(), n_occ)
        assert np.abs(D1.cpu().numpy().astype(np.float64) - ref["D1"]).max() <= 1e-3 * np.abs(ref["D1"]).max()
    else:
        D, r = h.density(H, n_occ)
    h.close()
    assert r["status"] == 0 and r["bounds_fallback"] == 0
    w = np.linalg.eigvalsh(H64)
    mu = np.trace(H64) / n
    assert r["eps_min"] <= w[0] and r["eps_max"] >= w[-1]                      # rigorous: an enclosure
    # the GPU interval is the oracle's radius widened by 1e-3 (22-bit squarings): never inside it, at most 2.5e-3 outside
    r_or, r_gpu = max(hi - mu, mu - lo), max(r["eps_max"] - mu, mu - r["eps_min"])
    g_lo, g_hi = oracle.gershgorin_bounds(H64)
    if lo > g_lo and hi < g_hi:                                                # not clipped by the discs
        assert r_or * (1 - 1e-6) <= r_gpu <= r_or * (1 + 2.5e-3)
    assert np.abs(D.cpu().numpy().astype(np.float64) - ref["D"]).max() <= 1e-4
    assert abs(r["tr_d"] - n_occ) <= 1e-3 and abs(r["tr_dh"] - ref["tr_dh"]) <= 1e-5 * abs(ref["tr_dh"])
    assert abs(r["layers"] - ref["layers"]) <= 6 and r["layers"] <= ref_g["layers"] - 3   # fewer layers than Gershgorin


@pytest.mark.parametrize("n_occ, hidden", [(40, -3.0), (150, 3.0)])
def test_power_trace_bounds_see_what_lanczos_misses(torch_cuda, sp2, n_occ, hidden):
    """The adversarial matrices of test_gpu_lanczos.py (an outlier eigenvalue whose eigenvector is orthogonal to the
    Lanczos start vector): the power-trace interval encloses the outlier, so the solve is right the first time --
    no SP2_ERR_BOUNDS inside the call, no fallback."""
    import oracle

    torch = torch_cuda
    n = 300
    H, lam = inputs.hidden_eigenvector_problem(n, n_occ, hidden, np.cos(0.7 * np.arange(n) + 0.3))
    ref = oracle.sp2_density(H, n_occ)
    h = sp2.Sp2Handle(n)
    h.set_options(power_squarings=4, lanczos_steps=12)            # the rigorous bounds take precedence over the estimate
    D, r = h.density(torch.from_numpy(H).cuda(), n_occ)
    h.close()
    assert r["status"] == 0 and r["bounds_fallback"] == 0
    assert r["eps_min"] <= lam.min() and r["eps_max"] >= lam.max()
    assert np.abs(D.cpu().numpy() - ref["D"]).max() <= 1e-4 and abs(r["tr_d"] - n_occ) <= 1e-3


def test_power_phase_edge_cases(torch_cuda, sp2):
    """H = c I (nothing to tighten: degenerate), non-finite input, trivial occupations, a sequence, and scale / offset."""
    torch = torch_cuda
    p = inputs.make_problem(inputs.scaled_config(inputs.CONFIGS[1], 200))
    n, n_occ = p["n"], p["n_occ"]
    H = torch.from_numpy(p["H"]).cuda()
    h = sp2.Sp2Handle(n)
    h.set_options(power_squarings=3)
    with pytest.raises(sp2.Sp2Error) as ei:
        h.density(3.0 * torch.eye(n, dtype=torch.float64, device="cuda"), n_occ)
    assert ei.value.status == sp2.SP2_ERR_DEGENERATE
    Hn = H.clone()
    Hn[3, 9] = float("nan")
    with pytest.raises(sp2.Sp2Error) as ei:
        h.density(Hn, n_occ)
    assert ei.value.status == sp2.SP2_ERR_NONFINITE
    D, r = h.density(H, 0)
    assert r["status"] == 0 and r["layers"] == 0
    D0, r0 = h.density(H, n_occ)
    Ds, rs = h.density(1e6 * H + 5e5 * torch.eye(n, dtype=H.dtype, device="cuda"), n_occ)
    assert rs["status"] == 0 and float((Ds - D0).abs().max()) <= 2e-6 and abs(rs["layers"] - r0["layers"]) <= 2
    h.sequence_begin(n, n_occ, n_steps_hint=2)
    outs = [torch.empty_like(H) for _ in range(2)]
    for o in outs:
        h.sequence_step(H, o)
    res = h.sequence_end()
    assert [x["status"] for x in res] == [0, 0] and torch.equal(outs[0], outs[1]) and float((outs[0] - D0).abs().max()) == 0.0
    h.close()
