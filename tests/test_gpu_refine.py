"""GPU parity of the float64 refinement layers: the refined D against the
oracle's plain float64 refinement of the SAME unrefined iterate (element by element), plus the properties the
paper wants from the step (eigenvalues purified: idempotency and trace errors collapse; D barely moves)."""
import numpy as np
import pytest

from paper_2107_02737_b200 import inputs

pytestmark = pytest.mark.gpu


# sizes: 6, 21 and 66 tiles (every tile split along k between the blocks), 171 tiles (one round of whole tiles on 148
# SMs, then the remaining 23 split), and a reduced grid (max_ctas: other split points, same result)
@pytest.mark.parametrize("n, base, max_ctas", [(384, 2, 0), (700, 3, 0), (700, 3, 40), (1300, 4, 0), (2304, 2, 0), (2304, 2, 100)])
def test_refinement_matches_oracle_layers(torch_cuda, sp2, n, base, max_ctas):
    import oracle

    torch = torch_cuda
    p = inputs.make_problem(inputs.scaled_config(inputs.CONFIGS[base], n), want_h1=False)
    n_occ = p["n_occ"]
    H = torch.from_numpy(p["H"].astype(np.float64)).cuda()
    h = sp2.Sp2Handle(n, refinement=True)
    h.set_options(max_ctas=max_ctas)
    D0, r0 = h.density(H, n_occ)                          # unrefined: exactly the iterate the refinement starts from
    h.set_options(refine_layers=2)
    D2, r2 = h.density(H, n_occ)
    h.close()
    assert r2["status"] == 0 and r2["refine_layers"] == 2 and r0["refine_layers"] == 0
    X0 = D0.cpu().numpy()
    ref, signs = oracle.sp2_refine_layers(X0, n_occ, layers=2)
    got = D2.cpu().numpy()
    assert np.abs(got - ref).max() <= 1e-13                # same float64 arithmetic up to summation order
    assert np.array_equal(got, got.T)
    # what the step is for: eigenvalues purified
    idem0 = np.linalg.norm(X0 @ X0 - X0)
    idem2 = np.linalg.norm(got @ got - got)
    assert idem2 < 1e-11 and idem2 < 1e-4 * idem0
    assert abs(r2["tr_d"] - n_occ) < 1e-9 and abs(np.trace(got) - r2["tr_d"]) < 1e-10
    assert abs(r2["idem_est"]) < 1e-9
    assert np.abs(got - X0).max() < 1e-5                   # eigenvectors untouched: D barely moves
    E = inputs.band_energy_closed_form(p["lam"], n_occ)
    assert abs(r2["tr_dh"] - E) <= 1e-5 * abs(E)
    assert r2["tr_dh"] == pytest.approx(float((got * p["H"].astype(np.float64)).sum()), rel=1e-12)


def test_refinement_needs_its_workspace_and_f32_output(torch_cuda, sp2):
    torch = torch_cuda
    p = inputs.make_problem(inputs.scaled_config(inputs.CONFIGS[3], 260))      # f32 input
    H = torch.from_numpy(p["H"]).cuda()
    h = sp2.Sp2Handle(260)
    h.set_options(refine_layers=2)
    with pytest.raises(sp2.Sp2Error) as ei:
        h.density(H, p["n_occ"])
    assert ei.value.status == sp2.SP2_ERR_WORKSPACE
    h.close()
    h = sp2.Sp2Handle(260, refinement=True)
    h.set_options(refine_layers=1)
    D, r = h.density(H, p["n_occ"])                        # f32 in, f32 out
    assert r["status"] == 0 and r["refine_layers"] == 1 and D.dtype == torch.float32
    assert abs(r["tr_d"] - p["n_occ"]) < 1e-4              # a single layer purifies one side of the spectrum only
    h.close()


def test_refinement_with_response_and_sequence(torch_cuda, sp2):
    """D is refined, D1 is left as the FP16 stack produced it; the sequence call refines every step."""
    torch = torch_cuda
    p = inputs.make_problem(inputs.scaled_config(inputs.CONFIGS[2], 300), want_h1=True)
    n, n_occ = p["n"], p["n_occ"]
    H = torch.from_numpy(p["H"]).cuda()
    H1 = torch.from_numpy(p["H1"]).cuda()
    h = sp2.Sp2Handle(n, response=True, refinement=True)
    D0, D10, r0 = h.response(H, H1, n_occ)
    h.set_options(refine_layers=2)
    D2, D12, r2 = h.response(H, H1, n_occ)
    assert torch.equal(D10, D12) and r2["tr_d1"] == r0["tr_d1"]
    assert abs(r2["tr_d"] - n_occ) < 1e-9 and float((D2 - D0).abs().max()) < 1e-5
    Ds = [torch.empty_like(H) for _ in range(3)]
    h.sequence_begin(n, n_occ, n_steps_hint=3)
    for k, Dk in enumerate(Ds):
        h.sequence_step(H + 1e-3 * k * H1, Dk)
    res = h.sequence_end()
    assert [r["refine_layers"] for r in res] == [2, 2, 2] and all(abs(r["tr_d"] - n_occ) < 1e-9 for r in res)
    assert torch.equal(Ds[0], D2)
    h.close()
