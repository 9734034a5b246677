"""GPU parity of the batched response: several perturbations of one H on
one stack of layers, against the oracle's one-stack loop (float64), element by element, through the C ABI.
Tolerances [north_star]: max|dD| <= 1e-4, |tr D - N_occ| <= 1e-3, rel d tr(DH) <= 1e-5, max|dD1_b| <= 1e-3 max|D1_b|."""
import numpy as np
import pytest

from paper_2107_02737_b200 import inputs

pytestmark = pytest.mark.gpu


def _check(r, ref, D, D1s, tr1, n_occ):
    assert r["status"] == 0
    assert np.abs(D.cpu().numpy().astype(np.float64) - ref["D"]).max() <= 1e-4
    assert abs(r["tr_d"] - n_occ) <= 1e-3
    assert abs(r["tr_dh"] - ref["tr_dh"]) <= 1e-5 * abs(ref["tr_dh"])
    assert abs(r["layers"] - ref["layers"]) <= 6
    for b, want in enumerate(ref["D1"]):
        got = D1s[b].cpu().numpy().astype(np.float64)
        s = np.abs(want).max()
        assert np.abs(got - want).max() <= 1e-3 * s, b
        assert np.abs(got - got.T).max() == 0.0                      # planes are bit-symmetric
        assert abs(tr1[b] - np.trace(got)) <= 1e-9 * s * len(got) + 1e-12
    assert r["tr_d1"] == tr1[0]


# sizes span several tiles and a ragged tail; engine 1 = the SIMT scaffold; cta_group 2 = CTA pairs
@pytest.mark.parametrize("n, nb, base, cta_group, engine", [
    (300, 3, 2, 0, 0), (640, 2, 2, 2, 0), (1000, 4, 3, 1, 0), (1100, 8, 2, 2, 0), (200, 3, 2, 0, 1)])
def test_batch_matches_oracle(torch_cuda, sp2, n, nb, base, cta_group, engine):
    import oracle

    torch = torch_cuda
    p = inputs.make_problem(inputs.scaled_config(inputs.CONFIGS[base], n), want_h1=False)
    n_occ = p["n_occ"]
    dt = p["H"].dtype
    H1s = inputs.perturbations(n, nb, seed=n, dtype=dt, decades=1.5)      # magnitudes 1e-2 ... 1e-12.5
    ref = oracle.sp2_response_batch(p["H"].astype(np.float64), n_occ, [a.astype(np.float64) for a in H1s])
    h = sp2.Sp2Handle(n, batch=nb)
    h.set_options(cta_group=cta_group, engine=engine)
    H = torch.from_numpy(p["H"]).cuda()
    D, D1s, tr1, r = h.response_batch(H, [torch.from_numpy(a).cuda() for a in H1s], n_occ)
    _check(r, ref, D, D1s, tr1, n_occ)
    # a smaller batch and the single-perturbation call on the same handle give the same matrices
    D2, D1s2, tr2, r2 = h.response_batch(H, [torch.from_numpy(H1s[nb - 1]).cuda()], n_occ)
    Ds, D1single, rs = h.response(H, torch.from_numpy(H1s[0]).cuda(), n_occ)
    h.close()
    # (the work schedule, hence the FP32 summation order of the split-k tail, depends on the batch size: the stop
    # rule may fire a layer apart, reading R4)
    assert abs(r2["layers"] - r["layers"]) <= 2 and abs(rs["layers"] - r["layers"]) <= 2
    assert float((D2 - D).abs().max()) <= 1e-6 and float((Ds - D).abs().max()) <= 1e-6
    s_last = float(D1s[nb - 1].abs().max())
    assert float((D1s2[0] - D1s[nb - 1]).abs().max()) <= 2e-5 * s_last
    assert float((D1single - D1s[0]).abs().max()) <= 2e-5 * float(D1s[0].abs().max())


def test_batch_f32_io_pitch_and_trivial_occupations(torch_cuda, sp2):
    import oracle

    torch = torch_cuda
    n, nb = 520, 3
    p = inputs.make_problem(inputs.scaled_config(inputs.CONFIGS[3], n), want_h1=False)   # float32 config
    n_occ = p["n_occ"]
    H1s = inputs.perturbations(n, nb, seed=11, dtype=np.float32)
    ref = oracle.sp2_response_batch(p["H"].astype(np.float64), n_occ, [a.astype(np.float64) for a in H1s])
    h = sp2.Sp2Handle(n + 8, batch=nb)
    ld = n + 24                                                         # pitched inputs and outputs
    Hbuf = torch.zeros((n, ld), dtype=torch.float32, device="cuda")
    Hbuf[:, :n] = torch.from_numpy(p["H"]).cuda()
    H1buf = []
    for a in H1s:
        t = torch.full((n, ld), float("nan"), dtype=torch.float32, device="cuda")
        t[:, :n] = torch.from_numpy(a).cuda()
        H1buf.append(t[:, :n])
    out = torch.full((n, ld), -7.0, dtype=torch.float32, device="cuda")[:, :n]
    out1 = [torch.full((n, ld), -7.0, dtype=torch.float32, device="cuda")[:, :n] for _ in range(nb)]
    D, D1s, tr1, r = h.response_batch(Hbuf[:, :n], H1buf, n_occ, out=out, out1s=out1)
    _check(r, ref, D, D1s, tr1, n_occ)
    assert float(out1[1].untyped_storage().nbytes()) > 0 and float(out1[1].as_strided((n, 24), (ld, 1), n).max()) == -7.0
    # trivial occupations: D = 0 / I and every D1_b = 0 (answered from the definition)
    for occ, diag in ((0, 0.0), (n, 1.0)):
        D, D1s, tr1, r = h.response_batch(Hbuf[:, :n], H1buf, occ)
        assert r["status"] == 0 and r["layers"] == 0
        assert float((D - diag * torch.eye(n, device="cuda")).abs().max()) == 0.0
        assert all(float(d.abs().max()) == 0.0 for d in D1s) and tr1 == [0.0] * nb
    h.close()


def test_batch_argument_errors(torch_cuda, sp2):
    torch = torch_cuda
    n = 256
    p = inputs.make_problem(inputs.scaled_config(inputs.CONFIGS[2], n), want_h1=False)
    H = torch.from_numpy(p["H"]).cuda()
    H1s = [torch.from_numpy(a).cuda() for a in inputs.perturbations(n, 3, seed=1)]
    h = sp2.Sp2Handle(n, batch=2)
    with pytest.raises(sp2.Sp2Error) as e:
        h.response_batch(H, H1s, p["n_occ"])                            # workspace was sized for 2
    assert e.value.status == sp2.SP2_ERR_WORKSPACE
    with pytest.raises(sp2.Sp2Error):
        h.response_batch(H, [], p["n_occ"])
    D, D1s, tr1, r = h.response_batch(H, H1s[:2], p["n_occ"])
    assert r["status"] == 0
    h.close()
    h = sp2.Sp2Handle(n)                                                # no response planes at all
    with pytest.raises(sp2.Sp2Error):
        h.response_batch(H, H1s[:1], p["n_occ"])
    h.close()
    # a NaN in the LAST perturbation is caught (every H1_b goes through the non-finite detector)
    h = sp2.Sp2Handle(n, batch=3)
    bad = H1s[2].clone()
    bad[5, 7] = float("nan")
    with pytest.raises(sp2.Sp2Error) as e:
        h.response_batch(H, [H1s[0], H1s[1], bad], p["n_occ"])
    assert e.value.status == sp2.SP2_ERR_NONFINITE
    h.close()


def test_batch_full_size_config4(torch_cuda, sp2):
    """BASELINE.json config 4 (N = 8192, gap 0.05) with 3 perturbations, in the launch configuration
    `bench.py --workload batch` times: sampled entries against the definitions the oracle evaluates one by one."""
    import oracle

    torch = torch_cuda
    p = inputs.make_problem(inputs.CONFIGS[4], device="cuda", want_h1=False)
    n, n_occ, nb = p["n"], p["n_occ"], 3
    H1n = inputs.perturbations(n, nb, seed=4, decades=2.0)
    H = torch.from_numpy(p["H"]).cuda()
    h = sp2.Sp2Handle(n, batch=nb)
    D, D1s, tr1, r = h.response_batch(H, [torch.from_numpy(a).cuda() for a in H1n], n_occ)
    h.close()
    rng = np.random.default_rng(3)
    rows = np.concatenate([rng.integers(0, n, 1500), [0, n - 1, 17]])
    cols = np.concatenate([rng.integers(0, n, 1500), [n - 1, n - 1, 17]])
    ri, ci = torch.from_numpy(rows).cuda(), torch.from_numpy(cols).cuda()
    De = oracle.density_from_eigenpairs(p["Q"], p["lam"], n_occ, rows, cols)
    assert r["status"] == 0 and 35 <= r["layers"] <= 52
    assert np.abs(D[ri, ci].cpu().numpy() - De).max() <= 1e-4
    assert abs(r["tr_d"] - n_occ) <= 1e-3
    E = inputs.band_energy_closed_form(p["lam"], n_occ)
    assert abs(r["tr_dh"] - E) <= 1e-5 * abs(E)
    for b in range(nb):
        want = oracle.response_closed_form_sampled(p["Q"], p["lam"], n_occ, H1n[b], rows, cols)
        s = float(D1s[b].abs().max())
        assert np.abs(D1s[b][ri, ci].cpu().numpy() - want).max() <= 1e-3 * s, b
        assert bool(torch.equal(D1s[b], D1s[b].T))
        assert abs(tr1[b]) <= 1e-3 * s * n ** 0.5                          # particle number conserved to first order


def test_batch_with_lanczos_bounds_and_refinement(torch_cuda, sp2):
    """The options compose: Lanczos bounds (fewer layers) and float64 refinement of D under a batched response."""
    import oracle

    torch = torch_cuda
    n, nb = 384, 3
    p = inputs.make_problem(inputs.scaled_config(inputs.CONFIGS[2], n), want_h1=False)
    n_occ = p["n_occ"]
    H1s = inputs.perturbations(n, nb, seed=21)
    lo, hi = oracle.lanczos_bounds(p["H"], 10)
    ref = oracle.sp2_response_batch(p["H"], n_occ, H1s, bounds=(lo, hi))
    ref_g = oracle.sp2_response_batch(p["H"], n_occ, H1s[:1])
    h = sp2.Sp2Handle(n, batch=nb, refinement=True)
    h.set_options(lanczos_steps=10, refine_layers=2)
    D, D1s, tr1, r = h.response_batch(torch.from_numpy(p["H"]).cuda(), [torch.from_numpy(a).cuda() for a in H1s], n_occ)
    h.close()
    assert r["status"] == 0 and r["refine_layers"] == 2 and r["layers"] <= ref_g["layers"] - 3
    Dn = D.cpu().numpy()
    assert np.abs(Dn - ref["D"]).max() <= 1e-6                        # refined: far inside the 1e-4 bar
    assert np.abs(Dn @ Dn - Dn).max() <= 1e-9
    for b in range(nb):
        assert np.abs(D1s[b].cpu().numpy() - ref["D1"][b]).max() <= 1e-3 * np.abs(ref["D1"][b]).max()
