"""GPU: sp2_density_noalloc (include/sp2.h), the entry point that allocates nothing.

Its scratch is a file-scope `static __device__` array inside the library instead of the caller's workspace; the kernel
is the one-CTA solve the handle path uses for N <= 128.  Checked here against that existing path (Sp2Handle.density,
default options) on the same seeded inputs, on consecutive calls that share the static array, within the tolerances of
tests/test_gpu_parity.py, and once against the float64 oracle.

The file name sorts last on purpose: the suite runs with `pytest -x`, and a failure here must not hide other tests.
"""
import numpy as np
import pytest

from paper_2107_02737_b200 import inputs

pytestmark = pytest.mark.gpu

TOL_D, TOL_TR, TOL_E = 1e-4, 1e-3, 1e-5          # BASELINE.json north_star, as in test_gpu_parity.py


@pytest.fixture(scope="module")
def torch_mod():
    import torch

    assert torch.cuda.is_available()
    return torch


@pytest.fixture(scope="module")
def sp2(torch_mod):
    from paper_2107_02737_b200 import sp2 as mod   # raises if libsp2_b200.so is missing: no fallback

    return mod


def _existing_path(sp2, torch, p):
    h = sp2.Sp2Handle(p["n"])
    D, r = h.density(torch.from_numpy(p["H"]).cuda(), p["n_occ"])
    out = D.cpu().numpy().astype(np.float64)
    h.close()
    return out, r


def _compare(D, r, D_ref, r_ref, n_occ):
    assert r["status"] == 0 and r_ref["status"] == 0
    assert np.abs(D - D_ref).max() <= TOL_D
    assert abs(r["tr_d"] - n_occ) <= TOL_TR
    assert abs(r["tr_dh"] - r_ref["tr_dh"]) <= TOL_E * abs(r_ref["tr_dh"])
    assert np.array_equal(D, D.T)                                      # bit-symmetric, like the handle path
    assert r["layers"] == r_ref["layers"] and r["signs"] == r_ref["signs"]
    assert r["eps_min"] == r_ref["eps_min"] and r["eps_max"] == r_ref["eps_max"]
    assert r["kernel_launches"] == 1


def test_noalloc_matches_the_handle_path_on_consecutive_calls(sp2, torch_mod):
    import oracle

    torch = torch_mod
    assert sp2.noalloc_max_n() == 128
    assert 0 < sp2.noalloc_scratch_bytes() <= 160 * 1024               # the "modest maximum" include/sp2.h states
    # two different problems back to back (the second call finds the first one's state in the shared scratch), then
    # the first one again: config 1 (N = 128, f64), a ragged f32 case with its own pitch, config 1 again
    pa = inputs.make_problem(inputs.CONFIGS[1])
    pb = inputs.make_problem(inputs.scaled_config(inputs.CONFIGS[3], 77))
    ref_a, ref_b = _existing_path(sp2, torch, pa), _existing_path(sp2, torch, pb)
    Ha = torch.from_numpy(pa["H"]).cuda()
    Hb_store = torch.zeros((77, 96), dtype=torch.float32, device="cuda")
    Hb = Hb_store[:, :77]
    Hb.copy_(torch.from_numpy(pb["H"]))
    Da, Da2 = torch.empty_like(Ha), torch.empty_like(Ha)
    Db = torch.empty((77, 77), dtype=torch.float32, device="cuda")
    d_res = torch.zeros(256, dtype=torch.uint8, device="cuda")
    sp2.density_noalloc(Ha, pa["n_occ"], out=torch.empty_like(Ha))    # first call on the device: one-time set-up
    sp2.density_noalloc(Hb, pb["n_occ"], out=torch.empty_like(Db))    # (and the lazy load of both kernel variants)
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]

    _, ra = sp2.density_noalloc(Ha, pa["n_occ"], out=Da)
    _, rb = sp2.density_noalloc(Hb, pb["n_occ"], out=Db)
    _, ra2 = sp2.density_noalloc(Ha, pa["n_occ"], out=Da2)
    # asynchronous form: nothing comes back to the host, the status lands in the caller's device buffer
    Da3 = torch.full_like(Ha, 7.0)
    sp2.density_noalloc(Ha, pa["n_occ"], out=Da3, d_result=d_res, blocking=False)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free_before                 # no device memory was taken by these calls

    _compare(Da.cpu().numpy(), ra, ref_a[0], ref_a[1], pa["n_occ"])
    _compare(Db.cpu().numpy().astype(np.float64), rb, ref_b[0], ref_b[1], pb["n_occ"])
    _compare(Da2.cpu().numpy(), ra2, ref_a[0], ref_a[1], pa["n_occ"])
    assert torch.equal(Da, Da2) and torch.equal(Da, Da3)               # no state leaks from one call into the next
    assert ra["tr_dh"] == ra2["tr_dh"]
    assert int(d_res[:4].cpu().numpy().view(np.int32)[0]) == 0         # sp2_result_t.status of the asynchronous call
    # the same kernel with the same inputs: the existing path's result bit for bit
    assert np.array_equal(Da.cpu().numpy(), ref_a[0])
    # and the paper's definition: the float64 oracle
    ref = oracle.sp2_density(pa["H"].astype(np.float64), pa["n_occ"])
    assert np.abs(Da.cpu().numpy() - ref["D"]).max() <= TOL_D
    assert abs(ra["tr_dh"] - ref["tr_dh"]) <= TOL_E * abs(ref["tr_dh"])


def test_noalloc_rejects_what_it_cannot_hold(sp2, torch_mod):
    torch = torch_mod
    H = torch.eye(129, dtype=torch.float64, device="cuda")
    D = torch.full_like(H, 3.0)
    with pytest.raises(sp2.Sp2Error) as e:
        sp2.density_noalloc(H, 5, out=D)
    assert e.value.status == sp2.SP2_ERR_TOO_LARGE and "static scratch" in str(e.value)
    torch.cuda.synchronize()
    assert bool((D == 3.0).all())                                      # nothing was launched
    H = torch.diag(torch.arange(8, dtype=torch.float64, device="cuda"))
    D = torch.empty_like(H)
    for n_occ in (0, 8, -1):                                           # the trivial projectors need no solve: rejected
        with pytest.raises(sp2.Sp2Error) as e:
            sp2.density_noalloc(H, n_occ, out=D)
        assert e.value.status == sp2.SP2_ERR_INVALID_ARG
    _, r = sp2.density_noalloc(H, 3, out=D)                            # closed form: projector on the 3 lowest levels
    assert r["status"] == 0
    want = np.diag([1.0, 1.0, 1.0, 0, 0, 0, 0, 0])
    assert np.abs(D.cpu().numpy() - want).max() <= TOL_D
