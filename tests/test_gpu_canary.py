"""Memory-safety net under every kernel (compute-sanitizer is not available on the GPU pool): the workspace and a
guard band either side of it are filled with a sentinel byte BEFORE sp2_create; after each kind of call the library
reports, per carved region, how many bytes that call was entitled to write (sp2_debug_layout: computed from the launch
geometry, not from the allocation formulas), and every other byte must still hold the sentinel:

    used <= reserved for every region,  tails of the regions, the padding between them and the guard bands untouched.

Sizes cover npad = 256 (where the round-1 slot array was 256 B short for a response solve: the layer kernel writes one
slot per CTA and class, the layout had kept a per-tile formula), ragged sizes, several tiles, both cta_group code
paths, and every entry point: density, response, batch(8), congruence, refinement, sequence, host buffers, the SIMT
scaffold, Lanczos and power-trace bounds and the trivial occupations.  Results are also checked (status, trace), so a kernel that
stays in bounds by doing nothing does not pass.
"""
import numpy as np
import pytest

from paper_2107_02737_b200 import inputs

pytestmark = pytest.mark.gpu

SENTINEL = 0xA5


def _assert_clean(h, what):
    bad = h.check_canary()
    assert not bad, f"after {what}: " + "; ".join(bad[:4])


@pytest.mark.parametrize("n", [2, 77, 256, 300, 641, 1100])
def test_workspace_canary_every_entry_point(torch_cuda, sp2, n):
    torch = torch_cuda
    n_occ = max(1, n // 2)
    cfg = inputs.Sp2Config("canary", 2, n, n_occ, (-1.5, -0.25), (0.25, 1.5), "f64", True)
    p = inputs.make_problem(cfg, want_h1=True)
    H = torch.from_numpy(p["H"]).cuda()
    H1s = [torch.from_numpy(a).cuda() for a in inputs.perturbations(n, 8, seed=3)]
    h = sp2.Sp2Handle(n, batch=8, host_staging=True, refinement=True, sentinel=SENTINEL)
    _assert_clean(h, "sp2_create")
    for cg in (1, 2):
        h.set_options()                                    # defaults: options persist across set_options(**kw) calls
        h.set_options(cta_group=cg)
        D, r = h.density(H, n_occ)
        assert r["status"] == 0 and abs(r["tr_d"] - n_occ) <= 1e-3, r
        _assert_clean(h, f"density cta_group={cg}")
        D, D1, r = h.response(H, H1s[0], n_occ)
        assert r["status"] == 0 and abs(r["tr_d"] - n_occ) <= 1e-3, r
        _assert_clean(h, f"response cta_group={cg}")
        for nb in (3, 8):
            D, D1b, tr1, r = h.response_batch(H, H1s[:nb], n_occ)
            assert r["status"] == 0 and len(D1b) == nb
            _assert_clean(h, f"batch({nb}) cta_group={cg}")
        C = h.congruence(H1s[1], H)
        assert bool(torch.isfinite(C).all())
        _assert_clean(h, f"congruence cta_group={cg}")
        h.set_options(cta_group=cg, refine_layers=2)
        D, r = h.density(H, n_occ)
        assert r["status"] == 0 and r["refine_layers"] == 2 and abs(r["tr_d"] - n_occ) <= 1e-6
        _assert_clean(h, f"refinement cta_group={cg}")
        h.set_options(cta_group=cg, refine_layers=0, lanczos_steps=8)
        D, r = h.density(H, n_occ)
        assert r["status"] == 0 and abs(r["tr_d"] - n_occ) <= 1e-3, r
        _assert_clean(h, f"lanczos cta_group={cg}")
        h.set_options(cta_group=cg, lanczos_steps=0, power_squarings=3)
        D, D1, r = h.response(H, H1s[0], n_occ)
        assert r["status"] == 0 and abs(r["tr_d"] - n_occ) <= 1e-3, r
        _assert_clean(h, f"power-trace bounds cta_group={cg}")
        h.set_options(cta_group=cg, power_squarings=0)
        h.sequence_begin(n, n_occ, n_steps_hint=3)
        Ds = [torch.empty_like(H) for _ in range(3)]
        for Dt in Ds:
            h.sequence_step(H, Dt)
        res = h.sequence_end()
        assert [x["status"] for x in res] == [0, 0, 0]
        _assert_clean(h, f"sequence cta_group={cg}")
    h.set_options()
    Dh, D1h = np.empty((n, n)), np.empty((n, n))
    h.response_host(p["H"], p["H1"], n_occ, Dh, D1h)
    _assert_clean(h, "response_host")
    D, r = h.density(H, 0)
    D, r = h.density(H, n)
    _assert_clean(h, "trivial occupations")
    if n <= 700:
        h.set_options(engine=sp2.SP2_ENGINE_SIMT_DEBUG)
        D, D1, r = h.response(H, H1s[0], n_occ)
        assert r["status"] == 0
        _assert_clean(h, "SIMT scaffold")
    # the bookkeeping itself: every region the calls above use reports a non-zero extent that fits
    lay = {r["name"]: r for r in h.debug_layout()}
    for name in ("plane0", "plane35", "slots", "slots2", "bslots", "fslots", "tiles", "items", "item_begin", "flags", "ctrl",
                 "ring", "staging0", "staging3", "lanczos", "refine0", "refine1", "refine_slots"):
        assert 0 < lay[name]["used"] <= lay[name]["reserved"], name
    h.close()


def test_canary_detects_a_write_outside_the_used_extent(torch_cuda, sp2):
    """The net has no hole where it matters: a stray byte in a region's tail, in a gap or in a guard band is reported."""
    torch = torch_cuda
    n = 256
    p = inputs.make_problem(inputs.Sp2Config("canary", 2, n, n // 2, (-1.5, -0.25), (0.25, 1.5), "f64", True))
    h = sp2.Sp2Handle(n, response=True, sentinel=SENTINEL)
    h.density(torch.from_numpy(p["H"]).cuda(), n // 2)
    assert not h.check_canary()
    lay = {r["name"]: r for r in h.debug_layout()}
    for name in ("slots", "plane4", "scratch"):                     # plane4 = Z.hi: untouched by a density call
        r = lay[name]
        assert r["used"] < r["reserved"]
        pos = h._ws_off + r["offset"] + r["reserved"] - 1
        old = int(h.workspace[pos])
        h.workspace[pos] = 0
        assert any(name in b for b in h.check_canary())
        h.workspace[pos] = old
    h.workspace[0] = 0                                              # guard band
    assert any("guard" in b for b in h.check_canary())
    h.close()


def test_layer_slot_array_fits_every_grid(torch_cuda, sp2):
    """One slot per CTA and product class: (1 + nb) * grid entries at any npad, including npad = 256 with a batch of 8
    (round 1 reserved 136 * (1 + nb) entries there for a grid of 148 CTAs)."""
    for n, nb in ((8, 1), (200, 3), (256, 8), (1000, 8)):
        h = sp2.Sp2Handle(n, batch=nb, sentinel=SENTINEL)
        lay = {r["name"]: r for r in h.debug_layout()}
        sms = torch_cuda.cuda.get_device_properties(0).multi_processor_count
        assert lay["slots"]["reserved"] >= (1 + nb) * sms * 32
        h.close()
