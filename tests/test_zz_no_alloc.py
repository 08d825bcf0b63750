"""ss_render_noalloc (include/ss.h): the allocation-free variant of ss_render -- no handle, no
workspace, scratch in a static device array of the library -- against the existing ss_render path
on the same fields, on two calls in a row.  The kernels and their arithmetic are the same, so
extrema and image agree exactly; the tolerance asserted for the extrema is the one
tests/test_render.py uses (1e-10 relative in fp64).  Collected last (file name) on purpose: the
suite runs with pytest -x."""
import gc

import numpy as np
import pytest
import torch

from paper_2603_24370_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _ss():
    from paper_2603_24370_b200 import ss
    return ss


def _existing(ss, w, fields, obs, strict=True):
    s = ss.solver_for(w)
    s.set_fields(fields[None])
    img, mm = s.render(obs, strict=strict)
    torch.cuda.synchronize()
    return img.cpu().numpy(), mm


def test_no_alloc_render_matches_ss_render_on_two_calls_in_a_row():
    ss = _ss()
    dev = "cuda:0"
    # call 1: a chiral-magnet lattice with one non-finite interior value (sets the scratch flag and
    # leaves 2 * 251 block partials behind); call 2: a smaller, clean Abelian-Higgs lattice, which
    # must see a cleared flag and none of call 1's partials
    w1 = W.cm_multi(N=250, count=3, margin=12.0, min_sep=14.0)
    f1 = w1.fields[0].copy()
    f1[2, 100, 57] = np.nan
    w2 = W.ah_vortices(N=150, h=0.1, lam=1.0, count=2, min_sep=2.0)
    f2 = w2.fields[0]
    d1 = torch.from_numpy(f1).to(dev)
    d2 = torch.from_numpy(f2).to(dev)
    # every output is the caller's, created before the calls
    mm = torch.zeros(2, 2, dtype=torch.float64, device=dev)
    flag = torch.full((2,), -1, dtype=torch.int32, device=dev)
    img1 = torch.zeros(w1.Ny, w1.Nx, 4, dtype=torch.uint8, device=dev)
    img2 = torch.zeros(w2.Ny, w2.Nx, 4, dtype=torch.uint8, device=dev)
    for obs in (ss.OBS_ENERGY, ss.OBS_CHARGE, ss.OBS_ORDER):
        # warm call (module load, address look-up: "one call per device before capturing"), then
        # nothing may be allocated: neither through torch nor on the device at all.  Objects of
        # earlier tests are collected first so that their release does not fall into the window.
        ss.render_noalloc(w1.theory, w1.h, d1, mm[0], rgba=img1, observable=obs, kappa=w1.kappa)
        ss.render_noalloc(w2.theory, w2.h, d2, mm[1], rgba=img2, observable=obs, lam=w2.lam)
        gc.collect()
        torch.cuda.synchronize()
        before = torch.cuda.memory_allocated(dev)
        free_before = torch.cuda.mem_get_info(dev)[0]
        ss.render_noalloc(w1.theory, w1.h, d1, mm[0], rgba=img1, nonfinite=flag[0:1], observable=obs,
                          kappa=w1.kappa, B=w1.B, K=w1.K)
        ss.render_noalloc(w2.theory, w2.h, d2, mm[1], rgba=img2, nonfinite=flag[1:2], observable=obs,
                          lam=w2.lam)
        torch.cuda.synchronize()
        assert torch.cuda.memory_allocated(dev) <= before
        assert torch.cuda.mem_get_info(dev)[0] >= free_before
        assert flag.tolist() == [1, 0]
        for w, f, img, k in ((w1, d1, img1, 0), (w2, d2, img2, 1)):
            want_img, (mn, mx) = _existing(ss, w, f, obs, strict=False)
            scale = max(abs(mn), abs(mx), 1e-300)
            got = mm[k].tolist()
            assert abs(got[0] - mn) <= 1e-10 * scale and abs(got[1] - mx) <= 1e-10 * scale
            assert (img.cpu().numpy() == want_img).all()
    # extrema only (no image), repeated: same numbers
    mm3 = torch.zeros(2, dtype=torch.float64, device=dev)
    ss.render_noalloc(w2.theory, w2.h, d2, mm3, observable=ss.OBS_ORDER, lam=w2.lam)
    torch.cuda.synchronize()
    assert mm3.tolist() == mm[1].tolist()


def test_no_alloc_render_rejects_sizes_beyond_the_maximum_and_bad_arguments():
    ss = _ss()
    dev = "cuda:0"
    mm = torch.zeros(2, dtype=torch.float64, device=dev)
    N = 2050                                        # 2050^2 > SS_NOALLOC_MAX_SITES = 2048^2
    assert N * N > ss.NOALLOC_MAX_SITES
    big = torch.zeros(3, N, N, dtype=torch.float64, device=dev)
    with pytest.raises(ss.SSError) as e:
        ss.render_noalloc(ss.THEORY_CHIRAL_MAGNET, 0.2, big, mm, kappa=1.0, B=0.6)
    assert e.value.code == ss.ERR_TOO_LARGE and "SS_NOALLOC_MAX_SITES" in str(e.value)
    ok = torch.zeros(3, 2048, 2048, dtype=torch.float64, device=dev)   # the maximum itself
    ok[2] = 1.0
    ss.render_noalloc(ss.THEORY_CHIRAL_MAGNET, 0.2, ok, mm, observable=ss.OBS_ORDER, kappa=1.0, B=0.6)
    torch.cuda.synchronize()
    assert mm.tolist() == [1.0, 1.0]
    small = torch.zeros(3, 64, 64, dtype=torch.float64, device=dev)
    with pytest.raises(ss.SSError) as e:
        ss.render_noalloc(ss.THEORY_CHIRAL_MAGNET, 0.2, small, mm, observable=3)
    assert e.value.code == ss.ERR_ARG
    with pytest.raises(ss.SSError) as e:
        ss.render_noalloc(ss.THEORY_CHIRAL_MAGNET, 0.0, small, mm)
    assert e.value.code == ss.ERR_ARG
