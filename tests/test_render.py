"""Headless visualisation (DESIGN R17).  The colour map is our own definition
(the paper gives none: parity of the map itself is unpinned); what IS pinned: the observables are
the oracle's pinned site densities, the extrema are exact, and the CPU restatement of the map
satisfies the properties a linear 5-stop map must have."""
import numpy as np
import pytest

import oracle
from paper_2603_24370_b200 import workloads as W


def test_colormap_properties_cpu():
    v = np.full((9, 11), np.nan)
    v[2:-2, 2:-2] = np.linspace(-3.0, 5.0, 5 * 7).reshape(5, 7)
    img, (mn, mx) = oracle.colormap(v)
    assert (mn, mx) == (-3.0, 5.0)
    assert (img[0, 0] == 0).all() and (img[4, 4, 3] == 255)          # halo transparent
    assert tuple(img[2, 2, :3]) == (0, 0, 128)                        # t = 0: first stop
    assert tuple(img[-3, -3, :3]) == (128, 0, 0)                      # t = 1: last stop
    mid = np.full((5, 5), np.nan)
    mid[2, 2] = 7.0                                                    # max == min -> t = 1/2
    assert tuple(oracle.colormap(mid)[0][2, 2, :3]) == (255, 255, 255)
    # monotone: red never decreases and blue never increases over the first three stops
    ramp = np.full((5, 1000 + 4), np.nan)
    ramp[2, 2:-2] = np.linspace(0.0, 1.0, 1000)
    rgb = oracle.colormap(ramp)[0][2, 2:-2, :3].astype(int)
    assert (np.diff(rgb[:500, 0]) >= 0).all() and (np.diff(rgb[500:, 2]) <= 0).all()
    assert np.abs(np.diff(rgb, axis=0)).max() <= 2                     # continuous


@pytest.mark.gpu
@pytest.mark.parametrize("case", ["cm", "ah", "cm_f32"])
def test_render_matches_cpu_restatement(case):
    import torch
    from paper_2603_24370_b200 import ss
    if case == "ah":
        w = W.ah_vortices(N=150, h=0.1, lam=1.0, count=2, min_sep=2.0)
    else:
        w = W.cm_multi(N=252 if case == "cm_f32" else 250, count=3, margin=12.0, min_sep=14.0)
    f32 = case == "cm_f32"
    s = ss.solver_for(w, dtype=ss.F32 if f32 else ss.F64)
    s.set_fields(torch.from_numpy(w.fields).to("cuda:0", dtype=torch.float32 if f32 else torch.float64))
    s.step(7)
    fl = oracle.Flow(oracle.model(w.theory, w.Nx, w.Ny, w.h, kappa=w.kappa, B=w.B, K=w.K,
                                  lam=w.lam), w.dt)
    fl.set_fields(w.fields[0])
    fl.step(7)
    phi = fl.get_fields()[0]
    for obs in (ss.OBS_ENERGY, ss.OBS_CHARGE, ss.OBS_ORDER):
        img, (mn, mx) = s.render(obs)
        vals = oracle.observable(fl.m, phi, obs)
        want, (omn, omx) = oracle.colormap(vals)
        tol = 1e-4 if f32 else 1e-10
        scale = max(abs(omn), abs(omx), 1e-300)
        assert abs(mn - omn) <= tol * scale and abs(mx - omx) <= tol * scale
        got = img.cpu().numpy()
        assert (got[..., 3] == want[..., 3]).all()                    # same halo mask
        diff = np.abs(got[..., :3].astype(int) - want[..., :3].astype(int))
        if f32:
            assert diff.max() <= 2
        else:
            # a byte flips only where x + 0.5 sits within rounding of an integer
            assert diff.max() <= 1 and (diff > 0).mean() < 1e-3
    fields_after = s.get_fields()[0].cpu().numpy()[0]
    s.step(3)                                                          # rendering left the flow alone
    fl.step(3)
    assert fields_after.shape == phi.shape
    if not f32:
        assert np.abs(s.get_fields()[0].cpu().numpy()[0] - fl.get_fields()[0]).max() <= 1e-11


@pytest.mark.gpu
def test_render_marks_non_finite_interior_values():
    # a NaN at an interior site is not the halo: it is drawn opaque magenta, stays out of the
    # extrema, and the call reports SS_ERR_NONFINITE; the halo is found by position
    import torch
    from paper_2603_24370_b200 import ss
    w = W.cm_single(N=64)
    f = w.fields.copy()
    f[0, 2, 30, 17] = np.nan
    s = ss.solver_for(w)
    s.set_fields(torch.from_numpy(f).to("cuda:0"))
    with pytest.raises(ss.SSError) as e:
        s.render(ss.OBS_ORDER)
    assert e.value.code == ss.ERR_NONFINITE
    img, (mn, mx) = s.render(ss.OBS_ORDER, strict=False)
    got = img.cpu().numpy()
    assert tuple(got[30, 17]) == (255, 0, 255, 255)
    ok = np.isfinite(f[0, 2]) & W.interior_mask(64, 64)
    assert (mn, mx) == (f[0, 2][ok].min(), f[0, 2][ok].max())
    assert (got[~W.interior_mask(64, 64)] == 0).all() and (got[ok][:, 3] == 255).all()
    vals = np.where(ok, f[0, 2], np.nan)
    want, _ = oracle.colormap(vals)
    assert (got[ok] == want[ok]).all()
