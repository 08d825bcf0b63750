"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times (default
flags: per-step CUDA graph, automatic segmentation).  The oracle runs the same seeded full-size
input for a few steps (seconds on the box's host cores); fields are compared element by element,
E / Q / KE through the canonical tree, arrest logs exactly.  Properties that hold at any size
(|n| = 1, frozen halo, tangent velocity) are checked on the GPU result as well."""
import numpy as np
import pytest
import torch

import oracle
from paper_2603_24370_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _ss():
    from paper_2603_24370_b200 import ss
    return ss


def _floor(m, phi, E):
    _, _, de, _ = oracle.energy_charge(m, phi, densities=True)
    return max(abs(E), m.h * m.h * float(np.abs(de).sum()), 1e-300)


def _check(w, steps, lattices=(0,), dtype=None, field_tol=1e-11, integrator="rk4", vel0=None):
    ss = _ss()
    s = ss.solver_for(w, integrator=ss.VERLET if integrator == "verlet" else ss.RK4)
    s.set_fields(torch.from_numpy(w.fields).to("cuda:0"),
                 None if vel0 is None else torch.from_numpy(vel0).to("cuda:0"))
    s.step(steps)
    phi, vel = s.get_fields()
    E, Q, KE = s.energy(), s.charge(), s.kinetic()
    assert s.status()["steps"] == steps
    mask = torch.from_numpy(~W.interior_mask(w.Nx, w.Ny)).to("cuda:0")
    for b in lattices:
        B = w.B if w.B_batch is None else float(w.B_batch[b])
        m = oracle.model(w.theory, w.Nx, w.Ny, w.h, kappa=w.kappa, B=B, K=w.K, lam=w.lam)
        fl = oracle.Flow(m, w.dt, integrator=integrator)
        fl.set_fields(w.fields[b], None if vel0 is None else vel0[b])
        fl.step(steps)
        ophi, ovel = fl.get_fields()
        gp, gv = phi[b].cpu().numpy(), vel[b].cpu().numpy()
        assert np.abs(gp - ophi).max() <= field_tol, b
        assert np.abs(gv - ovel).max() <= 10 * field_tol, b
        sc = fl.scalars()
        f = _floor(m, ophi, sc["E"])
        assert abs(E[b] - sc["E"]) <= 1e-9 * f
        assert abs(Q[b] - sc["Q"]) <= 1e-9 * max(1.0, abs(sc["Q"]))
        assert abs(KE[b] - sc["KE"]) <= 1e-9 * max(f, sc["KE"])
        assert s.arrests(b)[0] == fl.arrests()
        # any-size properties of the GPU result itself
        assert torch.equal(phi[b][:, mask], torch.from_numpy(w.fields[b]).to("cuda:0")[:, mask])
        assert float(vel[b][:, mask].abs().max()) == 0.0
        if w.theory == W.CM:
            inter = ~mask
            n2 = (phi[b] * phi[b]).sum(0)[inter]
            assert float((n2 - 1.0).abs().max()) < 1e-14
            if not s.status()["n_arrests"][b]:
                vn = (phi[b] * vel[b]).sum(0)[inter]
                assert float(vn.abs().max()) < 1e-12
    return s


def test_config4_cm_4096_fp64_full_size():
    _check(W.baseline_config(4), steps=3)


def test_config4_cm_4096_fp64_full_size_with_an_arrested_step():
    # The first arrest of config 4 is step 1226, so the 3-step test above never takes kernel Y's
    # arrested branch (vh = 0, a2 := a1, the skipped TMA boxes) at full size.  Start instead with
    # the uphill velocity v = -0.06 a(phi) (computed by the oracle): step 1 raises the energy, is
    # logged, and step 2 runs the arrested branch on all 4096 x 4096 sites.
    w = W.baseline_config(4)
    m = oracle.model(w.theory, w.Nx, w.Ny, w.h, kappa=w.kappa, B=w.B, K=w.K)
    vel = (-0.06 * oracle.accel(m, w.fields[0]))[None]
    s = _check(w, steps=3, vel0=vel)
    assert s.arrests(0)[0][:1] == [1]


def test_config4_cm_4096_full_size_verlet():
    _check(W.baseline_config(4), steps=4, integrator="verlet")


def test_config2_cm_1024_full_size():
    _check(W.baseline_config(2), steps=10)


def test_config3_ah_2048_full_size():
    _check(W.baseline_config(3), steps=3)


def test_config5_sweep_256x256_full_size_sampled_lattices():
    # all 256 lattices advance on the GPU; the oracle checks a sample of them one by one
    _check(W.baseline_config(5), steps=20, lattices=(0, 101, 255))


def test_config4_fp32_full_size_energy():
    ss = _ss()
    w = W.baseline_config(4)
    s = ss.solver_for(w, dtype=ss.F32)
    s.set_fields(torch.from_numpy(w.fields).to("cuda:0", dtype=torch.float32))
    m = oracle.model(w.theory, w.Nx, w.Ny, w.h, kappa=w.kappa, B=w.B, K=w.K)
    fl = oracle.Flow(m, w.dt)
    fl.set_fields(w.fields[0])
    s.step(3)
    fl.step(3)
    f = _floor(m, fl.get_fields()[0], fl.energy)
    assert abs(s.energy()[0] - fl.energy) <= 1e-4 * f
    assert abs(s.charge()[0] - fl.charge) <= 1e-4 * max(1.0, abs(fl.charge))
