"""Parity of the baby-Skyrme CUDA path (tile kernels of csrc/ss_bs.cuh, through the C ABI) with the
CPU oracle on the same seeded inputs, at the chiral-magnet tolerances of BASELINE.json: fp64
fields max-abs <= 1e-11 over the first 100 steps with identical arrest indices, E and Q within
1e-9 relative, fp32 energy within 1e-4 (SURVEY 8(f) NEXT-2b; DESIGN R18)."""
import numpy as np
import pytest
import torch

import oracle
from paper_2603_24370_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _ss():
    from paper_2603_24370_b200 import ss
    return ss


def _model(w):
    return oracle.model(oracle.BS, w.Nx, w.Ny, w.h, kappa=w.kappa, mu=w.mu, pot=w.pot, potN=w.potN)


def _floor(m, phi, E):
    _, _, de, _ = oracle.energy_charge(m, phi, densities=True)
    return max(abs(E), m.h * m.h * float(np.abs(de).sum()), 1e-300)


def _dev(a, dtype=torch.float64):
    return torch.from_numpy(np.ascontiguousarray(a)).to("cuda:0", dtype=dtype).contiguous()


def _ragged(w, Ny):
    """keep the first Ny rows of a square workload and restore the vacuum halo at the new edge"""
    f = w.fields[:, :, :Ny, :].copy()
    f[:, :, ~W.interior_mask(w.Nx, Ny)] = np.array([0.0, 0.0, 1.0])[None, :, None]
    w.fields, w.Ny = f, Ny
    return w


def _run(w, checkpoints, flags=0, integrator="rk4"):
    ss = _ss()
    s = ss.solver_for(w, flags=flags, integrator=ss.VERLET if integrator == "verlet" else ss.RK4)
    s.set_fields(_dev(w.fields))
    flows = []
    for b in range(w.batch):
        fl = oracle.Flow(_model(w), w.dt, integrator=integrator)
        fl.set_fields(w.fields[b])
        flows.append(fl)
        f0 = _floor(fl.m, w.fields[b], fl.energy)
        assert abs(s.energy()[b] - fl.energy) <= 1e-12 * f0
        assert abs(s.charge()[b] - fl.charge) <= 1e-12 * max(1.0, abs(fl.charge))
    done = 0
    for cp in checkpoints:
        s.step(cp - done)
        phi, vel = s.get_fields()
        E, Q, KE = s.energy(), s.charge(), s.kinetic()
        phi, vel = phi.cpu().numpy(), vel.cpu().numpy()
        for b, fl in enumerate(flows):
            fl.step(cp - done)
            ophi, ovel = fl.get_fields()
            assert np.abs(phi[b] - ophi).max() <= 1e-11, (cp, b)
            assert np.abs(vel[b] - ovel).max() <= 1e-10, (cp, b)
            sc = fl.scalars()
            f_ = _floor(fl.m, ophi, sc["E"])
            assert abs(E[b] - sc["E"]) <= 1e-9 * f_, (cp, b)
            assert abs(Q[b] - sc["Q"]) <= 1e-9 * max(1.0, abs(sc["Q"])), (cp, b)
            assert abs(KE[b] - sc["KE"]) <= 1e-9 * max(f_, sc["KE"]), (cp, b)
            got, cnt = s.arrests(b)
            assert got == fl.arrests() and cnt == sc["n_arrests"], (cp, b)
        done = cp
    return s, flows


@pytest.mark.parametrize("pot,potN", [(W.POT_STANDARD, 3), (W.POT_EASY_PLANE, 3), (W.POT_BROKEN, 3)])
def test_bs_first_100_steps_on_a_ragged_lattice(pot, potN):
    # 150 x 134: ragged against the 64 x 16 tiles in x and y; the first arrests fall in the window
    w = _ragged(W.bs_single(N=150, pot=pot, potN=potN), 134)
    s, flows = _run(w, (1, 2, 5, 10, 20, 50, 100))
    assert len(flows[0].arrests()) >= 1
    phi = s.get_fields(want_vel=False)
    assert float(((phi * phi).sum(1) - 1.0).abs().max()) < 1e-14


@pytest.mark.parametrize("pot", [W.POT_STANDARD, W.POT_BROKEN])
def test_bs_verlet_first_100_steps(pot):
    # the one-gradient-per-step integrator (DESIGN R15) through the stage-5 tile kernel
    w = _ragged(W.bs_single(N=150, pot=pot), 134)
    s, flows = _run(w, (1, 2, 5, 10, 20, 50, 100), integrator="verlet")
    assert len(flows[0].arrests()) >= 1
    w = W.bs_single(N=96, count=2, batch=2, kappa=0.8, mu=0.7)
    _run(w, (1, 5, 20), integrator="verlet")


def test_bs_batched_multi_skyrmion_and_smallest_lattices():
    w = W.bs_single(N=140, count=3, batch=2, kappa=0.8, mu=0.7)
    s, flows = _run(w, (1, 2, 5, 10, 20, 50))
    assert abs(flows[0].charge + 3.0) < 2e-2
    for Nx, Ny in ((6, 5), (10, 9), (8, 12)):
        rng = np.random.default_rng(Nx * 10 + Ny)
        f = rng.standard_normal((1, 3, Ny, Nx))
        f /= np.sqrt((f * f).sum(1, keepdims=True))
        w = W.Workload("tiny", W.BS, Nx, Ny, 0.2, 0.02, kappa=0.5, mu=1.0, fields=f)
        _run(w, (1, 2, 5))


def test_bs_vacuum_graph_vs_direct_and_unsupported():
    ss = _ss()
    vac = np.zeros((1, 3, 40, 70))
    vac[0, 2] = 1.0
    w = W.Workload("vac", W.BS, 70, 40, 0.2, 0.1, kappa=1.0, mu=1.0, pot=W.POT_BROKEN, fields=vac)
    s = ss.solver_for(w)
    s.set_fields(_dev(vac))
    s.step(3)
    assert s.energy() == [0.0] and s.charge() == [0.0] and s.kinetic() == [0.0]
    assert torch.equal(s.get_fields(want_vel=False).cpu(), torch.from_numpy(vac))
    w = W.bs_single(N=96)
    outs = []
    for flags in (0, ss.FLAG_NO_GRAPH):
        s = ss.solver_for(w, flags=flags)
        s.set_fields(_dev(w.fields))
        s.step(37)
        f, v = s.get_fields()
        outs.append((f.cpu(), v.cpu(), s.energy(), s.charge(), s.arrests(0)))
    assert torch.equal(outs[0][0], outs[1][0]) and torch.equal(outs[0][1], outs[1][1])
    assert outs[0][2:] == outs[1][2:]
    w.dmi = W.DMI_NEEL
    with pytest.raises(ss.SSError) as e:
        ss.solver_for(w)                                  # no DMI table in this theory
    assert e.value.code == ss.ERR_UNSUPPORTED
    with pytest.raises(ss.SSError) as e:
        ss.Solver(ss.THEORY_BABY_SKYRME, 64, 64, 0.2, pot=7)
    assert e.value.code == ss.ERR_ARG


def test_bs_fp32_energy_within_1e4_and_render():
    ss = _ss()
    w = W.bs_single(N=128)
    s = ss.solver_for(w, dtype=ss.F32)
    s.set_fields(_dev(w.fields, torch.float32))
    fl = oracle.Flow(_model(w), w.dt)
    fl.set_fields(w.fields[0])
    for _ in range(4):
        s.step(50)
        fl.step(50)
        phi = fl.get_fields()[0]
        assert abs(s.energy()[0] - fl.energy) <= 1e-4 * _floor(fl.m, phi, fl.energy)
    assert abs(s.charge()[0] - fl.charge) < 1e-4
    s = ss.solver_for(w)
    s.set_fields(_dev(w.fields))
    s.step(5)
    fl = oracle.Flow(_model(w), w.dt)
    fl.set_fields(w.fields[0])
    fl.step(5)
    for obs in (ss.OBS_ENERGY, ss.OBS_CHARGE, ss.OBS_ORDER):
        img, (mn, mx) = s.render(obs)
        want, (omn, omx) = oracle.colormap(oracle.observable(fl.m, fl.get_fields()[0], obs))
        scale = max(abs(omn), abs(omx))
        assert abs(mn - omn) <= 1e-10 * scale and abs(mx - omx) <= 1e-10 * scale
        diff = np.abs(img.cpu().numpy()[..., :3].astype(int) - want[..., :3].astype(int))
        assert diff.max() <= 1 and (diff > 0).mean() < 1e-3


def test_bs_2048_full_size_three_steps():
    # the size bench.py times (bs2048_f64), element by element against the oracle
    w = W.bs_bench()
    _run(w, (1, 3))
