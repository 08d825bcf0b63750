"""Demagnetisation on the GPU (csrc/ss_demag.cuh: multigrid Poisson solve inside the
one-gradient-per-step flow; eq. (5), :199-205 eq. (6); DESIGN R19; SURVEY 8(f)
NEXT-4) against the oracle, whose potential is an exact (conjugate-gradient) solve.

Tolerance: the device solves psi by a FIXED number of warm-started V-cycles (no host sync), so it
carries an algebraic error the exact oracle does not have.  Measured contraction per V-cycle:
0.26-0.28 for every lattice size (even and odd levels).  With 24 cycles per step that error is
below 1e-13 of psi; the tests use the chiral-magnet tolerances loosened by one decade (fields
1e-10, velocities and E, Q 1e-9).  The default of 8 cycles is chosen for throughput and tracks the
exact solve to ~1e-7 in the fields, ~1e-6 in the energy (asserted below)."""
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
    return oracle.model(oracle.CM, w.Nx, w.Ny, w.h, kappa=w.kappa, B=w.B, K=w.K, dmi=w.dmi,
                        demag=w.demag)


def _floor(m, phi, E):
    _, _, de, _ = oracle.energy_charge(m, phi, densities=True)
    return max(abs(E), m.h * m.h * float(np.abs(de).sum()), 1e-300)


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).to("cuda:0")


def _run(w, checkpoints, cycles, ftol, etol, integrator="verlet"):
    ss = _ss()
    s = ss.solver_for(w, integrator=ss.VERLET if integrator == "verlet" else ss.RK4,
                      demag_cycles=cycles)
    s.set_fields(_dev(w.fields))
    fl = oracle.Flow(_model(w), w.dt, integrator=integrator)
    fl.set_fields(w.fields[0])
    f0 = _floor(fl.m, w.fields[0], fl.energy)
    assert abs(s.energy()[0] - fl.energy) <= etol * f0
    done, worst = 0, 0.0
    for cp in checkpoints:
        s.step(cp - done)
        fl.step(cp - done)
        done = cp
        phi, vel = s.get_fields()
        ophi, ovel = fl.get_fields()
        d = np.abs(phi.cpu().numpy()[0] - ophi).max()
        worst = max(worst, d)
        assert d <= ftol, (cp, d)
        assert np.abs(vel.cpu().numpy()[0] - ovel).max() <= 10 * ftol, cp
        sc = fl.scalars()
        f_ = _floor(fl.m, ophi, sc["E"])
        assert abs(s.energy()[0] - sc["E"]) <= etol * f_, cp
        assert abs(s.charge()[0] - sc["Q"]) <= etol * max(1.0, abs(sc["Q"])), cp
        assert abs(s.kinetic()[0] - sc["KE"]) <= etol * max(f_, sc["KE"]), cp
        assert s.arrests(0)[0] == fl.arrests(), cp
    return s, fl, worst


@pytest.mark.parametrize("dmi", [None, "neel"])
def test_demag_verlet_parity_on_a_ragged_lattice(dmi):
    # 150 x 134: several multigrid levels with odd sizes (146 -> 73 -> 37 -> 19), ragged tiles
    w = W.cm_single(N=150, K=0.1)
    f = w.fields[:, :, :134, :].copy()
    f[:, :, ~W.interior_mask(150, 134)] = np.array([0.0, 0.0, 1.0])[None, :, None]
    w.fields, w.Ny = f, 134
    w.demag = 0.8
    if dmi:
        w.dmi = W.DMI_NEEL
    s, fl, _ = _run(w, (1, 2, 5, 10, 20, 50, 100), cycles=24, ftol=1e-10, etol=1e-9)
    assert len(fl.arrests()) >= 1
    psi = oracle.demag_potential(fl.m, fl.get_fields()[0])
    assert np.abs(psi).max() > 1e-2                      # the term is not negligible here


@pytest.mark.parametrize("dmi", [None, "neel"])
def test_demag_rk4_parity_one_solve_per_stage(dmi):
    # the paper's integrator with the demagnetising field: four Poisson solves per
    # step (stage fields 2, 3, 4 and the new field), 146 x 130 unknowns (odd multigrid levels)
    w = W.cm_single(N=150, K=0.1)
    f = w.fields[:, :, :134, :].copy()
    f[:, :, ~W.interior_mask(150, 134)] = np.array([0.0, 0.0, 1.0])[None, :, None]
    w.fields, w.Ny = f, 134
    w.demag = 0.8
    if dmi:
        w.dmi = W.DMI_NEEL
    s, fl, _ = _run(w, (1, 2, 5, 10, 20, 50), cycles=24, ftol=1e-10, etol=1e-9, integrator="rk4")
    assert s.schedule() != "resident-cluster" and len(fl.arrests()) >= 1


def test_default_cycle_count_tracks_the_exact_solve_to_1e7():
    w = W.cm_single(N=128)
    w.demag = 1.0
    w.dmi = W.DMI_NEEL
    _, _, worst = _run(w, (10, 50), cycles=0, ftol=2e-7, etol=2e-6)
    print("default cycles: worst field difference", worst)
    assert worst > 0.0


def test_demag_zero_coupling_equals_plain_verlet_and_unsupported_combinations():
    ss = _ss()
    w = W.cm_single(N=64)
    w.demag = 0.5
    with pytest.raises(ss.SSError) as e:
        ss.solver_for(w, integrator=ss.VERLET, dtype=ss.F32)
    assert e.value.code == ss.ERR_UNSUPPORTED
    with pytest.raises(ss.SSError) as e:
        ss.Solver(0, 64, 64, 0.2, demag=-1.0, integrator=ss.VERLET)
    assert e.value.code == ss.ERR_ARG
    # a tiny coupling changes nothing visible: the demag path reproduces the plain kernels
    a = ss.solver_for(W.cm_single(N=64), integrator=ss.VERLET)
    w.demag = 1e-300
    b = ss.solver_for(w, integrator=ss.VERLET)
    for s in (a, b):
        s.set_fields(_dev(w.fields))
        s.step(30)
    assert np.abs((a.get_fields()[0] - b.get_fields()[0]).cpu().numpy()).max() < 1e-12
    assert a.arrests(0) == b.arrests(0)


def test_paper_usage_example_shape_antiskyrmion_with_demag():
    """The paper's usage example (Fig. 1-2): a 320 x 320 lattice, D2d
    ("Heusler") DMI with the antiskyrmion ansatz, demagnetisation on, stepped five steps per
    frame.  (Its physical units and newtonflow=False are not reproduced: DESIGN R16, R19.)  Four
    frames of ss_step(5) against the oracle; the texture is an antiskyrmion, Q = +1."""
    w = W.cm_single(N=320, K=0.1, mirror=True)
    w.dmi, w.demag = W.DMI_D2D, 0.5
    s, fl, _ = _run(w, (5, 10, 15, 20), cycles=24, ftol=1e-10, etol=1e-9)
    assert abs(s.charge()[0] - 1.0) < 5e-3
    assert fl.energy < oracle.energy_charge(_model(w), w.fields[0])[0]


def test_batched_demag_with_per_lattice_B():
    # three lattices with their own B and their own potential psi (blockIdx.z through every
    # multigrid kernel, one coarsest-level CTA per lattice)
    ss = _ss()
    w = W.cm_sweep(batch=3, N=80)
    w.demag, w.dmi = 0.7, W.DMI_NEEL
    s = ss.solver_for(w, integrator=ss.VERLET, demag_cycles=24)
    s.set_fields(_dev(w.fields))
    flows = []
    for b in range(w.batch):
        m = oracle.model(oracle.CM, w.Nx, w.Ny, w.h, kappa=w.kappa, B=float(w.B_batch[b]), K=w.K,
                         dmi=w.dmi, demag=w.demag)
        fl = oracle.Flow(m, w.dt, integrator="verlet")
        fl.set_fields(w.fields[b])
        flows.append(fl)
    for k in (1, 9, 20):
        s.step(k)
        phi, vel = s.get_fields()
        E = s.energy()
        for b, fl in enumerate(flows):
            fl.step(k)
            ophi, _ = fl.get_fields()
            assert np.abs(phi[b].cpu().numpy() - ophi).max() <= 1e-10, (k, b)
            assert abs(E[b] - fl.energy) <= 1e-9 * _floor(fl.m, ophi, fl.energy), (k, b)
            assert s.arrests(b)[0] == fl.arrests()


def test_demag_bench_size_properties():
    """bench.py's demagnetisation workload (2048 x 2048, 64 skyrmions, Neel DMI, g = 1) in the
    launch configuration it times (default 8 V-cycles, CUDA graph).  The oracle's exact CG solve
    is minutes per step at this size, so this checks what holds at any size: E never rises except
    at the steps the device logged, |n| = 1, v.n = 0, the halo is frozen, and the default cycle
    count tracks a 24-cycle run of the same lattice to 1e-6."""
    ss = _ss()
    w = W.cm_demag_bench()
    x = _dev(w.fields)
    a = ss.solver_for(w, integrator=ss.VERLET)
    b = ss.solver_for(w, integrator=ss.VERLET, demag_cycles=24)
    for s in (a, b):
        s.set_fields(x)
    E = [a.energy()[0]]
    for _ in range(30):
        a.step(1)
        E.append(a.energy()[0])
    arrests = set(a.arrests(0)[0])
    for n in range(1, len(E)):
        assert (E[n] > E[n - 1]) == (n in arrests), n
    assert E[-1] < E[0] and a.status()["steps"] == 30
    b.step(30)
    fa, va = a.get_fields()
    fb, _ = b.get_fields()
    assert float((fa - fb).abs().max()) < 1e-6
    assert abs(a.energy()[0] - b.energy()[0]) < 1e-6 * abs(b.energy()[0])
    mask = torch.from_numpy(~W.interior_mask(w.Nx, w.Ny)).to("cuda:0")
    assert torch.equal(fa[0][:, mask], x[0][:, mask])
    assert float(((fa[0] * fa[0]).sum(0)[~mask] - 1.0).abs().max()) < 1e-14
    if not a.status()["n_arrests"][0] or 30 not in arrests:
        assert float((fa[0] * va[0]).sum(0)[~mask].abs().max()) < 1e-12
