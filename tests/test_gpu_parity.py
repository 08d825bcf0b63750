"""Parity of the CUDA path (through the C ABI) with the CPU oracle on the same seeded inputs.

Tolerances are BASELINE.json's: fp64 fields max-abs <= 1e-11 over the first 100 steps with
identical arrest-step indices; final E and Q within 1e-9 relative; fp32 runs within 1e-4
relative energy of the fp64 oracle.  Relative differences use the floor
max(|E|, h^2 sum |e_i|) because chiral-magnet energies cross zero during relaxation.
"""
import math

import numpy as np
import pytest
import torch

import oracle
from paper_2603_24370_b200 import workloads as W

pytestmark = pytest.mark.gpu

CHECKPOINTS = (1, 2, 5, 10, 20, 50, 100)


def _ss():
    from paper_2603_24370_b200 import ss
    return ss


def _model(w, b=0):
    B = w.B if w.B_batch is None else float(w.B_batch[b])
    return oracle.model(w.theory, w.Nx, w.Ny, w.h, kappa=w.kappa, B=B, K=w.K, lam=w.lam,
                        dmi=w.dmi)


def _floor(m, phi, E):
    _, _, de, _ = oracle.energy_charge(m, phi, densities=True)
    return max(abs(E), m.h * m.h * float(np.abs(de).sum()), 1e-300)


def _dev(a, dtype=torch.float64):
    return torch.from_numpy(np.ascontiguousarray(a)).to("cuda:0", dtype=dtype).contiguous()


def _run_parity(w, checkpoints=CHECKPOINTS, flags=0, field_tol=1e-11, lattices=None,
                integrator="rk4", vel0=None):
    ss = _ss()
    s = ss.solver_for(w, flags=flags, integrator=ss.VERLET if integrator == "verlet" else ss.RK4)
    s.set_fields(_dev(w.fields), None if vel0 is None else _dev(vel0))
    lattices = range(w.batch) if lattices is None else lattices
    flows = {}
    for b in lattices:
        fl = oracle.Flow(_model(w, b), w.dt, integrator=integrator)
        fl.set_fields(w.fields[b], None if vel0 is None else vel0[b])
        flows[b] = fl
    E0 = s.energy()
    Q0 = s.charge()
    for b, fl in flows.items():
        fl0 = _floor(fl.m, w.fields[b], fl.energy)
        assert abs(E0[b] - fl.energy) <= 1e-12 * fl0
        assert abs(Q0[b] - fl.charge) <= 1e-12 * max(1.0, abs(fl.charge))
    done = 0
    for cp in checkpoints:
        s.step(cp - done)
        phi, vel = s.get_fields()
        E, Q, KE = s.energy(), s.charge(), s.kinetic()
        phi, vel = phi.cpu().numpy(), vel.cpu().numpy()
        for b, fl in flows.items():
            fl.step(cp - done)
            ophi, ovel = fl.get_fields()
            assert np.abs(phi[b] - ophi).max() <= field_tol, (cp, b)
            assert np.abs(vel[b] - ovel).max() <= 10 * field_tol, (cp, b)
            sc = fl.scalars()
            fl_ = _floor(fl.m, ophi, sc["E"])
            assert abs(E[b] - sc["E"]) <= 1e-9 * fl_, (cp, b)
            assert abs(Q[b] - sc["Q"]) <= 1e-9 * max(1.0, abs(sc["Q"])), (cp, b)
            assert abs(KE[b] - sc["KE"]) <= 1e-9 * max(fl_, sc["KE"]), (cp, b)
            got, cnt = s.arrests(b)
            assert got == fl.arrests() and cnt == sc["n_arrests"], (cp, b)
        done = cp
    assert s.status()["steps"] == done
    return s, flows


def test_config1_cm_64_first_100_steps_and_final():
    w = W.baseline_config(1)
    s, flows = _run_parity(w)
    fl = flows[0]
    s.step(900)
    fl.step(900)
    phi = s.get_fields(want_vel=False).cpu().numpy()[0]
    E, Q = s.energy()[0], s.charge()[0]
    assert abs(E - fl.energy) <= 1e-9 * _floor(fl.m, phi, fl.energy)
    assert abs(Q - fl.charge) <= 1e-9 * abs(fl.charge)
    # after convergence late arrest decisions are rounding noise: fields agree only to ~sqrt(eps)
    assert np.abs(phi - fl.get_fields()[0]).max() <= 1e-5
    assert np.abs((phi * phi).sum(0) - 1.0).max() < 1e-14


def test_cm_multi_ragged_tiles():
    # config 2 recipe on a lattice that is not a multiple of the tile (ragged tail in x and y)
    w = W.cm_multi(N=250, count=3, margin=12.0, min_sep=14.0)
    _run_parity(w)


def test_cm_quench_with_anisotropy():
    # config 4 recipe (random unit vectors, K = 0.3), several tiles
    w = W.cm_quench(N=192)
    _run_parity(w, checkpoints=(1, 2, 5, 10, 20, 50))


def test_ah_vortices_lambda_1_and_2():
    for lam in (1.0, 2.0):
        w = W.ah_vortices(N=150, h=0.1, lam=lam, count=2, min_sep=2.0)
        _run_parity(w, checkpoints=(1, 2, 5, 10, 20, 50))


def test_batched_sweep_per_lattice_arrests():
    w = W.cm_sweep(batch=6, N=96)
    s, flows = _run_parity(w)
    logs = [tuple(s.arrests(b)[0]) for b in range(w.batch)]
    assert len(set(logs)) > 1            # different B -> different arrest histories


def test_batched_abelian_higgs():
    # batch dimension x C = 4 template path: three lattices with their own vortex positions
    ws = [W.ah_vortices(N=100, h=0.1, lam=1.0, count=2, min_sep=2.0, config=3 + 10 * k)
          for k in range(3)]
    w = ws[0]
    w.fields = np.concatenate([x.fields for x in ws], axis=0)
    w.batch = 3
    _run_parity(w, checkpoints=(1, 2, 5, 10, 20, 50))


def test_batched_dmi_table_with_per_lattice_B():
    # general-DMI kernels (kCMG) x batch x B_batch
    w = W.cm_sweep(batch=4, N=96)
    w.dmi = W.DMI_NEEL
    s, flows = _run_parity(w, checkpoints=(1, 2, 5, 10, 20, 50))
    assert len(set(s.energy())) == w.batch               # different B -> different lattices


def test_batched_fp32_with_per_lattice_B():
    # packed fp32 kernels x batch x B_batch: energies within 1e-4 of the fp64 oracle per lattice
    ss = _ss()
    w = W.cm_sweep(batch=5, N=96)
    s = ss.solver_for(w, dtype=ss.F32)
    s.set_fields(_dev(w.fields, torch.float32))
    flows = []
    for b in range(w.batch):
        fl = oracle.Flow(_model(w, b), w.dt)
        fl.set_fields(w.fields[b])
        flows.append(fl)
    for _ in range(3):
        s.step(40)
        E, Q = s.energy(), s.charge()
        for b, fl in enumerate(flows):
            fl.step(40)
            assert abs(E[b] - fl.energy) <= 1e-4 * _floor(fl.m, fl.get_fields()[0], fl.energy), b
            assert abs(Q[b] - fl.charge) <= 1e-4
    assert len(set(E)) == w.batch


def test_arrested_steps_from_an_uphill_velocity():
    # kernel Y's arrested branch (vh = 0, a2 := a1) right at steps 2.. on a ragged lattice: start
    # with v = -c a(phi) (uphill, from the oracle) so that step 1 is logged
    w = W.cm_quench(N=190)
    vel = (-0.06 * oracle.accel(_model(w), w.fields[0]))[None]
    s, flows = _run_parity(w, checkpoints=(1, 2, 3, 5, 10), vel0=vel)
    assert flows[0].arrests()[:1] == [1]


def test_extreme_aspect_ratios_at_the_size_limits():
    # widest and tallest lattices the reduction tree supports (include/ss.h "Limits"): Nx = 65536
    # (1024 segment partials per row) and Ny = 32768 (32 rows per thread in the y-tree)
    for Nx, Ny in ((65536, 6), (8, 32768)):
        rng = np.random.default_rng(Nx + Ny)
        f = rng.standard_normal((1, 3, Ny, Nx))
        f /= np.sqrt((f * f).sum(1, keepdims=True))
        f[:, :, ~W.interior_mask(Nx, Ny)] = np.array([0.0, 0.0, 1.0])[None, :, None]
        w = W.Workload("limit", W.CM, Nx, Ny, 0.2, 0.1, kappa=1.0, B=0.6, K=0.1, fields=f)
        _run_parity(w, checkpoints=(1, 2))


def test_verlet_cm_ragged_first_100_steps_with_arrests():
    # one-gradient-per-step integrator (DESIGN R15), same tolerances; config-1 recipe on a ragged
    # lattice; the first arrests fall inside the window
    w = W.cm_multi(N=250, count=3, margin=12.0, min_sep=14.0)
    s, flows = _run_parity(w, integrator="verlet")
    assert len(flows[0].arrests()) >= 1


def test_verlet_ah_and_batched():
    w = W.ah_vortices(N=150, h=0.1, lam=2.0, count=2, min_sep=2.0)
    _run_parity(w, checkpoints=(1, 2, 5, 10, 20, 50), integrator="verlet")
    w = W.cm_sweep(batch=5, N=96)
    s, flows = _run_parity(w, checkpoints=(1, 2, 5, 10, 20, 50), integrator="verlet")
    for Nx, Ny in ((6, 5), (8, 7)):
        rng = np.random.default_rng(Nx * 10 + Ny)
        f = rng.standard_normal((1, 3, Ny, Nx))
        f /= np.sqrt((f * f).sum(1, keepdims=True))
        w = W.Workload("tiny", W.CM, Nx, Ny, 0.2, 0.1, kappa=1.0, B=0.6, K=0.1, fields=f)
        _run_parity(w, checkpoints=(1, 2, 5), integrator="verlet")


def test_verlet_fp32_and_graph_vs_direct():
    ss = _ss()
    w = W.cm_single(N=64)
    s = ss.solver_for(w, dtype=ss.F32, integrator=ss.VERLET)
    s.set_fields(_dev(w.fields, torch.float32))
    fl = oracle.Flow(_model(w), w.dt, integrator="verlet")
    fl.set_fields(w.fields[0])
    for _ in range(3):
        s.step(100)
        fl.step(100)
        phi = fl.get_fields()[0]
        assert abs(s.energy()[0] - fl.energy) <= 1e-4 * _floor(fl.m, phi, fl.energy)
    outs = []
    for flags in (0, ss.FLAG_NO_GRAPH):
        s = ss.solver_for(w, flags=flags, integrator=ss.VERLET)
        s.set_fields(_dev(w.fields))
        s.step(41)
        f, v = s.get_fields()
        outs.append((f.cpu(), v.cpu(), s.energy(), s.charge(), s.arrests(0)))
    assert torch.equal(outs[0][0], outs[1][0]) and torch.equal(outs[0][1], outs[1][1])
    assert outs[0][2:] == outs[1][2:]


@pytest.mark.parametrize("table", ["neel", "d2d", "random", "bloch"])
def test_general_dmi_tables(table):
    # PAPER.md:196 eq. (5) with a (d_x, d_y) table (DESIGN R16): Neel and D2d ("Heusler", with the
    # mirrored = antiskyrmion ansatz), a random table, and the Bloch table through
    # the general kernels; ragged lattice, both integrators
    rng = np.random.default_rng(5)
    dmi = {"neel": W.DMI_NEEL, "d2d": W.DMI_D2D, "bloch": W.DMI_BLOCH,
           "random": tuple(map(tuple, rng.standard_normal((2, 3))))}[table]
    w = W.cm_single(N=90, K=0.2, mirror=(table == "d2d"))
    w.dmi = dmi
    s, flows = _run_parity(w, checkpoints=(1, 2, 5, 10, 20, 50))
    if table == "d2d":
        assert abs(s.charge()[0] - 1.0) < 5e-3           # antiskyrmion
    _run_parity(w, checkpoints=(1, 5, 20), integrator="verlet")


def test_graph_and_direct_launch_agree_bitwise():
    ss = _ss()
    w = W.cm_single(N=96)
    outs = []
    for flags in (0, ss.FLAG_NO_GRAPH):
        s = ss.solver_for(w, flags=flags)
        s.set_fields(_dev(w.fields))
        s.step(37)
        f, v = s.get_fields()
        outs.append((f.cpu(), v.cpu(), s.energy(), s.charge(), s.arrests(0)))
    assert torch.equal(outs[0][0], outs[1][0]) and torch.equal(outs[0][1], outs[1][1])
    assert outs[0][2:] == outs[1][2:]


@pytest.mark.parametrize("case", ["cm", "ah", "cm_verlet"])
def test_results_do_not_depend_on_the_segment_length(case):
    # The row segmentation of the flow kernels (chunks per CTA) only decides which CTA computes a
    # site; per-site arithmetic and the canonical reduction tree (DESIGN R10) are the same, so
    # fields, E, Q and the arrest log are bitwise identical for every segment length, including
    # one chunk per CTA, a length that does not divide the lattice and a single segment.
    ss = _ss()
    if case == "ah":
        w = W.ah_vortices(N=76, count=1)
    else:
        w = W.cm_single(N=100)
    integ = ss.VERLET if case == "cm_verlet" else ss.RK4
    outs = []
    for cps in (0, 1, 3, 7, 1000):
        s = ss.solver_for(w, cps=cps, integrator=integ)
        s.set_fields(_dev(w.fields))
        s.step(41)
        f, v = s.get_fields()
        outs.append((f.cpu(), v.cpu(), s.energy(), s.charge(), s.arrests(0)))
    for o in outs[1:]:
        assert torch.equal(outs[0][0], o[0]) and torch.equal(outs[0][1], o[1])
        assert outs[0][2:] == o[2:]


def test_fp32_energy_within_1e4_of_fp64_oracle():
    ss = _ss()
    w = W.cm_single(N=64)
    s = ss.solver_for(w, dtype=ss.F32)
    s.set_fields(_dev(w.fields, torch.float32))
    fl = oracle.Flow(_model(w), w.dt)
    fl.set_fields(w.fields[0])
    for _ in range(5):
        s.step(100)
        fl.step(100)
        phi = fl.get_fields()[0]
        assert abs(s.energy()[0] - fl.energy) <= 1e-4 * _floor(fl.m, phi, fl.energy)
    assert abs(s.charge()[0] - fl.charge) < 1e-4


@pytest.mark.parametrize("case", ["cm", "cm_neel", "cm_verlet", "ah"])
def test_fp32_fields_track_the_fp64_oracle_on_a_ragged_lattice(case):
    # the packed two-column fp32 kernels (chiral magnet) and the scalar fp32 kernels (Abelian
    # Higgs): fields after 12 steps within fp32 rounding of the fp64 oracle at EVERY site (edge
    # rings with their halo weights included), energy and charge within 1e-4
    ss = _ss()
    if case == "ah":
        w = W.ah_vortices(N=148, h=0.1, lam=1.0, count=2, min_sep=2.0)
    else:
        w = W.cm_multi(N=252, count=3, margin=12.0, min_sep=14.0)
        w.K = 0.2
        if case == "cm_neel":
            w.dmi = W.DMI_NEEL
    integ = "verlet" if case == "cm_verlet" else "rk4"
    s = ss.solver_for(w, dtype=ss.F32, integrator=ss.VERLET if integ == "verlet" else ss.RK4)
    s.set_fields(_dev(w.fields, torch.float32))
    fl = oracle.Flow(_model(w), w.dt, integrator=integ)
    fl.set_fields(w.fields[0])
    E0 = s.energy()[0]
    assert abs(E0 - fl.energy) <= 1e-5 * _floor(fl.m, w.fields[0], fl.energy)
    s.step(12)
    fl.step(12)
    phi, vel = s.get_fields()
    ophi, ovel = fl.get_fields()
    assert np.abs(phi.cpu().numpy()[0] - ophi).max() <= 2e-5
    assert np.abs(vel.cpu().numpy()[0] - ovel).max() <= 2e-4
    assert abs(s.energy()[0] - fl.energy) <= 1e-4 * _floor(fl.m, ophi, fl.energy)
    assert abs(s.charge()[0] - fl.charge) <= 1e-4 * max(1.0, abs(fl.charge))
    assert abs(s.kinetic()[0] - fl.scalars()["KE"]) <= 1e-3 * max(fl.scalars()["KE"], 1e-6)


@pytest.mark.timeout(120)
def test_fp32_smallest_and_odd_multiple_lattices():
    # smallest legal fp32 lattices (Nx % 4 == 0) and widths that are not a multiple of the strip
    ss = _ss()
    for Nx, Ny in ((8, 5), (8, 6), (12, 7), (68, 9), (132, 11)):
        rng = np.random.default_rng(Nx * 10 + Ny)
        f = rng.standard_normal((1, 3, Ny, Nx))
        f /= np.sqrt((f * f).sum(1, keepdims=True))
        w = W.Workload("tiny32", W.CM, Nx, Ny, 0.2, 0.1, kappa=1.0, B=0.6, K=0.1, fields=f)
        for integ in ("rk4", "verlet"):
            s = ss.solver_for(w, dtype=ss.F32, integrator=ss.VERLET if integ == "verlet" else ss.RK4)
            s.set_fields(_dev(f, torch.float32))
            fl = oracle.Flow(_model(w), w.dt, integrator=integ)
            fl.set_fields(f[0])
            s.step(5)
            fl.step(5)
            assert np.abs(s.get_fields()[0].cpu().numpy()[0] - fl.get_fields()[0]).max() <= 2e-5
            assert abs(s.energy()[0] - fl.energy) <= 1e-4 * _floor(fl.m, fl.get_fields()[0], fl.energy)


def test_checkpoint_roundtrip_is_bit_exact():
    ss = _ss()
    w = W.cm_single(N=80)
    a = ss.solver_for(w)
    a.set_fields(_dev(w.fields))
    a.step(9)
    assert a.status()["n_arrests"] == [0]
    f, v = a.get_fields()
    b = ss.solver_for(w)
    b.set_fields(f, v)
    f2, v2 = b.get_fields()
    assert torch.equal(f, f2) and torch.equal(v, v2)
    assert b.energy() == a.energy() and b.charge() == a.charge()
    a.step(5)
    b.step(5)
    assert torch.equal(a.get_fields()[0], b.get_fields()[0])
    # halo is frozen; halo velocities read as zero
    mask = torch.from_numpy(~W.interior_mask(80, 80)).to("cuda:0")
    fa, va = a.get_fields()
    assert torch.equal(fa[0][:, mask], _dev(w.fields)[0][:, mask])
    assert float(va[0][:, mask].abs().max()) == 0.0


def test_smallest_lattices_and_vacuum():
    ss = _ss()
    for Nx, Ny in ((6, 5), (6, 6), (8, 7)):
        rng = np.random.default_rng(Nx * 10 + Ny)
        f = rng.standard_normal((1, 3, Ny, Nx))
        f /= np.sqrt((f * f).sum(1, keepdims=True))
        w = W.Workload("tiny", W.CM, Nx, Ny, 0.2, 0.1, kappa=1.0, B=0.6, K=0.1, fields=f)
        _run_parity(w, checkpoints=(1, 2, 5))
    vac = np.zeros((1, 3, 40, 70))
    vac[0, 2] = 1.0
    w = W.Workload("vac", W.CM, 70, 40, 0.2, 0.1, kappa=1.0, B=0.6, K=0.3, fields=vac)
    s = ss.solver_for(w)
    s.set_fields(_dev(vac))
    s.step(3)
    assert s.energy() == [0.0] and s.charge() == [0.0] and s.kinetic() == [0.0]
    assert torch.equal(s.get_fields(want_vel=False).cpu(), torch.from_numpy(vac))


def test_error_paths():
    ss = _ss()
    with pytest.raises(ss.SSError) as e:
        ss.Solver(0, 63, 64, 0.2)                      # odd Nx in fp64
    assert e.value.code == ss.ERR_ARG
    with pytest.raises(ss.SSError):
        ss.Solver(7, 64, 64, 0.2)                      # unknown theory
    for kw in (dict(Nx=65538, Ny=64), dict(Nx=64, Ny=32770), dict(Nx=64, Ny=64, batch=65536)):
        with pytest.raises(ss.SSError) as e:           # over a limit of this build (ss.h "Limits")
            ss.Solver(0, kw["Nx"], kw["Ny"], 0.2, batch=kw.get("batch", 1))
        assert e.value.code == ss.ERR_UNSUPPORTED
        assert ss.workspace_bytes(0, kw["Nx"], kw["Ny"], batch=kw.get("batch", 1)) == 0
    with pytest.raises(ss.SSError) as e:
        ss.Solver(0, 64, 64, 0.2, flags=8)             # unknown flag bit
    assert e.value.code == ss.ERR_ARG
    s = ss.Solver(0, 64, 64, 0.2, kappa=1.0, B=0.6)
    with pytest.raises(ss.SSError) as e:
        s.step(1)                                      # before set_fields
    assert e.value.code == ss.ERR_STATE
    bad = np.full((1, 3, 64, 64), np.nan)
    s.set_fields(_dev(bad))
    with pytest.raises(ss.SSError) as e:
        s.energy()
    assert e.value.code == ss.ERR_NONFINITE
    assert math.isnan(s.energy(strict=False)[0])
