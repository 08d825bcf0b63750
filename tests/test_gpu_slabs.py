"""The row-slab schedule of the RK4 step (ss_api.cu `plan_slabs`: kernels Y and X split into four
row slabs each that overlap inside the CUDA graph) against the unsplit two-kernel schedule and
the oracle.  Only the launch geometry and the graph edges differ, so fields, E, Q, KE and the
arrest log must be bitwise identical; a missing edge would show as a race on the rows at a slab
seam.  The 4096^2 and 2048^2 full-size parity tests (tests/test_gpu_fullsize.py) run through this
schedule by default; here it is forced on smaller lattices with one chunk per segment."""
import numpy as np
import pytest
import torch

import oracle
from paper_2603_24370_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _ss():
    from paper_2603_24370_b200 import ss
    return ss


def _dev(a, dtype=torch.float64):
    return torch.from_numpy(np.ascontiguousarray(a)).to("cuda:0", dtype=dtype).contiguous()


def _cases():
    # (workload, fp32?, uphill start so that steps arrest early, steps)
    yield "cm", W.cm_quench(N=644), False, True, 12
    yield "cm_f32", W.cm_quench(N=900), True, False, 12
    yield "ah", W.ah_vortices(N=516, h=0.1, lam=2.0, count=2, min_sep=2.0), False, False, 8
    yield "cm_batched", W.cm_sweep(batch=3, N=324), False, False, 10


@pytest.mark.parametrize("case", ["cm", "cm_f32", "ah", "cm_batched"])
def test_slab_schedule_is_bitwise_identical_and_matches_the_oracle(case):
    ss = _ss()
    name, w, f32, uphill, steps = next(c for c in _cases() if c[0] == case)
    td = torch.float32 if f32 else torch.float64
    B0 = w.B if w.B_batch is None else float(w.B_batch[0])
    m = oracle.model(w.theory, w.Nx, w.Ny, w.h, kappa=w.kappa, B=B0, K=w.K, lam=w.lam)
    vel = (-0.06 * oracle.accel(m, w.fields[0]))[None] if uphill else None
    outs = {}
    for flags in (ss.FLAG_NO_SLABS, 0, ss.FLAG_NO_GRAPH):
        s = ss.solver_for(w, dtype=ss.F32 if f32 else ss.F64, flags=flags, cps=1)
        assert s.schedule() == ("two-kernel" if flags == ss.FLAG_NO_SLABS else "two-kernel, row slabs")
        s.set_fields(_dev(w.fields, td), None if vel is None else _dev(vel, td))
        s.step(steps)          # 8-step graph + single-step graphs
        f, v = s.get_fields()
        outs[flags] = (f.cpu(), v.cpu(), s.energy(), s.charge(), s.kinetic(), s.arrests(0))
    ref = outs[ss.FLAG_NO_SLABS]
    for flags in (0, ss.FLAG_NO_GRAPH):
        o = outs[flags]
        assert torch.equal(ref[0], o[0]) and torch.equal(ref[1], o[1]), flags
        assert ref[2:] == o[2:], flags
    if uphill:
        assert ref[5][0][:1] == [1]
    if not f32:
        fl = oracle.Flow(m, w.dt)
        fl.set_fields(w.fields[0], None if vel is None else vel[0])
        fl.step(steps)
        ophi, ovel = fl.get_fields()
        assert np.abs(outs[0][0][0].numpy() - ophi).max() <= 1e-11
        assert np.abs(outs[0][1][0].numpy() - ovel).max() <= 1e-10
        assert outs[0][5][0] == fl.arrests()


def test_slabs_are_not_used_where_they_do_not_pay():
    ss = _ss()
    assert ss.solver_for(W.cm_multi(N=1024)).schedule() == "two-kernel"          # < 2 waves
    assert ss.solver_for(W.cm_quench(N=1280)).schedule() == "two-kernel"
    assert ss.solver_for(W.cm_quench(N=1536)).schedule() == "two-kernel, row slabs"
    assert ss.solver_for(W.cm_sweep(batch=4, N=256)).schedule() == "two-kernel"   # small lattices
    assert ss.solver_for(W.cm_sweep(batch=4, N=1024)).schedule() == "two-kernel, row slabs"
    assert ss.solver_for(W.cm_quench(N=2048), integrator=ss.VERLET).schedule() == "one-kernel verlet"
    assert ss.solver_for(W.cm_quench(N=4096)).schedule() == "two-kernel, row slabs"


def test_slab_schedule_at_bench_size_is_bitwise_identical():
    # 4096^2 fp64 (the metric's workload) and 2048^2 Abelian Higgs with the default segment length:
    # 19 steps = two 8-step graphs + three single-step graphs, against whole-lattice launches
    ss = _ss()
    for w in (W.baseline_config(4), W.baseline_config(3)):
        outs = []
        for flags in (ss.FLAG_NO_SLABS, 0):
            s = ss.solver_for(w, flags=flags)
            s.set_fields(_dev(w.fields))
            s.step(19)
            f, v = s.get_fields()
            outs.append((f, v, s.energy(), s.charge(), s.kinetic(), s.arrests(0), s.schedule()))
            del s
        assert outs[0][6] == "two-kernel" and outs[1][6] == "two-kernel, row slabs"
        assert torch.equal(outs[0][0], outs[1][0]) and torch.equal(outs[0][1], outs[1][1])
        assert outs[0][2:6] == outs[1][2:6]
        del outs
        torch.cuda.empty_cache()


def test_profile_step_under_the_slab_schedule_advances_like_step():
    # ss_profile_step times whole-lattice launches of the same kernels (one by one); the state it
    # leaves must be the one ss_step leaves
    ss = _ss()
    w = W.cm_quench(N=644)
    a = ss.solver_for(w, cps=1)
    b = ss.solver_for(w, cps=1)
    assert a.schedule() == "two-kernel, row slabs"
    for s in (a, b):
        s.set_fields(_dev(w.fields))
        s.step(2)
    prof = a.profile_step(3)
    b.step(3)
    assert [n for n, _ in prof] == ["flow_y_stage34_combine_project_ke", "flow_x_grad_energy_charge_stage2",
                                    "row_reduce", "finalize_arrest"]
    a.step(4)
    b.step(4)
    fa, va = a.get_fields()
    fb, vb = b.get_fields()
    assert torch.equal(fa, fb) and torch.equal(va, vb)
    assert a.energy() == b.energy() and a.status()["steps"] == b.status()["steps"] == 9


@pytest.mark.parametrize("shape", [(6000, 1000, 1, "cm"), (66, 20000, 1, "cm"), (2002, 702, 3, "cm"),
                                   (518, 3000, 2, "ah")])
def test_slabs_on_ragged_non_square_and_batched_shapes(shape):
    # the default segment length and slab split on shapes whose sizes divide nothing evenly: wide,
    # tall and narrow, batched; random fields; bitwise against the unsplit step
    ss = _ss()
    Nx, Ny, batch, th = shape
    rng = np.random.default_rng(Nx + Ny)
    theory = W.AH if th == "ah" else W.CM
    f = rng.standard_normal((batch, 4 if th == "ah" else 3, Ny, Nx))
    if th == "cm":
        f /= np.sqrt((f * f).sum(1, keepdims=True))
        f[:, :, ~W.interior_mask(Nx, Ny)] = np.array([0.0, 0.0, 1.0])[None, :, None]
    else:
        f *= 0.3
        f[:, 0] += 1.0
    h = 0.1 if th == "ah" else 0.2
    w = W.Workload("shape", theory, Nx, Ny, h, 0.5 * h, kappa=1.0, B=0.6, K=0.1, lam=1.5, batch=batch,
                   fields=f)
    outs = []
    for flags in (ss.FLAG_NO_SLABS, 0):
        s = ss.solver_for(w, flags=flags)
        s.set_fields(_dev(w.fields))
        s.step(11)
        fo, vo = s.get_fields()
        outs.append((fo, vo, s.energy(), s.charge(), s.kinetic(), [s.arrests(k) for k in range(batch)],
                     s.schedule()))
        del s
    assert outs[0][6] == "two-kernel" and outs[1][6] == "two-kernel, row slabs"
    assert torch.equal(outs[0][0], outs[1][0]) and torch.equal(outs[0][1], outs[1][1])
    assert outs[0][2:6] == outs[1][2:6]
