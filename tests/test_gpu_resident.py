"""The resident-cluster schedule (csrc/ss_resident.cuh: one launch runs all k steps of a small
lattice out of shared memory) against the general schedule and the oracle.  It reuses the flow
kernels' per-site routines and the canonical tree order, so everything is bitwise identical to
the general path; config 1's 1000-step acceptance run goes through it."""
import json
import os

import numpy as np
import pytest
import torch

import oracle
from paper_2603_24370_b200 import workloads as W

pytestmark = pytest.mark.gpu
GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def _ss():
    from paper_2603_24370_b200 import ss
    return ss


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).to("cuda:0")


def _state(s):
    f, v = s.get_fields()
    return f.cpu(), v.cpu(), s.energy(), s.charge(), s.kinetic(), s.arrests(0), s.status()["steps"]


@pytest.mark.parametrize("shape", [(64, 64), (96, 80), (128, 128), (32, 24), (64, 6)])
def test_resident_is_bitwise_identical_to_the_general_schedule(shape):
    ss = _ss()
    Nx, Ny = shape
    w = W.cm_single(N=max(Nx, Ny), K=0.2)
    f = w.fields[:, :, :Ny, :Nx].copy()
    f[:, :, ~W.interior_mask(Nx, Ny)] = np.array([0.0, 0.0, 1.0])[None, :, None]
    w.fields, w.Nx, w.Ny = f, Nx, Ny
    a = ss.solver_for(w)
    b = ss.solver_for(w, flags=ss.FLAG_NO_RESIDENT)
    assert a.schedule() == "resident-cluster" and b.schedule() == "two-kernel"
    for s in (a, b):
        s.set_fields(_dev(w.fields))
    for k in (1, 2, 7, 40, 150):        # several launches, arrests inside (first at step ~17)
        a.step(k)
        b.step(k)
        sa, sb = _state(a), _state(b)
        assert torch.equal(sa[0], sb[0]) and torch.equal(sa[1], sb[1])
        assert sa[2:] == sb[2:]
    assert len(sa[5][0]) >= 1 or min(Nx, Ny) < 32


def test_resident_and_general_steps_can_be_mixed_and_batched():
    ss = _ss()
    w = W.cm_sweep(batch=3, N=64)
    a = ss.solver_for(w)
    b = ss.solver_for(w, flags=ss.FLAG_NO_RESIDENT)
    assert a.schedule() == "resident-cluster"
    for s in (a, b):
        s.set_fields(_dev(w.fields))
    a.step(30)
    b.step(30)
    a.profile_step(reps=3)               # three steps through the general kernels of the same handle
    b.step(3)
    a.step(20)
    b.step(20)
    fa, va = a.get_fields()
    fb, vb = b.get_fields()
    assert torch.equal(fa, fb) and torch.equal(va, vb)
    assert a.energy() == b.energy() and a.charge() == b.charge() and a.kinetic() == b.kinetic()
    for lat in range(3):
        assert a.arrests(lat) == b.arrests(lat)
    assert a.status()["steps"] == 53


def test_config1_acceptance_run_through_the_resident_schedule():
    ss = _ss()
    w = W.baseline_config(1)
    s = ss.solver_for(w)
    assert s.schedule() == "resident-cluster"
    s.set_fields(_dev(w.fields))
    fl = oracle.Flow(oracle.model(w.theory, w.Nx, w.Ny, w.h, kappa=w.kappa, B=w.B, K=w.K), w.dt)
    fl.set_fields(w.fields[0])
    done = 0
    for cp in (1, 2, 5, 10, 20, 50, 100):
        s.step(cp - done)
        fl.step(cp - done)
        done = cp
        phi, vel = s.get_fields()
        ophi, ovel = fl.get_fields()
        assert np.abs(phi.cpu().numpy()[0] - ophi).max() <= 1e-11
        assert np.abs(vel.cpu().numpy()[0] - ovel).max() <= 1e-10
        assert s.arrests(0)[0] == fl.arrests()
    s.step(w.steps - done)
    g = json.load(open(os.path.join(GOLD, "full_length_c1.json")))["runs"][0]
    floor = max(abs(g["E"]), g["abs_density_sum_h2"])
    assert abs(s.energy()[0] - g["E"]) <= 1e-9 * floor
    assert abs(s.charge()[0] - g["Q"]) <= 1e-9 * abs(g["Q"])
    assert [n for n in s.arrests(0)[0] if n <= 100] == [n for n in g["arrests_first"] if n <= 100]
