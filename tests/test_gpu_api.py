"""Semantics of the C ABI on the GPU (include/ss.h): streams, re-initialisation, arrest-log
capacity, zero-length calls, per-lattice parameters, host-buffer calls, independence of handles."""
import numpy as np
import pytest
import torch

import oracle
from paper_2603_24370_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _ss():
    from paper_2603_24370_b200 import ss
    return ss


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).to("cuda:0")


def test_non_default_stream_and_two_handles_interleaved():
    ss = _ss()
    w = W.cm_single(N=96)
    ref = ss.solver_for(w)
    ref.set_fields(_dev(w.fields))
    ref.step(30)
    want = ref.get_fields()[0].cpu()
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    x = _dev(w.fields)
    torch.cuda.synchronize()
    with torch.cuda.stream(s1):
        a = ss.Solver(w.theory, w.Nx, w.Ny, w.h, dt=w.dt, kappa=w.kappa, B=w.B, K=w.K, stream=s1)
        a.set_fields(x)
    with torch.cuda.stream(s2):
        b = ss.Solver(w.theory, w.Nx, w.Ny, w.h, dt=w.dt, kappa=w.kappa, B=w.B, K=w.K, stream=s2)
        b.set_fields(x)
    for _ in range(10):                     # interleave the two handles on their own streams
        a.step(3)
        b.step(3)
    assert torch.equal(a.get_fields()[0].cpu(), want)
    assert torch.equal(b.get_fields()[0].cpu(), want)
    assert a.energy() == ref.energy() and b.arrests(0) == ref.arrests(0)


def test_set_fields_again_resets_counters_and_log():
    ss = _ss()
    w = W.cm_single(N=64)
    s = ss.solver_for(w)
    s.set_fields(_dev(w.fields))
    s.step(40)
    first = (s.get_fields()[0].cpu(), s.energy(), s.arrests(0))
    assert first[2][1] >= 1
    s.set_fields(_dev(w.fields))
    st = s.status()
    assert st["steps"] == 0 and st["n_arrests"] == [0] and s.kinetic() == [0.0]
    s.step(0)                               # a zero-length call is a no-op
    assert s.status()["steps"] == 0
    s.step(40)
    assert torch.equal(s.get_fields()[0].cpu(), first[0])
    assert (s.energy(), s.arrests(0)) == first[1:]


def test_arrest_log_capacity_counts_but_does_not_overflow():
    ss = _ss()
    w = W.cm_single(N=64)
    s = ss.solver_for(w, log_cap=3)
    s.set_fields(_dev(w.fields))
    fl = oracle.Flow(oracle.model(w.theory, w.Nx, w.Ny, w.h, kappa=w.kappa, B=w.B, K=w.K), w.dt)
    fl.set_fields(w.fields[0])
    s.step(100)
    fl.step(100)
    logged, count = s.arrests(0)
    assert count == len(fl.arrests()) > 3
    assert logged == fl.arrests()[:3]


def test_per_lattice_B_matches_single_lattice_solvers():
    ss = _ss()
    w = W.cm_sweep(batch=4, N=64)
    s = ss.solver_for(w)
    s.set_fields(_dev(w.fields))
    s.step(25)
    f = s.get_fields()[0].cpu()
    E = s.energy()
    for b in range(w.batch):
        one = ss.Solver(w.theory, w.Nx, w.Ny, w.h, dt=w.dt, kappa=w.kappa, B=float(w.B_batch[b]))
        one.set_fields(_dev(w.fields[b:b + 1]))
        one.step(25)
        assert torch.equal(one.get_fields()[0].cpu()[0], f[b])
        assert one.energy()[0] == E[b]


def test_host_buffer_calls_equal_device_calls():
    ss = _ss()
    w = W.ah_vortices(N=96, h=0.1, lam=1.0, count=1)
    host = torch.from_numpy(w.fields).contiguous().pin_memory()
    a, b = ss.solver_for(w), ss.solver_for(w)
    a.set_fields(host.to("cuda:0"))
    b.set_fields_host(host)
    a.step(12)
    b.step(12)
    out_f, out_v = torch.empty_like(host), torch.empty_like(host)
    b.get_fields_host(out_f, out_v)
    fa, va = a.get_fields()
    assert torch.equal(out_f, fa.cpu()) and torch.equal(out_v, va.cpu())
    assert a.energy() == b.energy() and a.charge() == b.charge()


def test_velocity_input_halo_is_ignored_and_output_halo_is_zero():
    ss = _ss()
    w = W.cm_single(N=64)
    rng = np.random.default_rng(3)
    vel = 0.01 * rng.standard_normal(w.fields.shape)
    mask = W.interior_mask(64, 64)
    clean = vel.copy()
    clean[:, :, ~mask] = 0.0
    a, b = ss.solver_for(w), ss.solver_for(w)
    a.set_fields(_dev(w.fields), _dev(vel))
    b.set_fields(_dev(w.fields), _dev(clean))
    assert torch.equal(a.get_fields()[1], b.get_fields()[1])
    a.step(5)
    b.step(5)
    assert torch.equal(a.get_fields()[0], b.get_fields()[0])
    fl = oracle.Flow(oracle.model(w.theory, 64, 64, w.h, kappa=w.kappa, B=w.B, K=w.K), w.dt)
    fl.set_fields(w.fields[0], vel[0])
    fl.step(5)
    assert np.abs(a.get_fields()[0].cpu().numpy()[0] - fl.get_fields()[0]).max() <= 1e-11


def test_solver_on_a_non_current_device():
    # the library binds a solver to the device of its workspace: calls work with any
    # device current.  Needs two GPUs.
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two CUDA devices")
    ss = _ss()
    w = W.cm_single(N=64)
    ref = ss.solver_for(w)
    ref.set_fields(_dev(w.fields))
    ref.step(10)
    torch.cuda.set_device(0)
    s = ss.solver_for(w, device="cuda:1")
    s.set_fields(torch.from_numpy(w.fields).to("cuda:1"))
    s.step(10)
    assert torch.equal(s.get_fields()[0].cpu(), ref.get_fields()[0].cpu())
    assert s.energy() == ref.energy()
