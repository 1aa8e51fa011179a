"""far_mobility_real_noalloc (include/se_mobility.h): the real-space pair sum without a plan and without any allocation, its scratch
in a static device array of the library.  Collected last on purpose (the suite runs with pytest -x).  Checked against the
existing path -- far_mobility_apply with the wave, self and one-body parts switched off -- within the per-stage tolerance of the
parity tests, on two calls in a row that share the scratch (different systems, the larger one first, so that stale contents of
the first call would show in the second)."""
import numpy as np
import pytest

TOL_STAGE = 1e-12      # as tests/test_gpu_parity.py: relative L2 per output block of one stage


def _rel(a, b):
    return float(np.linalg.norm(np.asarray(a) - np.asarray(b)) / np.linalg.norm(np.asarray(b)))


def _existing_path(pk, torch, wl, dev):
    t = lambda a: torch.tensor(np.ascontiguousarray(a), device=dev, dtype=torch.float64)
    plan = pk.SePlan(wl.N, wl.L, wl.radii, wl.xi, wl.rc, wl.M, wl.P, wl.eta0)
    plan.set_flags(pk.SE_SKIP_WAVE | pk.SE_SKIP_SELF | pk.SE_SKIP_ONEBODY)
    U, W, E = (torch.full((wl.N, k), float("nan"), device=dev, dtype=torch.float64) for k in (3, 3, 5))
    plan.apply(t(wl.pos), t(wl.F), t(wl.T), t(wl.S), U, W, E)
    torch.cuda.synchronize()
    out = U.cpu().numpy(), W.cpu().numpy(), E.cpu().numpy()
    plan.destroy()
    return out


@pytest.mark.gpu
def test_no_alloc_real_space_sum_matches_the_plan_path_twice_in_a_row(workloads):
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_1506_08481_b200 as pk
    pk.load_library()
    dev = torch.device("cuda:0")
    t = lambda a: torch.tensor(np.ascontiguousarray(a), device=dev, dtype=torch.float64)
    cases = [workloads.make_workload("c2"), workloads.make_workload("c1")]          # N = 1000, then N = 100
    refs = [_existing_path(pk, torch, wl, dev) for wl in cases]
    # inputs and outputs are the caller's and are made before the calls; the calls themselves must not allocate on the device
    ins = [(t(wl.pos), t(wl.radii), t(wl.F), t(wl.T), t(wl.S)) for wl in cases]
    outs = [tuple(torch.full((wl.N, k), float("nan"), device=dev, dtype=torch.float64) for k in (3, 3, 5)) for wl in cases]
    # one call beforehand, so that the lazily loaded kernel code and the array's address are in place when memory is measured
    wl0, (pos, rad, F, T, S), (U, W, E) = cases[1], ins[1], outs[1]
    pk.real_noalloc(wl0.L, wl0.xi, wl0.rc, pos, rad, F, T, S, U, W, E, eta0=wl0.eta0)
    U.fill_(float("nan")); W.fill_(float("nan")); E.fill_(float("nan"))
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for wl, (pos, rad, F, T, S), (U, W, E) in zip(cases, ins, outs):                 # two calls in a row, same stream
        pk.real_noalloc(wl.L, wl.xi, wl.rc, pos, rad, F, T, S, U, W, E, eta0=wl.eta0)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free0, "the no-alloc entry point took device memory"
    for wl, ref, (U, W, E) in zip(cases, refs, outs):
        got = U.cpu().numpy(), W.cpu().numpy(), E.cpu().numpy()
        assert all(np.isfinite(g).all() for g in got)
        for g, r in zip(got, ref):
            assert _rel(g, r) <= TOL_STAGE, (wl.N, _rel(g, r))
    # the same call again gives the same bits (fixed summation order, scratch fully rewritten)
    wl, (pos, rad, F, T, S) = cases[0], ins[0]
    U2, W2, E2 = (torch.empty_like(x) for x in outs[0])
    pk.real_noalloc(wl.L, wl.xi, wl.rc, pos, rad, F, T, S, U2, W2, E2, eta0=wl.eta0)
    torch.cuda.synchronize()
    assert torch.equal(U2, outs[0][0]) and torch.equal(W2, outs[0][1]) and torch.equal(E2, outs[0][2])


@pytest.mark.gpu
def test_no_alloc_rejects_sizes_beyond_the_static_scratch():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_1506_08481_b200 as pk
    dev = torch.device("cuda:0")
    N = pk.SE_NOALLOC_MAX_N + 1
    z = lambda k: torch.zeros((N, k), device=dev, dtype=torch.float64)
    with pytest.raises(pk.SeError) as ei:
        pk.real_noalloc(100.0, 0.5, 4.0, z(3), torch.ones(N, device=dev, dtype=torch.float64), z(3), z(3), z(5), z(3), z(3), z(5))
    assert ei.value.status == 1 and "SE_NOALLOC_MAX_N" in str(ei.value)


@pytest.mark.gpu
def test_no_alloc_at_the_maximum_size_and_with_a_single_particle(workloads):
    """N = SE_NOALLOC_MAX_N exactly (the first 8192 particles of c3: the whole scratch array is in use, several candidate chunks
    per target in the all-pairs scan) against the plan path, and N = 1 (no pair at all: zeros, not stale scratch)."""
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_1506_08481_b200 as pk
    dev = torch.device("cuda:0")
    t = lambda a: torch.tensor(np.ascontiguousarray(a), device=dev, dtype=torch.float64)
    wl = workloads.make_workload("c3")
    N = pk.SE_NOALLOC_MAX_N
    assert wl.N >= N
    wl.N, wl.pos, wl.radii, wl.F, wl.T, wl.S = N, wl.pos[:N], wl.radii[:N], wl.F[:N], wl.T[:N], wl.S[:N]
    ref = _existing_path(pk, torch, wl, dev)
    U, W, E = (torch.full((N, k), float("nan"), device=dev, dtype=torch.float64) for k in (3, 3, 5))
    pk.real_noalloc(wl.L, wl.xi, wl.rc, t(wl.pos), t(wl.radii), t(wl.F), t(wl.T), t(wl.S), U, W, E, eta0=wl.eta0)
    torch.cuda.synchronize()
    for g, r in zip((U, W, E), ref):
        assert _rel(g.cpu().numpy(), r) <= TOL_STAGE
    # one particle, right after the full-size call
    U1, W1, E1 = (torch.full((1, k), float("nan"), device=dev, dtype=torch.float64) for k in (3, 3, 5))
    pk.real_noalloc(wl.L, wl.xi, wl.rc, t(wl.pos[:1]), t(wl.radii[:1]), t(wl.F[:1]), t(wl.T[:1]), t(wl.S[:1]), U1, W1, E1)
    torch.cuda.synchronize()
    assert float(U1.abs().sum() + W1.abs().sum() + E1.abs().sum()) == 0.0
