"""The chirp-table cache versus CUDA-graph capture (run with -m gpu).

While a stream is being captured the table builders are only RECORDED, and every replay rewrites the tables it
owns behind the host's back.  So a table (or the per-batch 1/lambda array) written under capture must never serve
an eager cache hit, and must never be handed to another key while its graph is alive.  Each test below fails on a
cache that treats captured builds like eager ones; expected values come from the oracle.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

N = 256


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch


@pytest.fixture(scope="module")
def B(torch_cuda):
    from paper_1806_06467_b200 import binding
    binding.lib()
    return binding


def rel(got, want):
    got = np.asarray(got).reshape(want.shape)
    return float(np.linalg.norm(got - want) / np.linalg.norm(want))


def setup(torch):
    from paper_1806_06467_b200 import inputs
    u = inputs.random_field(N, 8100, 1)
    opd = inputs.psd_map(N, 2e-5, 3.0, 30e-9, 8101)
    return u, opd, torch.from_numpy(opd).cuda()


def test_capture_without_warmup_then_eager_call_with_the_same_key(torch_cuda, B, oracle):
    """Capture first (nothing executes), then an EAGER call with the same (f, z, lambda) before any replay: it must
    build its own tables, not 'hit' the ones whose builders were only recorded."""
    torch = torch_cuda
    u, opd, dopd = setup(torch)
    dx, lam, f, z = np.array([2e-5]), np.array([600e-9]), 0.7, 0.05
    s = torch.cuda.Stream()
    plan = B.Plan(N, 1, "c128", stream=s)
    a = torch.from_numpy(u).cuda()
    b = torch.from_numpy(u).cuda()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.stream(s):
        s.synchronize()
        with torch.cuda.graph(g, stream=s):
            plan.surface_as(a, dx, lam, f, None, dopd, z)
        plan.surface_as(b, dx, lam, f, None, dopd, z)          # eager, same key, graph not yet replayed
        s.synchronize()
    want = oracle.surface_as(u[0], dx[0], lam[0], f, None, opd, z)
    assert rel(b.cpu().numpy(), want) <= 1e-11
    g.replay()
    torch.cuda.synchronize()
    assert rel(a.cpu().numpy(), want) <= 1e-11


def test_eager_replay_eager_with_different_wavelengths(torch_cuda, B, oracle):
    """Capture with wavelength A; eager call with B; replay (the graph's tables and 1/lambda hold A again); eager
    call with B once more: the host cache must not believe B is still resident where the replay wrote A."""
    torch = torch_cuda
    u, opd, dopd = setup(torch)
    dx, f, z = np.array([2e-5]), 0.9, 0.04
    lam_a, lam_b = np.array([500e-9]), np.array([650e-9])
    s = torch.cuda.Stream()
    plan = B.Plan(N, 1, "c128", stream=s)
    a = torch.from_numpy(u).cuda()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.stream(s):
        s.synchronize()
        with torch.cuda.graph(g, stream=s):
            plan.surface_as(a, dx, lam_a, f, None, dopd, z)
        want_b = oracle.surface_as(u[0], dx[0], lam_b[0], f, None, opd, z)
        for _ in range(2):
            b = torch.from_numpy(u).cuda()
            plan.surface_as(b, dx, lam_b, f, None, dopd, z)
            s.synchronize()
            assert rel(b.cpu().numpy(), want_b) <= 1e-11
            a.copy_(torch.from_numpy(u))
            s.synchronize()
            g.replay()
            torch.cuda.synchronize()
            want_a = oracle.surface_as(u[0], dx[0], lam_a[0], f, None, opd, z)
            assert rel(a.cpu().numpy(), want_a) <= 1e-11
        b = torch.from_numpy(u).cuda()
        plan.surface_as(b, dx, lam_b, f, None, dopd, z)        # eager after the replay
        s.synchronize()
        assert rel(b.cpu().numpy(), want_b) <= 1e-11


def test_graph_tables_survive_eager_cache_pressure(torch_cuda, B, oracle):
    """A captured surface keeps its tables while an eager train with more distinct tables than the plan caches
    churns through the least-recently-used slots; the replay afterwards is still right."""
    torch = torch_cuda
    from paper_1806_06467_b200.inputs import Surface
    u, opd, dopd = setup(torch)
    dx, lam, f, z = np.array([2e-5]), np.array([700e-9]), 0.6, 0.03
    s = torch.cuda.Stream()
    plan = B.Plan(N, 1, "c128", stream=s)
    a = torch.from_numpy(u).cuda()
    g = torch.cuda.CUDAGraph()
    r = np.random.Generator(np.random.PCG64(8102))
    surfs = [Surface(float(r.uniform(0.3, 2.0)), float(r.uniform(0.002, 0.02))) for _ in range(40)]
    with torch.cuda.stream(s):
        s.synchronize()
        with torch.cuda.graph(g, stream=s):
            plan.surface_as(a, dx, lam, f, None, dopd, z)
        b = torch.from_numpy(u).cuda()
        plan.system_run(b, dx, lam, surfs, methods=[B.METHOD_AS] * 40)      # 80 distinct tables
        s.synchronize()
    want_train, _, _ = oracle.system_run(u[0], dx[0], lam[0], surfs, methods=[0] * 40)
    assert rel(b.cpu().numpy(), want_train) <= 1e-11
    g.replay()
    torch.cuda.synchronize()
    want = oracle.surface_as(u[0], dx[0], lam[0], f, None, opd, z)
    assert rel(a.cpu().numpy(), want) <= 1e-11
    # released slots go back to the eager pool
    plan.release_graph_tables()
    del g
