"""Train-level pass fusion of fresnel_system_run (run with -m gpu): a run of L angular-spectrum surfaces is
scheduled as L+1 passes (rows_0 | cols_0, optic_1, cols_1 | rows_1, optic_2, rows_2 | ...), every inner pass
holding each line on chip through convolution -> optic -> convolution.  Expected values: the oracle's literal
surface-by-surface train (oracle.system_run), same seeded inputs; bar: the north-star tolerances plus the max-abs
bound of tests/test_gpu_parity.py.  The schedule itself (pass count, directions, maps per pass) is checked through
fresnel_plan_last_schedule.
"""
import math

import numpy as np
import pytest

from test_gpu_parity import assert_parity, field, map_dev, map_host, to_dev

pytestmark = pytest.mark.gpu


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


def make_train(N, dx, seed):
    """Six surfaces covering every optic a fused pass can meet: lens + both maps, lens only, OPD only, amplitude
    only (no lens), lens + OPD with z < 0, nothing but propagation."""
    from paper_1806_06467_b200 import inputs
    from paper_1806_06467_b200.inputs import Surface
    amp = inputs.circular_aperture(N, N / 3)
    amp2 = (inputs.centred_r2_px(N) > (N / 40) ** 2).astype(np.float64)
    opd = [inputs.psd_map(N, dx, 3.0, 12e-9, seed + i) for i in range(3)]
    zc = N * dx * dx / 1e-6
    return [Surface(0.7, 0.21 * zc, amp, opd[0]), Surface(-1.3, 0.13 * zc), Surface(math.inf, 0.17 * zc, None, opd[1]),
            Surface(math.inf, 0.09 * zc, amp2, None), Surface(0.9, -0.15 * zc, None, opd[2]), Surface(math.inf, 0.11 * zc)]


@pytest.mark.parametrize("dtype", ["c128", "c64"])
@pytest.mark.parametrize("N", [128, 512, 1024, 2048])
def test_fused_train_matches_the_oracle(torch_cuda, B, oracle, N, dtype):
    """N = 128 takes the per-thread-load column pass, N >= 512 the TMA column pass (map tiles by TMA: early-fetched
    into their own landing zone at N <= 1024, into the idle exchange space of the 16-byte-wide tiles at N = 2048); two
    wavelengths per call."""
    dx = 2e-5
    surfs = make_train(N, dx, 9000 + N)
    u = field(N, 9100 + N, 2, dtype)
    pix, lam = np.array([dx, dx]), np.array([0.9e-6, 0.75e-6])
    plan = B.Plan(N, 2, dtype)
    maps = [(map_dev(torch_cuda, s.amp, dtype), map_dev(torch_cuda, s.opd, dtype)) for s in surfs]
    d = to_dev(torch_cuda, u, dtype)
    px, used = plan.system_run(d, pix, lam, surfs, maps=maps, methods=[B.METHOD_AS] * len(surfs))
    assert used == [0] * len(surfs) and list(px) == [dx, dx]
    sched = plan.last_schedule()
    assert len(sched) == len(surfs) + 1                                  # L + 1 passes, not 2 L
    assert [k["direction"] for k in sched] == [i & 1 for i in range(len(sched))]
    assert [k["convolutions"] for k in sched] == [1] + [2] * (len(surfs) - 1) + [1]
    assert [k["maps_read"] for k in sched] == [2, 0, 1, 1, 1, 0, 0]
    got = d.cpu().numpy().reshape(2, N, N)
    hs = [type(s)(s.f, s.z, map_host(s.amp, dtype), map_host(s.opd, dtype)) for s in surfs]
    for b in range(2):
        want, _, _ = oracle.system_run(u[b], pix[b], lam[b], hs, methods=[0] * len(hs))
        assert_parity(got[b][None], want[None], dtype, f"wavelength {b}")


@pytest.mark.parametrize("dtype,N", [("c128", 4096), ("c64", 4096), ("c128", 8192), ("c64", 8192)])
def test_fused_train_large_grids(torch_cuda, B, oracle, dtype, N):
    """N = 4096 / 8192: the column tile is 16 bytes wide, narrower than (c128) or as wide as (c64) the 16-byte TMA
    minimum of a map box, and the map tile is fetched into the idle exchange space between the two convolutions.
    Three surfaces: both maps land in a column pass (surface 1) and in a row pass (surface 2)."""
    from paper_1806_06467_b200 import inputs
    from paper_1806_06467_b200.inputs import Surface
    dx = 1e-5
    amp = inputs.circular_aperture(N, N / 3)
    opd = inputs.psd_map(N, dx, 2.5, 15e-9, 9200 + N)
    zc = N * dx * dx / 633e-9
    surfs = [Surface(1.1, 0.2 * zc, None, opd), Surface(0.8, 0.1 * zc, amp, opd), Surface(-2.0, 0.15 * zc, amp, opd)]
    u = field(N, 9300 + N, 1, dtype)
    pix, lam = np.array([dx]), np.array([633e-9])
    plan = B.Plan(N, 1, dtype)
    da, do = map_dev(torch_cuda, amp, dtype), map_dev(torch_cuda, opd, dtype)
    maps = [(None, do), (da, do), (da, do)]
    d = to_dev(torch_cuda, u, dtype)
    plan.system_run(d, pix, lam, surfs, maps=maps, methods=[B.METHOD_AS] * 3)
    sched = plan.last_schedule()
    assert [(k["direction"], k["convolutions"], k["maps_read"]) for k in sched] == [(0, 1, 1), (1, 2, 2), (0, 2, 2), (1, 1, 0)]
    hs = [Surface(s.f, s.z, map_host(s.amp, dtype), map_host(s.opd, dtype)) for s in surfs]
    want, _, _ = oracle.system_run(u[0], dx, 633e-9, hs, methods=[0, 0, 0])
    assert_parity(d.cpu().numpy(), want[None], dtype)


def test_config3_full_size_fused_train(torch_cuda, B, oracle):
    """The step bench.py times: config 3 at full size (N=2048, complex128, 20 surfaces with their maps) as ONE
    fresnel_system_run -- 21 fused passes -- whole field against the oracle's surface-by-surface chain."""
    from paper_1806_06467_b200 import inputs
    wl = inputs.config3()
    plan = B.Plan(wl.N, 1, "c128")
    d = to_dev(torch_cuda, wl.field, "c128")
    maps = [(map_dev(torch_cuda, s.amp, "c128"), map_dev(torch_cuda, s.opd, "c128")) for s in wl.surfaces]
    plan.system_run(d, wl.dx, wl.lam, wl.surfaces, maps=maps, methods=[B.METHOD_AS] * 20)
    assert len(plan.last_schedule()) == 21
    want, _, _ = oracle.system_run(wl.field[0], wl.dx[0], wl.lam[0], wl.surfaces, methods=[0] * 20)
    assert_parity(d.cpu().numpy(), want[None], "c128")


def test_fused_train_breaks_at_direct_and_optic_only_surfaces(torch_cuda, B, oracle):
    """A direct-Fresnel surface and a z == 0 surface end a fused run; the runs on either side are fused on their
    own (2 + 1 passes each here), and the whole train still equals the oracle's."""
    from paper_1806_06467_b200 import inputs
    from paper_1806_06467_b200.inputs import Surface
    N, dx, lam = 512, 2e-5, 1e-6
    zc = N * dx * dx / lam
    opd = inputs.psd_map(N, dx, 3.0, 10e-9, 9400)
    surfs = [Surface(0.5, 0.3 * zc, None, opd), Surface(0.9, 0.2 * zc), Surface(1.5, 1.6 * zc, None, opd),
             Surface(math.inf, 0.0, None, opd), Surface(0.7, 0.5 * zc), Surface(-0.8, 0.4 * zc, None, opd)]
    methods = [B.METHOD_AS, B.METHOD_AS, B.METHOD_DIRECT, B.METHOD_AS, B.METHOD_AS, B.METHOD_AS]
    u = field(N, 9401, 1)
    plan = B.Plan(N, 1, "c128")
    do = map_dev(torch_cuda, opd, "c128")
    maps = [(None, do if s.opd is not None else None) for s in surfs]
    d = to_dev(torch_cuda, u, "c128")
    px, used = plan.system_run(d, [dx], [lam], surfs, maps=maps, methods=methods)
    assert used == [0, 0, 1, -1, 0, 0]
    kinds = [(k["direction"], k["convolutions"]) for k in plan.last_schedule()]
    assert kinds == [(0, 1), (1, 2), (0, 1), (0, 0), (1, 0), (0, 0), (0, 1), (1, 2), (0, 1)]
    want, dxo, _ = oracle.system_run(u[0], dx, lam, surfs, methods=[0, 0, 1, 0, 0, 0])
    assert px[0] == pytest.approx(dxo, rel=1e-14)
    assert_parity(d.cpu().numpy(), want[None], "c128")


def test_fused_train_as_one_cuda_graph_and_long_train_windows(torch_cuda, B, oracle):
    """(a) A fused train captured into one CUDA graph replays correctly (its tables are graph-owned).  (b) A train
    longer than the table pool allows at once (64 slots -> 30 surfaces per fused run) is split into runs."""
    torch = torch_cuda
    from paper_1806_06467_b200.inputs import Surface
    N, dx, lam = 256, np.array([2e-5]), np.array([0.8e-6])
    r = np.random.Generator(np.random.PCG64(9500))
    surfs = [Surface(float(r.uniform(0.3, 2.0)), float(r.uniform(0.002, 0.02))) for _ in range(40)]
    u = field(N, 9501, 1)
    want, _, _ = oracle.system_run(u[0], dx[0], lam[0], surfs, methods=[0] * 40)
    plan = B.Plan(N, 1, "c128")
    d = to_dev(torch, u, "c128")
    plan.system_run(d, dx, lam, surfs, methods=[B.METHOD_AS] * 40)
    assert len(plan.last_schedule()) == 31 + 11                          # runs of 30 and 10 surfaces
    assert_parity(d.cpu().numpy(), want[None], "c128")
    # (a) graph capture of the first 12 surfaces
    want12, _, _ = oracle.system_run(u[0], dx[0], lam[0], surfs[:12], methods=[0] * 12)
    s = torch.cuda.Stream()
    plan = B.Plan(N, 1, "c128", stream=s)
    d = to_dev(torch, u, "c128")
    src = d.clone()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.stream(s):
        s.synchronize()
        with torch.cuda.graph(g, stream=s):
            plan.system_run(d, dx, lam, surfs[:12], methods=[B.METHOD_AS] * 12)
    for _ in range(2):
        d.copy_(src)
        torch.cuda.synchronize()
        g.replay()
        torch.cuda.synchronize()
        assert_parity(d.cpu().numpy(), want12[None], "c128")
