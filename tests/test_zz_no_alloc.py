"""lb_check_state_static (include/lb.h): the state check that allocates nothing.  Its scratch
memory is a `static __device__` array inside the library; its output is compared here with the
existing path (lb_check_state, whose scratch the handle allocates), on two calls in a row and after
stepping.  The file sorts last on purpose: the suite runs with pytest -x."""
import re

import numpy as np
import pytest

import parity_util as pu
from paper_2005_12764_b200 import workloads as W

pytestmark = pytest.mark.gpu

# Both paths add the same per-site fp32 densities in double precision, in different orders: the
# sums agree to rounding of ~N^(1/2) additions of O(1) terms, far below this bound.
REL = 1e-12
MAX_SITES = 1 << 28       # the limit include/lb.h states


@pytest.fixture(scope="module")
def lbmod():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2005_12764_b200 import lb
    return lb


def _static(sim):
    import torch
    out = torch.full((3,), -7.0, dtype=torch.float64, device="cuda")   # garbage the call must overwrite
    sim.check_state_static(out)
    return out.cpu().numpy()


def _agree(sim, two=True):
    a = _static(sim)
    b = _static(sim)                      # second call in a row: the shared array holds the first call's sums
    mr, mb = sim.check_state()
    assert a[2] == 0.0 and b[2] == 0.0
    assert np.array_equal(a, b), (a, b)   # fixed summation order: the same bits
    assert abs(a[0] - mr) <= REL * abs(mr), (a, mr)
    if two:
        assert abs(a[1] - mb) <= REL * abs(mb), (a, mb)
    else:
        assert a[1] == 0.0 and mb == 0.0
    return a


@pytest.mark.parametrize("storage", ["ab", "aa"])
@pytest.mark.parametrize("name", ["c4-mini", "c1"])
def test_static_check_matches_check_state(lbmod, name, storage):
    w = W.get(name)                       # c4-mini: walls, 16 blocks of 8192 sites; c1: 64^3
    sim = pu.make_gpu(lbmod, w, storage)
    m0 = pu.masses(w.rho_r, w.rho_b)
    a = _agree(sim)
    if w.solid is None:
        assert abs(a[0] - m0[0]) / m0[0] < 1e-6 and abs(a[1] - m0[1]) / m0[1] < 1e-6
    for n in (1, 4):                      # odd and even step counts (AA: both layouts)
        sim.step(n)
        _agree(sim)


def test_static_check_ragged_single_component_and_two_handles(lbmod):
    rng = np.random.default_rng(5)
    nx, ny, nz = 36, 20, 13               # 9360 sites: one full block and a ragged one
    rho = (1.0 + 0.05 * rng.uniform(-1, 1, (nz, ny, nx))).astype(np.float32)
    u = (0.01 * rng.normal(size=(3, nz, ny, nx))).astype(np.float32)
    w = W.Workload("ragged", nx, ny, nz, 0.9, 0.9, 0.0, 0.0, 0.0, rho, None, u)
    sim = pu.make_gpu(lbmod, w)
    other = pu.make_gpu(lbmod, W.get("c4-mini"))
    a = _agree(sim, two=False)
    assert abs(a[0] - rho.astype(np.float64).sum()) / a[0] < 1e-6
    b = _agree(other)                     # another handle shares the array: nothing of `sim` leaks into it
    sim.step(3)
    assert np.array_equal(_agree(other), b)
    _agree(sim, two=False)


def test_static_check_allocates_nothing(lbmod):
    """No request reaches the allocator hook (PyTorch's caching allocator here) and the driver's
    free memory stays where it was (a cudaMalloc would lower it)."""
    import torch
    sim = pu.make_gpu(lbmod, W.get("c4-mini"))
    out = torch.zeros(3, dtype=torch.float64, device="cuda")
    sim.step(1)
    sim.check_state_static(out)           # first call on this device: resolves the array's address
    torch.cuda.synchronize()
    n0 = torch.cuda.memory_stats()["allocation.all.allocated"]
    free0 = torch.cuda.mem_get_info()[0]
    for _ in range(3):
        sim.step(1)
        sim.check_state_static(out)
    torch.cuda.synchronize()
    assert torch.cuda.memory_stats()["allocation.all.allocated"] == n0
    assert torch.cuda.mem_get_info()[0] == free0
    assert out[2].item() == 0.0 and out[0].item() > 0.0


def test_static_check_counts_non_finite_sites(lbmod):
    w = W.get("c1")
    sim = pu.make_gpu(lbmod, w)
    fr, fb = sim.get_populations(0), sim.get_populations(1)
    fr[3, 5, 6, 7] = np.nan
    fb[0, 9, 9, 9] = np.inf
    sim.set_populations(0, fr)
    sim.set_populations(1, fb)
    with pytest.raises(lbmod.LBError) as ei:
        sim.check_state()
    n_existing = float(re.search(r"([0-9]+) sites hold", str(ei.value)).group(1))
    a = _static(sim)                      # reports, never raises for the state
    assert a[2] == n_existing and a[2] >= 2.0
    assert np.array_equal(a, _static(sim))


def test_static_check_rejects_bad_arguments(lbmod):
    import torch
    out = torch.zeros(3, dtype=torch.float64, device="cuda")
    big = lbmod.LB(1024, 1024, 260)       # 272,629,760 sites > 2^28; lb_create allocates nothing
    with pytest.raises(lbmod.LBError) as ei:
        big.check_state_static(out)
    assert ei.value.code == lbmod.LB_EINVAL and str(MAX_SITES) in str(ei.value) and "maximum" in str(ei.value)
    sim = lbmod.LB(16, 16, 16)
    with pytest.raises(lbmod.LBError) as ei:
        sim.check_state_static(out)       # before lb_init
    assert ei.value.code == lbmod.LB_ESTATE
    sim = pu.make_gpu(lbmod, W.get("c4-mini"))
    with pytest.raises(lbmod.LBError) as ei:
        sim.check_state_static(np.zeros(3))          # a host pointer
    assert ei.value.code == lbmod.LB_EINVAL and "device pointer" in str(ei.value)
    with pytest.raises(lbmod.LBError) as ei:
        sim.check_state_static(None)
    assert ei.value.code == lbmod.LB_EINVAL
