"""rr_orbit_z_noalloc: the allocation-free variant of kernel 2 (scratch in a static device array,
include/roadrunner.h) against the existing rr_orbit_z, on two calls in a row.

Collected last on purpose (the suite runs with `pytest -x`: a failure here must not hide other
tests); passes alone in a fresh process and after the other GPU tests."""
import numpy as np
import pytest

import workloads

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def rr():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device (there is no CPU fallback)")
    import paper_2009_08500_b200 as m
    m.load()
    return m


def _tol(z):
    # the bar tests/test_gpu_parity.py holds rr_orbit_z to against the oracle; the two paths run the
    # same kernels, so they are expected to agree exactly
    return 1e-11 * max(1.0, float(np.nanmax(np.abs(z))))


@pytest.mark.parametrize("fp32_math", [False, True])
def test_no_alloc_orbit_matches_the_allocating_path_twice(rr, fp32_math):
    import torch
    wl = workloads.make_workload(3, npv=300, npt=6 * 150)       # eccentric, 6 light curves, ns up to 30
    gm = rr.RoadRunner.from_config(wl.model)
    gm.set_data(wl.times, wl.lc_index, wl.passband_index, wl.supersampling, wl.exposure_time)
    nsub = rr.rr_num_subsamples(gm.ctx)
    pv_a = wl.pv.copy()
    pv_a[7, 0] = 0.5                                            # an invalid row: NaN in both paths
    pv_b = np.ascontiguousarray(wl.pv[::-1][:211])              # second call: other rows, fewer of them
    refs = [gm.orbit_z(p, fp32_math=fp32_math).cpu().numpy() for p in (pv_a, pv_b)]
    torch.cuda.synchronize()
    outs = []
    for p in (pv_a, pv_b):                                      # two calls in a row, shared scratch
        pv_d = torch.as_tensor(p).cuda()
        z = torch.full((p.shape[0], nsub), -7.0, dtype=torch.float64, device="cuda")
        rr.rr_orbit_z_noalloc(gm.ctx, pv_d, z, fp32_math=fp32_math)
        outs.append(z)
    torch.cuda.synchronize()
    for ref, out in zip(refs, outs):
        got = out.cpu().numpy()
        assert got.shape == ref.shape
        assert np.array_equal(np.isnan(got), np.isnan(ref))
        ok = ~np.isnan(ref)
        assert np.max(np.abs(got[ok] - ref[ok])) <= _tol(ref)
        assert (np.abs(ref[ok]) < 1.2).sum() > 100              # transits are in the sample
    assert np.isnan(outs[0].cpu().numpy()[7]).all()
    # the first call again after the second: the stale rows of call two do not leak; with its tensors
    # made beforehand the device's free memory is the same before and after the call (no allocation)
    pv_d = torch.as_tensor(pv_a).cuda()
    z = torch.empty((pv_a.shape[0], nsub), dtype=torch.float64, device="cuda")
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    rr.rr_orbit_z_noalloc(gm.ctx, pv_d, z, fp32_math=fp32_math)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0
    assert torch.equal(torch.nan_to_num(z, nan=-1.0), torch.nan_to_num(outs[0], nan=-1.0))
    gm.close()


def test_no_alloc_orbit_rejects_sizes_beyond_the_static_scratch(rr):
    import torch
    wl = workloads.make_workload(1, npv=4, npt=64)
    gm = rr.RoadRunner.from_config(wl.model)
    gm.set_data(wl.times, wl.lc_index, wl.passband_index, wl.supersampling, wl.exposure_time)
    nsub = rr.rr_num_subsamples(gm.ctx)
    limit = 7709                                                # roadrunner.h: one k per pv
    assert ((200 * limit + 255) // 256) * 256 + 72 * limit <= rr.RR_NOALLOC_SCRATCH_BYTES \
        < ((200 * (limit + 1) + 255) // 256) * 256 + 72 * (limit + 1)
    pv = torch.as_tensor(np.tile(wl.pv, (limit // 4 + 2, 1))[:limit + 1]).cuda()
    z = torch.zeros((limit + 1, nsub), dtype=torch.float64, device="cuda")
    with pytest.raises(rr.RoadRunnerError) as e:
        rr.rr_orbit_z_noalloc(gm.ctx, pv, z)
    assert e.value.code == rr.RR_ESCRATCH and "static scratch" in str(e.value)
    assert float(z.abs().sum()) == 0.0                          # nothing was launched
    rr.rr_orbit_z_noalloc(gm.ctx, pv[:limit].contiguous(), z[:limit])   # the limit itself fits
    ref = gm.orbit_z(pv[:limit].contiguous())
    assert torch.equal(z[:limit], ref)
    gm.close()
