"""GPU test of pdv_mc_run_static, the run entry point that allocates no device memory (include/pdv.h).

Why the entry point exists: pdv_mc_run takes its per-call workspace from the device's memory pool.  A host program that has
already given all HBM to its own arena (a hydrocode running this library as an in-situ diagnostic, a framework whose caching
allocator owns the device) cannot afford that -- the pool may have nothing left, or growing it starves the host program -- and a
real-time caller wants the library's footprint fixed at load time.  pdv_mc_run_static therefore works in a fixed 2 MiB array
inside the library, shared by all calls on a device.

What is checked: on two calls in a row, of different shapes and seeds so that the second finds the first one's cursors and
tallies in the array, every output (hist, hist2, stats) equals pdv_mc_run's bit for bit -- the tallies are integer fixed point
and both paths launch the same kernels, so equality is the tolerance this suite uses for such pairs; that the free device
memory does not shrink across a call; and that requests beyond the array, gas clouds and host outputs are refused with a clear
message.  The file name sorts last on purpose: the test shares nothing with the others, and under `pytest -x` a failure here
must not hide them.
"""
import numpy as np
import pytest

import pdv_workloads as W

pytestmark = [pytest.mark.gpu, pytest.mark.usefixtures("_library_is_built")]


@pytest.fixture(scope="module")
def P():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2012_00963_b200 import build as pbuild
    pbuild.build()
    import paper_2012_00963_b200 as P
    return P


def _device_outputs(P, n_clouds, n_snap, n_bins):
    import torch
    dev = torch.device("cuda", torch.cuda.current_device())
    # filled with a pattern: whatever the call does not write would show
    hist = torch.full((n_clouds, n_snap, n_bins), -7.0, dtype=torch.float64, device=dev)
    hist2 = torch.full((n_clouds, n_snap, n_bins), -7.0, dtype=torch.float64, device=dev)
    stats = torch.full((n_clouds * n_snap * P.STATS_DTYPE.itemsize,), 0xAB, dtype=torch.uint8, device=dev)
    return hist, hist2, stats


def _both_paths(P, clouds, t_snap, n, seed, run):
    """-> ((hist, hist2, stats) of pdv_mc_run with device outputs, the same of pdv_mc_run_static), as numpy."""
    import torch
    out = []
    for call in (P.pdv_mc_run_device, P.pdv_mc_run_static):
        h, h2, st = _device_outputs(P, len(clouds), len(t_snap), run["n_bins"])
        call(clouds, t_snap, n, seed, run, h, h2, st)
        torch.cuda.synchronize()
        out.append((h.cpu().numpy(), h2.cpu().numpy(),
                    st.cpu().numpy().view(P.STATS_DTYPE).reshape(len(clouds), len(t_snap))))
    return out


def _assert_identical(ref, got):
    for a, b, name in zip(ref, got, ("hist", "hist2", "stats")):
        assert a.tobytes() == b.tobytes(), f"{name} of pdv_mc_run_static differs from pdv_mc_run"


def test_two_calls_in_a_row_match_the_allocating_path(P):
    import torch
    torch.cuda.set_device(0)
    mono = W.config(1)                                        # 5 um, 2 mg/cm^2 (the headline cloud)
    poly = W.scaled(W.config(2), 150_000, n_snap=3)           # 16 size classes, three snapshots in one launch
    c_mono = P.pdv_cloud_create(mono["clouds"][0])            # set-up: creating a cloud uploads it (and allocates)
    c_poly = P.pdv_cloud_create(poly["clouds"][0])

    # first call on this device (it also looks up the array's address): 3 units x 512 bins, 16-class kernel
    ref, got = _both_paths(P, [c_poly], poly["t_snap"], 150_000, 31, poly["run"])
    _assert_identical(ref, got)
    assert int(got[2]["histories"].sum()) == 3 * 150_000 and got[0].sum() > 0

    # second call, straight after: other kernel instantiation, ONE unit, 128 bins, other seed and id range, roulette on.
    # The array still holds call one's cursors (at 150 000) and tallies; had they not been cleared, unit 0 would start
    # with no photons left and bins full of the other spectrum.
    run2 = dict(mono["run"], n_bins=128, first_photon_id=12345, max_events=6, roulette_survival=0.25)
    h, h2, st = _device_outputs(P, 1, 1, 128)                 # the caller's buffers exist before the measurement
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    P.pdv_mc_run_static([c_mono], mono["t_snap"], 400_037, 77, run2, h, h2, st)
    torch.cuda.synchronize()
    free_after = torch.cuda.mem_get_info()[0]
    assert free_after >= free_before, f"device memory shrank by {free_before - free_after} bytes across a pdv_mc_run_static call"
    ref, got = _both_paths(P, [c_mono], mono["t_snap"], 400_037, 77, run2)
    _assert_identical(ref, got)
    assert got[0].tobytes() == h.cpu().numpy().tobytes()      # and the call is reproducible
    assert int(got[2]["histories"][0, 0]) == 400_037
    s = got[2][0, 0]
    resid = (s["detected"] + s["underflow"] + s["overflow"] + s["escaped"] + s["absorbed_particles"] + s["absorbed_surface"]
             + s["roulette_killed"] - s["roulette_gained"] + s["truncated"] - float(s["histories"]))
    assert resid == 0.0

    # an empty run leaves zeros, not the previous call's tallies
    h, h2, st = _device_outputs(P, 1, 1, 128)
    P.pdv_mc_run_static([c_mono], mono["t_snap"], 0, 77, run2, h, h2, st)
    torch.cuda.synchronize()
    assert float(h.abs().sum()) == 0.0 and float(h2.abs().sum()) == 0.0
    assert not st.cpu().numpy().any()


def test_requests_the_array_cannot_serve_are_refused(P):
    import torch
    torch.cuda.set_device(0)
    mono = W.config(1)
    c = P.pdv_cloud_create(mono["clouds"][0])
    # 40 snapshots x 4096 bins: 40 * 16 * 4096 bytes of tallies alone exceed the 2 MiB array
    run = dict(mono["run"], n_bins=4096)
    t = [1e-6 * (k + 1) for k in range(40)]
    h, h2, st = _device_outputs(P, 1, 40, 4096)
    with pytest.raises(P.PdvError) as e:
        P.pdv_mc_run_static([c], t, 1000, 1, run, h, h2, st)
    assert e.value.status == 4 and "static array holds" in str(e.value) and str(P.PDV_STATIC_SCRATCH_BYTES) in str(e.value)
    assert float(h[0, 0, 0]) == -7.0                          # outputs untouched on failure
    # the same request is fine for the allocating path
    P.pdv_mc_run_device([c], t, 1000, 1, run, h, h2, st)
    torch.cuda.synchronize()
    assert float(h.min()) >= 0.0
    # a cloud in a gas environment needs per-call uploads
    gas = P.pdv_cloud_create(dict(mono["clouds"][0], gas_density=1.2, drag_coefficient=0.5, n_depth_bins=256))
    h, h2, st = _device_outputs(P, 1, 1, 512)
    with pytest.raises(P.PdvError) as e:
        P.pdv_mc_run_static([gas], mono["t_snap"], 1000, 1, mono["run"], h, h2, st)
    assert e.value.status == 4 and "gas" in str(e.value)
