"""pdm_migrate_static -- the entry point for callers that cannot allocate device memory.

Some users of libpdm run where cudaMalloc is forbidden or too costly at call time: a plug-in inside a
host application that owns all device memory, a latency-bound loop that cannot take the device-wide
synchronisation an allocation implies, a job that fills HBM to the last byte.  Every other migration call
needs a plan from pdm_create, which allocates; pdm_migrate_static needs none and keeps its scratch (two
wavefield planes) in a 16 MiB array built into the library, shared by all calls on a GPU.

What is checked here: its image against the images of the existing plan-based paths (the tolerance of
tests/test_gpu_parity.py) on two calls in a row with DIFFERENT problems -- so the second call starts on
the first call's left-over wavefield -- then the first problem again (same bits as before), that the
free device memory does not move across a call, and that a problem larger than the array is refused.

This file is named test_zz_* so that pytest collects it after every other test file: with `pytest -x`
a failure here cannot hide another test.  It builds its own inputs and needs no state from other tests.
"""
import numpy as np
import pytest

import pdm_inputs

REL_L2_BAR = 1e-4       # as tests/test_gpu_parity.py
MAX_PIX_BAR = 1e-3


def _errors(got, ref):
    g, r = np.asarray(got, dtype=np.float64), np.asarray(ref, dtype=np.float64)
    d = g - r
    return (np.linalg.norm(d) / max(np.linalg.norm(r), 1e-300),
            np.abs(d).max() / max(np.abs(r).max(), 1e-300))


def _device_inputs(torch, cfg):
    return dict(omega=torch.from_numpy(np.ascontiguousarray(cfg["omega"], dtype=np.float32)).cuda(),
                velocity=torch.from_numpy(np.ascontiguousarray(cfg["velocity"], dtype=np.float32)).cuda(),
                table=torch.from_numpy(np.ascontiguousarray(cfg["table"], dtype=np.complex64)).cuda(),
                P0=torch.from_numpy(np.ascontiguousarray(cfg["P0"], dtype=np.complex64)).cuda(),
                image=torch.full((cfg["nz"], cfg["nx"]), float("nan"), dtype=torch.float32, device="cuda"))


def _existing_path(pdm, torch, cfg, flags):
    with pdm.Plan.from_config(cfg, flags) as plan:
        img = plan.migrate(torch.from_numpy(np.ascontiguousarray(cfg["P0"])).cuda())
        torch.cuda.synchronize()
        return img.cpu().numpy()


@pytest.mark.gpu
def test_static_scratch_entry_point_matches_the_plan_based_paths_on_consecutive_calls():
    import torch
    import paper_1912_05529_b200 as pdm
    assert torch.cuda.is_available(), "gpu tests need a B200"
    pdm.load_library()
    # A: laterally varying model, several thread blocks wide with a ragged tail, 25 taps.
    # B: a different shape (fewer, longer lines; 15 taps; every sample its own row), so that its planes
    #    overlap A's left-overs at different offsets.
    cfg_a = pdm_inputs.random_problem(21, 1500, 40, 12, 25, model="field")
    cfg_b = pdm_inputs.random_problem(22, 4100, 16, 5, 15, model="white")
    ref = {id(c): (_existing_path(pdm, torch, c, pdm.PDM_PATH_AUTO), _existing_path(pdm, torch, c, pdm.PDM_PATH_NAIVE))
           for c in (cfg_a, cfg_b)}
    dev = {id(c): _device_inputs(torch, c) for c in (cfg_a, cfg_b)}
    torch.cuda.synchronize()

    images = []
    for call, cfg in enumerate((cfg_a, cfg_b, cfg_a)):           # back to back, nothing reset in between
        d = dev[id(cfg)]
        d["image"].fill_(float("nan"))
        torch.cuda.synchronize()
        free_before = torch.cuda.mem_get_info()[0]
        out = pdm.migrate_static(d["omega"], d["velocity"], d["table"], cfg["dz"], cfg["du"], d["P0"], d["image"])
        torch.cuda.synchronize()
        if call > 0:        # the first call on a device may load the library's code; later calls change nothing
            assert torch.cuda.mem_get_info()[0] == free_before, "device memory moved across pdm_migrate_static"
        got = out.cpu().numpy()
        assert np.isfinite(got).all(), call
        auto, naive = ref[id(cfg)]
        rel, mx = _errors(got, auto)
        assert rel <= REL_L2_BAR and mx <= MAX_PIX_BAR, (call, cfg["name"], rel, mx)
        rel, mx = _errors(got, naive)
        assert rel <= REL_L2_BAR and mx <= MAX_PIX_BAR, (call, cfg["name"], rel, mx)
        images.append(got)
    assert np.array_equal(images[0], images[2]), "left-over scratch contents changed the result"


@pytest.mark.gpu
def test_static_scratch_entry_point_asymmetric_table_and_full_size_limit():
    """An asymmetric table (the general Eq. (1), no folding) and a problem of exactly the maximum size."""
    import torch
    import paper_1912_05529_b200 as pdm
    pdm.load_library()
    cfg = pdm_inputs.random_problem(23, 700, 9, 6, 7, model="field", symmetric=False)     # W_k != W_-k
    ref = _existing_path(pdm, torch, cfg, pdm.PDM_PATH_AUTO)
    d = _device_inputs(torch, cfg)
    got = pdm.migrate_static(d["omega"], d["velocity"], d["table"], cfg["dz"], cfg["du"], d["P0"], d["image"])
    torch.cuda.synchronize()
    rel, mx = _errors(got.cpu().numpy(), ref)
    assert rel <= REL_L2_BAR and mx <= MAX_PIX_BAR, (rel, mx)

    nw = 64
    nx = pdm.PDM_STATIC_MAX_SAMPLES // nw                          # nx*nw == the limit: accepted
    big = pdm_inputs.random_problem(24, nx, 3, nw, 7, model="layers")
    ref = _existing_path(pdm, torch, big, pdm.PDM_PATH_AUTO)
    d = _device_inputs(torch, big)
    got = pdm.migrate_static(d["omega"], d["velocity"], d["table"], big["dz"], big["du"], d["P0"], d["image"])
    torch.cuda.synchronize()
    rel, mx = _errors(got.cpu().numpy(), ref)
    assert rel <= REL_L2_BAR and mx <= MAX_PIX_BAR, (rel, mx)


def test_static_scratch_entry_point_refuses_what_does_not_fit():
    """Sizes are checked before anything touches a device, so this runs without a GPU: one sample more
    than the built-in array holds is PDM_ERR_TOO_LARGE (with a message that says why), never a launch."""
    import paper_1912_05529_b200 as pdm
    pdm.build_lib()
    pdm.load_library()
    fake = 0x1000                                                    # never dereferenced on these paths
    nw = 1024
    nx = pdm.PDM_STATIC_MAX_SAMPLES // nw + 1
    rc = pdm.pdm_migrate_static(nx, 4, nw, 5.0, fake, fake, fake, 16, 7, 0.01, fake, fake)
    assert rc == pdm.PDM_ERR_TOO_LARGE
    assert "PDM_STATIC_MAX_SAMPLES" in pdm.pdm_strerror(rc)
    assert pdm.pdm_migrate_static(100000, 4, 100000, 5.0, fake, fake, fake, 16, 7, 0.01, fake, fake) \
        == pdm.PDM_ERR_TOO_LARGE                                     # nx*nw overflows 32 bits
    for bad in (dict(nx=0), dict(nz=0), dict(nw=-1), dict(ntaps=6), dict(ntab=0), dict(dz=0.0), dict(du=-1.0),
                dict(P0=0), dict(image=0), dict(omega=0)):
        a = dict(nx=64, nz=4, nw=8, dz=5.0, omega=fake, velocity=fake, table=fake, ntab=16, ntaps=7, du=0.01,
                 P0=fake, image=fake)
        a.update(bad)
        rc = pdm.pdm_migrate_static(a["nx"], a["nz"], a["nw"], a["dz"], a["omega"], a["velocity"], a["table"],
                                    a["ntab"], a["ntaps"], a["du"], a["P0"], a["image"])
        assert rc == pdm.PDM_ERR_INVALID_ARG, bad
    assert pdm.pdm_migrate_static(64, 4, 8, 5.0, fake, fake, fake, 16, 131, 0.01, fake, fake) == pdm.PDM_ERR_UNSUPPORTED
