"""GPU parity of the prestack (shot-profile) variant, pdm_migrate_shot (
reading R17), against pdm_oracle_migrate_shot, element by element, at the north_star bar
(rel-L2 <= 1e-4, per-pixel <= 1e-3 of the image maximum)."""
import numpy as np
import pytest

import oracle
import pdm_inputs

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def pdm():
    import torch
    import paper_1912_05529_b200 as m
    assert torch.cuda.is_available(), "gpu tests need a B200"
    m.load_library()
    return m


def _fields(rng, nw, nx):
    def c():
        return (rng.standard_normal((nw, nx)) + 1j * rng.standard_normal((nw, nx))).astype(np.complex64)
    return c(), c()


def _errors(got, ref):
    d = got.astype(np.float64) - ref
    return np.linalg.norm(d) / np.linalg.norm(ref), np.abs(d).max() / np.abs(ref).max()


@pytest.mark.parametrize("T", [0, 1, 3])
@pytest.mark.parametrize("model,nx,nz,nw,ntaps,sym", [
    ("field", 300, 21, 7, 15, True),      # 14 lines: one full pack and a ragged one; nx below one tile
    ("white", 1000, 13, 10, 25, True),    # 3 x-tiles, every sample its own row
    ("layers", 2501, 10, 5, 7, True),     # odd nx, thread-uniform rows
    ("field", 700, 9, 8, 31, False),      # asymmetric table: the conjugate operator is NOT the mirrored one
    ("const", 129, 17, 3, 51, True),
])
def test_shot_matches_oracle(pdm, T, model, nx, nz, nw, ntaps, sym):
    import torch
    cfg = pdm_inputs.random_problem(53, nx, nz, nw, ntaps, model=model, symmetric=sym)
    rng = np.random.default_rng(nx + nw)
    S0, R0 = _fields(rng, nw, nx)
    ref = oracle.migrate_shot(cfg, S0, R0)
    flags = pdm.PDM_PRESTACK | ((pdm.PDM_PATH_PACKED | (T << pdm.PDM_CTAS_SHIFT)) if T else 0)
    with pdm.Plan.from_config(cfg, flags) as plan:
        info = plan.info
        assert info["path"] == pdm.PDM_PATH_PACKED and info["nw"] == nw
        s, r = torch.from_numpy(S0).cuda(), torch.from_numpy(R0).cuda()
        a = plan.migrate_shot(s, r).clone()
        b = plan.migrate_shot(s, r).clone()
        torch.cuda.synchronize()
        assert torch.equal(a, b)
        rel, mx = _errors(a.cpu().numpy(), ref)
        assert rel <= 1e-4 and mx <= 1e-3, (rel, mx, info)
        # the poststack call is refused on a prestack plan
        assert pdm.pdm_migrate(plan._h, r.data_ptr(), a.data_ptr(), 0) == pdm.PDM_ERR_INVALID_ARG


def test_shot_with_row_ranges_wider_than_any_slice_buffer(pdm):
    """Prestack plans have no other kernel form to fall back to: with 51 taps, 1024 table rows and
    independent samples (row range of a pack ~700 > the ~518 rows a slice holds) the plan must still
    exist -- on the build that reads tap rows from the global table."""
    import torch
    nx, nz, nw = 1100, 6, 9
    cfg = pdm_inputs.random_problem(71, nx, nz, nw, 51, ntab=1024, model="white")
    S0, R0 = _fields(np.random.default_rng(3), nw, nx)
    ref = oracle.migrate_shot(cfg, S0, R0)
    with pdm.Plan.from_config(cfg, pdm.PDM_PRESTACK) as plan:
        info = plan.info
        assert info["path"] == pdm.PDM_PATH_PACKED and info["taps_mode"] == 1, info
        a = plan.migrate_shot(torch.from_numpy(S0).cuda(), torch.from_numpy(R0).cuda())
        torch.cuda.synchronize()
        rel, mx = _errors(a.cpu().numpy(), ref)
    assert rel <= 1e-4 and mx <= 1e-3, (rel, mx, info)


@pytest.mark.parametrize("sym,T", [(True, 1), (False, 4)])
def test_shot_many_items_per_cta(pdm, sym, T):
    """~45 tiles x 8 packs on 148 CTAs: several items per CTA and depth block in the cross-correlation mode."""
    import torch
    nx, nz, nw = 20011, 5, 31
    cfg = pdm_inputs.random_problem(73, nx, nz, nw, 7, model="field", symmetric=sym)
    S0, R0 = _fields(np.random.default_rng(5), nw, nx)
    ref = oracle.migrate_shot(cfg, S0, R0)
    with pdm.Plan.from_config(cfg, pdm.PDM_PRESTACK | pdm.PDM_PATH_PACKED | (T << pdm.PDM_CTAS_SHIFT)) as plan:
        info = plan.info
        a = plan.migrate_shot(torch.from_numpy(S0).cuda(), torch.from_numpy(R0).cuda())
        torch.cuda.synchronize()
        rel, mx = _errors(a.cpu().numpy(), ref)
    assert rel <= 1e-4 and mx <= 1e-3, (rel, mx, info)


def test_shots_accumulate_into_one_image(pdm):
    import torch
    cfg = pdm_inputs.random_problem(59, 900, 14, 12, 25, model="field")
    rng = np.random.default_rng(4)
    shots = [_fields(rng, 12, 900) for _ in range(3)]
    ref = None
    for S0, R0 in shots:
        ref = oracle.migrate_shot(cfg, S0, R0, image=ref)
    with pdm.Plan.from_config(cfg, pdm.PDM_PRESTACK) as plan:
        img = None
        for S0, R0 in shots:
            img = plan.migrate_shot(torch.from_numpy(S0).cuda(), torch.from_numpy(R0).cuda(), image=img,
                                    accumulate=img is not None)
        torch.cuda.synchronize()
        rel, mx = _errors(img.cpu().numpy(), ref)
    assert rel <= 1e-4 and mx <= 1e-3, (rel, mx)


def test_prestack_argument_errors(pdm):
    import torch
    cfg = pdm_inputs.random_problem(61, 200, 5, 4, 15, model="layers")
    args = (cfg["nx"], cfg["nz"], cfg["nw"], cfg["dx"], cfg["dz"], cfg["omega"], cfg["velocity"], cfg["table"], cfg["du"])
    rc, h = pdm.pdm_create(*args, pdm.PDM_PRESTACK | pdm.PDM_PATH_SMEM)     # only the packed form does it
    assert rc == pdm.PDM_ERR_INVALID_ARG and h is None
    with pdm.Plan.from_config(cfg, 0) as plan:                              # a poststack plan refuses shots
        z = torch.zeros((4, 200), dtype=torch.complex64, device="cuda")
        img = torch.zeros((5, 200), dtype=torch.float32, device="cuda")
        assert pdm.pdm_migrate_shot(plan._h, z.data_ptr(), z.data_ptr(), img.data_ptr(), False, 0) == pdm.PDM_ERR_INVALID_ARG


@pytest.mark.slow
def test_shot_at_bench_size_sampled_frequencies(pdm):
    """The `bench.py --prestack` configuration (configs[4] field, nx = 4096, nw = 1024, 25 taps, AUTO T and
    CTA size): 16 sampled frequencies carry data (first / last, pack boundaries, CTA range boundaries), the
    other lines are zero, so the oracle only has to march those."""
    import torch
    from pdm_inputs.configs import sweep_point
    cfg = sweep_point(4096, 1024, 25)
    nw, nx = cfg["nw"], cfg["nx"]
    lines = sorted({0, 1, 7, 8, 9, 511, 512, 1015, 1016, 1023, 137, 138, 300, 666, 777, 901})
    rng = np.random.default_rng(99)
    S0 = np.zeros((nw, nx), np.complex64); R0 = np.zeros((nw, nx), np.complex64)
    s, r = _fields(rng, len(lines), nx)
    S0[lines] = s; R0[lines] = r
    sub = dict(cfg, nw=len(lines), omega=cfg["omega"][lines])
    ref = oracle.migrate_shot(sub, s, r)
    with pdm.Plan.from_config(cfg, pdm.PDM_PRESTACK) as plan:
        img = plan.migrate_shot(torch.from_numpy(S0).cuda(), torch.from_numpy(R0).cuda())
        torch.cuda.synchronize()
        rel, mx = _errors(img.cpu().numpy(), ref)
    assert rel <= 1e-4 and mx <= 1e-3, (rel, mx)
