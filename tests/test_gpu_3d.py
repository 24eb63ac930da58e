"""GPU parity of the 3-D variant (pdm3_create / pdm3_migrate; PAPER.md:41, :47;
reading R18) against pdm_oracle_migrate3d, element by element, at the north_star bar."""
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


def _errors(got, ref):
    d = got.astype(np.float64) - ref
    return np.linalg.norm(d) / np.linalg.norm(ref), np.abs(d).max() / np.abs(ref).max()


@pytest.mark.parametrize("model,nx,ny,nz,nw,ntaps", [
    ("field", 70, 19, 5, 3, 3),        # one ragged tile; every sample its own row
    ("white", 300, 20, 4, 5, 7),       # two x-tiles, three y-tiles; 7 x 7 operator
    ("layers", 513, 9, 6, 4, 5),       # odd nx: 8-byte copies; warp-uniform rows
    ("const", 64, 64, 3, 2, 15),       # the longest unrolled operator (15 x 15)
    ("field", 260, 33, 3, 9, 9),       # 9 x 9 runs on the 11 x 11 kernel with zero taps appended; several w groups
    ("field", 1, 1, 4, 2, 3),          # a single trace
])
def test_3d_matches_oracle(pdm, model, nx, ny, nz, nw, ntaps):
    import torch
    cfg = pdm_inputs.random_problem_3d(7, nx, ny, nz, nw, ntaps, model=model)
    ref = oracle.migrate3d(cfg)
    with pdm.Plan3D.from_config(cfg) as plan:
        info = plan.info
        p0 = torch.from_numpy(cfg["P0"]).cuda()
        a = plan.migrate(p0).clone()
        b = plan.migrate(p0).clone()
        torch.cuda.synchronize()
    assert torch.equal(a, b)
    rel, mx = _errors(a.cpu().numpy(), ref)
    assert np.isfinite(a.cpu().numpy()).all() and rel <= 1e-4 and mx <= 1e-3, (rel, mx, info)


@pytest.mark.parametrize("model,nx,ny,nz,nw,ntaps", [
    ("field", 70, 19, 5, 3, 3), ("white", 300, 20, 4, 5, 7), ("layers", 513, 9, 6, 4, 5),
    ("const", 64, 64, 3, 2, 15), ("field", 260, 33, 3, 9, 9), ("layers", 1, 5, 3, 2, 5),
])
def test_3d_doubly_symmetric_operators_run_folded(pdm, model, nx, ny, nz, nw, ntaps):
    """W[ky][kx] = W[-ky][kx] = W[ky][-kx] bit for bit: the folded kernels (rows y-ky and y+ky added while
    loaded, x-sum folded).  The oracle always applies the full (2L+1)^2 operator, so a folding mistake
    (a row pair counted twice, the centre row added to itself, a wrong tap pairing) fails here."""
    import torch
    cfg = pdm_inputs.random_problem_3d(17, nx, ny, nz, nw, ntaps, model=model, symmetric=True)
    t = cfg["table"]
    assert np.array_equal(t, t[:, ::-1, :]) and np.array_equal(t, t[:, :, ::-1])
    ref = oracle.migrate3d(cfg)
    with pdm.Plan3D.from_config(cfg, pdm.PDM_REQUIRE_SYMMETRIC) as plan:
        info = plan.info
        assert info["table_symmetric"] == 1
        img = plan.migrate(torch.from_numpy(cfg["P0"]).cuda())
        torch.cuda.synchronize()
    rel, mx = _errors(img.cpu().numpy(), ref)
    assert rel <= 1e-4 and mx <= 1e-3, (rel, mx, info)
    gen = pdm_inputs.random_problem_3d(17, nx, ny, nz, nw, ntaps, model=model)
    rc, h = pdm.pdm3_create(gen["nx"], gen["ny"], gen["nz"], gen["nw"], gen["dz"], gen["omega"], gen["velocity"],
                            gen["table"], gen["du"], pdm.PDM_REQUIRE_SYMMETRIC)
    assert rc == (pdm.PDM_ERR_TABLE_ASYMMETRIC if ntaps > 1 else pdm.PDM_OK) and h is None


def test_3d_designed_extrapolators_focus_a_diffractor_on_the_device(pdm):
    """A physically meaningful 3-D run: 15 x 15 extrapolators made from the designed 1-D rows
    by the McClellan transformation (pdm_inputs/filters.py::mcclellan_table), laterally varying velocity for
    parity with pdm_oracle_migrate3d, constant velocity for the focusing check of oracle pin T-P6 on the GPU."""
    import torch
    from pdm_inputs import filters
    from pdm_inputs.configs import dft_bin_omegas, ricker_spectrum, diffractor_volume
    nx, ny, nz, dx, dz, v = 56, 48, 40, 10.0, 10.0, 2000.0
    omega = dft_bin_omegas(256, 4e-3, 8.0, 45.0)
    ntab, ntaps = 64, 15
    x, y = np.arange(nx) * dx, np.arange(ny) * dx
    x0, y0, z0 = 310.0, 200.0, 250.0
    P0 = diffractor_volume(omega, ricker_spectrum(omega, 22.0), x, y, x0, y0, z0, v).astype(np.complex64)
    xs, ys = np.meshgrid(x, y)
    models = {"const": np.full((nz, ny, nx), 0.5 * v),
              "field": 0.5 * (v + 400.0 * np.sin(xs / 90.0 + ys / 130.0)[None] + 6.0 * np.arange(nz)[:, None, None])}
    for name, v_in in models.items():
        v_in = np.ascontiguousarray(v_in, dtype=np.float32)
        du = float(omega.max()) * dz / float(v_in.min()) / (ntab - 1)
        table = filters.mcclellan_table(filters.design_table(ntab, ntaps, du, dz / dx))
        cfg = dict(nx=nx, ny=ny, nz=nz, nw=omega.size, dz=dz, dx=dx, dy=dx, du=du, omega=omega, velocity=v_in,
                   table=table, ntab=ntab, ntaps=ntaps, P0=P0)
        ref = oracle.migrate3d(cfg)
        with pdm.Plan3D.from_config(cfg) as plan:
            assert plan.info["table_symmetric"] == 1                   # circularly built: the folded kernels
            img = plan.migrate(torch.from_numpy(P0).cuda()).cpu().numpy()
        rel, mx = _errors(img, ref)
        assert rel <= 1e-4 and mx <= 1e-3, (name, rel, mx)
        if name == "const":
            iz, iy, ix = np.unravel_index(np.argmax(np.abs(img)), img.shape)
            assert abs(ix - round(x0 / dx)) <= 1 and abs(iy - round(y0 / dx)) <= 1 and abs(iz - (round(z0 / dz) - 1)) <= 1


def test_3d_force_general_and_unaligned_input(pdm):
    import torch
    cfg = pdm_inputs.random_problem_3d(9, 200, 12, 4, 3, 5, model="layers")
    ref = oracle.migrate3d(cfg)
    with pdm.Plan3D.from_config(cfg) as fast, pdm.Plan3D.from_config(cfg, pdm.PDM_FORCE_GENERAL) as gen:
        p0 = torch.from_numpy(cfg["P0"]).cuda()
        store = torch.empty(p0.numel() + 1, dtype=p0.dtype, device="cuda")
        shifted = store[1:].view(p0.shape)
        shifted.copy_(p0)
        assert shifted.data_ptr() % 16 == 8
        a = fast.migrate(p0).clone()
        b = gen.migrate(p0).clone()
        c = fast.migrate(shifted).clone()
        torch.cuda.synchronize()
    assert torch.equal(a, b) and torch.equal(a, c)
    rel, mx = _errors(a.cpu().numpy(), ref)
    assert rel <= 1e-4 and mx <= 1e-3, (rel, mx)


def test_3d_error_codes(pdm):
    cfg = pdm_inputs.random_problem_3d(3, 16, 8, 2, 2, 3)
    args = (cfg["nx"], cfg["ny"], cfg["nz"], cfg["nw"], cfg["dz"], cfg["omega"], cfg["velocity"])
    rc, h = pdm.pdm3_create(*args, np.zeros((4, 17, 17), np.complex64), cfg["du"])      # 17 x 17: no unrolled kernel
    assert rc == pdm.PDM_ERR_UNSUPPORTED and h is None
    rc, h = pdm.pdm3_create(*args, cfg["table"][:, :2, :2], cfg["du"])                   # even ntaps
    assert rc == pdm.PDM_ERR_INVALID_ARG and h is None
    rc, h = pdm.pdm3_create(*args, cfg["table"], cfg["du"] * 0.5)                         # table too short
    assert rc == pdm.PDM_ERR_TABLE_RANGE and h is None


@pytest.mark.slow
@pytest.mark.parametrize("model,ntaps", [("layers", 7), ("field", 7), ("field", 15)])
def test_3d_at_bench_tile_counts(pdm, model, ntaps):
    """The `bench.py --3d` lateral size (256 x 256: 32 y-tiles, several frequency groups, the staged slice
    for the field model) on a shortened depth / frequency range the oracle finishes in seconds."""
    import torch
    cfg = pdm_inputs.random_problem_3d(5, 256, 256, 6, 5, ntaps, model=model)
    ref = oracle.migrate3d(cfg)
    with pdm.Plan3D.from_config(cfg) as plan:
        img = plan.migrate(torch.from_numpy(cfg["P0"]).cuda())
        torch.cuda.synchronize()
    rel, mx = _errors(img.cpu().numpy(), ref)
    assert rel <= 1e-4 and mx <= 1e-3, (rel, mx)


def test_3d_and_prestack_are_cuda_graph_capturable(pdm):
    """pdm3_migrate and pdm_migrate_shot only enqueue work (per-step launches; the cooperative packed
    kernel plus its interleave kernel): capture and replay."""
    import torch
    cfg3 = pdm_inputs.random_problem_3d(21, 130, 17, 4, 3, 5, model="field")
    cfg2 = pdm_inputs.random_problem(22, 900, 7, 6, 15, model="field")
    rng = np.random.default_rng(1)
    S0 = (rng.standard_normal((6, 900)) + 1j * rng.standard_normal((6, 900))).astype(np.complex64)
    with pdm.Plan3D.from_config(cfg3) as p3, pdm.Plan.from_config(cfg2, pdm.PDM_PRESTACK) as p2:
        a3 = torch.from_numpy(cfg3["P0"]).cuda()
        s, r = torch.from_numpy(S0).cuda(), torch.from_numpy(cfg2["P0"]).cuda()
        ref3 = p3.migrate(a3).clone()
        ref2 = p2.migrate_shot(s, r).clone()
        img3, img2 = torch.zeros_like(ref3), torch.zeros_like(ref2)
        torch.cuda.synchronize()
        st = torch.cuda.Stream()
        with torch.cuda.stream(st):
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g, stream=st):
                p3.migrate(a3, img3, stream=st)
                p2.migrate_shot(s, r, img2, stream=st)
        img3.zero_(); img2.zero_()
        torch.cuda.synchronize()
        g.replay()
        torch.cuda.synchronize()
        assert torch.equal(img3, ref3) and torch.equal(img2, ref2)
