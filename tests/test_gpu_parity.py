"""GPU parity: the CUDA path (through the C ABI) against the FP64 oracle, element by element.

Bar (BASELINE.json north_star): relative L2 error <= 1e-4 over the whole image and per-pixel
error <= 1e-3 of the image maximum.  The table index is taken in FP32 on both sides (reading
R3), so the only differences are FP32 rounding and summation order (reading R13).
"""
import numpy as np
import pytest

import oracle
import pdm_inputs

pytestmark = pytest.mark.gpu

REL_L2_BAR = 1e-4
MAX_PIX_BAR = 1e-3


@pytest.fixture(scope="module")
def pdm():
    import torch
    import paper_1912_05529_b200 as m
    assert torch.cuda.is_available(), "gpu tests need a B200"
    m.load_library()           # raises if libpdm.so is missing: no fallback
    return m


def errors(gpu_img, ref):
    g = np.asarray(gpu_img, dtype=np.float64)
    d = g - ref
    rel = np.linalg.norm(d) / max(np.linalg.norm(ref), 1e-300)
    mx = np.abs(d).max() / max(np.abs(ref).max(), 1e-300)
    return rel, mx


def gpu_migrate(pdm, cfg, flags=0, P0=None, want_info=False):
    import torch
    with pdm.Plan.from_config(cfg, flags) as plan:
        p0 = torch.from_numpy(np.ascontiguousarray(cfg["P0"] if P0 is None else P0)).cuda()
        img = plan.migrate(p0)
        torch.cuda.synchronize()
        out = img.cpu().numpy()
        info = plan.info
    return (out, info) if want_info else out


def assert_parity(pdm, cfg, flags=0, ref=None, expect_path=None):
    img, info = gpu_migrate(pdm, cfg, flags, want_info=True)
    if expect_path is not None:
        assert info["path"] == expect_path, info
    ref = oracle.migrate(cfg) if ref is None else ref
    rel, mx = errors(img, ref)
    assert np.isfinite(img).all()
    assert rel <= REL_L2_BAR and mx <= MAX_PIX_BAR, (cfg["name"], flags, rel, mx, info)
    return rel, mx


PATHS = ["naive", "smem_global", "smem_staged", "tiled", "cluster", "packed"]


def path_flags(pdm, name):
    return {"naive": pdm.PDM_PATH_NAIVE,
            "smem_global": pdm.PDM_PATH_SMEM | pdm.PDM_TAPS_GLOBAL,
            "smem_staged": pdm.PDM_PATH_SMEM | pdm.PDM_TAPS_SLICE,
            "tiled": pdm.PDM_PATH_TILED,
            "cluster": pdm.PDM_PATH_CLUSTER,
            "packed": pdm.PDM_PATH_PACKED}[name]


# ---------------------------------------------------------------- every kernel form, small inputs
@pytest.mark.parametrize("path", PATHS)
@pytest.mark.parametrize("model,nx,nz,nw,ntaps", [
    ("field", 300, 40, 7, 15),        # ragged tail: nx not a multiple of the 8-sample group
    ("white", 1000, 24, 5, 25),       # every sample its own table row (general gather path)
    ("layers", 2500, 30, 6, 31),      # warp-uniform rows; several tiles in the tiled form
    ("const", 129, 50, 3, 35),        # one sample past a group boundary
    ("field", 4100, 12, 4, 51),       # two passes per depth step in the SMEM form, 3 x-tiles
])
def test_every_path_matches_oracle(pdm, path, model, nx, nz, nw, ntaps):
    cfg = pdm_inputs.random_problem(11, nx, nz, nw, ntaps, model=model)
    assert_parity(pdm, cfg, path_flags(pdm, path))


@pytest.mark.parametrize("path", PATHS)
@pytest.mark.parametrize("L", [1, 2, 3])
def test_short_filters_and_tiny_grids(pdm, path, L):
    for seed, nx in ((1, 9), (2, 1), (3, 17), (4, 64)):
        cfg = pdm_inputs.tiny_random_problem(seed, nx=nx, nz=5, nw=3, L=L, ntab=9)
        assert_parity(pdm, cfg, path_flags(pdm, path))


def test_filter_lengths_without_their_own_unrolled_kernel(pdm):
    """Lengths between two instantiations run on the next longer one with zero taps appended (every
    kernel form); lengths beyond the longest fall back to the scaffold."""
    for L, nx in ((5, 40), (10, 333), (20, 1200), (24, 2600)):     # -> kernels for L = 7, 12, 25, 25
        cfg = pdm_inputs.tiny_random_problem(7 + L, nx=nx, nz=6, nw=3, L=L, ntab=11)
        ref = oracle.migrate(cfg)
        assert_parity(pdm, cfg, 0, ref=ref, expect_path=pdm.PDM_PATH_SMEM)
        for path in ("smem_global", "tiled", "cluster"):
            assert_parity(pdm, cfg, path_flags(pdm, path), ref=ref)
    cfg = pdm_inputs.tiny_random_problem(9, nx=50, nz=4, nw=2, L=30, ntab=9)   # 61 taps: longer than any
    assert_parity(pdm, cfg, 0, expect_path=pdm.PDM_PATH_NAIVE)
    rc, h = pdm.pdm_create(cfg["nx"], cfg["nz"], cfg["nw"], cfg["dx"], cfg["dz"], cfg["omega"],
                           cfg["velocity"], cfg["table"], cfg["du"], pdm.PDM_PATH_SMEM)
    assert rc == pdm.PDM_ERR_UNSUPPORTED and h is None


@pytest.mark.parametrize("nx,nz,nw,ntaps,model,ctas", [
    (200, 37, 700, 15, "field", 1),     # 148 CTAs, 4.7 lines each: tail + whole lines + head per CTA
    (520, 23, 151, 25, "layers", 1),    # 1.02 lines each: most CTAs own only a tail and a head
    (300, 16, 449, 7, "white", 3),      # 444 CTAs (3 per SM), 5 lines over
])
def test_depth_split_balancing_matches_oracle_and_whole_line_schedule(pdm, nx, nz, nw, ntaps, model, ctas):
    """Lines split between CTAs at a depth (hand-off through HBM) give the same image as whole
    lines per CTA, up to the summation order of the partial images, and both match the oracle."""
    cfg = pdm_inputs.random_problem(17, nx, nz, nw, ntaps, model=model)
    ref = oracle.migrate(cfg)
    base = pdm.PDM_PATH_SMEM | (ctas << pdm.PDM_CTAS_SHIFT)
    img_b, info_b = gpu_migrate(pdm, cfg, base, want_info=True)
    img_w, info_w = gpu_migrate(pdm, cfg, base | pdm.PDM_NO_BALANCE, want_info=True)
    assert info_b["grid_ctas"] == info_w["grid_ctas"] == 148 * ctas
    for img in (img_b, img_w):
        rel, mx = errors(img, ref)
        assert rel <= REL_L2_BAR and mx <= MAX_PIX_BAR, (rel, mx)
    # run the balanced plan twice more: the hand-off flags must be back to empty after each call
    import torch
    with pdm.Plan.from_config(cfg, base) as plan:
        p0 = torch.from_numpy(cfg["P0"]).cuda()
        a = plan.migrate(p0).clone()
        b = plan.migrate(p0).clone()
        torch.cuda.synchronize()
        assert torch.equal(a, b) and np.array_equal(a.cpu().numpy(), img_b)


@pytest.mark.parametrize("nx,warps,ntaps,model", [
    (3000, 2, 25, "layers"),     # 375 groups on 2 warps: 6 passes per warp, ragged last pass
    (1000, 3, 15, "field"),      # 125 groups on 3 warps: the last warp is partly idle
    (700, 12, 7, "white"),       # 88 groups on 12 warps: warps 3..11 idle (always-ahead flags)
])
def test_neighbour_flag_marching_with_forced_thread_counts(pdm, nx, warps, ntaps, model):
    """The marching kernel synchronises depth steps with per-warp progress flags between
    neighbouring warps (no CTA barrier); force odd warp/pass layouts and check parity and
    bit-identical repeats."""
    import torch
    cfg = pdm_inputs.random_problem(23, nx, 40, 5, ntaps, model=model)
    flags = pdm.PDM_PATH_SMEM | (warps << pdm.PDM_THREADS_SHIFT)
    ref = oracle.migrate(cfg)
    with pdm.Plan.from_config(cfg, flags) as plan:
        assert plan.info["threads_per_cta"] == 32 * warps
        p0 = torch.from_numpy(cfg["P0"]).cuda()
        a = plan.migrate(p0).clone()
        b = plan.migrate(p0).clone()
        torch.cuda.synchronize()
    assert torch.equal(a, b)
    rel, mx = errors(a.cpu().numpy(), ref)
    assert rel <= REL_L2_BAR and mx <= MAX_PIX_BAR, (rel, mx)


def test_tiled_path_with_unaligned_plane_pointer(pdm):
    """Even nx but a P0 that is only 8-byte aligned: the tiled kernel must take its 8-byte
    async-copy variant and still match the 16-byte one bit for bit."""
    import torch
    cfg = pdm_inputs.random_problem(29, 2600, 12, 6, 25, model="field")
    with pdm.Plan.from_config(cfg, pdm.PDM_PATH_TILED) as plan:
        p0 = torch.from_numpy(cfg["P0"]).cuda()
        store = torch.empty(p0.numel() + 1, dtype=p0.dtype, device="cuda")
        shifted = store[1:].view(p0.shape)
        shifted.copy_(p0)
        assert shifted.data_ptr() % 16 == 8
        a = plan.migrate(p0).clone()
        b = plan.migrate(shifted).clone()
        torch.cuda.synchronize()
    assert torch.equal(a, b)
    rel, mx = errors(a.cpu().numpy(), oracle.migrate(cfg))
    assert rel <= REL_L2_BAR and mx <= MAX_PIX_BAR, (rel, mx)


@pytest.mark.parametrize("T", [0, 1, 2, 3, 4, 8])
@pytest.mark.parametrize("model,nx,nz,nw,ntaps", [
    ("field", 300, 21, 7, 15),        # nx below one tile, one ragged pack, nz not a multiple of T
    ("white", 1000, 13, 19, 25),      # 3 packs (the last ragged), 3 x-tiles, every sample its own row
    ("layers", 2501, 10, 9, 7),       # odd nx: P0 is repacked for TMA; thread-uniform rows
    ("field", 1900, 9, 16, 35),       # two whole packs; kernel for L = 17
    ("const", 129, 17, 3, 51),        # halo of 4 groups fetched per side; T*L far beyond the line
])
def test_packed_path_matches_oracle_for_every_block_depth(pdm, T, model, nx, nz, nw, ntaps):
    """T depth steps per tile visit with recomputed halos, 8
    adjacent frequencies per quarter warp, tiles moved by TMA with zero fill at the edges (R5); forced
    T = 1, 2, 3, 4, 8 and the default, ragged nx / nw / nz; parity and bit-identical repeats."""
    import torch
    cfg = pdm_inputs.random_problem(37, nx, nz, nw, ntaps, model=model)
    flags = pdm.PDM_PATH_PACKED | (T << pdm.PDM_CTAS_SHIFT)
    ref = oracle.migrate(cfg)
    with pdm.Plan.from_config(cfg, flags) as plan:
        info = plan.info
        assert info["path"] == pdm.PDM_PATH_PACKED
        p0 = torch.from_numpy(cfg["P0"]).cuda()
        a = plan.migrate(p0).clone()
        b = plan.migrate(p0).clone()
        torch.cuda.synchronize()
    assert torch.equal(a, b)
    rel, mx = errors(a.cpu().numpy(), ref)
    assert np.isfinite(a.cpu().numpy()).all() and rel <= REL_L2_BAR and mx <= MAX_PIX_BAR, (rel, mx, info)


@pytest.mark.parametrize("model,nx,nz,nw,ntaps,n,T", [
    ("field", 300, 21, 7, 15, 20, 0),       # one tile: both edges inside it
    ("white", 1000, 13, 19, 25, 40, 2),     # three tiles: the taper zones sit in the first and the last
    ("layers", 2501, 10, 9, 7, 255, 4),     # the widest taper; odd nx
    ("const", 129, 17, 3, 51, 100, 1),      # taper zones overlap in the middle (n > nx/2)
    ("field", 1900, 9, 16, 35, 1, 0),       # one sample per side
])
def test_edge_taper_variant_matches_oracle(pdm, model, nx, nz, nw, ntaps, n, T):
    """Reading R5b (optional): absorbing cosine taper over n samples per side applied
    after every depth step, in the packed form, against pdm_oracle_migrate_taper."""
    cfg = pdm_inputs.random_problem(47, nx, nz, nw, ntaps, model=model)
    flags = (n << pdm.PDM_TAPER_SHIFT) | ((pdm.PDM_PATH_PACKED | (T << pdm.PDM_CTAS_SHIFT)) if T else 0)
    img, info = gpu_migrate(pdm, cfg, flags, want_info=True)
    assert info["path"] == pdm.PDM_PATH_PACKED
    ref = oracle.migrate(cfg, ntaper=n)
    rel, mx = errors(img, ref)
    assert rel <= REL_L2_BAR and mx <= MAX_PIX_BAR, (rel, mx, info)
    plain = oracle.migrate(cfg)
    assert np.abs(plain - ref).max() > 1e-3 * np.abs(ref).max()       # the taper does something here
    args = (cfg["nx"], cfg["nz"], cfg["nw"], cfg["dx"], cfg["dz"], cfg["omega"], cfg["velocity"], cfg["table"], cfg["du"])
    for bad in (pdm.PDM_PATH_SMEM, pdm.PDM_PATH_TILED, pdm.PDM_PRESTACK):
        rc, h = pdm.pdm_create(*args, (n << pdm.PDM_TAPER_SHIFT) | bad)
        assert rc == pdm.PDM_ERR_INVALID_ARG and h is None


@pytest.mark.parametrize("sym", [True, False])
def test_packed_form_with_row_ranges_wider_than_any_slice_buffer(pdm, sym):
    """51 taps, ntab = 1024, independent samples with a 3.3x velocity spread: at the top frequencies one
    pack's rows on a tile visit span ~700 table rows, more than the ~518 the shared-memory slice holds.
    Forced PDM_PATH_PACKED and PDM_TAPER plans then run the build that reads tap rows from the global
    table (pdm_info.taps_mode = 1) instead of failing; AUTO poststack takes another form."""
    cfg = pdm_inputs.random_problem(61, 1100, 7, 19, 51, ntab=1024, model="white", symmetric=sym)
    ref = oracle.migrate(cfg)
    img, info = gpu_migrate(pdm, cfg, pdm.PDM_PATH_PACKED, want_info=True)
    assert info["path"] == pdm.PDM_PATH_PACKED and info["taps_mode"] == 1 and info["threads_per_cta"] == 256, info
    rel, mx = errors(img, ref)
    assert rel <= REL_L2_BAR and mx <= MAX_PIX_BAR, (rel, mx, info)
    img2, info2 = gpu_migrate(pdm, cfg, pdm.PDM_PATH_PACKED | (3 << pdm.PDM_CTAS_SHIFT) | pdm.PDM_FORCE_GENERAL, want_info=True)
    assert info2["taps_mode"] == 1
    rel, mx = errors(img2, ref)
    assert rel <= REL_L2_BAR and mx <= MAX_PIX_BAR, (rel, mx, info2)
    n = 30
    timg, tinfo = gpu_migrate(pdm, cfg, n << pdm.PDM_TAPER_SHIFT, want_info=True)
    assert tinfo["path"] == pdm.PDM_PATH_PACKED and tinfo["taps_mode"] == 1, tinfo
    rel, mx = errors(timg, oracle.migrate(cfg, ntaper=n))
    assert rel <= REL_L2_BAR and mx <= MAX_PIX_BAR, (rel, mx, tinfo)
    _, auto = gpu_migrate(pdm, cfg, 0, want_info=True)              # AUTO still plans (any form), staged or not
    assert auto["path"] != pdm.PDM_PATH_NAIVE
    args = (cfg["nx"], cfg["nz"], cfg["nw"], cfg["dx"], cfg["dz"], cfg["omega"], cfg["velocity"], cfg["table"], cfg["du"])
    rc, h = pdm.pdm_create(*args, pdm.PDM_PATH_PACKED | (16 << pdm.PDM_THREADS_SHIFT))   # the global-row build is 256 threads only
    assert rc == pdm.PDM_ERR_UNSUPPORTED and h is None


@pytest.mark.parametrize("sym,T,n", [(True, 1, 0), (True, 4, 25), (False, 4, 0), (False, 1, 25), (True, 0, 0)])
def test_packed_form_many_items_per_cta(pdm, sym, T, n):
    """nitems = tiles x packs far above the 148-CTA grid (here ~45 x 8 = 360): every CTA runs several
    items per depth block, so the double-buffered TMA refill (issue(k+2) by the last warp), the mbarrier
    parities across items and blocks, slice reuse over packs, the image flush on a tile change and the
    progress flags carried across items all run -- with asymmetric tables, the taper and forced T."""
    cfg = pdm_inputs.random_problem(67, 20011, 6, 61, 7, model="field", symmetric=sym)
    flags = pdm.PDM_PATH_PACKED | (T << pdm.PDM_CTAS_SHIFT) | (n << pdm.PDM_TAPER_SHIFT)
    img, info = gpu_migrate(pdm, cfg, flags, want_info=True)
    assert info["path"] == pdm.PDM_PATH_PACKED and info["grid_ctas"] <= info["sm_count"], info
    ref = oracle.migrate(cfg, ntaper=n)
    rel, mx = errors(img, ref)
    assert rel <= REL_L2_BAR and mx <= MAX_PIX_BAR, (rel, mx, info)
    again = gpu_migrate(pdm, cfg, flags)
    assert np.array_equal(img, again)


@pytest.mark.parametrize("model,nx,nz,nw,ntaps,sym", [
    ("field", 300, 21, 7, 15, True), ("white", 1000, 13, 5, 25, False), ("layers", 129, 9, 3, 51, True),
    ("const", 64, 5, 2, 61, True),
])
def test_interpolated_table_lookup_matches_oracle(pdm, model, nx, nz, nw, ntaps, sym):
    """PDM_TABLE_INTERP (reading R3c): the operator is the linear blend of the two rows
    bracketing u; against pdm_oracle_migrate_interp, and visibly different from the nearest-row image."""
    cfg = pdm_inputs.random_problem(83, nx, nz, nw, ntaps, ntab=64, model=model, symmetric=sym)
    img, info = gpu_migrate(pdm, cfg, pdm.PDM_TABLE_INTERP, want_info=True)
    assert info["path"] == pdm.PDM_PATH_NAIVE
    ref = oracle.migrate(cfg, interp=True)
    rel, mx = errors(img, ref)
    assert rel <= REL_L2_BAR and mx <= MAX_PIX_BAR, (rel, mx)
    if model != "const":
        assert errors(img, oracle.migrate(cfg))[0] > 10 * REL_L2_BAR
    args = (cfg["nx"], cfg["nz"], cfg["nw"], cfg["dx"], cfg["dz"], cfg["omega"], cfg["velocity"], cfg["table"], cfg["du"])
    for bad in (pdm.PDM_PATH_SMEM, pdm.PDM_PATH_PACKED, pdm.PDM_PRESTACK, 9 << pdm.PDM_TAPER_SHIFT):
        rc, h = pdm.pdm_create(*args, pdm.PDM_TABLE_INTERP | bad)
        assert rc == pdm.PDM_ERR_INVALID_ARG and h is None


def test_packed_path_with_unaligned_p0_pointer(pdm):
    """Even nx but a P0 that is only 8-byte aligned: TMA cannot address it, so the library repacks it
    into its own plane first; same image bit for bit as the direct descriptor on an aligned P0."""
    import torch
    cfg = pdm_inputs.random_problem(29, 2600, 12, 21, 25, model="field")
    with pdm.Plan.from_config(cfg, pdm.PDM_PATH_PACKED) as plan:
        p0 = torch.from_numpy(cfg["P0"]).cuda()
        store = torch.empty(p0.numel() + 1, dtype=p0.dtype, device="cuda")
        shifted = store[1:].view(p0.shape)
        shifted.copy_(p0)
        assert shifted.data_ptr() % 16 == 8
        a = plan.migrate(p0).clone()
        b = plan.migrate(shifted).clone()
        torch.cuda.synchronize()
    assert torch.equal(a, b)
    rel, mx = errors(a.cpu().numpy(), oracle.migrate(cfg))
    assert rel <= REL_L2_BAR and mx <= MAX_PIX_BAR, (rel, mx)


@pytest.mark.parametrize("steps", [1, 2])
@pytest.mark.parametrize("model,nx,nz,nw,ntaps,sym", [
    ("layers", 2500, 31, 6, 15, True),     # odd nz: the last step runs alone; 2 x-tiles of 8 x 240 samples
    ("field", 300, 8, 7, 25, True),        # halo of 2 groups: 28 of 32 groups kept; nx below one warp tile
    ("white", 5000, 5, 3, 31, True),       # L = 15: the longest filter of the two-step kernel
    ("const", 129, 12, 3, 7, False),       # general (asymmetric) table
    ("layers", 1921, 6, 40, 3, True),      # odd nx: 8-byte copies; several frequency groups
])
def test_tiled_path_two_depth_steps_per_launch(pdm, steps, model, nx, nz, nw, ntaps, sym):
    """SURVEY 8(f) N2 at warp granularity: pdm_tiled_step2 keeps a warp's sub-tile on chip for two depth
    steps (planes cross HBM once per two steps); forced 1 and 2 steps per launch must both match the
    oracle, and agree with each other bit for bit (same arithmetic, same summation order)."""
    cfg = pdm_inputs.random_problem(41, nx, nz, nw, ntaps, model=model, symmetric=sym)
    flags = pdm.PDM_PATH_TILED | (steps << pdm.PDM_CTAS_SHIFT)
    img, info = gpu_migrate(pdm, cfg, flags, want_info=True)
    assert info["path"] == pdm.PDM_PATH_TILED
    assert info["launches_per_migrate"] == (nz if steps == 1 else nz // 2 + nz % 2) + 1
    rel, mx = errors(img, oracle.migrate(cfg))
    assert rel <= REL_L2_BAR and mx <= MAX_PIX_BAR, (rel, mx, info)
    if steps == 2:
        one = gpu_migrate(pdm, cfg, pdm.PDM_PATH_TILED | (1 << pdm.PDM_CTAS_SHIFT))
        assert np.array_equal(one, img)


@pytest.mark.parametrize("nx,nz,nw,ntaps,model,csize", [
    (1000, 24, 5, 25, "white", 4),       # 125 groups over 4 CTAs of one warp: ragged last CTA
    (129, 50, 3, 35, "const", 8),        # 17 groups over 8 CTAs: most CTAs of a cluster idle
    (9000, 20, 300, 25, "layers", 4),    # more lines than clusters: partial-image accumulation
    (20000, 10, 3, 15, "field", 0),      # a line too long for one CTA: auto cluster size
    (4100, 12, 4, 51, "field", 2),       # halo of 4 groups pushed through DSMEM, 2 passes per CTA
])
def test_cluster_path_matches_oracle(pdm, nx, nz, nw, ntaps, model, csize):
    """Line split over a thread-block cluster: halos pushed into the neighbour CTA's shared memory,
    step counters published with release.cluster stores; parity and bit-identical repeats."""
    import torch
    cfg = pdm_inputs.random_problem(13, nx, nz, nw, ntaps, model=model)
    flags = pdm.PDM_PATH_CLUSTER | (csize << pdm.PDM_CTAS_SHIFT)
    ref = oracle.migrate(cfg)
    with pdm.Plan.from_config(cfg, flags) as plan:
        assert plan.info["path"] == pdm.PDM_PATH_CLUSTER
        p0 = torch.from_numpy(cfg["P0"]).cuda()
        a = plan.migrate(p0).clone()
        b = plan.migrate(p0).clone()
        torch.cuda.synchronize()
    assert torch.equal(a, b)
    rel, mx = errors(a.cpu().numpy(), ref)
    assert rel <= REL_L2_BAR and mx <= MAX_PIX_BAR, (rel, mx)


@pytest.mark.parametrize("path", PATHS + ["auto"])
@pytest.mark.parametrize("model,nx,nz,nw,ntaps", [
    ("field", 300, 20, 5, 15), ("white", 1000, 12, 4, 25), ("layers", 2500, 16, 5, 31),
    ("const", 129, 30, 3, 35), ("field", 4100, 10, 3, 51), ("layers", 77, 9, 2, 3)])
def test_asymmetric_tables_run_on_the_general_kernels(pdm, path, model, nx, nz, nw, ntaps):
    """SURVEY 8(f) N3 (Eq. (1) literally): a table with W_k != W_-k is no longer
    refused -- every kernel form has a general (unfolded) build.  The oracle applies the full row in
    the x-k orientation (R11), so a transposed operand or a swapped W_k/W_-k fails here."""
    cfg = pdm_inputs.random_problem(19, nx, nz, nw, ntaps, model=model, symmetric=False)
    L = (ntaps - 1) // 2
    assert not np.array_equal(cfg["table"][:, :L][:, ::-1], cfg["table"][:, L + 1:])
    flags = 0 if path == "auto" else path_flags(pdm, path)
    img, info = gpu_migrate(pdm, cfg, flags, want_info=True)
    assert info["table_symmetric"] == 0
    rel, mx = errors(img, oracle.migrate(cfg))
    assert rel <= REL_L2_BAR and mx <= MAX_PIX_BAR, (path, rel, mx, info)
    # the symmetric twin of the same problem still reports the folded kernels
    sym = pdm_inputs.random_problem(19, nx, nz, nw, ntaps, model=model)
    with pdm.Plan.from_config(sym, flags) as plan:
        assert plan.info["table_symmetric"] == 1
    rc, h = pdm.pdm_create(cfg["nx"], cfg["nz"], cfg["nw"], cfg["dx"], cfg["dz"], cfg["omega"],
                           cfg["velocity"], cfg["table"], cfg["du"], flags | pdm.PDM_REQUIRE_SYMMETRIC)
    assert rc == pdm.PDM_ERR_TABLE_ASYMMETRIC and h is None


def test_auto_small_problem_with_a_huge_table_keeps_a_consistent_layout(pdm):
    """nx <= 1024, few lines (the R = 4 regime) and a table so large that the row map alone would not
    fit shared memory: the outputs-per-thread choice must follow the path actually chosen (R = 4 exists
    for the single-CTA marching form only), and the row map must not count against a plan whose rows
    stay global."""
    for nx, nw, ntab in ((640, 6, 120000), (1024, 3, 131072), (512, 40, 110000)):
        cfg = pdm_inputs.random_problem(81, nx, 10, nw, 15, ntab=ntab, model="field")
        ref = oracle.migrate(cfg)
        img, info = gpu_migrate(pdm, cfg, 0, want_info=True)
        rel, mx = errors(img, ref)
        assert rel <= REL_L2_BAR and mx <= MAX_PIX_BAR, (nx, nw, ntab, rel, mx, info)
        for path in ("tiled", "cluster", "smem_global"):
            assert_parity(pdm, cfg, path_flags(pdm, path), ref=ref)


@pytest.mark.parametrize("path", ["smem_staged", "smem_global", "tiled", "cluster", "packed"])
def test_force_general_flag_takes_the_per_output_gather(pdm, path):
    """PDM_FORCE_GENERAL: a warp-uniform model (layers) run through the per-output tap gather must
    give the same image bit for bit as the thread-uniform fast path (same taps, same order)."""
    cfg = pdm_inputs.random_problem(83, 1300, 18, 5, 25, model="layers")
    flags = path_flags(pdm, path)
    fast = gpu_migrate(pdm, cfg, flags)
    general = gpu_migrate(pdm, cfg, flags | pdm.PDM_FORCE_GENERAL)
    assert np.array_equal(fast, general)
    rel, mx = errors(general, oracle.migrate(cfg))
    assert rel <= REL_L2_BAR and mx <= MAX_PIX_BAR, (rel, mx)


def test_auto_policy_picks_the_measured_best_form(pdm):
    """pdm_create's AUTO choice (flags = 0) for the regimes measured in profiles/r01_sweep_config4.md."""
    def path_of(nx, nw, ntaps, model):
        cfg = pdm_inputs.random_problem(71, nx, 4, nw, ntaps, model=model)
        with pdm.Plan.from_config(cfg, 0) as plan:
            return plan.info
    assert path_of(2048, 300, 25, "layers")["path"] == pdm.PDM_PATH_SMEM        # plenty of lines
    small = path_of(512, 100, 31, "layers")                                     # few short lines: R = 4
    assert small["path"] == pdm.PDM_PATH_SMEM and small["threads_per_cta"] == 128
    assert path_of(4096, 40, 25, "layers")["path"] == pdm.PDM_PATH_CLUSTER      # too few lines for 148 SMs
    assert path_of(16384, 592, 15, "layers")["path"] == pdm.PDM_PATH_CLUSTER    # a line fits a pair of CTAs
    assert path_of(16384, 200, 15, "layers")["path"] == pdm.PDM_PATH_TILED      # ... but 200 lines waste a round
    assert path_of(32768, 400, 15, "layers")["path"] == pdm.PDM_PATH_TILED      # north_star: forced x-tiled
    # every sample its own table row (profiles/r02_sweep_config4.md)
    assert path_of(4096, 1024, 15, "field")["path"] == pdm.PDM_PATH_PACKED      # dense frequency list
    assert path_of(4096, 300, 15, "field")["path"] == pdm.PDM_PATH_SMEM         # too few items for 148 CTAs
    assert path_of(1024, 2048, 15, "field")["path"] == pdm.PDM_PATH_SMEM        # short lines: tile quantisation
    assert path_of(32768, 400, 25, "field")["path"] == pdm.PDM_PATH_PACKED      # would be x-tiled otherwise


# ---------------------------------------------------------------- BASELINE.json configs
def test_config0_all_paths(pdm, config0):
    ref = oracle.migrate(config0)
    for path in PATHS:
        assert_parity(pdm, config0, path_flags(pdm, path), ref=ref)
    assert_parity(pdm, config0, 0, ref=ref, expect_path=pdm.PDM_PATH_SMEM)


def test_config1_auto_and_tiled(pdm):
    cfg = pdm_inputs.make_config(1)
    ref = oracle.migrate(cfg)
    assert_parity(pdm, cfg, 0, ref=ref, expect_path=pdm.PDM_PATH_SMEM)
    assert_parity(pdm, cfg, pdm.PDM_PATH_TILED, ref=ref)


@pytest.mark.slow
def test_config2_full(pdm):
    cfg = pdm_inputs.make_config(2)
    assert_parity(pdm, cfg, 0, expect_path=pdm.PDM_PATH_SMEM)


def _subset_parity(pdm, cfg, lines, flags=0, expect_path=None):
    """Full-size launch configuration, sampled frequencies: P0 is zero except on `lines`, so the
    image is the sum of exactly those lines' contributions, which the oracle computes one by one."""
    P0 = np.zeros_like(cfg["P0"])
    P0[lines] = cfg["P0"][lines]
    img, info = gpu_migrate(pdm, cfg, flags, P0=P0, want_info=True)
    if expect_path is not None:
        assert info["path"] == expect_path
    ref = oracle.migrate(cfg, omega_index=np.asarray(lines, dtype=np.int32))
    rel, mx = errors(img, ref)
    assert rel <= REL_L2_BAR and mx <= MAX_PIX_BAR, (cfg["name"], rel, mx, info)


@pytest.mark.slow
def test_config3_full_image_in_the_bench_configuration(pdm):
    """The whole configs[3] image (6144 x 1500, all 803 frequencies), in the launch configuration
    bench.py times (AUTO: balanced SMEM marching), against the full FP64 oracle run."""
    cfg = pdm_inputs.make_config(3)
    rel, mx = assert_parity(pdm, cfg, 0, expect_path=pdm.PDM_PATH_SMEM)
    assert rel <= 1e-5 and mx <= 1e-5, (rel, mx)          # measured ~1.5e-6: well inside the 1e-4 bar


@pytest.mark.slow
def test_config3_full_size_sampled_frequencies(pdm):
    cfg = pdm_inputs.make_config(3)
    nw = cfg["nw"]
    lines = sorted({0, 1, nw // 7, nw // 2, nw - 150, nw - 2, nw - 1})
    _subset_parity(pdm, cfg, lines, 0, expect_path=pdm.PDM_PATH_SMEM)


def _sample_lines(info, nw, want=16):
    """Frequency lines for a sampled-line parity check at full size: the first and last lines, the
    lines at (and next to) the boundaries between CTAs' work ranges -- with depth-split balancing the
    line floor(nw*c/grid) is the one CTA c-1 and CTA c share (head on one, tail on the other); on the
    x-tiled path the same lines sit at frequency-group boundaries -- the lines around the first wrap
    of the round-robin cluster schedule, and an even fill up to `want`."""
    lines = {0, 1, nw - 2, nw - 1}
    grid = max(1, info["grid_ctas"])
    for c in (1, 2, grid // 3, grid // 2, grid - 1):
        b = nw * c // grid
        lines |= {b - 1, b, b + 1}
    for wrap in (37, 74, 148, 296):
        lines |= {wrap - 1, wrap}
    lines = {l for l in lines if 0 <= l < nw}
    fill = [int(round(t)) for t in np.linspace(0, nw - 1, want)]
    for l in fill:
        if len(lines) >= want:
            break
        lines.add(l)
    return sorted(lines)[:max(want, 24)]


# the four corners and the diagonal of the (nx, nw) sweep for each filter length
CONFIG4_POINTS = [(1024, 64), (1024, 2048), (32768, 64), (32768, 2048), (4096, 256), (16384, 1024)]


@pytest.mark.slow
@pytest.mark.parametrize("ntaps", [15, 25, 51])
@pytest.mark.parametrize("nx,nw", CONFIG4_POINTS)
def test_config4_corners_and_diagonal(pdm, nx, nw, ntaps):
    """BASELINE.json configs[4] at FULL size in the launch configuration bench.py --sweep times (AUTO):
    (a) >= 16 sampled frequency lines (CTA range boundaries, split lines, first/last) against the
        oracle, the other lines zero -- the oracle computes exactly those lines;
    (b) ALL lines non-zero: the AUTO image against the scaffold kernel (PDM_PATH_NAIVE: one thread per
        sample, unfolded 2L+1 row, one launch per level -- an independent kernel that shares only the
        index rule), whose own sampled lines are oracle-checked in (c).  A defect tied to particular
        CTAs or lines (hand-off of split lines, last-round clusters, frequency-group tails) cannot
        hide behind zero-filled lines here."""
    import torch
    cfg = pdm_inputs.sweep_point(nx, nw, ntaps)
    with pdm.Plan.from_config(cfg, 0) as plan:
        info = plan.info
        if nx <= 4096:
            assert info["path"] == pdm.PDM_PATH_SMEM or (nw == 64 and info["path"] == pdm.PDM_PATH_CLUSTER), info
        elif (nx == 32768 and nw >= 256) or (nx, nw) == (16384, 1024):
            # per-sample rows, lines too long for one CTA or a frequency list dense against the table:
            # the frequency-packed, temporally blocked x-tiled form (conflict-free tap gather)
            assert info["path"] == pdm.PDM_PATH_PACKED, info
        lines = _sample_lines(info, nw)
        assert len(lines) >= min(16, nw)
        full = torch.from_numpy(cfg["P0"]).cuda()
        sub = torch.zeros_like(full)
        idx = torch.as_tensor(lines, device="cuda")
        sub[idx] = full[idx]
        img_sub = plan.migrate(sub).cpu().numpy()
        img_full = plan.migrate(full).cpu().numpy()
    ref = oracle.migrate(cfg, omega_index=np.asarray(lines, dtype=np.int32))
    rel, mx = errors(img_sub, ref)
    assert rel <= REL_L2_BAR and mx <= MAX_PIX_BAR, ("sampled lines", cfg["name"], rel, mx, info)
    with pdm.Plan.from_config(cfg, pdm.PDM_PATH_NAIVE) as naive:
        ref_full = naive.migrate(full).cpu().numpy().astype(np.float64)
        ref_sub = naive.migrate(sub).cpu().numpy()
    rel, mx = errors(ref_sub, ref)                                      # (c) the scaffold itself
    assert rel <= REL_L2_BAR and mx <= MAX_PIX_BAR, ("scaffold", cfg["name"], rel, mx)
    rel, mx = errors(img_full, ref_full)                                # (b) every line
    assert rel <= REL_L2_BAR and mx <= MAX_PIX_BAR, ("all lines vs scaffold", cfg["name"], rel, mx, info)


@pytest.mark.slow
@pytest.mark.parametrize("nx,nw,ntaps,model,flags_name", [
    (32768, 1024, 15, "layers", "auto"),     # the point the x-tiled path's HBM fraction is quoted on
    (16384, 1024, 15, "field", "tiled"),     # the x-tiled alternative AUTO's pair policy is measured against
    (16384, 64, 15, "field", "auto"),        # few long lines: cluster form
    (32768, 256, 25, "field", "auto"),
])
def test_config4_more_points_sampled_frequencies(pdm, nx, nw, ntaps, model, flags_name):
    cfg = pdm_inputs.sweep_point(nx, nw, ntaps, model=model)
    flags = 0 if flags_name == "auto" else path_flags(pdm, flags_name)
    with pdm.Plan.from_config(cfg, flags) as plan:
        info = plan.info
    if (nx, nw, model) == (32768, 1024, "layers"):
        assert info["path"] == pdm.PDM_PATH_TILED
    _subset_parity(pdm, cfg, _sample_lines(info, nw), flags)


# The other 28 points of the 48-point field sweep ("for the remaining points verify parity on a
# seeded omega-subset"), each with the kernel form AUTO chose when profiles/r02_sweep_config4.md section 1 was
# measured: S = SMEM marching, C = cluster, T = x-tiled, P = frequency-packed.
CONFIG4_REST = [
    (1024, 256, 15, "S"), (1024, 1024, 15, "S"), (4096, 64, 15, "C"), (4096, 1024, 15, "P"),
    (4096, 2048, 15, "P"), (16384, 256, 15, "C"), (16384, 2048, 15, "P"), (32768, 256, 15, "P"),
    (32768, 1024, 15, "P"), (1024, 256, 25, "S"), (1024, 1024, 25, "S"), (4096, 64, 25, "C"),
    (4096, 1024, 25, "P"), (4096, 2048, 25, "P"), (16384, 64, 25, "T"), (16384, 256, 25, "P"),
    (16384, 2048, 25, "P"), (32768, 1024, 25, "P"), (1024, 256, 51, "S"), (1024, 1024, 51, "S"),
    (4096, 64, 51, "C"), (4096, 1024, 51, "P"), (4096, 2048, 51, "P"), (16384, 64, 51, "T"),
    (16384, 256, 51, "P"), (16384, 2048, 51, "P"), (32768, 256, 51, "P"), (32768, 1024, 51, "P"),
]


@pytest.mark.slow
@pytest.mark.parametrize("nx,nw,ntaps,form", CONFIG4_REST)
def test_config4_remaining_points_sampled_frequencies(pdm, nx, nw, ntaps, form):
    """Full size, AUTO launch configuration (what bench.py --sweep times): >= 8 sampled frequency lines
    (first / last, CTA work-range boundaries) against the oracle, and the path the sweep table reports."""
    cfg = pdm_inputs.sweep_point(nx, nw, ntaps)
    with pdm.Plan.from_config(cfg, 0) as plan:
        info = plan.info
    want = {"S": pdm.PDM_PATH_SMEM, "C": pdm.PDM_PATH_CLUSTER, "T": pdm.PDM_PATH_TILED, "P": pdm.PDM_PATH_PACKED}[form]
    assert info["path"] == want, info
    lines = _sample_lines(info, nw, want=8)[:12]
    assert len(lines) >= 8
    _subset_parity(pdm, cfg, lines, 0, expect_path=want)


@pytest.mark.slow
def test_randomized_parity_over_forms_shapes_and_filter_lengths(pdm):
    """Seeded fuzz: random (nx, nz, nw, taps, model, kernel form) -- ragged sizes around the 8-sample
    group and the 32-group warp, filter lengths with and without their own instantiation, every
    cluster size -- each against the oracle at the north_star bar."""
    import torch
    rng = np.random.default_rng(2024)
    forms = [0, pdm.PDM_PATH_SMEM, pdm.PDM_PATH_SMEM | pdm.PDM_TAPS_GLOBAL, pdm.PDM_PATH_TILED,
             pdm.PDM_PATH_CLUSTER, pdm.PDM_PATH_CLUSTER | (4 << pdm.PDM_CTAS_SHIFT),
             pdm.PDM_PATH_CLUSTER | (8 << pdm.PDM_CTAS_SHIFT),
             pdm.PDM_PATH_PACKED, pdm.PDM_PATH_PACKED | (1 << pdm.PDM_CTAS_SHIFT),
             pdm.PDM_PATH_PACKED | (5 << pdm.PDM_CTAS_SHIFT)]
    for i in range(64):
        nx = int(rng.choice([1, 7, 8, 9, 63, 64, 65, 255, 257, 700, 1023, 1500, 2049, 3333, 5000]))
        nz = int(rng.integers(1, 24))
        nw = int(rng.choice([1, 2, 5, 37, 150, 310]))
        ntaps = int(rng.choice([3, 5, 7, 9, 11, 15, 21, 25, 31, 35, 41, 51]))
        model = str(rng.choice(["field", "white", "layers", "const"]))
        flags = int(rng.choice(forms))
        if nx * nz * nw > 4e6:
            nw = max(1, int(4e6 // (nx * nz)))
        cfg = pdm_inputs.random_problem(1000 + i, nx, nz, nw, ntaps, model=model)
        img = gpu_migrate(pdm, cfg, flags)
        rel, mx = errors(img, oracle.migrate(cfg))
        assert np.isfinite(img).all() and rel <= REL_L2_BAR and mx <= MAX_PIX_BAR, \
            (i, nx, nz, nw, ntaps, model, hex(flags), rel, mx)


# ---------------------------------------------------------------- properties of the GPU path itself
def test_plan_that_cannot_fit_fails_with_nomem_and_leaks_nothing(pdm):
    """The main form keeps one partial image per CTA (grid*nz*nx*4 B).  A plan whose partial images exceed
    the free device memory must fail with PDM_ERR_NOMEM (checked before the allocation is attempted) and
    give back everything it had allocated by then."""
    import torch
    nx, nz, nw = 4096, 90000, 160                       # 148 CTAs x 90000 x 4096 x 4 B = 218 GB
    cfg = pdm_inputs.tiny_random_problem(3, nx=64, nz=2, nw=2, L=3, ntab=64)
    omega = np.linspace(20.0, 60.0, nw).astype(np.float32)
    vel = np.full((nz, nx), 2000.0, dtype=np.float32)
    du = float(omega.max()) * 10.0 / 2000.0 / 63
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    assert 148 * nz * nx * 4 > free0
    rc, h = pdm.pdm_create(nx, nz, nw, 10.0, 10.0, omega, vel, cfg["table"], du, pdm.PDM_PATH_SMEM)
    assert rc == pdm.PDM_ERR_NOMEM and h is None, rc
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free0 - (64 << 20)          # nothing of the failed plan is left
    small = pdm_inputs.random_problem(5, 300, 8, 5, 15)
    assert_parity(pdm, small, pdm.PDM_PATH_SMEM)                       # and the library is still usable


def test_delta_table_is_identity_on_gpu(pdm):
    cfg = pdm_inputs.random_problem(3, 520, 9, 4, 25, model="field")
    cfg = dict(cfg, table=pdm_inputs.filters.delta_table(cfg["ntab"], cfg["ntaps"]))
    want = cfg["P0"].real.astype(np.float64).sum(axis=0)
    for path in PATHS:
        img = gpu_migrate(pdm, cfg, path_flags(pdm, path))
        for z in range(cfg["nz"]):
            np.testing.assert_allclose(img[z], want, rtol=0, atol=1e-5)


@pytest.mark.parametrize("path", PATHS)
def test_gpu_path_properties_superposition_mirror_additivity(pdm, path):
    """Properties that hold for the method at any size, checked on the GPU path itself (no oracle):
    real-linear superposition, x-mirror symmetry (symmetric taps + zero edges), and additivity over
    a split of the frequency list."""
    flags = path_flags(pdm, path)
    cfg = pdm_inputs.random_problem(37, 777, 14, 6, 25, model="field")
    rng = np.random.default_rng(5)
    A = cfg["P0"]
    B = (rng.standard_normal(A.shape) + 1j * rng.standard_normal(A.shape)).astype(np.complex64)
    img_a = gpu_migrate(pdm, cfg, flags).astype(np.float64)
    img_b = gpu_migrate(pdm, cfg, flags, P0=B).astype(np.float64)
    img_c = gpu_migrate(pdm, cfg, flags, P0=(2.0 * A - 0.5 * B).astype(np.complex64)).astype(np.float64)
    scale = np.abs(img_a).max() + np.abs(img_b).max()
    assert np.abs(img_c - (2.0 * img_a - 0.5 * img_b)).max() <= 2e-5 * scale
    # mirror: reverse x in the data and in the velocity -> the image is reversed
    mir = dict(cfg, velocity=np.ascontiguousarray(cfg["velocity"][:, ::-1]))
    img_m = gpu_migrate(pdm, mir, flags, P0=np.ascontiguousarray(A[:, ::-1])).astype(np.float64)
    assert np.abs(img_m[:, ::-1] - img_a).max() <= 2e-5 * np.abs(img_a).max()
    # frequency additivity: image(all) = image(first half) + image(second half)
    h = cfg["nw"] // 2
    parts = []
    for sl in (slice(0, h), slice(h, None)):
        sub = dict(cfg, omega=np.ascontiguousarray(cfg["omega"][sl]), nw=len(cfg["omega"][sl]),
                   P0=np.ascontiguousarray(A[sl]))
        parts.append(gpu_migrate(pdm, sub, flags).astype(np.float64))
    assert np.abs(parts[0] + parts[1] - img_a).max() <= 2e-5 * np.abs(img_a).max()


@pytest.mark.parametrize("name,nx,nz,nw,ntaps,model,path", [
    ("smem balanced", 700, 20, 300, 15, "field", "auto"),
    ("smem whole lines", 333, 10, 5, 25, "layers", "smem_staged"),
    ("tiled", 2600, 8, 6, 25, "field", "tiled"),
    ("cluster", 5000, 8, 6, 25, "layers", "cluster"),
    ("packed", 2600, 9, 20, 15, "field", "packed"),
])
def test_migrate_is_cuda_graph_capturable(pdm, name, nx, nz, nw, ntaps, model, path):
    """pdm_migrate only enqueues work (no allocation, no host sync, no copies): capture it in a CUDA
    graph -- cooperative and cluster launches included -- and replay it."""
    import torch
    cfg = pdm_inputs.random_problem(43, nx, nz, nw, ntaps, model=model)
    flags = 0 if path == "auto" else path_flags(pdm, path)
    with pdm.Plan.from_config(cfg, flags) as plan:
        p0 = torch.from_numpy(cfg["P0"]).cuda()
        img = torch.empty((nz, nx), dtype=torch.float32, device="cuda")
        ref = plan.migrate(p0).clone()
        torch.cuda.synchronize()
        s = torch.cuda.Stream()
        with torch.cuda.stream(s):
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g, stream=s):
                plan.migrate(p0, img, stream=s)
        img.zero_()
        torch.cuda.synchronize()
        g.replay()
        g.replay()
        torch.cuda.synchronize()
        assert torch.equal(img, ref), name


@pytest.mark.parametrize("name,nx,nz,nw,ntaps,model,path,csize", [
    ("march balanced", 3000, 40, 500, 25, "layers", "auto", 0),
    ("march dedup", 2048, 30, 320, 15, "field", "auto", 0),
    ("march R=4", 512, 60, 100, 31, "layers", "auto", 0),
    ("cluster of 4", 9000, 30, 40, 25, "layers", "cluster", 4),
    ("cluster of 8", 20000, 20, 12, 15, "field", "cluster", 8),
])
def test_flag_synchronised_kernels_repeat_bit_identically(pdm, name, nx, nz, nw, ntaps, model, path, csize):
    """The depth steps are ordered by progress flags (between warps, between CTAs of a cluster and,
    with depth-split balancing, between CTAs through HBM), not by barriers: a missing fence would
    show up as run-to-run differences.  60 repeats of full-machine grids must be bit-identical."""
    import torch
    cfg = pdm_inputs.random_problem(61, nx, nz, nw, ntaps, model=model)
    flags = 0 if path == "auto" else (path_flags(pdm, path) | (csize << pdm.PDM_CTAS_SHIFT))
    with pdm.Plan.from_config(cfg, flags) as plan:
        p0 = torch.from_numpy(cfg["P0"]).cuda()
        ref = plan.migrate(p0).clone()
        img = torch.empty_like(ref)
        for _ in range(60):
            plan.migrate(p0, img)
            assert torch.equal(img, ref), name
    assert torch.isfinite(ref).all()


def test_repeated_migrate_is_bit_identical_and_plans_are_independent(pdm):
    import torch
    a = pdm_inputs.random_problem(21, 700, 20, 300, 15, model="field")
    b = pdm_inputs.random_problem(22, 333, 10, 5, 25, model="layers")
    with pdm.Plan.from_config(a) as pa, pdm.Plan.from_config(b) as pb:
        xa = torch.from_numpy(a["P0"]).cuda(); xb = torch.from_numpy(b["P0"]).cuda()
        s = torch.cuda.Stream()
        with torch.cuda.stream(s):
            ia1 = pa.migrate(xa, stream=s)
            ib = pb.migrate(xb, stream=s)
            ia2 = pa.migrate(xa, stream=s).clone()
        s.synchronize()
        ia3 = pa.migrate(xa)
        torch.cuda.synchronize()
        assert torch.equal(ia1, ia2) and torch.equal(ia1, ia3)
        rel, mx = errors(ib.cpu().numpy(), oracle.migrate(b))
        assert rel <= REL_L2_BAR and mx <= MAX_PIX_BAR
        rel, mx = errors(ia1.cpu().numpy(), oracle.migrate(a))
        assert rel <= REL_L2_BAR and mx <= MAX_PIX_BAR


def test_migrate_host_equals_device_call(pdm):
    import torch
    cfg = pdm_inputs.random_problem(31, 600, 16, 9, 31, model="field")
    with pdm.Plan.from_config(cfg) as plan:
        dev = plan.migrate(torch.from_numpy(cfg["P0"]).cuda())
        torch.cuda.synchronize()
        pinned = torch.from_numpy(cfg["P0"]).pin_memory()
        host = plan.migrate_host(pinned)
        assert np.array_equal(host, dev.cpu().numpy())
        host2 = plan.migrate_host(cfg["P0"])
        assert np.array_equal(host2, host)
        # both buffers pinned: the main form reads P0 and writes the image through the host mapping
        # (no staging copies); same bits
        out = torch.empty((cfg["nz"], cfg["nx"]), dtype=torch.float32).pin_memory()
        assert plan.info["path"] == pdm.PDM_PATH_SMEM
        plan.migrate_host(pinned, out)
        assert np.array_equal(out.numpy(), host)


def test_gpu_index_rule_matches_oracle_bit_for_bit(pdm):
    rng = np.random.default_rng(12)
    n = 200000
    ntab, dz, du = 1024, 10.0, 3.1e-3
    omega = rng.uniform(10.0, 630.0, n).astype(np.float32)
    vel = rng.uniform(700.0, 2500.0, n).astype(np.float32)
    # force exact .5 products: q is a power of two, omega a half-integer multiple of 1/q
    vel[:64] = np.float32(dz / (0.25 * du))
    omega[:64] = (np.arange(64, dtype=np.float32) + 0.5) * 4.0
    got = pdm.pdm_debug_table_index(omega, vel, dz, du, ntab)
    want = np.array([oracle.table_index(omega[i], vel[i], dz, du, ntab) for i in range(0, n, 37)])
    assert np.array_equal(got[::37], want)
    want64 = np.array([oracle.table_index(omega[i], vel[i], dz, du, ntab) for i in range(64)])
    assert np.array_equal(got[:64], want64)


def test_error_codes_on_device(pdm):
    c = pdm_inputs.tiny_random_problem(5, nx=40, nz=4, nw=3, L=2, ntab=9)
    args = (c["nx"], c["nz"], c["nw"], c["dx"], c["dz"], c["omega"], c["velocity"], c["table"])
    rc, h = pdm.pdm_create(*args, c["du"] * 0.5)                     # u exceeds the table
    assert rc == pdm.PDM_ERR_TABLE_RANGE and h is None
    rc, h = pdm.pdm_create(*args, c["du"], pdm.PDM_PATH_CLUSTER | (3 << pdm.PDM_CTAS_SHIFT))
    assert rc == pdm.PDM_ERR_UNSUPPORTED and h is None              # cluster sizes are 2, 4, 8
    big = pdm_inputs.random_problem(1, 40000, 2, 1, 15, model="const")
    rc, h = pdm.pdm_create(big["nx"], big["nz"], big["nw"], big["dx"], big["dz"], big["omega"],
                           big["velocity"], big["table"], big["du"], pdm.PDM_PATH_SMEM)
    assert rc == pdm.PDM_ERR_UNSUPPORTED and h is None              # line cannot fit shared memory
    rc, h = pdm.pdm_create(*args, c["du"])
    assert rc == pdm.PDM_OK
    assert pdm.pdm_migrate(h, 0, 0, 0) == pdm.PDM_ERR_INVALID_ARG
    assert pdm.pdm_destroy(h) == pdm.PDM_OK


def test_create_destroy_does_not_leak(pdm):
    import torch
    cfg = pdm_inputs.random_problem(41, 2048, 64, 32, 25, model="field")
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(5):
        with pdm.Plan.from_config(cfg) as plan:
            plan.migrate(torch.from_numpy(cfg["P0"]).cuda())
            torch.cuda.synchronize()
    torch.cuda.empty_cache()
    free1, _ = torch.cuda.mem_get_info()
    assert free0 - free1 < 64 << 20
