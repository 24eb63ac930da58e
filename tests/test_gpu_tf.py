"""GPU parity of the time -> frequency transform (pdm_tf_*) against its FP64
oracle, element by element.

Tolerance: the kernel accumulates nt FP32 products of a section sample with a twiddle
rounded once from double, sequentially in n.  Sequential FP32 summation of random-sign terms has a
rounding error of ~ 2^-24 * sqrt(sum_k |s_k|^2) with partial sums |s_k| ~ sqrt(k) * rms(d), i.e.
~ 2^-24 * nt/sqrt(2) * rms(d), against |P0| ~ sqrt(nt) * rms(d): relative ~ 2^-24 * sqrt(nt/2)
(2.7e-6 at nt = 4096; measured 1.1e-6), plus ~1e-7 from the rounded twiddles.  Bar: rel-L2 <=
2^-24 * sqrt(nt) + 2e-7 and every element within 10x that of the largest |P0| -- two orders of
magnitude inside the 1e-4 image bar the transform feeds.
"""
import numpy as np
import pytest

import oracle
import pdm_inputs

pytestmark = pytest.mark.gpu



def bars(nt):
    rel = 2.0 ** -24 * np.sqrt(nt) + 2e-7
    return rel, 10.0 * rel


@pytest.fixture(scope="module")
def pdm():
    import torch
    import paper_1912_05529_b200 as m
    assert torch.cuda.is_available(), "gpu tests need a B200"
    m.load_library()
    return m


def gpu_forward(pdm, section, bins):
    import torch
    nt, nx = section.shape
    with pdm.SectionTransform(nt, nx, bins) as tf:
        out = tf.forward(torch.from_numpy(section).cuda())
        torch.cuda.synchronize()
        return out.cpu().numpy()


@pytest.mark.parametrize("nt,nx,bins", [
    (200, 301, [0, 1, 2, 7, 50, 99, 100]),                 # nt not a power of two, odd nx, DC and Nyquist
    (1024, 520, list(range(20, 245))),                     # configs[1]-like band: several bin tiles, ragged
    (64, 1, [3]),                                          # one trace, one bin
    (4096, 130, list(range(8, 410, 3))),                   # long traces; 2 x-tiles with a 2-sample tail
    (37, 129, list(range(0, 19))),                         # odd nt: every bin of the real spectrum
    (2048, 77, [0, 1, 5, 300, 1023, 1024]),                # FFT form, odd log2(nt): a last radix-2 stage; odd nx
    (8192, 36, list(range(100, 1500, 7)) + [4096]),        # longest record: 2 pairs of traces per CTA
    (32, 1000, list(range(0, 17))),                        # short record: 16 pairs per CTA, every bin
    (8, 19, [0, 1, 2, 3, 4]),
    (4, 2, [0, 1, 2]),
])
def test_transform_matches_oracle(pdm, nt, nx, bins):
    rng = np.random.default_rng(nt * 7 + nx)
    section = rng.standard_normal((nt, nx)).astype(np.float32)
    bins = np.asarray(bins, dtype=np.int32)
    got = gpu_forward(pdm, section, bins).astype(np.complex128)
    ref = oracle.section_to_fx(section, bins)
    rel = np.linalg.norm(got - ref) / np.linalg.norm(ref)
    mx = np.abs(got - ref).max() / np.abs(ref).max()
    rel_bar, max_bar = bars(nt)
    assert rel <= rel_bar and mx <= max_bar, (rel, mx, rel_bar)


def test_cosine_and_repeat_determinism(pdm):
    import torch
    nt, nx, j0 = 512, 260, 33
    n = np.arange(nt, dtype=np.float64)[:, None]
    section = (1.5 * np.cos(2 * np.pi * j0 * n / nt + 0.4) * np.ones((1, nx))).astype(np.float32)
    bins = np.arange(0, nt // 2 + 1, dtype=np.int32)
    with pdm.SectionTransform(nt, nx, bins) as tf:
        s = torch.from_numpy(section).cuda()
        a = tf.forward(s).clone()
        b = tf.forward(s).clone()
        torch.cuda.synchronize()
    assert torch.equal(torch.view_as_real(a), torch.view_as_real(b))
    got = a.cpu().numpy()
    want = np.zeros_like(got)
    want[j0] = 1.5 * nt / 2 * np.exp(0.4j)
    assert np.abs(got - want).max() <= 2e-5 * 1.5 * nt / 2


def test_section_to_image_end_to_end(pdm):
    """t-x section -> (GPU transform) -> P0 -> (GPU migration) -> image, against the oracle chain."""
    import torch
    cfg = pdm_inputs.random_problem(9, 700, 30, 40, 25, model="layers")
    nt, dt = 512, 0.004
    bins = np.arange(10, 50, dtype=np.int32)
    omega = (2 * np.pi * bins / (nt * dt)).astype(np.float32)
    rng = np.random.default_rng(4)
    section = rng.standard_normal((nt, cfg["nx"])).astype(np.float32)
    scale = 1.0                                            # P0 is the unscaled transform
    # frequencies of the record's own bins; the table abscissa must still cover omega*q
    cfg = dict(cfg, omega=omega, nw=bins.size,
               du=float(omega.max() * cfg["dz"] / cfg["velocity"].min() / (cfg["ntab"] - 1)))
    P0_ref = (oracle.section_to_fx(section, bins) * scale).astype(np.complex64)
    ref = oracle.migrate(dict(cfg, P0=P0_ref))
    with pdm.SectionTransform(nt, cfg["nx"], bins) as tf, pdm.Plan.from_config(dict(cfg, P0=P0_ref)) as plan:
        P0 = tf.forward(torch.from_numpy(section).cuda()) * scale
        img = plan.migrate(P0.contiguous())
        torch.cuda.synchronize()
        got = img.cpu().numpy().astype(np.float64)
        img2 = plan.migrate_section(tf, torch.from_numpy(section).cuda())               # one-call form
        torch.cuda.synchronize()
        assert np.array_equal(img2.cpu().numpy(), img.cpu().numpy())
    rel = np.linalg.norm(got - ref) / np.linalg.norm(ref)
    mx = np.abs(got - ref).max() / np.abs(ref).max()
    assert rel <= 1e-4 and mx <= 1e-3, (rel, mx)


def test_tf_error_codes_on_device(pdm):
    rc, h = pdm.pdm_tf_create(64, 8, 2, np.array([1, 2], dtype=np.int32))
    assert rc == pdm.PDM_OK
    assert pdm.pdm_tf_forward(h, 0, 0, 0) == pdm.PDM_ERR_INVALID_ARG
    assert pdm.pdm_tf_destroy(h) == pdm.PDM_OK
    assert pdm.pdm_tf_destroy(None) == pdm.PDM_OK


def test_transform_into_an_output_that_is_only_8_byte_aligned(pdm):
    """Even nx but a P0 buffer at an address = 8 mod 16 (pdm_migrate accepts such a P0): the kernel
    must fall back to 8-byte stores and give the same values as the aligned call."""
    import torch
    nt, nx = 256, 260
    bins = np.arange(3, 60, dtype=np.int32)
    rng = np.random.default_rng(77)
    section = torch.from_numpy(rng.standard_normal((nt, nx)).astype(np.float32)).cuda()
    with pdm.SectionTransform(nt, nx, bins) as tf:
        aligned = tf.forward(section)
        store = torch.empty(bins.size * nx + 1, dtype=torch.complex64, device="cuda")
        shifted = store[1:].view(bins.size, nx)
        assert shifted.data_ptr() % 16 == 8
        tf.forward(section, out=shifted)
        torch.cuda.synchronize()
    assert torch.equal(aligned, shifted)
