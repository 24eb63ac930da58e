"""CPU-side checks of the C-ABI library: it loads, exports every symbol include/pdm.h declares,
validates arguments before touching a device, and fails loudly when no B200 is present."""
import ctypes
import os
import re

import numpy as np
import pytest

import pdm_inputs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    import paper_1912_05529_b200 as pdm
    pdm.build_lib()
    return pdm.load_library()


def _declared_functions():
    text = open(os.path.join(ROOT, "include", "pdm.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(pdm3?_[a-z0-9_]+)\s*\(", text)))


def test_header_declares_the_boundary():
    names = _declared_functions()
    for must in ("pdm_create", "pdm_migrate", "pdm_destroy", "pdm_get_info", "pdm_strerror"):
        assert must in names


def test_library_exports_every_declared_symbol(lib):
    import paper_1912_05529_b200 as pdm
    declared = _declared_functions()
    assert sorted(pdm.EXPORTED_SYMBOLS) == declared
    for name in declared:
        assert hasattr(lib, name), name


def test_info_struct_matches_header_field_order():
    import paper_1912_05529_b200 as pdm
    text = open(os.path.join(ROOT, "include", "pdm.h")).read()
    head = text[:text.index("} pdm_info;")]
    body = head[head.rindex("typedef struct {") + len("typedef struct {"):]
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    fields = []
    for decl in body.split(";"):
        decl = decl.strip()
        if not decl:
            continue
        typ, names = decl.split(None, 1)
        fields += [(n.strip(), typ) for n in names.split(",")]
    ctype = {"int": ctypes.c_int, "double": ctypes.c_double}
    assert [(n, ctype[t]) for n, t in fields] == list(pdm.PdmInfo._fields_)


def test_strerror_is_total(lib):
    import paper_1912_05529_b200 as pdm
    for code in range(-8, 2):
        s = pdm.pdm_strerror(code)
        assert isinstance(s, str) and s


def test_argument_validation_happens_before_any_device_use(lib):
    import paper_1912_05529_b200 as pdm
    c = pdm_inputs.tiny_random_problem(5)
    args = (c["nx"], c["nz"], c["nw"], c["dx"], c["dz"], c["omega"], c["velocity"], c["table"], c["du"])
    bad_omega = c["omega"].copy(); bad_omega[0] = -1.0
    bad_v = c["velocity"].copy(); bad_v[1, 2] = np.nan
    even = c["table"][:, :-1]
    asym = c["table"].copy(); asym[3, 0] += np.complex64(1e-3)
    cases = [
        ((*args[:5], bad_omega, *args[6:]), pdm.PDM_ERR_INVALID_ARG),
        ((*args[:6], bad_v, *args[7:]), pdm.PDM_ERR_INVALID_ARG),
        ((*args[:7], even, args[8]), pdm.PDM_ERR_INVALID_ARG),
        ((*args[:7], asym, args[8], pdm.PDM_REQUIRE_SYMMETRIC), pdm.PDM_ERR_TABLE_ASYMMETRIC),
        ((*args[:8], -1.0), pdm.PDM_ERR_INVALID_ARG),
        ((*args[:8], float("nan")), pdm.PDM_ERR_INVALID_ARG),
    ]
    for a, want in cases:
        rc, h = pdm.pdm_create(*a)
        assert rc == want and h is None
    for bad_flags in (1 << 31, 6, 15):            # unknown bits; undefined path numbers
        rc, h = pdm.pdm_create(*args, flags=bad_flags)
        assert rc == pdm.PDM_ERR_INVALID_ARG and h is None, bad_flags
    # NULL handles
    assert lib.pdm_migrate(None, None, None, None) == pdm.PDM_ERR_INVALID_ARG
    assert lib.pdm_destroy(None) == pdm.PDM_OK
    assert lib.pdm_get_info(None, None) == pdm.PDM_ERR_INVALID_ARG


def test_no_cpu_fallback_without_a_b200(lib):
    """On a box without a CC 10.x device the product path must fail loudly, never compute."""
    import torch
    import paper_1912_05529_b200 as pdm
    if torch.cuda.is_available() and torch.cuda.get_device_capability()[0] == 10:
        pytest.skip("a B200 is present")
    c = pdm_inputs.tiny_random_problem(6)
    rc, h = pdm.pdm_create(c["nx"], c["nz"], c["nw"], c["dx"], c["dz"], c["omega"], c["velocity"],
                           c["table"], c["du"])
    assert rc == pdm.PDM_ERR_UNSUPPORTED and h is None
    with pytest.raises(pdm.PdmError):
        pdm.Plan.from_config(c)
    with pytest.raises(pdm.PdmError):
        pdm.pdm_fp32_peak(True, 10, 1)


def test_product_package_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_1912_05529_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text, f
                assert "pdm_oracle" not in text, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_1912_05529_b200" not in text and "libpdm.so" not in text, f


def test_tf_create_rejects_bad_arguments_before_touching_the_device(lib):
    import numpy as np
    import paper_1912_05529_b200 as pdm
    ok = np.array([1, 2, 3], dtype=np.int32)
    assert pdm.pdm_tf_create(0, 8, 3, ok)[0] == pdm.PDM_ERR_INVALID_ARG
    assert pdm.pdm_tf_create(16, 0, 3, ok)[0] == pdm.PDM_ERR_INVALID_ARG
    assert pdm.pdm_tf_create(16, 8, 0, ok[:0])[0] == pdm.PDM_ERR_INVALID_ARG
    assert pdm.pdm_tf_create(16, 8, 3, np.array([1, 9, 3], dtype=np.int32))[0] == pdm.PDM_ERR_INVALID_ARG
    assert pdm.pdm_tf_create(16, 8, 3, np.array([1, -1, 3], dtype=np.int32))[0] == pdm.PDM_ERR_INVALID_ARG
    assert pdm.pdm_tf_create(1 << 14, 8, 3, ok)[0] == pdm.PDM_ERR_UNSUPPORTED      # nt > PDM_TF_MAX_NT
    assert pdm.pdm_tf_destroy(None) == pdm.PDM_OK
