"""Host-side checks that need no GPU: the C-ABI library builds, loads and exports every symbol include/lsm.h declares,
argument validation that happens before any CUDA call, and that the product path fails loudly without a device."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import paper_2201_04565_b200 as lsm
from paper_2201_04565_b200.binding import LsmDesc, LsmInfo

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "lsm.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(lsm_[a-z_]+)\s*\(", src)) - {"lsm_alloc_fn", "lsm_free_fn"})


def test_library_exports_every_declared_symbol():
    L = lsm.library()
    names = _declared()
    assert set(names) == set(lsm.EXPORTS)
    for n in names:
        assert hasattr(L, n), n
    assert lsm.lsm_abi_version() == 5


def test_desc_layout_matches_header_field_order():
    hdr = open(os.path.join(ROOT, "include", "lsm.h")).read()
    body = hdr[hdr.index("typedef struct lsm_desc {"):hdr.index("} lsm_desc;")]
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    fields = []
    for decl in body.split("{", 1)[1].split(";"):
        decl = decl.strip()
        if not decl:
            continue
        for part in decl.split(","):
            fields.append(re.findall(r"[A-Za-z_0-9]+", part)[-1])
    assert fields == [f[0] for f in LsmDesc._fields_]
    assert C.sizeof(LsmDesc) % 8 == 0


def test_create_validation_before_cuda():
    L = lsm.library()
    h = C.c_void_p()
    d = LsmDesc()
    d.struct_size = 12
    assert L.lsm_create(C.byref(d), C.byref(h)) == -1 and not h.value
    assert b"ABI" in L.lsm_last_error(None)
    d.struct_size = C.sizeof(LsmDesc)
    d.dim = 4
    assert L.lsm_create(C.byref(d), C.byref(h)) == -1            # dim must be 2 or 3
    d.dim = 3
    d.force_mode = lsm.FORCE_SCATTER
    assert L.lsm_create(C.byref(d), C.byref(h)) == -7            # LSM_E_UNSUPPORTED: 3-D has no scatter path
    d.force_mode = lsm.FORCE_AUTO
    d.dim = 2
    d.n_particles = 0
    assert L.lsm_create(C.byref(d), C.byref(h)) == -1
    assert L.lsm_create(None, C.byref(h)) == -1
    assert L.lsm_step(None, 1) == -1
    assert L.lsm_get_info(None, C.byref(LsmInfo())) == -1


@pytest.mark.skipif(__import__("torch").cuda.is_available(), reason="only meaningful on a box without a GPU")
def test_no_cpu_fallback():
    x = np.zeros((2, 2)); x[1, 0] = 1.0
    with pytest.raises(lsm.LsmError) as ei:
        lsm.lsm_create(x, [0], [1], 1.0, 1.0, 2.0, 0.01)
    assert ei.value.status == -4 and "no CPU fallback" in str(ei.value)


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2201_04565_b200")
    for dp, _, fns in os.walk(pkg):
        for fn in fns:
            if fn.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                txt = open(os.path.join(dp, fn)).read()
                # the word may appear in comments ("bit-identical to the oracle"); what must not appear is any way of
                # reaching it: an import, an include, a path, a dlopen name, one of its symbols
                for needle in ("import oracle", "from oracle", "olsm", "oracle/", "oracle\\", "liboracle", "oracle."):
                    assert needle not in txt, (fn, needle)
