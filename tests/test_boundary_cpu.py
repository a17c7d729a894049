"""CPU-only checks of the boundary: the C-ABI library loads, exports every symbol include/*.h declares,
validates inputs, normalises like the oracle, and refuses to compute without a GPU (no CPU fallback)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_2406_11185_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def api():
    from paper_2406_11185_b200 import build, api as _api
    build.build()
    return _api


def test_exports_every_declared_symbol(api):
    inc = os.path.join(ROOT, "include")
    hdr = "\n".join(open(os.path.join(inc, f)).read() for f in sorted(os.listdir(inc)) if f.endswith(".h"))
    declared = sorted(n for n in set(re.findall(r"\b(adft_[a-z0-9_]+)\s*\(", hdr)) if not n.endswith("_t"))
    assert "adft_basis_create" in declared and "adft_shellpairs_build" in declared and "adft_jk_build" in declared
    assert "adft_cart_to_spherical_noalloc" in declared
    L = api.lib()
    for name in declared:
        assert hasattr(L, name), f"{name} declared in include/*.h but not exported"
    assert set(api.EXPORTS) <= set(declared)


def test_basis_validation_codes(api):
    w = W.make(0)
    sh = w.shells_struct()
    with pytest.raises(api.AdftError) as e:
        bad = sh.copy(); bad[0, 1] = 5
        api.Basis(w.atoms, bad, w.exponents, w.coefficients)
    assert e.value.status == 2
    with pytest.raises(api.AdftError) as e:
        bad = sh.copy(); bad[0, 0] = 7
        api.Basis(w.atoms, bad, w.exponents, w.coefficients)
    assert e.value.status == 1
    with pytest.raises(api.AdftError) as e:
        ex = w.exponents.copy(); ex[1] = -1.0
        api.Basis(w.atoms, sh, ex, w.coefficients)
    assert e.value.status == 1
    L = api.lib()
    h = C.c_void_p()
    rc = L.adft_basis_create(C.c_int32(3), None, C.c_int32(9), None, None, None, C.c_uint32(0), C.byref(h))
    assert rc == 1 and not h
    assert L.adft_status_string(2) == b"unsupported angular momentum"
    assert L.adft_jk_build(None, None, None, None, C.c_double(0.0), None) == 1


@pytest.mark.parametrize("cfg", [0, 1, 3])
def test_normalisation_and_offsets_match_oracle(api, orc, cfg):
    w = W.make(cfg)
    b = api.Basis.from_workload(w, normalize=True)
    assert b.nbf == w.nbf
    np.testing.assert_array_equal(b.shell_offsets(), w.bf_offsets())
    ref = orc.normalize(w.shell_l, w.shell_nprim, w.shell_off, w.exponents, w.coefficients)
    np.testing.assert_allclose(b.coefficients(), ref, rtol=1e-14)
    b2 = api.Basis.from_workload(w, normalize=False)
    np.testing.assert_array_equal(b2.coefficients(), w.coefficients)


def test_no_cpu_fallback(api):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    b = api.Basis.from_workload(W.make(0))
    with pytest.raises(api.AdftError) as e:
        api.ShellPairs(b, stream=0)
    assert e.value.status == 4


def test_codegen_model_flops_table():
    import json
    metas = json.load(open(os.path.join(ROOT, "paper_2406_11185_b200", "csrc", "generated", "classes.json")))
    tags = {m["tag"] for m in metas}
    assert {"0000", "1000", "2110", "2222"} <= tags
    for m in metas:
        assert m["vrr_ops"] > 0 and m["nint"] > 0
