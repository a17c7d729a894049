"""adft_cart_to_spherical_noalloc (include/adft_noalloc.h): the Cartesian -> spherical transform with its working memory
in the library's static device array, for callers that cannot call cudaMalloc.  Checked against the existing path,
adft_cart_to_spherical: same kernel and tables, so the results are compared bit for bit (the bar of the byte / index
work), and against the oracle's transform within the tolerance of tests/test_gpu_g.py::test_g_spherical_output.

Collected last on purpose (the suite runs with pytest -x); it depends on nothing the other tests leave behind and
passes alone in a fresh process as well as after them: every call rebuilds what it reads from the shared array.
"""
import numpy as np
import pytest

from paper_2406_11185_b200 import workloads as W

pytestmark = pytest.mark.gpu

ATOMS = np.array([[0.0, 0.1, -0.2], [1.3, -0.4, 0.5], [-0.6, 1.1, 0.9], [0.7, 0.8, -1.2]])


@pytest.fixture(scope="module")
def api():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2406_11185_b200 import api as _api
    _api.lib()
    return _api


def _handles(api, w):
    b = api.Basis.from_workload(w)
    return b, api.ShellPairs(b)


def _random_symmetric(n, seed):
    import torch
    g = torch.Generator().manual_seed(seed)
    M = torch.randn(n, n, dtype=torch.float64, generator=g)
    return (M + M.T).cuda()


def test_noalloc_matches_existing_path_two_calls_in_a_row(api):
    """Two calls in a row on one basis, then a basis of another shape (the shared array is rebuilt by every call and
    keeps nothing a later call relies on), then the first one again; every result equal to adft_cart_to_spherical's."""
    import torch
    from oracle import sph
    wa = W.make_custom(ATOMS, [(0, 4), (1, 2), (2, 4), (3, 1), (0, 0), (2, 3)], seed=41, emin=0.2, emax=8.0, nprim=2)
    wb = W.make(1)
    ba, spa = _handles(api, wa)
    bb, spb = _handles(api, wb)
    for rep, (w, sp) in enumerate([(wa, spa), (wa, spa), (wb, spb), (wa, spa)]):
        M = _random_symmetric(w.nbf, 100 + rep)
        ref = sp.cart_to_spherical(M)                                  # existing path (allocates per handle)
        out = torch.full_like(ref, float("nan"))
        got = sp.cart_to_spherical_noalloc(M, out)
        torch.cuda.synchronize()
        assert got is out and torch.equal(out, ref), (rep, float((out - ref).abs().max()))
        T = sph.transform_matrix(w.shell_l)                            # and the definition, to the GPU tests' tolerance
        Mo = M.cpu().numpy()
        assert np.abs(out.cpu().numpy() - T.T @ Mo @ T).max() <= 4e-10 * np.abs(T).max() ** 2 * max(1.0, np.abs(Mo).max())
    spa.close(); ba.close(); spb.close(); bb.close()


def test_noalloc_allocates_nothing(api):
    """After the first call on the device (set-up), calls leave the device's free memory and torch's allocator untouched."""
    import torch
    w = W.make(1)
    b, sp = _handles(api, w)
    M = _random_symmetric(w.nbf, 7)
    n = sp.cart_to_spherical(M).shape[0]
    out = torch.empty(n, n, dtype=torch.float64, device="cuda")
    sp.cart_to_spherical_noalloc(M, out)                               # set-up happens here at the latest
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    alloc0 = torch.cuda.memory_allocated()
    for _ in range(5):
        sp.cart_to_spherical_noalloc(M, out)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0 and torch.cuda.memory_allocated() == alloc0
    sp.close(); b.close()


def test_noalloc_on_a_side_stream_and_argument_errors(api):
    import torch
    w = W.make(0)
    b, sp = _handles(api, w)
    M = _random_symmetric(w.nbf, 9)
    ref = sp.cart_to_spherical(M)
    out = torch.zeros_like(ref)
    st = torch.cuda.Stream()
    st.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(st):
        sp.cart_to_spherical_noalloc(M, out, stream=st)
    st.synchronize()
    assert torch.equal(out, ref)
    import ctypes as C
    L = api.lib()
    rc = L.adft_cart_to_spherical_noalloc(sp._h, C.c_void_p(M.data_ptr()), None, None)
    assert rc == 1 and b"NULL" in L.adft_last_error()
    sq = torch.zeros(w.nbf, w.nbf, dtype=torch.float64, device="cuda")
    rc = L.adft_cart_to_spherical_noalloc(sp._h, C.c_void_p(sq.data_ptr()), C.c_void_p(sq.data_ptr()), None)
    assert rc == 1 and b"alias" in L.adft_last_error()
    sp.close(); b.close()


def test_noalloc_rejects_a_basis_beyond_the_limit(api):
    """8193 s shells (one more than ADFT_NOALLOC_MAX_SHELLS): refused with ADFT_ERR_INVALID_ARG and a message that names
    the limit, output untouched; the existing path takes the same basis."""
    import torch
    ns = 8193
    g = int(np.ceil(ns ** (1 / 3)))
    atoms = np.array([[i, j, k] for i in range(g) for j in range(g) for k in range(g)], float)[:ns] * 3.0
    shells = np.stack([np.arange(ns), np.zeros(ns), np.ones(ns), np.arange(ns)], 1).astype(np.int32)
    b = api.Basis(atoms, shells, np.full(ns, 1.3), np.ones(ns))
    sp = api.ShellPairs(b)
    M = torch.eye(ns, dtype=torch.float64, device="cuda")
    out = torch.full((ns, ns), 7.0, dtype=torch.float64, device="cuda")
    with pytest.raises(api.AdftError) as e:
        sp.cart_to_spherical_noalloc(M, out)
    assert e.value.status == 1 and "8192 shells" in str(e.value) and "16384 spherical functions" in str(e.value)
    torch.cuda.synchronize()
    assert bool((out == 7.0).all())
    assert torch.equal(sp.cart_to_spherical(M), M)             # s shells: T = 1
    sp.close(); b.close()
