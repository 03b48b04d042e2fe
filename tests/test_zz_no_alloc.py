"""lgf_measure_static: theta and F for callers that cannot let the library allocate device memory.

Who they are: a production Monte Carlo job whose own pool holds all of the HBM (a library cudaMalloc fails there although
the job has memory to spare), a program under a framework's caching allocator (PyTorch's cached blocks are invisible to
cudaMalloc), and a measurement hook inside a running update loop (cudaMalloc/cudaFree synchronise the whole device).  The
entry point needs no context and keeps its block partial sums in a fixed 2 MiB array inside the library, shared by all
calls -- so what is checked here is (i) the result against the existing context path lgf_measure, within the tolerances
of tests/test_gpu_parity.py, on calls made one after the other on lattices of DIFFERENT sizes (a stale partial sum left
by the larger lattice must not leak into the smaller one), (ii) that a repeated call gives the same bits, (iii) that
the call leaves the free device memory as it found it, (iv) the size limit.

This file sorts last on purpose (pytest -x stops at the first failure; a failure here must not hide the parity tests)
and depends on nothing the other tests leave behind: it passes alone in a fresh process and at the end of the suite.
"""
import ctypes as C

import numpy as np
import pytest

import ensembles as E
import paper_1301_3460_b200 as lgf

F_TOL = 1e-12          # |dF|, as tests/test_gpu_parity.py (north star)
TOL = 1e-15


def theta_close(t_new, t_ref):
    return abs(t_new - t_ref) <= 1e-9 * max(t_ref, TOL)


def _static_measure(U_dev, dims, out):
    """One call on torch's current stream; U_dev complex128 [V,4,3,3] on the device, out float64 [2] on the device."""
    import torch
    lgf.measure_static(U_dev.data_ptr(), dims, out.data_ptr(), torch.cuda.current_stream().cuda_stream)


def _context_measure(U_dev, dims, storage):
    """The existing path: a context (which allocates), lgf_load_links_device, lgf_measure."""
    gf = lgf.GaugeFixer(dims, storage)
    gf.load_links_device(U_dev.data_ptr())
    F, th, _ = gf.measure()
    gf.destroy()
    return F, th


@pytest.mark.gpu
def test_static_measure_equals_the_context_path_on_consecutive_calls():
    import torch
    big, small = (8, 16, 8, 16), (4, 8, 4, 8)              # 128 and 8 blocks of 128 sites
    Ub = torch.from_numpy(E.noisy(big, 11, 0.35)).cuda()
    Us = torch.from_numpy(E.noisy(small, 12, 0.2)).cuda()
    ref_b = _context_measure(Ub, big, lgf.LGF_STORE_18)
    ref_s = _context_measure(Us, small, lgf.LGF_STORE_18)
    ref_s12 = _context_measure(Us, small, lgf.LGF_STORE_12)
    out = torch.full((3, 2), float("nan"), dtype=torch.float64, device="cuda")
    # two calls in a row on one stream, larger lattice first: the second call finds the first call's 128 partial sums in
    # the shared array and must read only the 8 it wrote itself
    _static_measure(Ub, big, out[0])
    _static_measure(Us, small, out[1])
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    _static_measure(Ub, big, out[2])                        # third call: same input as the first
    torch.cuda.synchronize()
    free1 = torch.cuda.mem_get_info()[0]
    o = out.cpu().numpy()
    for (F, th), (F_ref, th_ref) in ((o[0], ref_b), (o[1], ref_s), (o[1], ref_s12), (o[2], ref_b)):
        assert abs(F - F_ref) <= F_TOL, (F, F_ref)
        assert theta_close(th, th_ref), (th, th_ref)
    assert np.array_equal(o[0], o[2])                       # fixed summation order: a repeated call repeats its bits
    assert free1 >= free0                                   # the call took no device memory
    assert lgf.lib().lgf_measure_static_error() == b""


@pytest.mark.gpu
def test_static_measure_on_extents_the_contexts_do_not_take():
    """Any extents, not only powers of two, and a volume that is not a multiple of the 128-site block: against the oracle
    (the contexts refuse such a lattice).  A gauge copy of the trivial configuration has F = 1 - O(eps^2) and theta > 0."""
    import oracle
    import torch
    dims = (6, 5, 3, 7)                                     # 630 sites: 5 blocks, the last one ragged
    U = E.noisy(dims, 13, 0.3)
    o = oracle.Oracle(dims, 18)
    o.load(U)
    F_ref, th_ref = o.measure()
    out = torch.empty(2, dtype=torch.float64, device="cuda")
    _static_measure(torch.from_numpy(U).cuda(), dims, out)
    torch.cuda.synchronize()
    F, th = out.cpu().numpy()
    assert abs(F - F_ref) <= F_TOL and theta_close(th, th_ref)


@pytest.mark.gpu
def test_static_measure_at_the_maximum_size():
    """LGF_STATIC_MAX_SITES = 64^4 (configs[4]): every entry of the scratch array is in use; same device array into both
    paths."""
    import torch
    cfg = E.CONFIGS["C4"]
    dims = tuple(cfg["dims"])
    assert int(np.prod(dims)) == lgf.LGF_STATIC_MAX_SITES
    Ud = E.noisy_device(dims, cfg["seed"], cfg["eps"], cfg.get("stream", 0))
    out = torch.empty(2, dtype=torch.float64, device="cuda")
    _static_measure(Ud, dims, out)
    torch.cuda.synchronize()
    F, th = out.cpu().numpy()
    F_ref, th_ref = _context_measure(Ud, dims, cfg["storage"])
    del Ud
    torch.cuda.empty_cache()
    assert abs(F - F_ref) <= F_TOL and theta_close(th, th_ref)


def test_static_measure_refuses_what_it_cannot_hold():
    """Argument checks come before any device work, so they run without a GPU: one site more than the array holds is
    LGF_ERR_UNSUPPORTED with a text that names the limit; NULL pointers and non-positive extents are INVALID_ARG."""
    L = lgf.lib()
    d = lambda *v: (C.c_int * 4)(*v)
    p = C.c_void_p(256)                                     # never dereferenced: the calls below fail before any launch
    assert L.lgf_measure_static(p, d(64, 64, 64, 128), None, p) == lgf.LGF_ERR_UNSUPPORTED
    assert b"LGF_STATIC_MAX_SITES" in L.lgf_measure_static_error()
    assert L.lgf_measure_static(p, d(257, 256, 256, 1), None, p) == lgf.LGF_ERR_UNSUPPORTED
    assert L.lgf_measure_static(p, d(1 << 16, 1 << 16, 1 << 16, 1 << 16), None, p) == lgf.LGF_ERR_UNSUPPORTED   # no overflow
    assert L.lgf_measure_static(None, d(8, 8, 8, 8), None, p) == lgf.LGF_ERR_INVALID_ARG
    assert L.lgf_measure_static(p, d(8, 8, 8, 8), None, None) == lgf.LGF_ERR_INVALID_ARG
    assert L.lgf_measure_static(p, None, None, p) == lgf.LGF_ERR_INVALID_ARG
    assert L.lgf_measure_static(p, d(8, 0, 8, 8), None, p) == lgf.LGF_ERR_INVALID_ARG
    assert len(L.lgf_measure_static_error()) > 0
    with pytest.raises(lgf.LgfError) as e:
        lgf.measure_static(256, (128, 64, 64, 64), 256)
    assert e.value.status == lgf.LGF_ERR_UNSUPPORTED and "LGF_STATIC_MAX_SITES" in str(e.value)
