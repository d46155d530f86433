"""spgpe_norm_noalloc (include/spgpe.h): the component norms through the entry point that allocates nothing (its
scratch is a fixed device array inside the library) against the existing path, spgpe_norm of a handle holding the same
order parameter.  Tolerance: rtol 1e-13, the one tests/test_gpu_parity.py uses for norms (the two paths sum in the same
order, so the results are in fact bit-identical).  Two calls in a row on different sizes: the second finds the first
call's contents in the shared scratch.  The file name sorts last, so a failure here cannot hide another test under
`pytest -x`; it passes alone in a fresh process and after the other tests."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

RTOL_NORM = 1e-13


@pytest.fixture(scope="module")
def sp():
    import torch
    assert torch.cuda.is_available(), "the gpu tests need a CUDA device"
    import paper_2010_15069_b200 as sp_
    sp_.lib()  # fails loudly if libspgpe.so is missing
    return sp_


def _state(nx, ny, seed, cdt):
    r = np.random.default_rng(seed)
    psi = (r.standard_normal((ny, nx, 2)) + 1j * r.standard_normal((ny, nx, 2))) * np.array([1.0, 0.37])
    return np.ascontiguousarray(psi.astype(cdt))


def _existing_path(sp, psi, Lx, Ly):
    """spgpe_norm of a handle that holds psi (allocates: the path the new entry point is compared with)."""
    ny, nx, _ = psi.shape
    dt = sp.SPGPE_C128 if psi.dtype == np.complex128 else sp.SPGPE_C64
    h = sp.spgpe_create(nx, ny, Lx, Ly, dt)
    sp.spgpe_set_psi_host(h, psi)
    n = sp.spgpe_norm(h)
    sp.spgpe_destroy(h)
    return n


@pytest.mark.parametrize("cdt", [np.complex128, np.complex64])
def test_two_calls_in_a_row_match_the_existing_path(sp, cdt):
    import torch
    Lx, Ly = 12.0, 10.0
    out = torch.full((2,), -1.0, dtype=torch.float64, device="cuda")
    # first call: a large grid fills every slot of the scratch with large partial sums ...
    big = _state(1024, 512, 1, cdt)
    d_big = torch.from_numpy(big).cuda()
    sp.spgpe_norm_noalloc(d_big, Lx, Ly, out)
    torch.cuda.synchronize()
    got_big = out.cpu().numpy().copy()
    np.testing.assert_allclose(got_big, _existing_path(sp, big, Lx, Ly), rtol=RTOL_NORM)
    # ... second call right after it: a small grid (most CTAs have no point and must overwrite their slots with zeros)
    small = 1e-3 * _state(64, 128, 2, cdt)
    d_small = torch.from_numpy(np.ascontiguousarray(small)).cuda()
    sp.spgpe_norm_noalloc(d_small, Lx, Ly, out)
    torch.cuda.synchronize()
    got_small = out.cpu().numpy().copy()
    np.testing.assert_allclose(got_small, _existing_path(sp, np.ascontiguousarray(small), Lx, Ly), rtol=RTOL_NORM)
    assert got_small.max() < 1e-3 * got_big.min()  # nothing of the first call is left in the result
    # and against the plain definition (numpy, fp64), so that both paths are not wrong together
    cell = (Lx / 64) * (Ly / 128)
    want = cell * (np.abs(small.astype(np.complex128)) ** 2).sum(axis=(0, 1))
    np.testing.assert_allclose(got_small, want, rtol=1e-12)


def test_on_a_side_stream_and_a_non_power_of_two_grid(sp):
    import torch
    psi = _state(96, 50, 3, np.complex128)  # no power-of-two requirement here
    d_psi = torch.from_numpy(psi).cuda()
    out = torch.zeros(2, dtype=torch.float64, device="cuda")
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    sp.spgpe_norm_noalloc(d_psi, 3.0, 7.0, out, stream=s.cuda_stream)
    s.synchronize()
    cell = (3.0 / 96) * (7.0 / 50)
    np.testing.assert_allclose(out.cpu().numpy(), cell * (np.abs(psi) ** 2).sum(axis=(0, 1)), rtol=1e-12)


def test_sizes_beyond_the_maximum_are_rejected(sp):
    import ctypes
    import torch
    L = sp.lib()
    d = torch.zeros(16, dtype=torch.float64, device="cuda")
    out = torch.full((2,), 7.0, dtype=torch.float64, device="cuda")
    # the size check comes first: nothing is read or written, so a small buffer is enough to probe it
    for nx, ny in ((8193, 64), (64, 16384)):
        rc = L.spgpe_norm_noalloc(d.data_ptr(), sp.SPGPE_C128, nx, ny, 1.0, 1.0, out.data_ptr(), ctypes.c_void_p(0))
        assert rc == -7
        assert b"maximum" in L.spgpe_strerror(rc)
    assert L.spgpe_norm_noalloc(d.data_ptr(), 5, 64, 64, 1.0, 1.0, out.data_ptr(), ctypes.c_void_p(0)) == -1
    assert L.spgpe_norm_noalloc(None, sp.SPGPE_C128, 64, 64, 1.0, 1.0, out.data_ptr(), ctypes.c_void_p(0)) == -1
    torch.cuda.synchronize()
    assert out.cpu().numpy().tolist() == [7.0, 7.0]
