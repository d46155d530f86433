"""spgpe_step under CUDA stream capture (small-grid path of SURVEY.md 3(d) / 7 step 9: a caller that replays a graph of
one spgpe_step(n) call instead of enqueueing 2n or 3n launches).  spgpe_step only enqueues kernels on the handle's stream
(include/spgpe.h): no allocation, no synchronisation, no host read-back, and the imaginary-time rescale factors travel
through device memory, so a captured call replays correctly.  Two conditions, stated in include/spgpe.h: the k-space
tables of (dt, imag) are built by the first call that uses them, so one plain call precedes the capture; an annealed
schedule (spgpe_set_annealing) bakes its event indices into the graph and must not be replayed.

Checked here: the state after `plain call + k replays` equals the oracle's after the same number of steps (tolerances of
tests/test_gpu_parity.py) and is bit-identical with the same steps enqueued plainly on a second handle.
"""
import numpy as np
import pytest

import oracle as orc
from test_gpu_parity import TOL_C128, TOL_C64, assert_parity, random_problem, sp  # noqa: F401

pytestmark = pytest.mark.gpu


def _solver_on(sp, stream, psi, V, Om, De, p, dtype):
    h = sp.spgpe_create(p.nx, p.ny, p.Lx, p.Ly, dtype, p.g_uu, p.g_dd, p.g_ud, p.k_L, p.norm_mode,
                        stream=stream.cuda_stream)
    cdt, rdt = h._np_dtypes
    sp.spgpe_set_potential(h, np.ascontiguousarray(V, dtype=rdt))
    sp.spgpe_set_raman(h, np.ascontiguousarray(Om, dtype=rdt))
    sp.spgpe_set_zeeman(h, np.ascontiguousarray(De, dtype=rdt))
    sp.spgpe_set_psi_host(h, np.ascontiguousarray(psi, dtype=cdt))
    return h


@pytest.mark.parametrize("nx,ny,imag,storage", [(64, 64, 0, "c128"), (64, 64, 1, "c128"), (256, 256, 0, "c128"),
                                                (256, 128, 1, "c128"), (1024, 64, 0, "c128"), (256, 256, 0, "c64")])
def test_captured_step_replays_like_plain_calls(sp, nx, ny, imag, storage):
    import torch
    psi, V, Om, De, p, _ = random_problem(nx, ny, seed=11 * nx + ny + imag)
    dtype = sp.SPGPE_C128 if storage == "c128" else sp.SPGPE_C64
    if storage == "c64":  # both sides start from the values the complex64 arrays hold (R-14)
        psi = psi.astype(np.complex64).astype(np.complex128)
        V, Om, De = (a.astype(np.float32).astype(np.float64) for a in (V, Om, De))
    s = torch.cuda.Stream()
    n, dt, replays = 3, 1e-3, 2
    with torch.cuda.stream(s):
        h = _solver_on(sp, s, psi, V, Om, De, p, dtype)
        hp = _solver_on(sp, s, psi, V, Om, De, p, dtype)
        sp.spgpe_step(h, 1, dt, imag)  # builds the tables of (dt, imag) outside the capture
        sp.spgpe_synchronize(h)
        launches = sp.spgpe_launch_count(h)
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=s):
            sp.spgpe_step(h, n, dt, imag)
        assert sp.spgpe_launch_count(h) > launches  # the library's own launches were recorded, not executed
        s.synchronize()
        for _ in range(replays):
            g.replay()
        got = sp.spgpe_get_psi_host(h)
        sp.spgpe_step(hp, 1, dt, imag)
        for _ in range(replays):
            sp.spgpe_step(hp, n, dt, imag)
        plain = sp.spgpe_get_psi_host(hp)
    total = 1 + replays * n
    # the oracle renormalises after every imaginary-time step, so the chain of calls equals one call of `total` steps
    if imag:
        ref = orc.step(psi, V, Om, De, p, total, dt, 1, targets=orc.norm(psi, p))
    else:
        ref = orc.step(psi, V, Om, De, p, total, dt, 0)
    assert_parity(got, ref, TOL_C128 if storage == "c128" else TOL_C64)
    assert np.array_equal(got, plain)
    sp.spgpe_destroy(h)
    sp.spgpe_destroy(hp)
