"""Pins of the oracle functions behind SURVEY.md 8(f): the nested second-order real-space split (NEXT-1, PAPER.md
L138), the observables of Eq. 14 and of k space (NEXT-2) and the annealing noise (NEXT-3, PAPER.md
L223).  No expected value below comes from the oracle or from the CUDA path: they are scipy matrix exponentials,
closed forms, numpy sums, and the independent numpy implementation of the splitmix64 stream in workloads/.
"""
import numpy as np
import pytest
from scipy.linalg import expm
from scipy import stats

import oracle as orc
import workloads as wl
from workloads import configs as wcfg

SX = np.array([[0, 1], [1, 0]], dtype=complex)


def rel_l2(a, b):
    return np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel())


def _random_state(seed, ny, nx, scale=1.0):
    r = np.random.default_rng(seed)
    return scale * (r.standard_normal((ny, nx, 2)) + 1j * r.standard_normal((ny, nx, 2)))


# ---------------------------------------------------------------- NEXT-1: nested split D(tau/2) X(tau) D(tau/2)
def _diag_factor(u, d, V, de, g, s, imag):
    """exp(-i s diag(d_up, d_dn)) applied with scipy expm; densities of (u, d) (Eqs. 6-7)."""
    nu, nd = abs(u) ** 2, abs(d) ** 2
    D = np.diag([V + g[0] * nu + g[2] * nd + de / 2, V + g[1] * nd + g[2] * nu - de / 2]).astype(complex)
    U = expm(-D * s) if imag else expm(-1j * D * s)
    return U @ np.array([u, d])


@pytest.mark.parametrize("imag,tau", [(0, 0.037), (0, -0.02), (1, 0.05)])
def test_nested_half_step_is_the_product_of_three_matrix_exponentials(imag, tau):
    r = np.random.default_rng(21)
    ny, nx = 3, 4
    psi = _random_state(22, ny, nx)
    V, Om, de = r.uniform(0, 3, (ny, nx)), r.uniform(-2, 2, (ny, nx)), r.uniform(-1, 1, (ny, nx))
    g = (1.3, 0.7, 0.4)
    p = orc.params(nx, ny, 1.0, 1.0, *g, rs_split=1)
    got = orc.half(psi, V, Om, de, p, tau, imag)
    np.testing.assert_array_equal(got, orc.half_nested(psi, V, Om, de, p, tau, imag))  # dispatch on rs_split
    for iy in range(ny):
        for ix in range(nx):
            q = _diag_factor(*psi[iy, ix], V[iy, ix], de[iy, ix], g, tau / 2, imag)
            X = expm(-(Om[iy, ix] / 2) * SX * tau) if imag else expm(-1j * (Om[iy, ix] / 2) * SX * tau)
            q = X @ q
            q = _diag_factor(q[0], q[1], V[iy, ix], de[iy, ix], g, tau / 2, imag)  # refreshed densities
            np.testing.assert_allclose(got[iy, ix], q, rtol=0, atol=1e-13)


def test_nested_equals_the_single_exponential_where_the_factors_commute():
    """Omega = 0: both are the same diagonal phase; V = delta = g = 0: both are the same sigma_x rotation."""
    psi = _random_state(23, 4, 8)
    r = np.random.default_rng(24)
    V, Om, de = r.uniform(0, 3, (4, 8)), r.uniform(-2, 2, (4, 8)), r.uniform(-1, 1, (4, 8))
    for imag in (0, 1):
        p0 = orc.params(8, 4, 1.0, 1.0, 1.3, 0.7, 0.4, rs_split=0)
        p1 = orc.params(8, 4, 1.0, 1.0, 1.3, 0.7, 0.4, rs_split=1)
        if not imag:  # imaginary time changes the densities inside D, so only the unitary case is an identity
            np.testing.assert_allclose(orc.half(psi, V, None, de, p1, 0.03, imag),
                                       orc.half(psi, V, None, de, p0, 0.03, imag), rtol=0, atol=2e-14)
        q0 = orc.params(8, 4, 1.0, 1.0, rs_split=0)
        q1 = orc.params(8, 4, 1.0, 1.0, rs_split=1)
        np.testing.assert_allclose(orc.half(psi, None, Om, None, q1, 0.03, imag),
                                   orc.half(psi, None, Om, None, q0, 0.03, imag), rtol=0, atol=2e-14)


def _config2_like(n=32):
    w = wl.make_workload(2, n=n)
    return w


def test_nested_split_is_second_order_where_the_single_exponential_is_not():
    """Config 2's parameters (Omega != 0, unequal g): the error against a fine reference falls by 4 per halving of dt
    for the nested split (order 2.0 +- 0.1); the frozen-density single exponential stays below order 1.9 (SURVEY.md
    8(c) item 5).  Both converge to the same solution."""
    w = _config2_like(32)
    T = 0.04
    p_n, p_s = orc.params_of(w, rs_split=1), orc.params_of(w, rs_split=0)
    ref = orc.step(w.psi0, w.V, w.Omega, w.delta, p_n, 2048, T / 2048, 0)
    err_n, err_s = [], []
    for n in (8, 16, 32):
        err_n.append(rel_l2(orc.step(w.psi0, w.V, w.Omega, w.delta, p_n, n, T / n, 0), ref))
        err_s.append(rel_l2(orc.step(w.psi0, w.V, w.Omega, w.delta, p_s, n, T / n, 0), ref))
    order_n = np.log2(err_n[0] / err_n[1]), np.log2(err_n[1] / err_n[2])
    order_s = np.log2(err_s[1] / err_s[2])
    assert all(abs(o - 2.0) < 0.1 for o in order_n), (order_n, err_n)
    assert order_s < 1.9, (order_s, err_s)
    # the single exponential converges to the same limit (first order): its error keeps falling
    assert err_s[2] < err_s[1] < err_s[0] and err_s[2] < 30 * err_n[2] + 1e-3


def test_nested_split_is_exactly_reversible_with_unequal_g_and_raman_coupling():
    """Every factor of D X D is inverted exactly by the same factor with -tau (a diagonal phase keeps the densities it
    was built from), so step(n, dt) then step(n, -dt) is the identity; the single exponential is not (3.9e-6 in the
    survey probe)."""
    w = _config2_like(32)
    p_n, p_s = orc.params_of(w, rs_split=1), orc.params_of(w, rs_split=0)
    dt = 2e-3
    fwd = orc.step(w.psi0, w.V, w.Omega, w.delta, p_n, 40, dt, 0)
    back = orc.step(fwd, w.V, w.Omega, w.delta, p_n, 40, -dt, 0)
    assert rel_l2(back, w.psi0) < 5e-13
    back_s = orc.step(orc.step(w.psi0, w.V, w.Omega, w.delta, p_s, 40, dt, 0), w.V, w.Omega, w.delta, p_s, 40, -dt, 0)
    assert rel_l2(back_s, w.psi0) > 1e-9
    # the total norm is conserved by the nested split as well (the Raman term moves atoms between the components)
    np.testing.assert_allclose(orc.norm(fwd, p_n).sum(), orc.norm(w.psi0, p_n).sum(), rtol=1e-12)


# ---------------------------------------------------------------- NEXT-3: annealing noise
def _noise_by_numpy(seed, event, amp, ny, nx):
    """The stated generator evaluated with the independent numpy splitmix64 of workloads/configs.py: element e of
    event k uses the uniforms 2q, 2q+1 of the stream, q = k * (2 nx ny) + e."""
    E = ny * nx * 2
    u = wcfg.uniforms(seed, 2 * event * E, 2 * E).reshape(E, 2)
    r = np.sqrt(-2.0 * np.log1p(-u[:, 0]))
    z = r * np.exp(2j * np.pi * u[:, 1])
    return (amp / np.sqrt(2.0)) * z.reshape(ny, nx, 2)


def test_anneal_noise_follows_the_stated_counter_stream():
    ny, nx = 6, 10
    p = orc.params(nx, ny, 1.0, 1.0)
    psi = _random_state(31, ny, nx)
    for seed, event, amp in ((12345, 1, 1e-2), (2**63 + 17, 3, 0.5), (7, 1000, 1.0)):
        got = orc.anneal_noise(psi, p, seed, event, amp) - psi
        np.testing.assert_allclose(got, _noise_by_numpy(seed, event, amp, ny, nx), rtol=0, atol=1e-14 * max(1.0, amp))
    # different events and different seeds give different noise
    a = orc.anneal_noise(0 * psi, p, 5, 1, 1.0)
    assert np.abs(a - orc.anneal_noise(0 * psi, p, 5, 2, 1.0)).min() > 0
    assert np.abs(a - orc.anneal_noise(0 * psi, p, 6, 1, 1.0)).min() > 0


def test_anneal_noise_is_complex_gaussian_of_variance_amp_squared():
    ny = nx = 128
    p = orc.params(nx, ny, 1.0, 1.0)
    amp = 0.3
    z = orc.anneal_noise(np.zeros((ny, nx, 2), dtype=complex), p, 99, 2, amp).ravel()
    n = z.size
    assert abs(np.mean(np.abs(z) ** 2) / amp**2 - 1.0) < 5.0 / np.sqrt(n)          # <|noise|^2> = amp^2
    assert abs(z.real.mean()) < 5 * amp / np.sqrt(2 * n) and abs(z.imag.mean()) < 5 * amp / np.sqrt(2 * n)
    assert abs(np.mean(z.real * z.imag)) < 5 * amp**2 / 2 / np.sqrt(n)              # re, im uncorrelated
    assert abs(np.mean(z[:-1].real * z[1:].real)) < 5 * amp**2 / 2 / np.sqrt(n)     # neighbours uncorrelated
    for part in (z.real, z.imag):
        assert stats.kstest(part / (amp / np.sqrt(2.0)), "norm").pvalue > 1e-3


def test_step_anneal_places_the_events_and_continues_across_calls():
    w = wl.make_workload(1, n=16)
    p = orc.params_of(w)
    dt, every, amp, seed = 1e-2, 2, 1e-2, 4242
    t = orc.norm(w.psi0, p)
    got = orc.step_anneal(w.psi0, w.V, None, None, p, 5, dt, every, amp, seed)
    # by hand: steps 0..4; noise enters steps 2 (event 1) and 4 (event 2)
    q = orc.step(w.psi0, w.V, None, None, p, 2, dt, 1, targets=t)
    q = orc.step(orc.anneal_noise(q, p, seed, 1, amp), w.V, None, None, p, 2, dt, 1, targets=t)
    q = orc.step(orc.anneal_noise(q, p, seed, 2, amp), w.V, None, None, p, 1, dt, 1, targets=t)
    np.testing.assert_allclose(got, q, rtol=0, atol=1e-14)
    # every = 0: no noise at all
    np.testing.assert_allclose(orc.step_anneal(w.psi0, w.V, None, None, p, 3, dt, 0, amp, seed),
                               orc.step(w.psi0, w.V, None, None, p, 3, dt, 1), rtol=0, atol=1e-14)
    # 3 steps then 2 more with first_step = 3 equal 5 steps
    a = orc.step_anneal(w.psi0, w.V, None, None, p, 3, dt, every, amp, seed)
    b = orc.step_anneal(a, w.V, None, None, p, 2, dt, every, amp, seed, first_step=3, targets=t)
    np.testing.assert_allclose(b, got, rtol=0, atol=1e-14)
    # the renormalisation at the end of a noisy step restores the norms
    np.testing.assert_allclose(orc.norm(got, p), t, rtol=1e-13)


def test_annealed_then_plain_imaginary_time_still_finds_the_harmonic_ground_state():
    """The paper's two-segment protocol on config 1's trap: E/N -> hbar omega = 1."""
    w = wl.make_workload(1)
    p = orc.params_of(w)
    q = orc.step_anneal(w.psi0, w.V, None, None, p, 300, 1e-2, 50, 1e-3, 77)
    q = orc.step(q, w.V, None, None, p, 600, 1e-2, 1)
    e = orc.energy(q, w.V, None, None, p)[0] / orc.norm(q, p).sum()
    assert abs(e - 1.0) < 1e-4


# ---------------------------------------------------------------- NEXT-2: observables
def test_phase_separation_parameter_on_mixed_and_separated_states():
    nx, ny, L = 32, 16, 8.0
    p = orc.params(nx, ny, L, L)
    A = L * L
    # uniform densities a, b: I_uu = a^2 A, I_dd = b^2 A, I_ud = a b A, s = 0 (completely mixed)
    psi = np.empty((ny, nx, 2), dtype=complex)
    psi[..., 0] = np.sqrt(0.7) * np.exp(0.3j)
    psi[..., 1] = -np.sqrt(0.2)
    o = orc.observables(psi, p)
    np.testing.assert_allclose(o[:5], [0.7 * A, 0.2 * A, 0.49 * A, 0.04 * A, 0.14 * A], rtol=1e-13)
    assert abs(o[5]) < 1e-14
    # disjoint supports: I_ud = 0, s = 1 (completely separated)
    psi[:, : nx // 2, 1] = 0
    psi[:, nx // 2:, 0] = 0
    o = orc.observables(psi, p)
    assert o[4] == 0.0 and o[5] == 1.0
    np.testing.assert_allclose(o[:4], [0.35 * A, 0.1 * A, 0.245 * A, 0.02 * A], rtol=1e-13)


def test_observables_of_gaussians_have_their_closed_forms():
    """rho = N e^{-r^2/s^2}/(pi s^2): int rho^2 = N^2/(2 pi s^2); two Gaussians of widths s1, s2:
    int rho_1 rho_2 = N1 N2/(pi (s1^2 + s2^2)), so s = 1 - 2 s1 s2/(s1^2 + s2^2)."""
    n, L = 128, 24.0
    p = orc.params(n, n, L, L)
    x = orc.xgrid(n, L)
    X, Y = np.meshgrid(x, x)
    r2 = X * X + Y * Y
    N1, N2, s1, s2 = 3.0, 5.0, 1.0, 1.7
    psi = np.empty((n, n, 2), dtype=complex)
    psi[..., 0] = np.sqrt(N1 / (np.pi * s1**2)) * np.exp(-r2 / (2 * s1**2)) * np.exp(0.2j * X)
    psi[..., 1] = np.sqrt(N2 / (np.pi * s2**2)) * np.exp(-r2 / (2 * s2**2))
    o = orc.observables(psi, p)
    want = [N1, N2, N1**2 / (2 * np.pi * s1**2), N2**2 / (2 * np.pi * s2**2), N1 * N2 / (np.pi * (s1**2 + s2**2))]
    np.testing.assert_allclose(o[:5], want, rtol=1e-12)
    np.testing.assert_allclose(o[5], 1 - 2 * s1 * s2 / (s1**2 + s2**2), rtol=1e-12)


def test_kspace_observables_of_plane_waves_and_a_gaussian():
    nx, ny, Lx, Ly, k_L = 32, 16, 10.0, 6.0, 0.8
    p = orc.params(nx, ny, Lx, Ly, k_L=k_L)
    x, y = orc.xgrid(nx, Lx), orc.xgrid(ny, Ly)
    X, Y = np.meshgrid(x, y)
    kx, ky = orc.kgrid(nx, Lx), orc.kgrid(ny, Ly)
    a_u, a_d, (mu, nu), (md, nd) = 0.6, 0.9, (3, -2), (-5, 7)
    psi = np.empty((ny, nx, 2), dtype=complex)
    psi[..., 0] = a_u * np.exp(1j * (kx[mu] * X + ky[nu] * Y))
    psi[..., 1] = a_d * np.exp(1j * (kx[md] * X + ky[nd] * Y))
    o = orc.kspace_observables(np.fft.fft2(psi, axes=(0, 1)), p)
    A = Lx * Ly
    want = [a_u**2 * A, a_d**2 * A,
            a_u**2 * A * ((kx[mu] + k_L) ** 2 + ky[nu] ** 2) / 2, a_d**2 * A * ((kx[md] - k_L) ** 2 + ky[nd] ** 2) / 2,
            a_u**2 * A * kx[mu], a_d**2 * A * kx[md]]
    np.testing.assert_allclose(o, want, rtol=1e-12)
    # Gaussian e^{-r^2/2} boosted by e^{i q x}: T = N (1/2 + q^2/2) without recoil, P = N q
    n, L, q = 64, 16.0, 2 * np.pi * 4 / 16.0
    p = orc.params(n, n, L, L)
    x = orc.xgrid(n, L)
    X, Y = np.meshgrid(x, x)
    psi = np.zeros((n, n, 2), dtype=complex)
    psi[..., 0] = np.exp(-(X * X + Y * Y) / 2) * np.exp(1j * q * X)
    psi[..., 1] = 2 * np.exp(-(X * X + Y * Y) / 2)
    o = orc.kspace_observables(np.fft.fft2(psi, axes=(0, 1)), p)
    np.testing.assert_allclose(o, [np.pi, 4 * np.pi, np.pi * (0.5 + q * q / 2), 4 * np.pi * 0.5, np.pi * q, 0.0],
                               rtol=1e-12, atol=1e-12)


@pytest.mark.parametrize("imag", [0, 1])
def test_step_observe_reports_the_final_state_and_the_middle_of_the_last_step(imag):
    w = wl.make_workload(2, n=32)
    p = orc.params_of(w)
    dt, n = 2e-3, 4
    t = orc.norm(w.psi0, p)
    psi, o_r, o_k = orc.step_observe(w.psi0, w.V, w.Omega, w.delta, p, n, dt, imag)
    ref = orc.step(w.psi0, w.V, w.Omega, w.delta, p, n, dt, imag)
    np.testing.assert_allclose(psi, ref, rtol=0, atol=1e-14 * np.abs(ref).max())
    # real space: plain numpy sums on the final state
    w_ = (w.Lx / w.nx) * (w.Ly / w.ny)
    ru, rd = np.abs(ref[..., 0]) ** 2, np.abs(ref[..., 1]) ** 2
    want = [w_ * ru.sum(), w_ * rd.sum(), w_ * (ru**2).sum(), w_ * (rd**2).sum(), w_ * (ru * rd).sum()]
    np.testing.assert_allclose(o_r[:5], want, rtol=1e-12)
    # s = 1 - (a ratio close to 1): an absolute bound (the sums' rounding, 1e-16 of 1, is not small relative to s)
    np.testing.assert_allclose(o_r[5], 1 - (ru * rd).sum() / np.sqrt((ru**2).sum() * (rd**2).sum()), rtol=0, atol=1e-13)
    # k space: numpy.fft of the state after the first half-step of the last step
    mid = orc.half(orc.step(w.psi0, w.V, w.Omega, w.delta, p, n - 1, dt, imag, targets=t),
                   w.V, w.Omega, w.delta, p, dt / 2, imag)
    hat = np.fft.fft2(mid, axes=(0, 1))
    kx, ky = orc.kgrid(w.nx, w.Lx), orc.kgrid(w.ny, w.Ly)
    KX, KY = np.meshgrid(kx, ky)
    wk = w_ / (w.nx * w.ny)
    hu, hd = np.abs(hat[..., 0]) ** 2, np.abs(hat[..., 1]) ** 2
    want_k = [wk * hu.sum(), wk * hd.sum(), wk * ((((KX + w.k_L) ** 2 + KY**2) / 2) * hu).sum(),
              wk * ((((KX - w.k_L) ** 2 + KY**2) / 2) * hd).sum(), wk * (KX * hu).sum(), wk * (KX * hd).sum()]
    np.testing.assert_allclose(o_k, want_k, rtol=1e-11, atol=1e-11)
    if not imag:  # Parseval and the unit modulus of the k-space phase: M_c is the norm of the mid-step state
        np.testing.assert_allclose(o_k[:2], orc.norm(mid, p), rtol=1e-12)
