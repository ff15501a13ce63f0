"""Pins for the fp64 oracle against what the paper and the mathematics fix.

Every check here compares ``oracle/gmmnlse_oracle.py`` with something other
than itself: a closed form, a brute-force sum, an invariant, a convergence
order, or a library routine used as an independent witness.  CPU only.
"""
import math

import numpy as np
import pytest

from oracle import gmmnlse_oracle as O
from paper_1708_05324_b200 import workloads as W

KAPPA = W.N2 * W.OMEGA0 / W.C_LIGHT


def rel(a, b):
    return np.linalg.norm(np.ravel(a) - np.ravel(b)) / np.linalg.norm(np.ravel(b))


# ------------------------------------------------------------------ transforms
@pytest.mark.parametrize("N", [1, 2, 4, 8, 32, 64])
@pytest.mark.parametrize("sign", [+1, -1])
def test_fft_vs_direct_dft(N, sign):
    rng = np.random.default_rng(N + 7)
    x = rng.standard_normal((3, N)) + 1j * rng.standard_normal((3, N))
    assert np.allclose(O.fft_radix2(x, sign), O.dft_direct(x, sign), rtol=0, atol=1e-12 * N)


@pytest.mark.parametrize("N", [1, 2, 8, 64])
def test_transforms_vs_direct_dft(N):
    # to_freq / to_time (library FFT as the step) against the O(N^2) definition, sign and 1/N included
    rng = np.random.default_rng(N + 11)
    x = rng.standard_normal((3, N)) + 1j * rng.standard_normal((3, N))
    assert np.allclose(O.to_freq(x), O.dft_direct(x, +1), rtol=0, atol=1e-12 * N)
    assert np.allclose(O.to_time(x), O.dft_direct(x, -1) / N, rtol=0, atol=1e-12)


@pytest.mark.parametrize("log2N", range(0, 15))
def test_transforms_vs_written_out_radix2(log2N):
    # every power of two the configurations use (up to 16384): library transform == the recursion written out above it
    N = 1 << log2N
    rng = np.random.default_rng(100 + log2N)
    x = rng.standard_normal((2, N)) + 1j * rng.standard_normal((2, N))
    assert rel(O.to_freq(x), O.fft_radix2(x, +1)) < 1e-14 * max(1, log2N)
    assert rel(O.to_time(x), O.fft_radix2(x, -1) / N) < 1e-14 * max(1, log2N)


def test_fft_convention_round_trip_and_parseval():
    rng = np.random.default_rng(1)
    x = rng.standard_normal((2, 256)) + 1j * rng.standard_normal((2, 256))
    assert rel(O.to_time(O.to_freq(x)), x) < 1e-13
    # Parseval: sum |X|^2 = N sum |x|^2
    assert abs(np.sum(abs(O.to_freq(x)) ** 2) / (256 * np.sum(abs(x) ** 2)) - 1) < 1e-13
    # a real, even input has a real spectrum; a delta at n=1 gives exp(+2 pi i k/N)  (sign of the exponent)
    d = np.zeros(16); d[1] = 1.0
    assert np.allclose(O.to_freq(d), np.exp(+2j * np.pi * np.arange(16) / 16), atol=1e-14)
    assert np.allclose(O.fft_radix2(d, +1), np.exp(+2j * np.pi * np.arange(16) / 16), atol=1e-14)


def test_single_tone_lands_in_expected_bin():
    # A_n = exp(-i w_k t_n) must land in bin k under F{f} = sum f exp(+i w t)
    N, dt, k = 64, 1e-15, 5
    w = O.omega_grid(N, dt)
    t = np.arange(N) * dt
    X = O.to_freq(np.exp(-1j * w[k] * t))
    assert abs(X[k] - N) < 1e-9 and np.sum(abs(X)) - abs(X[k]) < 1e-8
    assert w[N // 2] < 0 and np.isclose(w[N // 2], -math.pi / dt)      # S9


# ---------------------------------------------------------------- linear part
def _linear(A0, z, beta, dt, steps=4):
    P = A0.shape[0]
    S = np.zeros((P, P, P, P))
    return O.rk4ip_propagate(A0, z, z / steps, beta, S, 0.0, W.OMEGA0, 0.0, None, dt, shock=False)


@pytest.mark.parametrize("b2", [-20e-27, +20e-27])
def test_gaussian_gvd_closed_form(b2):
    # A(z,t) = T0/sqrt(T0^2 - i b2 z) exp(-t^2 / (2 (T0^2 - i b2 z)))   ([47]; Eq. 9)
    N, dt, T0, z = 2048, 10e-15, 100e-15, 1.3
    t = (np.arange(N) - N // 2) * dt
    A0 = np.exp(-t ** 2 / (2 * T0 ** 2))[None, :].astype(complex)
    A = _linear(A0, z, np.array([[0, 0, b2]]), dt)
    q = T0 ** 2 - 1j * b2 * z
    exact = T0 / np.sqrt(q) * np.exp(-t ** 2 / (2 * q))
    assert rel(A[0], exact) < 1e-12
    # Eq. 9: T(z) = T0 sqrt(1 + (z |b2| / T0^2)^2), T from the 1/e intensity half-width^2 = 2<t^2>
    I = abs(A[0]) ** 2
    T_meas = math.sqrt(2 * np.sum(t ** 2 * I) / np.sum(I))
    assert abs(T_meas / (T0 * math.sqrt(1 + (z * abs(b2) / T0 ** 2) ** 2)) - 1) < 1e-10


def test_walkoff_and_beating_signs():
    # Eq. 8: pulse in mode p becomes S(t - db1 z); Eq. 7 (101-110): A_p -> A_p exp(i db0 z)
    N, dt, T0, z = 1024, 10e-15, 100e-15, 0.5
    t = (np.arange(N) - N // 2) * dt
    A0 = np.tile(np.exp(-t ** 2 / (2 * T0 ** 2)), (2, 1)).astype(complex)
    db1, db0 = 1.0e-12, -37.0
    A = _linear(A0, z, np.array([[0.0, 0.0], [db0, db1]]), dt)
    assert rel(A[0], A0[0]) < 1e-13
    shifted = np.exp(-(t - db1 * z) ** 2 / (2 * T0 ** 2)) * np.exp(1j * db0 * z)
    assert rel(A[1], shifted) < 1e-10
    cen = np.sum(t * abs(A[1]) ** 2) / np.sum(abs(A[1]) ** 2)
    assert abs(cen - db1 * z) < 1e-3 * dt


def test_higher_order_dispersion_spectral_phase():
    N, dt, z = 256, 5e-15, 0.2
    rng = np.random.default_rng(3)
    A0 = (rng.standard_normal((1, N)) + 1j * rng.standard_normal((1, N)))
    b3, b4 = 40e-42, 3e-56
    A = _linear(A0, z, np.array([[0, 0, 0, b3, b4]]), dt)
    w = O.omega_grid(N, dt)
    want = O.to_freq(A0) * np.exp(1j * (b3 * w ** 3 / 6 + b4 * w ** 4 / 24) * z)
    assert rel(O.to_freq(A), want) < 1e-12


# ------------------------------------------------------------- nonlinear part
def test_spm_closed_form_and_kerr_sign():
    # dispersion off, P = 1:  A(z,t) = A(0,t) exp(i kappa S_1111 |A|^2 z)
    N, dt = 256, 10e-15
    t = (np.arange(N) - N // 2) * dt
    A0 = (30.0 * np.exp(-t ** 2 / (2 * (200e-15) ** 2)))[None, :].astype(complex)
    S = np.full((1, 1, 1, 1), 1 / 50e-12)
    z = 0.4
    A = O.rk4ip_propagate(A0, z, z / 200, np.zeros((1, 3)), S, KAPPA, W.OMEGA0, 0.0, None, dt, shock=False)
    exact = A0 * np.exp(1j * KAPPA * S[0, 0, 0, 0] * abs(A0) ** 2 * z)
    assert rel(A, exact) < 1e-9
    # one operator evaluation is exactly i kappa S |A|^2 A
    dA = O.nonlinear_op(A0, S, KAPPA, W.OMEGA0, 0.0, None, dt, shock=False)
    assert rel(dA, 1j * KAPPA * S[0, 0, 0, 0] * abs(A0) ** 2 * A0) < 1e-13


def test_xpm_factor_two_and_no_energy_exchange():
    # two CW modes, only S_pppp and the XPM entries S_ppnn(+perms) non-zero:
    # phase rate of mode p = kappa (S_pppp |A_p|^2 + 2 S_ppnn |A_n|^2); |A_p| constant.
    N, dt = 16, 10e-15
    S = np.zeros((2, 2, 2, 2))
    s11, s22, sx = 2.0e10, 1.5e10, 0.8e10
    S[0, 0, 0, 0], S[1, 1, 1, 1] = s11, s22
    for idx in [(0, 0, 1, 1), (0, 1, 0, 1), (0, 1, 1, 0), (1, 1, 0, 0), (1, 0, 1, 0), (1, 0, 0, 1)]:
        S[idx] = sx
    a = np.array([3.0 * np.exp(0.3j), 2.0 * np.exp(-1.1j)])
    A0 = np.tile(a[:, None], (1, N))
    Nt = O.nonlinear_term(A0, S)
    # terms ~ A_p^* A_n^2 (from S_pnnp... = S[p][n][n][p]) are FWM-like; exclude them as the paper does by
    # checking the XPM/SPM-only tensor: zero the (p,n,n,p)-type entry and re-evaluate.
    S2 = S.copy()
    S2[0, 1, 1, 0] = S2[1, 0, 0, 1] = 0.0
    Nt2 = O.nonlinear_term(A0, S2)
    want0 = (s11 * abs(a[0]) ** 2 + 2 * sx * abs(a[1]) ** 2) * a[0]
    want1 = (s22 * abs(a[1]) ** 2 + 2 * sx * abs(a[0]) ** 2) * a[1]
    assert np.allclose(Nt2[0], want0, rtol=1e-13) and np.allclose(Nt2[1], want1, rtol=1e-13)
    # full symmetric tensor adds the S_pnnp A_n A_n A_p^* term
    assert np.allclose(Nt[0], want0 + sx * a[1] ** 2 * np.conj(a[0]), rtol=1e-13)
    z = 0.05
    A = O.rk4ip_propagate(A0, z, z / 100, np.zeros((2, 3)), S2, KAPPA, W.OMEGA0, 0.0, None, dt, shock=False)
    assert np.allclose(abs(A[:, 0]), abs(a), rtol=1e-10)
    ph = np.angle(A[:, 0] / a)
    assert np.allclose(ph, KAPPA * z * np.array([want0 / a[0], want1 / a[1]]).real, rtol=1e-8)


@pytest.mark.parametrize("P,N,fR", [(2, 8, 0.0), (3, 16, 0.18), (4, 8, 0.3)])
def test_staged_sum_vs_literal_quadruple_loop(P, N, fR):
    rng = np.random.default_rng(P * 100 + N)
    A = rng.standard_normal((P, N)) + 1j * rng.standard_normal((P, N))
    S = rng.standard_normal((P, P, P, P))          # NO symmetry: a transposed index would show
    h = rng.standard_normal(N) if fR else None
    dt = 0.37
    a = O.nonlinear_term(A, S, fR, h, dt)
    b = O.nonlinear_term_literal(A, S, fR, h, dt)
    assert rel(a, b) < 1e-13
    if fR:
        c = O.nonlinear_term(A, S, fR, h, dt, direct_conv=True)
        assert rel(c, b) < 1e-13


def test_raman_cw_modulated_and_causal():
    N, dt = 4096, 10e-12 / 4096
    h = W.raman_response(N, dt)
    assert abs(dt * h.sum() - 1) < 1e-14
    # CW: h (*) T = T  => operator identical to fR = 0
    S = np.full((1, 1, 1, 1), 2e10)
    A = np.full((1, N), 5.0 + 2.0j)
    assert rel(O.nonlinear_term(A, S, 0.18, h, dt), O.nonlinear_term(A, S, 0.0)) < 1e-13
    # T = 1 + eps cos(W t)  =>  1 + eps Re[ht(W) exp(-i W t)], ht analytic damped oscillator
    k = 40
    Om = 2 * math.pi * k / (N * dt)
    t = np.arange(N) * dt
    T = (1 + 0.1 * np.cos(Om * t))[None, :].astype(complex)
    R = O.raman_convolve(T, h, dt)[0]
    t1, t2 = W.TAU1, W.TAU2
    ht = (t1 ** 2 + t2 ** 2) / (t1 ** 2 * t2 ** 2) / ((1 / t2 - 1j * Om) ** 2 + 1 / t1 ** 2)
    want = 1 + 0.1 * np.real(ht * np.exp(-1j * Om * t))
    # sampling + rescaling of h_R differs from the continuous transform at O(dt^2/tau1^2) ~ 4e-3 (S6)
    assert np.max(abs(R.real - want)) < 0.1 * 1.5e-2 and np.max(abs(R.imag)) < 1e-13
    # sign of the imaginary part of ht (Raman gain on the red side) is what a conjugated transform would flip
    assert np.sign(O.raman_transfer(h, dt)[k].imag) == np.sign(ht.imag) != 0
    # causality: impulse in T at t0 responds only at t >= t0 (until the decayed tail wraps)
    imp = np.zeros((1, N), complex)
    imp[0, 1000] = 1.0
    R = O.raman_convolve(imp, h, dt)[0]
    assert np.max(abs(R[:1000])) < 1e-6 * np.max(abs(R)) and abs(R[1001]) > 1e-2 * np.max(abs(R))
    # the FFT route equals the literal circular sum
    Ns = 32
    hs = W.raman_response(Ns, 4e-15)
    Ts = np.random.default_rng(5).standard_normal((2, Ns)) + 0j
    assert rel(O.raman_convolve(Ts, hs, 4e-15), O.raman_convolve_direct(Ts, hs, 4e-15)) < 1e-13


def test_shock_term_against_analytic_derivative():
    # dA = i kappa S (1 + i/w0 d_t)(|A|^2 A)   (Eq. 1) for a chirped Gaussian
    N, dt = 1024, 4e-15
    t = (np.arange(N) - N // 2) * dt
    T0, C = 80e-15, 0.7
    q = (1 + 1j * C) / (2 * T0 ** 2)
    A = 20 * np.exp(-q * t ** 2)
    f = abs(A) ** 2 * A                                   # = 8000 exp(-(2 Re q + q) t^2)
    dfdt = -2 * (2 * q.real + q) * t * f
    S = np.full((1, 1, 1, 1), 2e10)
    w0 = 1.0e15
    want = 1j * KAPPA * 2e10 * (f + 1j / w0 * dfdt)
    got = O.nonlinear_op(A[None, :], S, KAPPA, w0, 0.0, None, dt, shock=True)[0]
    assert rel(got, want) < 1e-11


# ------------------------------------------------------------------ integrators
def test_fundamental_soliton_config1():
    # BASELINE config 1 over its full 5 dispersion lengths (1000 steps): |A| invariant, phase z / (2 L_D)
    wl = W.make_config(1)
    assert abs(wl.meta["P0"] - 712.737) < 1e-3 and abs(wl.meta["L_D"] - 0.5) < 1e-12
    assert abs(wl.kappa * wl.S[0, 0, 0, 0] - 2.80608e-3) < 1e-8
    z = 5.0 * wl.meta["L_D"]
    assert abs(z - wl.L) < 1e-12 and abs(z / wl.dz - 1000) < 1e-9
    A = O.rk4ip_propagate(wl.A0, z, wl.dz, wl.beta, wl.S, wl.kappa, wl.omega0, 0.0, None, wl.dt, shock=False)
    exact = wl.A0 * np.exp(1j * z / (2 * wl.meta["L_D"]))
    assert rel(A, exact) < 5e-9
    assert abs(rel(np.abs(A), np.abs(wl.A0))) < 5e-9                 # shape-invariant
    # the MPA reaches the same soliton at second order in dz (implicit trapezoid rule): error / 4 on halving dz
    zs = 0.5 * wl.meta["L_D"]
    ex = wl.A0 * np.exp(1j * zs / (2 * wl.meta["L_D"]))
    errs = []
    for k in (1, 2):
        Am = O.mpa_propagate(wl.A0, zs, wl.dz / k, 10, wl.beta, wl.S, wl.kappa, wl.omega0, 0.0, None, wl.dt,
                             shock=False, tol=1e-12)
        errs.append(rel(Am, ex))
    assert errs[0] < 1e-5 and 3.5 < errs[0] / errs[1] < 4.5


def test_mpa_not_converged_branch_and_predictor():
    """(i) max_iter reached: the last iterate is used, converged = False, the step is counted (reading R2) -- and that
    iterate IS the fixed_iter = max_iter result.  (ii) the predictor of reading S11 changes the first iterate only:
    same fixed point to the tolerance, never more iterations, first large step untouched."""
    wl = _small_mm()
    L = 3 * 10 * wl.dz
    args = (wl.beta, wl.S, wl.kappa, wl.omega0, wl.f_R, wl.h_R, wl.dt)
    st = {}
    A2 = O.mpa_propagate(wl.A0, L, wl.dz, 10, *args, tol=1e-12, max_iter=2, stats=st)
    assert st["not_converged"] == 3 and st["iterations"] == 6 and st["large_steps"] == 3 and st["last_err"] > 1e-12
    Af = O.mpa_propagate(wl.A0, L, wl.dz, 10, *args, fixed_iter=2)
    assert np.array_equal(A2, Af)
    omega = O.omega_grid(wl.N, wl.dt)
    D = O.dispersion_operator(wl.beta, omega)
    K = 1j * wl.kappa * (1 + omega / wl.omega0)
    nlt = lambda A: O.nonlinear_term(A, wl.S, wl.f_R, wl.h_R, wl.dt)
    _, n_it, err, conv = O.mpa_large_step(O.to_freq(wl.A0), 10, wl.dz, D, nlt, K, tol=1e-12, max_iter=1)
    assert n_it == 1 and not conv and err > 1e-6
    # predictor
    s0, s1 = {}, {}
    Lp = 6 * 10 * wl.dz
    ref = O.mpa_propagate(wl.A0, Lp, wl.dz, 10, *args, tol=1e-8, stats=s0)
    got = O.mpa_propagate(wl.A0, Lp, wl.dz, 10, *args, tol=1e-8, stats=s1, predictor=1)
    assert rel(got, ref) < 5e-8 and s1["iterations"] <= s0["iterations"] and s1["not_converged"] == 0
    one0 = O.mpa_propagate(wl.A0, 10 * wl.dz, wl.dz, 10, *args, tol=1e-8)
    one1 = O.mpa_propagate(wl.A0, 10 * wl.dz, wl.dz, 10, *args, tol=1e-8, predictor=1)
    assert np.array_equal(one0, one1)                                # no history yet: the paper's psi_j = psi_0


def _small_mm(P=3, N=256, seed=0, shock=True, fR=0.18):
    wl = W.make_config(2, N=N, max_group=1)
    assert wl.P == 3
    return wl


def test_invariants_energy_and_photon_number():
    wl = _small_mm()
    L, dz = 2e-3, 50e-6
    args = (wl.beta, wl.S, wl.kappa, wl.omega0, wl.f_R, wl.h_R, wl.dt)
    # the ODE conserves these exactly; RK4IP to O(dz^4): small, and shrinking >8x on halving dz
    A = O.rk4ip_propagate(wl.A0, L, dz, *args, shock=False)          # Raman on, shock off: energy
    d1 = abs(O.energy(A, wl.dt) / O.energy(wl.A0, wl.dt) - 1)
    A = O.rk4ip_propagate(wl.A0, L, dz / 2, *args, shock=False)
    d2 = abs(O.energy(A, wl.dt) / O.energy(wl.A0, wl.dt) - 1)
    assert d1 < 1e-8 and d2 < d1 / 8
    q0 = O.photon_number(wl.A0, wl.dt, wl.omega0)
    A = O.rk4ip_propagate(wl.A0, L, dz / 2, *args, shock=True)       # shock on: photon number
    p2 = abs(O.photon_number(A, wl.dt, wl.omega0) / q0 - 1)
    A = O.rk4ip_propagate(wl.A0, L, dz, *args, shock=True)
    p1 = abs(O.photon_number(A, wl.dt, wl.omega0) / q0 - 1)
    assert p1 < 1e-8 and p2 < p1 / 8
    assert abs(O.energy(A, wl.dt) / O.energy(wl.A0, wl.dt) - 1) > 1e-8   # ...and energy is not
    assert rel(A, wl.A0) > 1e-2                                      # something happened


def test_rk4ip_order4_mpa_order2_and_m_independence():
    wl = _small_mm()
    L = 2e-3
    args = (wl.beta, wl.S, wl.kappa, wl.omega0, wl.f_R, wl.h_R, wl.dt)
    ref = O.rk4ip_propagate(wl.A0, L, 12.5e-6, *args)
    e1 = rel(O.rk4ip_propagate(wl.A0, L, 100e-6, *args), ref)
    e2 = rel(O.rk4ip_propagate(wl.A0, L, 50e-6, *args), ref)
    assert 12 < e1 / e2 < 20
    m1 = rel(O.mpa_propagate(wl.A0, L, 100e-6, 10, *args, tol=1e-12), ref)
    m2 = rel(O.mpa_propagate(wl.A0, L, 50e-6, 10, *args, tol=1e-12), ref)
    assert 3.5 < m1 / m2 < 4.5                                     # MPA -> RK4IP at second order
    a = O.mpa_propagate(wl.A0, L, 100e-6, 10, *args, tol=1e-13)
    b = O.mpa_propagate(wl.A0, L, 100e-6, 1, *args, tol=1e-13)
    c = O.mpa_propagate(wl.A0, L, 100e-6, 4, *args, tol=1e-13)
    assert rel(a, b) < 1e-10 and rel(a, c) < 1e-10                 # implicit trapezoid, independent of M


def test_mpa_first_iterate_is_linear_and_error_law():
    wl = _small_mm()
    args = (wl.beta, wl.S, wl.kappa, wl.omega0, wl.f_R, wl.h_R, wl.dt)
    M, dz = 10, 50e-6
    hist, stats = [], {}
    O.mpa_propagate(wl.A0, M * dz, dz, M, *args, tol=1e-12, stats=stats, history=hist)
    planes = hist[0]
    # after iteration 1 psi_j = psi_0 + dz * trapezoid of integrands evaluated on *linear* propagation
    omega = O.omega_grid(wl.N, wl.dt)
    D = O.dispersion_operator(wl.beta, omega)
    K = 1j * wl.kappa * (1 + omega / wl.omega0)
    psi0 = O.to_freq(wl.A0)
    G = [K * np.exp(-D * j * dz) * O.to_freq(O.nonlinear_term(O.to_time(psi0 * np.exp(D * j * dz)),
                                                               wl.S, wl.f_R, wl.h_R, wl.dt)) for j in range(M + 1)]
    want = psi0 + dz * (0.5 * G[0] + sum(G[1:M]) + 0.5 * G[M])
    assert rel(planes[0][M], want) < 1e-13
    # successive corrections shrink geometrically (~ (L/z_nl)^n)
    d = [np.linalg.norm(planes[i + 1][M] - planes[i][M]) for i in range(len(planes) - 1)]
    assert len(d) >= 2 and all(d[i + 1] < 0.2 * d[i] for i in range(len(d) - 1))
    assert 2 <= stats["iterations"] <= 8 and stats["not_converged"] == 0


def test_mpa_ragged_last_step_and_fixed_iter():
    wl = _small_mm()
    args = (wl.beta, wl.S, wl.kappa, wl.omega0, wl.f_R, wl.h_R, wl.dt)
    st = {}
    a = O.mpa_propagate(wl.A0, 13 * 50e-6, 50e-6, 5, *args, tol=1e-13, stats=st)
    assert st["large_steps"] == 3
    b = O.mpa_propagate(wl.A0, 13 * 50e-6, 50e-6, 13, *args, tol=1e-13)
    assert rel(a, b) < 1e-10
    st = {}
    O.mpa_propagate(wl.A0, 10 * 50e-6, 50e-6, 5, *args, fixed_iter=3, stats=st)
    assert st["iterations"] == 6


# ------------------------------------------------------------ general form (S^K != S^R, complex, no symmetry)
@pytest.mark.parametrize("P,N,fR,cplx", [(2, 8, 0.0, False), (3, 8, 0.18, False), (3, 8, 0.3, True)])
def test_general_term_vs_literal_loop_and_reductions(P, N, fR, cplx):
    rng = np.random.default_rng(7 * P + N)
    A = rng.standard_normal((P, N)) + 1j * rng.standard_normal((P, N))
    mk = lambda: rng.standard_normal((P,) * 4) + (1j * rng.standard_normal((P,) * 4) if cplx else 0)
    SK, SR = mk(), mk()
    h = rng.standard_normal(N) if fR else None
    dt = 0.41
    a = O.nonlinear_term_general(A, SK, SR, fR, h, dt)
    assert rel(a, O.nonlinear_term_general_literal(A, SK, SR, fR, h, dt)) < 1e-13
    # tuple dispatch through the common entry, and S^K = S^R = real S reduces to the scalar-mode term (Eq. 2)
    assert rel(O.nonlinear_term(A, (SK, SR), fR, h, dt), a) < 1e-15
    S = rng.standard_normal((P,) * 4)
    assert rel(O.nonlinear_term_general(A, S, S, fR, h, dt), O.nonlinear_term(A, S, fR, h, dt)) < 1e-13
    if fR:
        # linear in each tensor; the Raman tensor acts only through h_R (*) T: CW fields see the blended tensor
        z = np.zeros_like(SK)
        assert rel(O.nonlinear_term_general(A, SK, z, fR, h, dt) + O.nonlinear_term_general(A, z, SR, fR, h, dt), a) < 1e-13
        Acw = (rng.standard_normal((P, 1)) + 1j * rng.standard_normal((P, 1))) * np.ones((1, N))
        hn = np.abs(rng.standard_normal(N)); hn /= dt * hn.sum()           # dt sum h = 1
        blend = (1 - fR) * SK + fR * SR
        assert rel(O.nonlinear_term_general(Acw, SK, SR, fR, hn, dt),
                   O.nonlinear_term_general(Acw, blend, blend, 0.0, None, dt)) < 1e-12


def test_general_form_conserves_energy_for_a_hermitian_tensor():
    """With S_plmn = conj(S_lpnm) (what an overlap integral of F_p* F_l F_m* F_n-type products gives) and no shock,
    sum_p int A_p* N_p is real, so the energy is conserved: an invariant of the general path's integrators."""
    rng = np.random.default_rng(5)
    P, N = 3, 64
    dt = 5e-15
    S0 = rng.standard_normal((P,) * 4) + 1j * rng.standard_normal((P,) * 4)
    S = 0.5 * (S0 + np.conj(S0.transpose(1, 0, 3, 2))) * 1e9
    t = (np.arange(N) - N // 2) * dt
    A0 = (rng.standard_normal((P, 1)) + 1j * rng.standard_normal((P, 1))) * np.exp(-(t / 40e-15) ** 2)[None, :] * 30.0
    beta = np.zeros((P, 3)); beta[:, 2] = 2e-26
    out = O.rk4ip_propagate(A0, 0.02, 0.0005, beta, (S, S), KAPPA, W.OMEGA0, 0.0, None, dt, shock=False)
    assert abs(O.energy(out, dt) / O.energy(A0, dt) - 1) < 1e-8
    assert rel(out, A0) > 1e-3            # the propagation did something


# ------------------------------------------------------------ NEXT-3: gain g_p A_p and linear coupling i Q_np A_n
def test_gain_closed_form_with_dispersion():
    """g_p A_p is linear and diagonal: the Gaussian of Eq. 9 broadens exactly as without gain and its
    field grows as exp(g z); a negative g is loss."""
    N, dt, T0, b2, z = 1024, 4e-15, 60e-15, 2e-26, 0.08
    t = (np.arange(N) - N // 2) * dt
    A0 = np.stack([np.exp(-t ** 2 / (2 * T0 ** 2)), 0.5 * np.exp(-t ** 2 / (2 * T0 ** 2))]).astype(complex)
    g = np.array([3.0, -7.0])
    beta = np.array([[0, 0, b2], [0, 0, b2]])
    S0 = np.zeros((2, 2, 2, 2))
    q = T0 ** 2 - 1j * b2 * z
    exact = T0 / np.sqrt(q) * np.exp(-t ** 2 / (2 * q))
    for out in (O.rk4ip_propagate(A0, z, z / 8, beta, S0, KAPPA, W.OMEGA0, 0.0, None, dt, shock=False, gain=g),
                O.mpa_propagate(A0, z, z / 8, 4, beta, S0, KAPPA, W.OMEGA0, 0.0, None, dt, shock=False, gain=g)):
        assert rel(out[0], np.exp(g[0] * z) * exact) < 1e-10
        assert rel(out[1], 0.5 * np.exp(g[1] * z) * exact) < 1e-10


def test_linear_coupling_two_mode_coupler_closed_form():
    """i sum_n Q_np A_n with Q = [[0, k], [k, 0]] and a propagation-constant mismatch D: the
    textbook directional coupler, P_2(z) = k^2/(k^2 + (D/2)^2) sin^2(sqrt(k^2 + (D/2)^2) z); energy conserved
    for a hermitian Q; the sign (A_2 leads by +i for D = 0) fixes the 'i' of the term."""
    N, dt = 64, 5e-15
    A0 = np.zeros((2, N), complex); A0[0] = 1.0
    kap, Dm, z = 40.0, 50.0, 0.03
    Qc = np.array([[0, kap], [kap, 0]], dtype=complex)
    S0 = np.zeros((2, 2, 2, 2))
    for Dm_ in (0.0, Dm):
        beta = np.array([[0.0], [Dm_]])
        Om = np.hypot(kap, Dm_ / 2)
        p2 = kap ** 2 / Om ** 2 * np.sin(Om * z) ** 2
        rk = O.rk4ip_propagate(A0, z, z / 400, beta, S0, KAPPA, W.OMEGA0, 0.0, None, dt, shock=False, coupling=Qc)
        mp = O.mpa_propagate(A0, z, z / 400, 8, beta, S0, KAPPA, W.OMEGA0, 0.0, None, dt, shock=False, coupling=Qc,
                             tol=1e-12)
        for out, tol in ((rk, 1e-9), (mp, 2e-5)):
            assert abs(np.abs(out[1, 0]) ** 2 - p2) < tol
            assert abs(np.sum(np.abs(out[:, 0]) ** 2) - 1.0) < tol
        if Dm_ == 0.0:
            assert abs(rk[1, 0] - 1j * np.sin(kap * z)) < 1e-9 and abs(rk[0, 0] - np.cos(kap * z)) < 1e-9
    # index order: Q[n][p] couples n -> p; a one-way (non-hermitian) Q feeds only its target mode
    Q1 = np.zeros((2, 2), complex); Q1[0, 1] = kap
    out = O.rk4ip_propagate(A0, z, z / 100, np.zeros((2, 1)), S0, KAPPA, W.OMEGA0, 0.0, None, dt, shock=False, coupling=Q1)
    assert abs(out[0, 0] - 1.0) < 1e-12 and abs(out[1, 0] - 1j * kap * z) < 1e-9


# ------------------------------------------ section F: gain saturation and z-dependent coupling
def test_gain_saturation_logistic_energy_closed_form():
    """P = 1, no dispersion, no Kerr: dA/dz = g A - g_sat S E(z) A with E = int |A|^2 dt, so the energy obeys the
    logistic law E(z) = E0 e^{2gz} / [1 + (g_sat S E0 / g)(e^{2gz} - 1)] and the pulse keeps its shape
    (PAPER.md:297-299 with reading S22)."""
    N, dt = 256, 10e-15
    t = (np.arange(N) - N // 2) * dt
    A0 = (30.0 * np.exp(-t ** 2 / (2 * (80e-15) ** 2)))[None, :].astype(np.complex128)
    S = np.full((1, 1, 1, 1), 2.0e10)
    g, z = 4.0, 0.3
    E0 = O.energy(A0, dt)
    g_sat = 0.6 * g / (S[0, 0, 0, 0] * E0)                      # saturation is strong: g_sat S E0 = 0.6 g
    beta = np.zeros((1, 3))
    for integ in ("rk", "mpa"):
        if integ == "rk":
            A = O.rk4ip_propagate(A0, z, z / 60, beta, S, 0.0, W.OMEGA0, 0.0, None, dt, shock=False, gain=[g], g_sat=g_sat)
        else:
            A = O.mpa_propagate(A0, z, z / 600, 10, beta, S, 0.0, W.OMEGA0, 0.0, None, dt, shock=False, gain=[g],
                                g_sat=g_sat, tol=1e-12)
        Ez = E0 * np.exp(2 * g * z) / (1 + (g_sat * S[0, 0, 0, 0] * E0 / g) * (np.exp(2 * g * z) - 1))
        assert abs(O.energy(A, dt) / Ez - 1) < (1e-7 if integ == "rk" else 1e-5)
        assert rel(A, A0 * np.sqrt(Ez / E0)) < (1e-7 if integ == "rk" else 1e-5)
    # the literal triple sum of the printed term on a small multimode field
    rng = np.random.default_rng(5)
    P = 3
    Sm = rng.standard_normal((P, P, P, P))
    Am = rng.standard_normal((P, 16)) + 1j * rng.standard_normal((P, 16))
    lit = np.zeros_like(Am)
    for p in range(P):
        for l in range(P):
            for m in range(P):
                for n in range(P):
                    lit[p] -= 0.7 * Sm[p, l, m, n] * Am[l] * (dt * np.sum(Am[m] * np.conj(Am[n])))
    assert rel(O.saturation_term(Am, Sm, 0.7, dt), lit) < 1e-13


def test_z_dependent_coupling_against_library_ode_solver():
    """Two modes, no nonlinearity, Q(z) = f(z) Q0 with a grating profile f: per frequency the field
    obeys a 2 x 2 linear ODE, integrated here by scipy's solve_ivp as an independent witness; a grating whose period
    matches the modes' beat length transfers power that the unmodulated coupler (strongly mismatched) cannot."""
    from scipy.integrate import solve_ivp
    N, dt = 64, 5e-15
    A0 = np.zeros((2, N), np.complex128)
    A0[0] = 1.0
    Dm, kap, z = 900.0, 25.0, 0.05
    beta = np.array([[0.0], [Dm]])
    Q0 = np.array([[0, kap], [kap, 0]], dtype=complex)
    f = lambda zz: 2.0 * np.cos(Dm * zz)
    S0 = np.zeros((2, 2, 2, 2))
    rhs = lambda zz, a: 1j * np.array([0.0, Dm]) * a + 1j * f(zz) * (Q0.T @ a)
    sol = solve_ivp(rhs, (0, z), np.array([1.0 + 0j, 0.0 + 0j]), rtol=1e-11, atol=1e-13)
    want = sol.y[:, -1]
    A = O.rk4ip_propagate(A0, z, z / 400, beta, S0, 0.0, W.OMEGA0, 0.0, None, dt, shock=False, coupling=(Q0, f))
    assert np.abs(A[:, 3] - want).max() < 2e-7                       # O(h^4) of the 400-step RK4IP against the 1e-11 witness
    Am = O.mpa_propagate(A0, z, z / 2000, 10, beta, S0, 0.0, W.OMEGA0, 0.0, None, dt, shock=False, coupling=(Q0, f),
                         tol=1e-12)
    assert np.abs(Am[:, 3] - want).max() < 2e-5
    assert abs(want[1]) ** 2 > 0.7                                    # phase matched by the grating: sin^2(kap z) = 0.90
    flat = O.rk4ip_propagate(A0, z, z / 400, beta, S0, 0.0, W.OMEGA0, 0.0, None, dt, shock=False, coupling=Q0)
    assert abs(flat[1, 3]) ** 2 < 0.02                                # without it: 4 kap^2 / D^2 at most
    # a constant profile is the constant coupler
    same = O.rk4ip_propagate(A0, z, z / 400, beta, S0, 0.0, W.OMEGA0, 0.0, None, dt, shock=False,
                             coupling=(Q0, lambda zz: 1.0))
    assert np.array_equal(same, flat)


# ------------------------------------------------------------------ Eq. 2
def test_overlap_tensor_closed_forms_and_symmetries():
    """Eq. 2 on the GRIN Hermite-Gauss modes of the configurations: S_1111 = 1 / (pi w^2) (the Gaussian
    mode's effective area), S_2222 = 3/4 S_1111 (HG10), S_1122 = 1/2 S_1111; all 24 index permutations equal
    (PAPER.md:60-63); staged matmul form = the literal four loops."""
    F, dA, _ = W.grin_modes(2)                                   # 6 modes on the 256 x 256 grid
    S = O.overlap_tensor(F, dA)
    w0 = W.grin_spot_size()
    s1111 = 1.0 / (math.pi * w0 ** 2)
    assert abs(S[0, 0, 0, 0] / s1111 - 1) < 1e-12
    assert abs(S[1, 1, 1, 1] / (0.75 * s1111) - 1) < 1e-12
    assert abs(S[0, 0, 1, 1] / (0.5 * s1111) - 1) < 1e-12
    import itertools
    for perm in itertools.permutations(range(4)):
        assert np.allclose(S, S.transpose(perm), rtol=0, atol=1e-12 * s1111)
    rng = np.random.default_rng(3)
    Fr = rng.standard_normal((3, 40))
    assert np.allclose(O.overlap_tensor(Fr, 0.3), O.overlap_tensor_literal(Fr, 0.3), rtol=1e-13, atol=0)
    # scale invariance: the normalisation removes the units of F
    assert np.allclose(O.overlap_tensor(7.0 * Fr, 0.3), O.overlap_tensor(Fr, 0.3), rtol=1e-13, atol=0)


def test_aposteriori_stop_rule_keeps_the_result_within_tol_and_saves_iterations():
    """Reading S25: stopping on the a-posteriori bound err rho / (1 - rho) instead of the raw difference of the last
    two iterates.  (i) the bound holds: at every iteration the distance of the iterate to the fixed point (taken from a
    run converged to 1e-13) is below it; (ii) the propagated field differs from the S12 result by less than tol;
    (iii) it never takes more iterations, and fewer where the last S12 iteration only confirmed convergence."""
    wl = W.make_config(2, N=256, max_group=1)
    args = (wl.beta, wl.S, wl.kappa, wl.omega0, wl.f_R, wl.h_R, wl.dt)
    omega = O.omega_grid(wl.N, wl.dt)
    D = O.dispersion_operator(wl.beta, omega)
    K = 1j * wl.kappa * (1 + omega / wl.omega0)
    nlt = lambda A: O.nonlinear_term(A, wl.S, wl.f_R, wl.h_R, wl.dt)
    psi0 = O.to_freq(3.0 * wl.A0)                                   # stronger nonlinearity: more iterations to look at
    hist, keep = [], []
    O.mpa_large_step(psi0, 10, wl.dz, D, nlt, K, tol=1e-13, history=hist, planes_out=keep)
    star = keep[0]
    dist = [max(np.linalg.norm(h[j] - star[j]) / np.linalg.norm(star[j]) for j in range(1, 11)) for h in hist]
    errs = [max(np.linalg.norm(hist[i][j] - (hist[i - 1][j] if i else psi0)) / np.linalg.norm(hist[i][j])
                for j in range(1, 11)) for i in range(len(hist))]
    for i in range(2, len(hist) - 2):
        rho = max(errs[i] / errs[i - 1], errs[i - 1] / errs[i - 2])      # the ratios alternate: take the larger
        assert rho < 1 and dist[i] <= errs[i] * rho / (1 - rho), i
        assert dist[i] < errs[i]                                     # the raw difference over-estimates the error
    L = 6 * 10 * wl.dz
    s0, s1 = {}, {}
    ref = O.mpa_propagate(wl.A0, L, wl.dz, 10, *args, tol=1e-6, stats=s0)
    got = O.mpa_propagate(wl.A0, L, wl.dz, 10, *args, tol=1e-6, stats=s1, stop_rule=1)
    assert rel(got, ref) < 1e-6 and s1["not_converged"] == 0
    assert s1["iterations"] < s0["iterations"] and s1["large_steps"] == s0["large_steps"]
    # never more iterations, whatever the strength of the nonlinearity
    for amp in (0.3, 3.0):
        a0, a1 = {}, {}
        r0 = O.mpa_propagate(amp * wl.A0, L, wl.dz, 10, *args, tol=1e-6, stats=a0)
        r1 = O.mpa_propagate(amp * wl.A0, L, wl.dz, 10, *args, tol=1e-6, stats=a1, stop_rule=1)
        assert a1["iterations"] <= a0["iterations"] and rel(r1, r0) < 1e-6
