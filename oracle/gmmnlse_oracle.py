"""fp64 CPU oracle for the GMMNLSE / MPA hot path  --  TEST INFRASTRUCTURE ONLY.

This file is the plain, slow, obviously-correct statement of what the CUDA path
in ``paper_1708_05324_b200/csrc`` computes.  It is written from the paper
(Wright et al., arXiv 1708.05324; citations are ``PAPER.md:<line>``) and shares
no code with the CUDA path.  Only ``tests/``, ``__graft_entry__.smoke()`` and
``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may import it; the
product path never does.

Everything is complex128 / float64 numpy.  There is no blocking, packing or
symmetry exploitation: the nonlinear term is the ordered P^2-pair sum of Eq. 1.
Library primitives serve as steps where the definition is a textbook one: the
matmul of the (m,n) sum and the FFT (``to_freq`` / ``to_time``; the recursive
radix-2 transform written out below and the O(N^2) DFT are their pins).

Conventions (S1; fixed by Eq. 1 <-> Eq. 12 consistency,
PAPER.md:53 vs PAPER.md:209: ``(1 + i/w0 d_t)  <->  (1 + w/w0)`` i.e.
``d_t <-> -i w``):

    to-frequency   At_k = sum_n A_n exp(+2 pi i k n / N)          (un-normalised)
    to-time        A_n  = (1/N) sum_k At_k exp(-2 pi i k n / N)
    w_k = 2 pi k' / (N dt),  k' = k for k < N/2 else k - N
    D_w^(p) = i [ dbeta0 + dbeta1 w + sum_{k>=2} beta_k w^k / k! ]

Parity pins for every function live in ``tests/test_oracle_*.py`` (closed
forms, brute force, invariants, convergence orders).  Nothing here is
"parity unpinned".  (The step-index LP-mode S *values* produced by the input
generator are unpinned, but S is an input to both sides -- see DESIGN.md.)
"""
from __future__ import annotations

import math
import numpy as np

__all__ = [
    "dft_direct", "fft_radix2", "to_freq", "to_time", "omega_grid",
    "overlap_tensor", "overlap_tensor_literal",
    "dispersion_operator", "coupling_term", "coupling_at", "saturation_term", "raman_transfer", "pair_products",
    "raman_convolve_direct", "raman_convolve", "nonlinear_term",
    "nonlinear_term_literal", "nonlinear_term_general", "nonlinear_term_general_literal",
    "nonlinear_op", "nonlinear_op_freq",
    "rk4ip_step", "rk4ip_propagate", "mpa_large_step", "mpa_propagate",
    "energy", "photon_number", "conserved_quantity",
]


# --------------------------------------------------------------------------- O1
def dft_direct(x: np.ndarray, sign: int) -> np.ndarray:
    """O(N^2) DFT along the last axis: X_k = sum_n x_n exp(sign 2 pi i k n / N).

    Used only to check :func:`fft_radix2` on tiny N (and for tiny-N pins).
    """
    x = np.asarray(x, dtype=np.complex128)
    N = x.shape[-1]
    n = np.arange(N)
    W = np.exp(sign * 2j * np.pi * np.outer(n, n) / N)     # W[k, n]
    return x @ W.T


def fft_radix2(x: np.ndarray, sign: int) -> np.ndarray:
    """Recursive radix-2 decimation-in-time FFT along the last axis (N = 2^q).

    X_k = sum_n x_n exp(sign 2 pi i k n / N); un-normalised for both signs.
    Textbook Cooley-Tukey: X_k = E_k + w^k O_k, X_{k+N/2} = E_k - w^k O_k.
    """
    x = np.asarray(x, dtype=np.complex128)
    N = x.shape[-1]
    if N == 1:
        return x.copy()
    if N & (N - 1):
        raise ValueError("N must be a power of two")
    even = fft_radix2(x[..., 0::2], sign)
    odd = fft_radix2(x[..., 1::2], sign)
    w = np.exp(sign * 2j * np.pi * np.arange(N // 2) / N)
    t = w * odd
    return np.concatenate([even + t, even - t], axis=-1)


def to_freq(A: np.ndarray) -> np.ndarray:
    """At_k = sum_n A_n exp(+2 pi i k n/N)  (the paper's F{.}, reading S1).

    The library FFT serves as the step (numpy's pocketfft: ``ifft`` carries exp(+i..) and 1/N, undone here).  It is
    pinned against :func:`dft_direct` (N <= 64) and against the written-out :func:`fft_radix2` at every power of
    two up to 16384 (``tests/test_oracle_pins.py``); rounding differs from the recursion at the 1e-16 level only.
    """
    A = np.asarray(A, dtype=np.complex128)
    return np.fft.ifft(A, axis=-1) * A.shape[-1]


def to_time(At: np.ndarray) -> np.ndarray:
    """A_n = (1/N) sum_k At_k exp(-2 pi i k n/N)."""
    At = np.asarray(At, dtype=np.complex128)
    return np.fft.fft(At, axis=-1) / At.shape[-1]


def omega_grid(N: int, dt: float) -> np.ndarray:
    """Angular-frequency offset of bin k; Nyquist bin is -N/2 (reading S9)."""
    k = np.arange(N)
    kp = np.where(k < N // 2, k, k - N)
    return 2.0 * np.pi * kp / (N * dt)


# ------------------------------------------------------------------ Eq. 2
def overlap_tensor(F: np.ndarray, dA: float) -> np.ndarray:
    """S_plmn = int F_p F_l F_m F_n dA / [int F_p^2 dA int F_l^2 dA int F_m^2 dA int F_n^2 dA]^(1/2)  (PAPER.md:60,
    Eq. 2) for real scalar mode fields F[p][grid] by the rectangle (midpoint) rule on the grid: all P^2 ORDERED pair
    functions F_p F_l, one matmul over the grid, no symmetry used."""
    F = np.asarray(F, dtype=np.float64)
    P = F.shape[0]
    f = F.reshape(P, -1)
    nrm = np.sqrt(np.sum(f * f, axis=1) * dA)
    pair = (f[:, None, :] * f[None, :, :]).reshape(P * P, -1)         # [(p l)][g]
    S = (pair @ pair.T) * dA
    S = S.reshape(P, P, P, P) / (nrm[:, None, None, None] * nrm[None, :, None, None] *
                                 nrm[None, None, :, None] * nrm[None, None, None, :])
    return S


def overlap_tensor_literal(F: np.ndarray, dA: float) -> np.ndarray:
    """The same as four nested loops over the modes (tiny P only)."""
    F = np.asarray(F, dtype=np.float64)
    P = F.shape[0]
    f = F.reshape(P, -1)
    S = np.zeros((P, P, P, P))
    for p in range(P):
        for l in range(P):
            for m in range(P):
                for n in range(P):
                    num = np.sum(f[p] * f[l] * f[m] * f[n]) * dA
                    den = math.sqrt(np.sum(f[p] ** 2) * dA * np.sum(f[l] ** 2) * dA * np.sum(f[m] ** 2) * dA *
                                    np.sum(f[n] ** 2) * dA)
                    S[p, l, m, n] = num / den
    return S


# ------------------------------------------------------------------ linear part
def dispersion_operator(beta: np.ndarray, omega: np.ndarray, gain=None) -> np.ndarray:
    """D_w^(p) = i[dbeta0 + dbeta1 w + sum_{k>=2} beta_k w^k / k!]  [+ g_p].

    ``gain[p]`` (optional, 1/m): the small-signal FIELD gain (loss if negative) of the added term
    ``g_p A_p`` (section F.2); being linear and diagonal it joins D as its real part.

    ``beta[p][k]`` = beta_k^(p) in s^k/m (k=0: dbeta0 [1/m], k=1: dbeta1 [s/m]).
    Follows from Eq. 1's first three terms with d_t -> -i w:
    -dbeta1 d_t -> +i dbeta1 w;  i^{m+1} beta_m/m! d_t^m -> i beta_m w^m / m!.
    """
    beta = np.atleast_2d(np.asarray(beta, dtype=np.float64))
    P, nb = beta.shape
    D = np.zeros((P, omega.shape[0]), dtype=np.float64)
    for k in range(nb):
        D += beta[:, k:k + 1] * omega[None, :] ** k / math.factorial(k)
    if gain is not None:
        return 1j * D + np.asarray(gain, dtype=np.float64).reshape(P, 1)
    return 1j * D


def coupling_term(At: np.ndarray, Qc) -> np.ndarray:
    """C_p = i sum_n Q_np A_n  (section F.1; Eq. 13 defines Q_np): the linear mode-coupling term added
    to the right-hand side.  ``Qc[n][p]`` = Q_np [1/m], constant over the call and over frequency, so the sum
    reads the same in the time and the frequency domain."""
    return 1j * (np.asarray(Qc, dtype=np.complex128).T @ At)


def coupling_at(coupling, z):
    """Q_np at position z (measured from the start of the call).  ``coupling`` is a constant matrix, a callable z -> matrix,
    or a pair (Q0, f) meaning Q(z) = f(z) Q0: the separable perturbation eps(x, y) f(z) of PAPER.md:277 (gratings:
    f periodic; disorder: f a stochastic function)."""
    if callable(coupling):
        return np.asarray(coupling(z), dtype=np.complex128)
    if isinstance(coupling, tuple):
        return float(coupling[1](z)) * np.asarray(coupling[0], dtype=np.complex128)
    return np.asarray(coupling, dtype=np.complex128)


def saturation_term(A: np.ndarray, S, g_sat: float, dt: float) -> np.ndarray:
    """First-order gain saturation (section F.2): the Taylor expansion of
    g(I) = g0 / [1 + int dt I / I_sat] projected on the modes adds, beside g_p A_p,

        - g_sat sum_lmn S_plmn A_l(t) int dtau A_m(tau) A_n*(tau),      g_sat = g0 / I_sat  [m/J]

    (reading S22: the paper prints the term without its gain prefactor; with S in 1/m^2 and the integral in J the sum is
    J/m^2, so the coefficient that makes it a gain per length is g0 / I_sat).  The time integral is the rectangle sum
    dt sum_t over the periodic window.  Linear in A_l with a matrix that depends on the field only through its
    time-integrated pair products, so it reads the same in the time and the frequency domain."""
    A = np.asarray(A, dtype=np.complex128)
    S = np.asarray(S[1] if isinstance(S, tuple) else S)          # general form: the Raman tensor, as printed
    E = dt * (A @ np.conj(A).T)                                   # E_mn = int A_m A_n* dtau
    W = np.einsum("plmn,mn->pl", S, E)
    return -g_sat * (W @ A)


# ---------------------------------------------------------------- nonlinear part
def raman_transfer(h_R: np.ndarray, dt: float) -> np.ndarray:
    """ht_R(w_k) = dt * F{h_R}_k  with h_R sampled at t_j = j dt (reading S6/S7)."""
    return dt * to_freq(np.asarray(h_R, dtype=np.float64))


def pair_products(A: np.ndarray) -> np.ndarray:
    """T_mn(t) = A_m(t) A_n*(t) for all P^2 ordered pairs (Eq. 1)."""
    return A[:, None, :] * np.conj(A[None, :, :])


def raman_convolve_direct(T: np.ndarray, h_R: np.ndarray, dt: float) -> np.ndarray:
    """R[i] = dt sum_j h_R[j] T[(i-j) mod N]  -- the literal circular sum (S7).

    Discretisation of  int_0^inf h_R(tau) T(t - tau) dtau  (Eq. 1) on the
    periodic grid.  O(N^2): tiny N only.
    """
    N = T.shape[-1]
    R = np.zeros_like(T, dtype=np.complex128)
    for i in range(N):
        for j in range(N):
            R[..., i] += h_R[j] * T[..., (i - j) % N]
    return dt * R


def raman_convolve(T: np.ndarray, h_R: np.ndarray, dt: float) -> np.ndarray:
    """Same circular convolution through O1 (convolution theorem)."""
    return to_time(raman_transfer(h_R, dt) * to_freq(T))


def nonlinear_term(A, S, f_R=0.0, h_R=None, dt=1.0, direct_conv=False):
    """N_p(t) = sum_{lmn} S_plmn A_l [(1-fR) A_m A_n* + fR (h_R (*) A_m A_n*)].

    Eq. 1 bracket with S^K = S^R = S (Eq. 2; reading
    S8).  Staged exactly as the definition reads: all P^2 ordered pair streams
    T_mn, their Raman convolution, the blend, the sum over (m,n) (a matmul
    step), the sum over l.  No symmetry of S is used.
    """
    if isinstance(S, tuple):                              # (S^K, S^R): the general form of Eq. 1
        return nonlinear_term_general(A, S[0], S[1], f_R, h_R, dt, direct_conv)
    A = np.asarray(A, dtype=np.complex128)
    S = np.asarray(S, dtype=np.float64)
    P, N = A.shape
    T = pair_products(A)                                  # [m][n][t]
    if f_R != 0.0:
        R = (raman_convolve_direct if direct_conv else raman_convolve)(T, h_R, dt)
        B = (1.0 - f_R) * T + f_R * R
    else:
        B = T
    U = S.reshape(P * P, P * P) @ B.reshape(P * P, N)     # U[(p l)][t]
    U = U.reshape(P, P, N)
    return np.einsum("plt,lt->pt", U, A)


def nonlinear_term_literal(A, S, f_R=0.0, h_R=None, dt=1.0):
    """The same sum as four nested Python loops + the literal convolution.

    Brute-force cross-check of :func:`nonlinear_term` for P <= 4, N <= 32.
    """
    A = np.asarray(A, dtype=np.complex128)
    P, N = A.shape
    out = np.zeros((P, N), dtype=np.complex128)
    for p in range(P):
        for l in range(P):
            for m in range(P):
                for n in range(P):
                    s = S[p, l, m, n]
                    if s == 0.0:
                        continue
                    T = A[m] * np.conj(A[n])
                    term = (1.0 - f_R) * T
                    if f_R != 0.0:
                        R = np.zeros(N, dtype=np.complex128)
                        for i in range(N):
                            acc = 0.0
                            for j in range(N):
                                acc += h_R[j] * T[(i - j) % N]
                            R[i] = dt * acc
                        term = term + f_R * R
                    out[p] += s * A[l] * term
    return out


def nonlinear_term_general(A, SK, SR, f_R=0.0, h_R=None, dt=1.0, direct_conv=False):
    """N_p(t) = sum_{lmn} A_l [(1-fR) S^K_plmn A_m A_n* + fR S^R_plmn (h_R (*) A_m A_n*)].

    Eq. 1 before the scalar-mode simplification of Eq. 2: separate Kerr and Raman
    tensors, real or complex, with no index symmetry assumed (S^K and S^R differ once the
    modes carry polarisation).  Two polarisations per spatial mode are 2P fields
    with the corresponding (2P)^4 tensors.  Staged as the definition reads: all P^2 ordered pair
    streams, their convolution, one matmul per tensor, the sum over l.
    """
    A = np.asarray(A, dtype=np.complex128)
    SK = np.asarray(SK, dtype=np.complex128)
    SR = np.asarray(SR, dtype=np.complex128)
    P, N = A.shape
    T = pair_products(A).reshape(P * P, N)                # [(m n)][t]
    U = (1.0 - f_R) * (SK.reshape(P * P, P * P) @ T)
    if f_R != 0.0:
        R = (raman_convolve_direct if direct_conv else raman_convolve)(T, h_R, dt)
        U = U + f_R * (SR.reshape(P * P, P * P) @ R)
    return np.einsum("plt,lt->pt", U.reshape(P, P, N), A)


def nonlinear_term_general_literal(A, SK, SR, f_R=0.0, h_R=None, dt=1.0):
    """Four nested loops + the literal convolution for the general form (tiny P, N only)."""
    A = np.asarray(A, dtype=np.complex128)
    P, N = A.shape
    out = np.zeros((P, N), dtype=np.complex128)
    for p in range(P):
        for l in range(P):
            for m in range(P):
                for n in range(P):
                    T = A[m] * np.conj(A[n])
                    term = (1.0 - f_R) * SK[p, l, m, n] * T
                    if f_R != 0.0:
                        R = np.zeros(N, dtype=np.complex128)
                        for i in range(N):
                            acc = 0.0
                            for j in range(N):
                                acc += h_R[j] * T[(i - j) % N]
                            R[i] = dt * acc
                        term = term + f_R * SR[p, l, m, n] * R
                    out[p] += A[l] * term
    return out


def _shock_factor(omega, omega0, shock):
    return (1.0 + omega / omega0) if shock else np.ones_like(omega)


def nonlinear_op_freq(At, S, kappa, omega, omega0, f_R, h_R, dt, shock=True):
    """N^(At) = i kappa (1 + w/w0) F{ N_p[F^-1 At] }  (Eq. 12 prefactor)."""
    A = to_time(At)
    Nt = nonlinear_term(A, S, f_R, h_R, dt)
    return 1j * kappa * _shock_factor(omega, omega0, shock) * to_freq(Nt)


def nonlinear_op(A, S, kappa, omega0, f_R, h_R, dt, shock=True):
    """dA_p(t) = i kappa (1 + i/w0 d_t) N_p[A](t): last term of Eq. 1, time in/out."""
    A = np.asarray(A, dtype=np.complex128)
    omega = omega_grid(A.shape[-1], dt)
    return to_time(nonlinear_op_freq(to_freq(A), S, kappa, omega, omega0, f_R, h_R, dt, shock))


# ------------------------------------------------------------------- O3: RK4IP
def rk4ip_step(At, h, D, nl, z=None):
    """One RK4IP step (textbook interaction-picture RK4; named by north_star).

    ``nl(At)`` is the frequency-domain nonlinear operator; E = exp(D h / 2).  With ``z`` given (a right-hand side
    that depends on position: z-dependent coupling) it is called as ``nl(At, z_stage)`` at z, z + h/2, z + h/2, z + h.
    """
    f = nl if z is None else None
    E = np.exp(D * (h / 2.0))
    AI = E * At
    k1 = E * (h * (f(At) if f else nl(At, z)))
    k2 = h * (f(AI + k1 / 2.0) if f else nl(AI + k1 / 2.0, z + h / 2.0))
    k3 = h * (f(AI + k2 / 2.0) if f else nl(AI + k2 / 2.0, z + h / 2.0))
    k4 = h * (f(E * (AI + k3)) if f else nl(E * (AI + k3), z + h))
    return E * (AI + k1 / 6.0 + k2 / 3.0 + k3 / 3.0) + k4 / 6.0


def rk4ip_propagate(A0, L, dz, beta, S, kappa, omega0, f_R, h_R, dt, shock=True, n_steps=None,
                    gain=None, coupling=None, g_sat=0.0):
    """Propagate A0[p][t] over L with fixed step dz using RK4IP; returns A(L)[p][t].

    ``gain`` joins D; ``coupling`` (Q_np, see :func:`coupling_at`) and the saturation term (``g_sat``,
    :func:`saturation_term`) are integrated with the nonlinear term (they do not commute with D)."""
    A0 = np.asarray(A0, dtype=np.complex128)
    N = A0.shape[-1]
    omega = omega_grid(N, dt)
    D = dispersion_operator(beta, omega, gain)
    if n_steps is None:
        n_steps = int(round(L / dz))
    nl0 = lambda X: nonlinear_op_freq(X, S, kappa, omega, omega0, f_R, h_R, dt, shock)
    if coupling is None and g_sat == 0.0:
        At = to_freq(A0)
        for _ in range(n_steps):
            At = rk4ip_step(At, dz, D, nl0)
        return to_time(At)

    def nl(X, z):
        out = nl0(X)
        if coupling is not None:
            out = out + coupling_term(X, coupling_at(coupling, z))
        if g_sat != 0.0:
            out = out + to_freq(saturation_term(to_time(X), S, g_sat, dt))
        return out
    At = to_freq(A0)
    for i in range(n_steps):
        At = rk4ip_step(At, dz, D, nl, z=i * dz)
    return to_time(At)


# --------------------------------------------------------------------- O4: MPA
def mpa_large_step(psi0, M, dz, D, nl_time, K, tol=1e-6, max_iter=None, fixed_iter=0,
                   history=None, coupling=None, first_iterate=None, planes_out=None, z0=0.0, extra_time=None,
                   stop_rule=0):
    """One MPA large step z0 -> z0 + M dz  (Eqs. 11-12).

    psi0[p][w] = At(z0).  Planes j = 0..M (reading S10).  ``nl_time(A_t)`` returns
    N_p[A](t); ``K[w] = i kappa (1 + w/w0)``.  Returns (At(z0 + M dz), n_iter,
    last_err, converged).

      first iterate      psi_j = psi_0; ``first_iterate[j]`` (optional,
                         [M+1][P][N], plane 0 ignored) replaces it: the predictor of reading S11, see mpa_propagate
      each iteration     A_j = psi_j exp(D j dz)            (Eq. 11)
                         G_j = K exp(-D j dz) F{N[A_j]}     (Eq. 12 integrand)
                         psi_j <- psi_0 + dz [G_0/2 + G_1 + .. + G_{j-1} + G_j/2]
                                                            (trapezoid)
      stop when err = max_j ||psi_j^new - psi_j|| / ||psi_j^new|| < tol   (S12)
      ``stop_rule=1`` (reading S25, an option: off by default): the paper stops "once the accuracy reaches a given
      threshold", and the accuracy of the iterate just formed is its distance to the fixed point,
      which the difference of the last two iterates over-estimates.  With a contraction ratio rho < 1 the fixed-point
      iteration gives the a-posteriori bound  ||psi^(n) - psi*|| <= err_n rho / (1 - rho).  The ratios err_n / err_{n-1}
      of this iteration alternate between odd and even n (measured: 0.098, 0.18, 0.056, 0.11, 0.042, ..), so rho is
      the LARGER of the last two ratios (needs n >= 3); stop when the bound (or err_n itself) is below tol.  The
      result differs from the S12 result by less than tol; it takes one iteration less whenever the last S12
      iteration only confirmed convergence.
    """
    P, N = psi0.shape
    if max_iter is None:
        max_iter = 2 * M + 4
    psi = np.broadcast_to(psi0, (M + 1, P, N)).copy()
    if first_iterate is not None:
        psi[1:] = first_iterate[1:]
    G = np.zeros((M + 1, P, N), dtype=np.complex128)
    # extra right-hand-side terms (linear coupling at the plane's position z0 + j dz; ``extra_time``: a term given in the
    # time domain, e.g. the gain saturation), rotated like the nonlinear one
    def extra(Af, j):
        out = 0.0
        if coupling is not None:
            out = out + coupling_term(Af, coupling_at(coupling, z0 + j * dz))
        if extra_time is not None:
            out = out + to_freq(extra_time(to_time(Af)))
        return out
    G[0] = K * to_freq(nl_time(to_time(psi0))) + extra(psi0, 0)   # depends on psi_0 only (S10)
    n_iter, err, converged = 0, np.inf, False
    err_prev, rho_prev = np.inf, np.inf
    while True:
        for j in range(1, M + 1):
            Afj = psi[j] * np.exp(D * (j * dz))
            G[j] = np.exp(-D * (j * dz)) * (K * to_freq(nl_time(to_time(Afj))) + extra(Afj, j))
        new = np.empty_like(psi)
        new[0] = psi0
        for j in range(1, M + 1):
            acc = 0.5 * G[0] + 0.5 * G[j]
            for i in range(1, j):
                acc = acc + G[i]
            new[j] = psi0 + dz * acc
        err = 0.0
        for j in range(1, M + 1):
            num = np.sqrt(np.sum(np.abs(new[j] - psi[j]) ** 2))
            den = np.sqrt(np.sum(np.abs(new[j]) ** 2))
            err = max(err, num / den if den > 0 else 0.0)
        psi = new
        n_iter += 1
        if history is not None:
            history.append(psi.copy())
        est = err
        rho_now = err / err_prev if err_prev > 0 else 0.0           # inf / inf on the first iteration -> nan: unused
        if stop_rule == 1 and n_iter >= 3:
            rho = max(rho_now, rho_prev)
            if rho < 1.0:
                est = err * rho / (1.0 - rho)
        err_prev, rho_prev = err, rho_now
        if fixed_iter > 0:
            if n_iter >= fixed_iter:
                converged = True
                break
        elif err < tol or est < tol:
            converged = True
            break
        elif n_iter >= max_iter:
            break
    if planes_out is not None:
        planes_out.append(psi)
    return psi[M] * np.exp(D * (M * dz)), n_iter, err, converged


def mpa_propagate(A0, L, dz, M, beta, S, kappa, omega0, f_R, h_R, dt, shock=True,
                  tol=1e-6, max_iter=None, fixed_iter=0, stats=None, history=None, gain=None, coupling=None,
                  predictor=0, g_sat=0.0, stop_rule=0):
    """Propagate with MPA; the last large step uses M' = (L/dz) mod M planes.

    ``predictor`` (reading S11: an optimisation of the first iterate, off by default = the paper's psi_j = psi_0):
    1 starts the planes of a large step from the previous large step's converged increments carried into the new
    interaction picture, psi_j^(1) = psi_0' + exp(D M dz) (psi_j^prev - psi_0^prev): the increment of plane j is
    dz times the trapezoid sum of G, and under linear propagation over one large step every phase-matched term of
    G_p picks up the phase of mode p (the factor exp(D M dz)); what is left for the iteration is the change of the
    envelopes over one large step and the non-phase-matched terms.  Same fixed point, same stopping rule."""
    A0 = np.asarray(A0, dtype=np.complex128)
    N = A0.shape[-1]
    omega = omega_grid(N, dt)
    D = dispersion_operator(beta, omega, gain)
    K = 1j * kappa * _shock_factor(omega, omega0, shock)
    nl_time = lambda A: nonlinear_term(A, S, f_R, h_R, dt)
    n_small = int(round(L / dz))
    psi0 = to_freq(A0)
    done = 0
    tot_it, n_large, n_noconv, last_err = 0, 0, 0, 0.0
    prev = None                                           # (planes, psi_0) of the previous large step
    while done < n_small:
        Mc = min(M, n_small - done)
        hist = [] if history is not None else None
        first = None
        if predictor == 1 and prev is not None and prev[0].shape[0] == Mc + 1:
            first = psi0[None] + np.exp(D * (prev[0].shape[0] - 1) * dz)[None] * (prev[0] - prev[1][None])
        keep = []
        start = psi0
        sat = None if g_sat == 0.0 else (lambda A: saturation_term(A, S, g_sat, dt))
        psi0, it, last_err, conv = mpa_large_step(psi0, Mc, dz, D, nl_time, K, tol,
                                                   max_iter, fixed_iter, hist, coupling, first, keep,
                                                   z0=done * dz, extra_time=sat, stop_rule=stop_rule)
        prev = (keep[0], start)
        if history is not None:
            history.append(hist)
        tot_it += it
        n_large += 1
        n_noconv += 0 if conv else 1
        done += Mc
    if stats is not None:
        stats.update(large_steps=n_large, iterations=tot_it, last_err=last_err,
                     not_converged=n_noconv)
    return to_time(psi0)


# ------------------------------------------------------------------ invariants
def energy(A, dt):
    """sum_p sum_n |A_p(t_n)|^2 dt  [J]  -- conserved with shock off (S15)."""
    return float(np.sum(np.abs(A) ** 2) * dt)


def photon_number(A, dt, omega0):
    """sum_p sum_k |At_p,k|^2 / (1 + w_k/w0)  -- conserved with shock on (S15)."""
    At = to_freq(np.asarray(A, dtype=np.complex128))
    w = omega_grid(A.shape[-1], dt)
    return float(np.sum(np.abs(At) ** 2 / (1.0 + w / omega0)))


def conserved_quantity(A, dt, omega0, shock):
    return photon_number(A, dt, omega0) if shock else energy(A, dt)
