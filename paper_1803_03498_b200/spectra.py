"""Linear absorption (Eq. 56) on top of the C-ABI path.

The propagation -- the HEOM right-hand side and RK4 of every auxiliary density matrix, and the dipole trace
Tr(mu_p sigma_0(t)) -- runs in the CUDA kernels through `Heom`; this module only marshals arguments, loops over
the three polarisation directions of Eq. 55 (independent replicas) and Fourier-transforms the resulting
correlation function on the host (a few thousand numbers).
"""
import numpy as np

from .binding import Heom

HBAR_CM_FS = 5308.8   # cm^-1 fs (BASELINE.json config 1)


def linear_absorption(H_cm, bath_state, dipoles, lambda_cm, nu_per_fs, T_kelvin, K, D, dt_fs, steps, pad=4,
                      device=0, **options):
    """<LA(omega)>_rot = Re sum_p int_0^inf dt exp(i omega t) Tr[mu_p(t) mu_p(0) rho(0)]  (Eq. 56).

    H_cm [N+1][N+1] with the ground state as state 0 (Eq. 48); bath_state as heom_create_sites; dipoles [N][3]
    (d_m of Eq. 53).  sigma_0(0) = mu_p |0><0|, all ADOs zero.  Returns (t [steps+1] fs,
    corr [steps+1] complex, omega [cm^-1], spectrum): corr = sum_p Tr(mu_p sigma_0(t)); the integral is the
    trapezoid rule on the zero-padded correlation function, omega = 2 pi hbar k / (n dt)."""
    H = np.asarray(H_cm, dtype=np.float64)
    n = H.shape[0]
    d = np.asarray(dipoles, dtype=np.float64)
    if d.shape != (n - 1, 3):
        raise ValueError("dipoles must be [n_states-1][3]")
    corr = np.zeros(steps + 1, dtype=np.complex128)
    g = Heom(H, lambda_cm, nu_per_fs, T_kelvin, K, D, device=device, bath_state=bath_state, **options).bind()
    try:
        for p in range(3):
            mu = np.zeros((n, n), dtype=np.complex128)
            mu[1:, 0] = d[:, p]
            mu[0, 1:] = d[:, p]
            s0 = np.zeros((n, n), dtype=np.complex128)
            s0[:, 0] = mu[:, 0]                      # mu_p |0><0|
            g.set_state(s0)
            corr[0] += g.expectation(mu)
            for q in range(1, steps + 1):
                g.rk4_steps(dt_fs, 1)
                corr[q] += g.expectation(mu)
    finally:
        g.close()
    t = dt_fs * np.arange(steps + 1)
    nfft = int(pad) * (steps + 1)
    f = corr.copy()
    f[0] *= 0.5                                      # trapezoid end point; the padded tail is zero
    spec = (np.fft.ifft(f, nfft) * nfft * dt_fs).real   # sum_q f_q exp(+i omega_k t_q) dt
    omega = 2.0 * np.pi * HBAR_CM_FS * np.fft.fftfreq(nfft, d=dt_fs)
    order = np.argsort(omega)
    return t, corr, omega[order], spec[order]
