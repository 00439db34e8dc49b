"""overlap_oracle.py -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Plain numpy (fp64) statement of steps iv-v of the paper's likelihood evaluation (arXiv 2505.09600):
Fourier transform of the TDI channels A, E, T, the analytic "Sangria" noise PSDs of Sec. II C and the
noise-weighted inner product, overlap, mismatch and SNR of Eqs. (5.1), (5.2), (6.1).  "P:n" = line n of
/root/reference/PAPER.md; readings G24-G27 are listed in DESIGN.md.  It shares nothing with the CUDA path; only
tests/, __graft_entry__.smoke() and bench.py's cpu_baseline legs may import it.  numpy.fft.rfft is used as a
library primitive for the discrete Fourier transform, everything else is the definition written out.

Pins (tests/test_oracle_overlap.py): Lambda relation S^{2.0} = 4 sin^2(2x) S^{1.5} and the stated low-frequency
power laws; printed constants; zeros of the PSD at x = n pi; Parseval (white PSD: <x|y> = 2 sum x y dt);
closed form <h|h> = A^2 T / S_n(f0) for a bin-centred sinusoid; overlap = 1 / -1 for y = +-c x, symmetry,
Cauchy-Schwarz; SNR additivity over channels (6.1).
Parity unpinned: absolute PSD levels of Fig. 2 (an image; no value is printed in the text).
"""
import numpy as np

C_LIGHT = 299792458.0            # m/s
SQRT_S_ACC = 2.4e-15             # m s^-2 Hz^-1/2
SQRT_S_OMS = 7.9e-12             # m Hz^-1/2
GAL_A = 1.28265531e-44
GAL_ALPHA = 1.62966700
GAL_F2 = 4.81078093e-4           # Hz
GAL_A1, GAL_B1 = -0.223499956, -2.70408439
GAL_AK, GAL_BK = -0.360976122, -2.37822436


def s_pm(f):
    """Eq. (2.10a): proof-mass noise (relative frequency units)."""
    f = np.asarray(f, dtype=np.float64)
    return SQRT_S_ACC ** 2 * (2.0 * np.pi * f * C_LIGHT) ** -2 * (1.0 + (0.0004 / f) ** 2) * (1.0 + (f / 0.008) ** 4)


def s_op(f):
    """Eq. (2.10b): optical-path noise."""
    f = np.asarray(f, dtype=np.float64)
    return SQRT_S_OMS ** 2 * (2.0 * np.pi * f / C_LIGHT) ** 2 * (1.0 + (0.002 / f) ** 4)


def s_gal(f, arm_m, t_obs_yr):
    """Eqs. (2.11), (2.12): galactic foreground, x = 2 pi f L / c, T_obs in years (G26)."""
    f = np.asarray(f, dtype=np.float64)
    x = 2.0 * np.pi * f * arm_m / C_LIGHT
    f1 = 10.0 ** (GAL_A1 * np.log10(t_obs_yr) + GAL_B1)
    fknee = 10.0 ** (GAL_AK * np.log10(t_obs_yr) + GAL_BK)
    return (2.0 * x ** 2 * np.sin(x) ** 2 * GAL_A * f ** (-7.0 / 3.0) * np.exp(-(f / f1) ** GAL_ALPHA)
            * (1.0 + np.tanh((fknee - f) / GAL_F2)))


def psd_aet(f, gen, arm_m=2.5e9, t_obs_yr=1.0, galactic=True):
    """Eqs. (2.13a), (2.13b): S_n^{A,E}(f), S_n^T(f); Lambda = 4 sin^2(2x) (TDI 2.0) or 1 (TDI 1.5).
    f > 0.  Returns (S_AE, S_T)."""
    f = np.asarray(f, dtype=np.float64)
    x = 2.0 * np.pi * f * arm_m / C_LIGHT
    lam = 4.0 * np.sin(2.0 * x) ** 2 if gen == 20 else np.ones_like(x)
    gal = s_gal(f, arm_m, t_obs_yr) if galactic else np.zeros_like(x)
    pm, op = s_pm(f), s_op(f)
    s_ae = (8.0 * lam * np.sin(x) ** 2 * (2.0 * (3.0 + 2.0 * np.cos(x) + np.cos(2.0 * x)) * pm + (2.0 + np.cos(x)) * op)
            + 1.5 * lam * gal)
    s_t = 16.0 * lam * np.sin(x) ** 2 * ((1.0 - np.cos(x)) * op + 8.0 * np.sin(x / 2.0) ** 4 * pm) + lam * gal
    return s_ae, s_t


def spectrum(x, dt):
    """Step iv: x~(f_k) = dt sum_n x_n exp(-2 pi i f_k n dt), f_k = k / (N dt), k = 0 .. N/2 (G24: the series as
    it stands, margins zero, no window)."""
    return dt * np.fft.rfft(np.asarray(x, dtype=np.float64), axis=-1)


def inner(xa, xb, dt, s_n, fmin, fmax):
    """Eq. (5.1): <x|y> = 4 Re int_{fmin}^{fmax} conj(x~) y~ / S_n df as the rectangle rule over the bins with
    fmin <= f_k <= fmax (G25); s_n is sampled on f_k = k df (entry 0 is never used: f = 0 is outside any band)."""
    n = np.asarray(xa).shape[-1]
    df = 1.0 / (n * dt)
    fa, fb = spectrum(xa, dt), spectrum(xb, dt)
    k = np.arange(fa.shape[-1])
    f = k * df
    band = (f >= fmin) & (f <= fmax) & (k > 0)
    integrand = (np.conj(fa) * fb).real[..., band] / np.asarray(s_n)[band]
    return 4.0 * df * np.sum(integrand, axis=-1)


def products(a, b, dt, gen, fmin, fmax, arm_m=2.5e9, t_obs_yr=1.0, galactic=True):
    """For two responses a, b = dict(A, E, T) of arrays [batch][n]: per source and channel <a|a>, <b|b>, <a|b>,
    the overlap (5.2) and the mismatch 1 - |O|.  Returns array [batch][3][5]."""
    n = np.asarray(a["A"]).shape[-1]
    f = np.arange(n // 2 + 1) / (n * dt)
    s_ae, s_t = np.full_like(f, np.inf), np.full_like(f, np.inf)
    s_ae[1:], s_t[1:] = psd_aet(f[1:], gen, arm_m, t_obs_yr, galactic)
    out = np.zeros((np.atleast_2d(a["A"]).shape[0], 3, 5))
    for c, ch in enumerate("AET"):
        s_n = s_t if ch == "T" else s_ae
        xa, xb = np.atleast_2d(a[ch]), np.atleast_2d(b[ch])
        aa, bb, ab = inner(xa, xa, dt, s_n, fmin, fmax), inner(xb, xb, dt, s_n, fmin, fmax), inner(xa, xb, dt, s_n, fmin, fmax)
        with np.errstate(invalid="ignore", divide="ignore"):
            ov = ab / (np.sqrt(aa) * np.sqrt(bb))
        out[:, c, 0], out[:, c, 1], out[:, c, 2], out[:, c, 3], out[:, c, 4] = aa, bb, ab, ov, 1.0 - np.abs(ov)
    return out


def snr(prod_self):
    """Eq. (6.1): rho = sqrt(<A|A> + <E|E> + <T|T>) from the [batch][3] self products."""
    return np.sqrt(np.sum(np.asarray(prod_self), axis=-1))


def log_likelihood(prod):
    """Eq. (D4): ln L = -1/2 <d - h|d - h> = -1/2 (<d|d> + <h|h> - 2 <d|h>), summed over A, E, T, from the
    [batch][3][>=3] products with a = d and b = h."""
    p = np.asarray(prod)
    return -0.5 * np.sum((p[:, :, 0] + p[:, :, 1]) - 2.0 * p[:, :, 2], axis=-1)
