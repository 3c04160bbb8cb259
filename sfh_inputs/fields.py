"""Seeded random fields and pointwise samplers for the synthetic initial conditions.

Recipes: DESIGN.md "Synthetic inputs" (SURVEY.md readings S23, S24, S21).  No method arithmetic.
"""
import numpy as np


def gaussian_random_field(n, slope, seed):
    """Periodic Gaussian random field on n^3 cells, 3-D power spectrum P(k) ~ k^slope on
    1 <= |k| <= n/2 (zero elsewhere), zero mean, unit variance.  Returned as [z,y,x] float64."""
    rng = np.random.default_rng(seed)
    white = rng.standard_normal((n, n, n))
    fk = np.fft.rfftn(white)
    del white
    kx = np.fft.rfftfreq(n, 1.0 / n)
    ky = np.fft.fftfreq(n, 1.0 / n)
    k2 = ky[:, None, None] ** 2 + ky[None, :, None] ** 2 + kx[None, None, :] ** 2
    amp = np.zeros_like(k2)
    band = (k2 >= 1.0) & (k2 <= (n / 2) ** 2)
    amp[band] = k2[band] ** (slope / 4.0)          # sqrt(P) = k^(slope/2) = (k^2)^(slope/4)
    fk *= amp
    del amp, k2, band
    f = np.fft.irfftn(fk, s=(n, n, n), axes=(0, 1, 2))
    del fk
    f -= f.mean()
    f /= f.std()
    return f


def lognormal_density(n, sigma, seed):
    """rho = exp(s), s = sigma*g - sigma^2/2 with g a k^-3 Gaussian field; discrete mean exactly 1."""
    g = gaussian_random_field(n, -3.0, seed)
    rho = np.exp(sigma * g - 0.5 * sigma * sigma)
    rho /= rho.mean()
    return rho


def velocity_field(n, mach, seed):
    """Three independent k^-4 Gaussian components, mean removed, scaled to rms |v| = mach (c0 = 1)."""
    from concurrent.futures import ThreadPoolExecutor
    with ThreadPoolExecutor(3) as ex:      # the FFTs release the GIL; same values as the serial loop
        v = list(ex.map(lambda d: gaussian_random_field(n, -4.0, seed + 101 * d), range(3)))
    rms = np.sqrt(sum((c * c).mean() for c in v))
    return [c * (mach / rms) for c in v]


def _splitmix64(x):
    x = (x + np.uint64(0x9E3779B97F4A7C15)) & np.uint64(0xFFFFFFFFFFFFFFFF)
    z = x
    z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
    z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
    return z ^ (z >> np.uint64(31))


def hash_normal(seed, level, I, J, K, d):
    """Counter-based N(0,1): a pure function of (seed, level, global cell index, component)."""
    with np.errstate(over="ignore"):
        I = np.asarray(I, dtype=np.uint64)
        J = np.asarray(J, dtype=np.uint64)
        K = np.asarray(K, dtype=np.uint64)
        ctr = (((I * np.uint64(1 << 21)) + J) * np.uint64(1 << 21) + K) * np.uint64(64) \
            + np.uint64(8 * level + d)
        a = _splitmix64(ctr ^ _splitmix64(np.uint64(seed)))
        b = _splitmix64(a)
    u1 = ((a >> np.uint64(11)).astype(np.float64) + 0.5) / 9007199254740992.0
    u2 = ((b >> np.uint64(11)).astype(np.float64) + 0.5) / 9007199254740992.0
    return np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * np.pi * u2)


def prim_to_cons(rho, vx, vy, vz, P, gamma):
    """Stack (rho, rho v, rho E) along axis 1 of [b][k][j][i] arrays; rho E per eq. (8)."""
    E = P / (gamma - 1.0) + 0.5 * rho * (vx * vx + vy * vy + vz * vz)
    return np.stack([rho, rho * vx, rho * vy, rho * vz, E], axis=1)


def trilinear_sample(base, x, y, z):
    """Periodic trilinear interpolation of a cell-centred base field [nz,ny,nx] (unit box) at points."""
    n = base.shape[0]
    out = None
    fx = x * n - 0.5
    fy = y * n - 0.5
    fz = z * n - 0.5
    ix = np.floor(fx).astype(np.int64)
    iy = np.floor(fy).astype(np.int64)
    iz = np.floor(fz).astype(np.int64)
    wx = fx - ix
    wy = fy - iy
    wz = fz - iz
    for dz in (0, 1):
        for dy in (0, 1):
            for dx in (0, 1):
                w = (wx if dx else 1.0 - wx) * (wy if dy else 1.0 - wy) * (wz if dz else 1.0 - wz)
                t = w * base[(iz + dz) % n, (iy + dy) % n, (ix + dx) % n]
                out = t if out is None else out + t
    return out
