"""Seeded synthetic inputs shared by the CUDA path, the oracle tests and bench.py.

This module holds NONE of the method's arithmetic (no CIC, no force, no growth, no time
stepping): it only draws random numbers and shapes them into inputs.  numpy/scipy only,
no torch, no CUDA, and it imports neither the product binding nor the oracle.

The inputs stand in for the paper's LambdaCDM workloads (Fig. 2,
L428-432 Table 1, L478 Fig. 3), whose Eisenstein-Hu power spectrum is not in the
container: a power-law spectrum with a Gaussian cut-off replaces it (BASELINE.json
configs; recipe in DESIGN.md "Input recipe").
"""
import numpy as np
import scipy.fft as sfft

# BASELINE.json configs[0..3]; a-schedules per DESIGN.md "Input recipe".
CONFIGS = {
    0: dict(name="cfg0_32p_64m_eds_16steps", lattice=(32, 32, 32), mesh=(64, 64, 64), omega_m=1.0,
            n_steps=16, a0=1.0 / 16),
    1: dict(name="cfg1_128p_256m_lcdm_63steps", lattice=(128,) * 3, mesh=(256,) * 3, omega_m=0.3,
            n_steps=63, a0=1.0 / 64),
    2: dict(name="cfg2_256p_512m_lcdm_63steps", lattice=(256,) * 3, mesh=(512,) * 3, omega_m=0.3,
            n_steps=63, a0=1.0 / 64),
    3: dict(name="cfg3_512p_1024m_lcdm_100steps", lattice=(512,) * 3, mesh=(1024,) * 3, omega_m=0.3,
            n_steps=100, a0=1.0 / 64),
}


def a_schedule(a0, n_steps, a1=1.0):
    """n_steps+1 scale factors linearly spaced in a, a0 .. a1 inclusive."""
    return a0 + (a1 - a0) * np.arange(n_steps + 1, dtype=np.float64) / float(n_steps)


def config(idx):
    c = dict(CONFIGS[idx])
    c["a"] = a_schedule(c["a0"], c["n_steps"])
    return c


def _signed_modes(n):
    m = np.arange(n)
    return np.where(m < (n + 1) // 2, m, m - n)


def _colored_field(shape, cell_per_site, seed, rms):
    """Gaussian random field on a grid of `shape` sites, spacing `cell_per_site` cells.

    white noise omega(q) ~ N(0,1), default_rng(seed) -> FFT -> times sqrt(P(k)),
    P(k) = k^-1.5 exp(-(2k)^2), k in rad/cell; delta(k=0) = 0 (eq. 6).
    Returns (delta_k, kvec list, k2) for further shaping; rms is applied by callers.
    """
    rng = np.random.default_rng(seed)
    w = rng.standard_normal(shape)
    wk = sfft.rfftn(w, workers=-1)
    del w
    ks = []
    for d in range(3):
        m = _signed_modes(shape[d]).astype(np.float64)
        if d == 2:
            m = np.arange(shape[2] // 2 + 1, dtype=np.float64)
        ks.append(2.0 * np.pi * m / (shape[d] * cell_per_site[d]))
    kx, ky, kz = np.meshgrid(*ks, indexing="ij", sparse=True)
    k2 = kx * kx + ky * ky + kz * kz
    k2[0, 0, 0] = 1.0
    k = np.sqrt(k2)
    amp = np.sqrt(k ** -1.5 * np.exp(-(2.0 * k) ** 2))
    amp[0, 0, 0] = 0.0
    wk *= amp
    return wk, ks, k2


def zeldovich_displacement(lattice, mesh, seed, rms=0.3):
    """s0[N_p, 3] float32: Zel'dovich (first-order, eq. 3-4) displacement on the
    particle lattice, in cells, scaled so sqrt(mean_j |s_j|^2) = rms (3-D norm).

    s(k) = i k~ delta1(k) / k^2 with k~ = 0 on the lattice Nyquist planes, so that the field is real.
    Particle j = (jx*Ly + jy)*Lz + jz.
    """
    lattice = tuple(int(v) for v in lattice)
    cps = [mesh[d] / lattice[d] for d in range(3)]
    dk, ks, k2 = _colored_field(lattice, cps, seed, rms)
    out = np.empty((lattice[0] * lattice[1] * lattice[2], 3), dtype=np.float64)
    for d in range(3):
        kd = ks[d].copy()
        if lattice[d] % 2 == 0:
            kd[lattice[d] // 2] = 0.0
        shp = [1, 1, 1]
        shp[d] = -1
        sk = 1j * kd.reshape(shp) * dk / k2
        out[:, d] = sfft.irfftn(sk, s=lattice, workers=-1).reshape(-1)
        del sk
    out *= rms / np.sqrt(np.mean(np.sum(out * out, axis=1)))
    return out.astype(np.float32)


def lognormal_target(mesh, seed, sigma=1.0):
    """delta_target[Nx, Ny, Nz] float32 for the larger configs: exp(G - var/2) - 1 with G a Gaussian
    field of the same power-law spectrum on the mesh (std = sigma).  A positive-density,
    non-Gaussian field "from a second seed" (BASELINE.json configs) that needs neither the oracle
    nor the CUDA path to make.  Mean is removed exactly so that sum(delta) = 0."""
    mesh = tuple(int(v) for v in mesh)
    dk, _, _ = _colored_field(mesh, (1.0, 1.0, 1.0), seed, 1.0)
    g = sfft.irfftn(dk, s=mesh, workers=-1)
    del dk
    g *= sigma / g.std()
    rho = np.exp(g)
    rho /= rho.mean()
    return (rho - 1.0).astype(np.float32)


def blob_positions(n_particles, mesh, seed=3, n_blobs=20000, frac_blobs=0.7, mass_max=512.0,
                   order="generation"):
    """configs[4] kernel-sweep positions x[N_p, 3] float32 in [0, mesh): 70 % of the particles in
    n_blobs Gaussian blobs (masses ~ M^-2 on [1, mass_max], radius 0.5 M^(1/3) cell in [0.5, 4]),
    30 % uniform.  order = "generation" (blob after blob, then the uniform ones) or "random".
    """
    rng = np.random.default_rng(seed)
    mesh = np.asarray(mesh, dtype=np.float64)
    u = rng.random(n_blobs)
    M = 1.0 / (1.0 - u * (1.0 - 1.0 / mass_max))
    sig = 0.5 * M ** (1.0 / 3.0)
    centres = rng.random((n_blobs, 3)) * mesh
    n_in = int(np.floor(frac_blobs * n_particles))
    share = M / M.sum() * n_in
    cnt = np.floor(share).astype(np.int64)
    rem = n_in - int(cnt.sum())
    if rem > 0:  # largest remainder
        idx = np.argsort(-(share - cnt), kind="stable")[:rem]
        cnt[idx] += 1
    x = np.empty((n_particles, 3), dtype=np.float32)
    which = np.repeat(np.arange(n_blobs), cnt)
    chunk = 1 << 24
    for lo in range(0, n_in, chunk):
        hi = min(n_in, lo + chunk)
        w = which[lo:hi]
        pos = centres[w] + sig[w, None] * rng.standard_normal((hi - lo, 3))
        x[lo:hi] = np.mod(pos, mesh).astype(np.float32)
    for lo in range(n_in, n_particles, chunk):
        hi = min(n_particles, lo + chunk)
        x[lo:hi] = (rng.random((hi - lo, 3)) * mesh).astype(np.float32)
    # float32 rounding can land exactly on mesh (== N); fold back
    for d in range(3):
        col = x[:, d]
        col[col >= np.float32(mesh[d])] = 0.0
    if order == "random":
        x = x[rng.permutation(n_particles)]
    elif order != "generation":
        raise ValueError(order)
    return x


def uniform_positions(n_particles, mesh, seed=3):
    rng = np.random.default_rng(seed + 1000)
    mesh = np.asarray(mesh, dtype=np.float64)
    x = np.empty((n_particles, 3), dtype=np.float32)
    chunk = 1 << 24
    for lo in range(0, n_particles, chunk):
        hi = min(n_particles, lo + chunk)
        x[lo:hi] = (rng.random((hi - lo, 3)) * mesh).astype(np.float32)
    for d in range(3):
        col = x[:, d]
        col[col >= np.float32(mesh[d])] = 0.0
    return x
