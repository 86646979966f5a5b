"""Seeded synthetic inputs shaped like the paper's workloads (BASELINE.json configs).

The paper's particle data (cosmological boxes: near-uniform early, strongly clustered late,
PAPER.md:172) are not available; these generators are the stand-ins BASELINE.json names.  They hold
NONE of the method's arithmetic — only random draws — and serve the CUDA path and the oracle alike.
All draws are fp64 from numpy.random.Generator(PCG64(seed)), cast once to fp32.

Seeds: SEED0 + config number; subsample seeds: +100.
"""
import numpy as np

SEED0 = 14072600


def _rng(cfg, extra=0):
    return np.random.Generator(np.random.PCG64(SEED0 + cfg + extra))


def subsample(cfg, n, k):
    """fixed sink subsample: k distinct particle indices (sorted)"""
    k = min(k, n)
    return np.sort(_rng(cfg, 100).choice(n, size=k, replace=False)).astype(np.int64)


def uniform_box(n=32768, cfg=1):
    """C1: isolated uniform random box, equal masses 1/n."""
    rng = _rng(cfg)
    pos = rng.random((n, 3), dtype=np.float32)
    mass = np.full(n, 1.0 / n, dtype=np.float32)
    return pos, mass


def _plummer_radii(rng, n, a, cut):
    r = np.empty(n)
    todo = np.arange(n)
    while todo.size:
        u = rng.random(todo.size)
        u = np.clip(u, 1e-300, 1.0)
        rr = a / np.sqrt(np.maximum(u ** (-2.0 / 3.0) - 1.0, 1e-300))
        ok = rr <= cut * a
        r[todo[ok]] = rr[ok]
        todo = todo[~ok]
    return r


def _isotropic(rng, n):
    ct = rng.uniform(-1.0, 1.0, n)
    ph = rng.uniform(0.0, 2.0 * np.pi, n)
    st = np.sqrt(1.0 - ct * ct)
    return np.stack([st * np.cos(ph), st * np.sin(ph), ct], axis=1)


def plummer_sphere(n=1 << 20, a=0.01, cut=20.0, cfg=2):
    """C2: isolated Plummer sphere, M = 1, scale radius a, cut at cut*a, centred in the unit box."""
    rng = _rng(cfg)
    r = _plummer_radii(rng, n, a, cut)
    pos = 0.5 + r[:, None] * _isotropic(rng, n)
    pos = pos.astype(np.float32)
    mass = np.full(n, 1.0 / n, dtype=np.float32)
    return pos, mass


def perturbed_lattice(ng=128, rms=0.2, cfg=3):
    """C3: periodic ng^3 lattice displaced by a Gaussian random field with P(k) ~ k^-2, rms
    3-D displacement `rms` grid spacings.  Unit box."""
    rng = _rng(cfg)
    n = ng ** 3
    kx = np.fft.fftfreq(ng, d=1.0 / ng)
    kz = np.fft.rfftfreq(ng, d=1.0 / ng)
    KX, KY, KZ = np.meshgrid(kx, kx, kz, indexing="ij")
    k2 = KX ** 2 + KY ** 2 + KZ ** 2
    kk = np.sqrt(k2)
    amp = np.zeros_like(kk)
    m = (kk >= 1.0) & (kk <= ng / 2)
    amp[m] = kk[m] ** -1.0                       # sqrt(P), P ~ k^-2
    shape = kk.shape
    dk = (rng.standard_normal(shape) + 1j * rng.standard_normal(shape)) * amp
    k2s = np.where(k2 > 0, k2, 1.0)
    psi = []
    for K in (KX, KY, KZ):
        psi.append(np.fft.irfftn(1j * K * dk / k2s, s=(ng, ng, ng), axes=(0, 1, 2)))
    psi = np.stack(psi, axis=-1).reshape(n, 3)
    psi *= (rms / ng) / np.sqrt(np.mean(np.sum(psi ** 2, axis=1)))
    q = (np.arange(ng) + 0.5) / ng
    Q = np.stack(np.meshgrid(q, q, q, indexing="ij"), axis=-1).reshape(n, 3)
    pos = np.mod(Q + psi, 1.0).astype(np.float32)
    pos[pos >= 1.0] = 0.0
    mass = np.full(n, 1.0 / n, dtype=np.float32)
    return pos, mass


def clustered_box(ng=256, nhalo=2000, cfg=4):
    """C4/C5: periodic unit box, half the particles in `nhalo` Plummer halos (dN/dM ~ M^-1.9 over
    a factor 1000 in mass, r200 from overdensity 200, a = r200/5, cut at 10a, centres uniform), half
    a uniform background."""
    rng = _rng(cfg)
    n = ng ** 3
    nh_tot = n // 2
    # inverse CDF of dN/dM ~ M^-1.9 on [1, 1000]
    u = rng.random(nhalo)
    g = -0.9
    M = (1.0 + u * (1000.0 ** g - 1.0)) ** (1.0 / g)
    cnt = np.rint(nh_tot * M / M.sum()).astype(np.int64)
    cnt[np.argmax(cnt)] += nh_tot - cnt.sum()
    centres = rng.random((nhalo, 3))
    parts = []
    for k in range(nhalo):
        nk = int(cnt[k])
        if nk <= 0:
            continue
        r200 = (3.0 * (nk / n) / (4.0 * np.pi * 200.0)) ** (1.0 / 3.0)
        a = r200 / 5.0
        r = _plummer_radii(rng, nk, a, 10.0)
        parts.append(centres[k] + r[:, None] * _isotropic(rng, nk))
    parts.append(rng.random((n - nh_tot, 3)))
    pos = np.mod(np.concatenate(parts, axis=0), 1.0).astype(np.float32)
    pos[pos >= 1.0] = 0.0
    pos = pos[rng.permutation(n)]
    mass = np.full(n, 1.0 / n, dtype=np.float32)
    return pos, mass


def perfect_lattice(k=8):
    """k^3 perfect cubic lattice in the unit box (zero net periodic force by symmetry)."""
    q = (np.arange(k) + 0.5) / k
    pos = np.stack(np.meshgrid(q, q, q, indexing="ij"), axis=-1).reshape(-1, 3).astype(np.float32)
    mass = np.full(k ** 3, 1.0 / k ** 3, dtype=np.float32)
    return pos, mass


# The five BASELINE.json configs: (generator kwargs, solver parameters)
CONFIGS = {
    1: dict(name="C1 isolated uniform box", N=32768, box=1.0, periodic=False, eps=1e-3, theta=0.5, p=4),
    2: dict(name="C2 isolated Plummer sphere", N=1 << 20, box=1.0, periodic=False, eps=1e-4, theta=0.5, p=4),
    3: dict(name="C3 periodic perturbed lattice", N=128 ** 3, box=1.0, periodic=True, eps=1.0 / (40 * 128), theta=0.5, p=4),
    4: dict(name="C4 periodic clustered box", N=256 ** 3, box=1.0, periodic=True, eps=1.0 / (40 * 256), theta=0.5, p=6),
    5: dict(name="C5 periodic clustered run", N=512 ** 3, box=1.0, periodic=True, eps=1.0 / (40 * 512), theta=0.6, p=4),
}


def make(cfg, scale=1.0):
    """positions, masses of config `cfg`; `scale` < 1 shrinks N (same recipe) for parity tests."""
    if cfg == 1:
        return uniform_box(max(1, int(round(32768 * scale))), 1)
    if cfg == 2:
        return plummer_sphere(max(1, int(round((1 << 20) * scale))), cfg=2)
    if cfg == 3:
        return perturbed_lattice(max(2, int(round(128 * scale ** (1 / 3)))), cfg=3)
    if cfg == 4:
        ng = max(4, int(round(256 * scale ** (1 / 3))))
        return clustered_box(ng, max(1, int(round(2000 * min(1.0, scale * 4)))), cfg=4)
    if cfg == 5:
        ng = max(4, int(round(512 * scale ** (1 / 3))))
        return clustered_box(ng, max(1, int(round(2000 * min(1.0, scale * 32)))), cfg=5)
    raise ValueError(cfg)
