"""Zel'dovich-displaced Lagrangian lattices and other seeded particle sets.

Positions are returned as C-contiguous arrays indexed [i, j, k, component] with particle
(i,j,k) the one whose Lagrangian (unperturbed) position is (i,j,k) * L/N -- i.e. already
"sorted by ID" in the sense of PAPER.md:60.

Displacement field (BASELINE.json configs; reading stated in DESIGN.md "Input recipe"):
    psi(q) = s * sum_m (g_m / |k_m|^2) * k_m * sin(2 pi k_m . q / L + phi_m)
with M distinct integer wavevectors k_m drawn without replacement from the half ball
0 < |k| <= k_max (first non-zero component positive), g_m ~ N(0,1), phi_m ~ U[0, 2 pi),
and s such that the rms over all 3 N^3 displacement components is r * L / N.

RNG: SplitMix64 in counter mode (stream position i -> mix(seed + (i+1)*GOLDEN)), Box-Muller
for normals.  Everything is a pure function of (seed, parameters).
"""
from __future__ import annotations

import hashlib

import numpy as np

_GOLDEN = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)

BASE_SEED = 161209491

# (name, N, G, n_modes, k_max, rms in lattice spacings, dtype, stride)
CONFIGS = [
    dict(name="cfg0_32_64", N=32, G=64, modes=64, kmax=4, rms=0.3, dtype="float64", stride=3),
    dict(name="cfg1_128_256", N=128, G=256, modes=64, kmax=8, rms=1.5, dtype="float32", stride=4),
    dict(name="cfg2_256_512", N=256, G=512, modes=128, kmax=16, rms=4.0, dtype="float32", stride=4),
    dict(name="cfg3_256_patches", N=256, G=128, modes=128, kmax=16, rms=4.0, dtype="float32",
         stride=4, patches=dict(base_G=128, P=16, max_level=2, factor=4.0), same_particles_as=2),
    dict(name="cfg4_512_1024", N=512, G=1024, modes=256, kmax=32, rms=6.0, dtype="float32",
         stride=4),
    # not in BASELINE.json: the paper's own analytic weak-scaling workload (PAPER.md:175,
    # SURVEY.md 8(f) row 1): 512^3 particles on a lattice + independent uniform offsets of up to
    # one lattice spacing per axis, deposited on 256^3 cells (G = N/2: most tets inside one cell)
    dict(name="paper_weak_512_256", N=512, G=256, kind="jitter", amplitude=1.0, dtype="float32",
         stride=4),
]


def splitmix64(seed: int, start: int, count: int) -> np.ndarray:
    """count 64-bit outputs of SplitMix64 at stream positions start .. start+count-1."""
    with np.errstate(over="ignore"):
        idx = np.arange(start + 1, start + count + 1, dtype=np.uint64)
        z = np.uint64(seed) + idx * _GOLDEN
        z = (z ^ (z >> np.uint64(30))) * _M1
        z = (z ^ (z >> np.uint64(27))) * _M2
        z = z ^ (z >> np.uint64(31))
    return z


def _uniform(seed: int, start: int, count: int) -> np.ndarray:
    """U[0,1) doubles with 53 random bits."""
    return (splitmix64(seed, start, count) >> np.uint64(11)).astype(np.float64) * 2.0 ** -53


def _half_ball(kmax: int) -> np.ndarray:
    r = np.arange(-kmax, kmax + 1)
    kx, ky, kz = np.meshgrid(r, r, r, indexing="ij")
    k = np.stack([kx.ravel(), ky.ravel(), kz.ravel()], axis=1)
    n2 = (k * k).sum(axis=1)
    keep = (n2 > 0) & (n2 <= kmax * kmax)
    k = k[keep]
    # first non-zero component positive
    first = np.where(k[:, 0] != 0, k[:, 0], np.where(k[:, 1] != 0, k[:, 1], k[:, 2]))
    return k[first > 0]


def _draw_modes(seed: int, n_modes: int, kmax: int):
    cand = _half_ball(kmax)
    if n_modes > cand.shape[0]:
        raise ValueError("more modes requested than the half ball holds")
    # Fisher-Yates with the counter RNG (stream positions 0 .. len-2)
    u = _uniform(seed, 0, cand.shape[0])
    perm = np.arange(cand.shape[0])
    for i in range(cand.shape[0] - 1, 0, -1):
        j = int(u[i] * (i + 1))
        perm[i], perm[j] = perm[j], perm[i]
    k = cand[perm[:n_modes]]
    base = 1 << 20
    u1 = _uniform(seed, base, n_modes)
    u2 = _uniform(seed, base + n_modes, n_modes)
    g = np.sqrt(-2.0 * np.log(1.0 - u1)) * np.cos(2.0 * np.pi * u2)  # Box-Muller
    phi = 2.0 * np.pi * _uniform(seed, base + 2 * n_modes, n_modes)
    return k.astype(np.int64), g, phi


def displacement_direct(N: int, k, g, phi) -> np.ndarray:
    """Unscaled psi on the lattice, by the defining sum (small N only). Shape (N,N,N,3)."""
    n = np.arange(N, dtype=np.float64)
    psi = np.zeros((N, N, N, 3))
    for km, gm, pm in zip(k, g, phi):
        th = (2.0 * np.pi / N) * (km[0] * n[:, None, None] + km[1] * n[None, :, None]
                                  + km[2] * n[None, None, :]) + pm
        a = gm / float(km @ km)
        s = np.sin(th)
        for c in range(3):
            if km[c]:
                psi[..., c] += (a * km[c]) * s
    return psi


def displacement_fft(N: int, k, g, phi) -> np.ndarray:
    """Same field through one inverse FFT per component (any N >= 2*k_max+1)."""
    from scipy import fft as sfft
    psi = np.empty((N, N, N, 3))
    amp = g / (k * k).sum(axis=1)
    ph = np.exp(1j * phi)
    for c in range(3):
        spec = np.zeros((N, N, N), dtype=np.complex128)
        np.add.at(spec, (k[:, 0] % N, k[:, 1] % N, k[:, 2] % N), amp * k[:, c] * ph)
        f = sfft.ifftn(spec, workers=-1, overwrite_x=True)
        psi[..., c] = f.imag * float(N) ** 3
        del spec, f
    return psi


def zeldovich_positions(N: int, n_modes: int, kmax: int, rms_cells: float, seed: int,
                        L: float = 1.0, dtype="float32", stride: int = 4, method: str = "auto",
                        return_info: bool = False):
    k, g, phi = _draw_modes(seed, n_modes, kmax)
    if method == "auto":
        method = "direct" if N <= 32 else "fft"
    psi = displacement_direct(N, k, g, phi) if method == "direct" else displacement_fft(N, k, g, phi)
    rms = np.sqrt(np.mean(psi * psi))
    psi *= (rms_cells * L / N) / rms
    q = np.arange(N, dtype=np.float64) * (L / N)
    psi[..., 0] += q[:, None, None]
    psi[..., 1] += q[None, :, None]
    psi[..., 2] += q[None, None, :]
    np.mod(psi, L, out=psi)
    out = np.zeros((N, N, N, stride), dtype=dtype)
    out[..., :3] = psi
    if return_info:
        return out, dict(k=k, g=g, phi=phi, scale=(rms_cells * L / N) / rms)
    return out


def config_positions(index: int, N_override: int | None = None):
    """Positions of BASELINE.json configs[index] (cfg3 uses cfg2's particles)."""
    cfg = CONFIGS[index]
    if cfg.get("kind") == "jitter":
        return jittered_lattice(N_override or cfg["N"], BASE_SEED + index, cfg["amplitude"],
                                dtype=cfg["dtype"], stride=cfg["stride"])
    src = cfg.get("same_particles_as", index)
    c = CONFIGS[src]
    N = N_override or c["N"]
    return zeldovich_positions(N, c["modes"], c["kmax"], c["rms"], BASE_SEED + src,
                               dtype=c["dtype"], stride=c["stride"])


def lattice(N: int, L: float = 1.0, shift=(0.0, 0.0, 0.0), dtype="float64", stride: int = 3,
            shear_xy: int = 0) -> np.ndarray:
    """Unperturbed lattice q = (i,j,k) L/N, rigidly shifted (and wrapped); optional integer
    torus shear x -> x + shear_xy * y (mod L)."""
    q = np.arange(N, dtype=np.float64) * (L / N)
    out = np.zeros((N, N, N, stride), dtype=np.float64)
    out[..., 0] = q[:, None, None] + shear_xy * q[None, :, None]
    out[..., 1] = q[None, :, None]
    out[..., 2] = q[None, None, :]
    out[..., :3] += np.asarray(shift, dtype=np.float64)
    out[..., :3] = np.mod(out[..., :3], L)
    return out.astype(dtype)


def jittered_lattice(N: int, seed: int, amplitude_cells: float = 1.0, L: float = 1.0,
                     dtype="float32", stride: int = 4) -> np.ndarray:
    """lattice plus independent uniform offsets in [-a, a] cell widths per axis."""
    u = _uniform(seed, 0, 3 * N ** 3).reshape(N, N, N, 3)
    out = np.zeros((N, N, N, stride), dtype=np.float64)
    q = np.arange(N, dtype=np.float64) * (L / N)
    out[..., 0] = q[:, None, None]
    out[..., 1] = q[None, :, None]
    out[..., 2] = q[None, None, :]
    out[..., :3] += (2.0 * u - 1.0) * (amplitude_cells * L / N)
    out[..., :3] = np.mod(out[..., :3], L)
    return out.astype(dtype)


def sha256_of(a: np.ndarray) -> str:
    return hashlib.sha256(np.ascontiguousarray(a).tobytes()).hexdigest()
