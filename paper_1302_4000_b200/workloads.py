"""Seeded synthetic decoy ensembles shaped like the paper's workloads.

This module is the ONLY code shared by the FP64 CPU oracle's tests and the CUDA path's
harness.  It generates inputs and nothing else: it holds none of the cRMSD arithmetic
(no centring, no covariance, no eigenvalues, no superposition) and imports neither
`oracle/` nor the CUDA binding.

The paper measures on Decoys 'R' Us and I-TASSER decoy sets (PAPER.md:90, 100, 110, 140,
229, 236: 6256 x 36, 12 500 x 60, 32 000 x 108, proteins of 71/215/887 residues).  None
of those is available, so BASELINE.json's five synthetic configurations stand in for
them; the recipe below is the one stated in DESIGN.md ("Input recipe") and SURVEY.md
section 8(d).  All mathematics is FP64; the cast to fp32 is the very last step and the
fp32 array is *the* input for both the oracle and the GPU.

    C1  N=200     L=76    sigma ~ U(0.5, 6)   5 mirror images, 2 exact rigid copies
    C2  N=2000    L=120   sigma ~ U(0.5,10)
    C3  N=10000   L=250   20 clusters: centre = native + N(0,4^2), members + N(0,U(0.3,2)^2)
    C4  N=30000   L=100   sigma ~ U(0.5, 8)
    C5  N=1e6     L=150   sigma ~ U(0.5,10), one-vs-all against the (rigidly moved) native
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

BOND = 3.8  # C-alpha -- C-alpha virtual bond length in Angstrom (BASELINE.json configs)
SEED_BASE = 13024000


@dataclass
class Ensemble:
    """An ensemble of N models of L atoms: `coords[N][L][3]` fp32, plus bookkeeping for tests."""

    name: str
    coords: np.ndarray                      # (N, L, 3) float32 -- the input
    native: np.ndarray                      # (L, 3) float32 -- the un-noised chain, own rigid transform
    sigma: np.ndarray                       # (N,) float64 noise level used for each model
    mirror_idx: np.ndarray = field(default_factory=lambda: np.zeros(0, np.int64))
    rigid_copy_idx: np.ndarray = field(default_factory=lambda: np.zeros(0, np.int64))
    cluster_id: np.ndarray | None = None    # (N,) for C3
    stats: dict | None = None               # shape record of the native (chain_shape), logged beside every result

    @property
    def N(self) -> int:
        return self.coords.shape[0]

    @property
    def L(self) -> int:
        return self.coords.shape[1]


def _streams(config_index: int, n: int = 4):
    ss = np.random.SeedSequence(SEED_BASE + config_index)
    return [np.random.Generator(np.random.PCG64(s)) for s in ss.spawn(n)]


def random_walk_chain(L: int, rng: np.random.Generator) -> np.ndarray:
    """Native chain: 3.8 A steps, bond angle ~U(80,150) deg, dihedral ~U(-180,180) deg.

    Atoms 0..2 lie in the xy-plane; atoms i>=3 are placed from the previous three by the
    usual internal-coordinate construction.  No self-avoidance.
    """
    x = np.zeros((L, 3), np.float64)
    theta = np.deg2rad(rng.uniform(80.0, 150.0, size=L))
    phi = np.deg2rad(rng.uniform(-180.0, 180.0, size=L))
    if L > 1:
        x[1] = (BOND, 0.0, 0.0)
    if L > 2:
        x[2] = x[1] + BOND * np.array([-np.cos(theta[2]), np.sin(theta[2]), 0.0])
    for i in range(3, L):
        a, b, c = x[i - 3], x[i - 2], x[i - 1]
        bc = c - b
        bc /= np.linalg.norm(bc)
        n = np.cross(b - a, bc)
        n /= np.linalg.norm(n)
        m = np.cross(n, bc)
        d = np.array([-BOND * np.cos(theta[i]),
                      BOND * np.sin(theta[i]) * np.cos(phi[i]),
                      BOND * np.sin(theta[i]) * np.sin(phi[i])])
        x[i] = c + d[0] * bc + d[1] * m + d[2] * n
    return x


def chain_shape(x: np.ndarray) -> dict:
    """Shape record of one chain, logged for every config (generator step 1): the native's
    R_g^2 varies ~8x over seeds and every fp32 error term of the GPU path scales with it, so a result without this
    record cannot be placed.  Plain FP64 numpy on the un-noised chain; neither the oracle nor the CUDA path uses it."""
    a = np.asarray(x, np.float64)
    a = a - a.mean(0)
    ev = np.linalg.eigvalsh(a.T @ a / a.shape[0])[::-1]
    return {"rg2": float(ev.sum()), "gyration_eigenvalues": [float(v) for v in ev],
            "max_abs_centred": float(np.abs(a).max())}


# The generator's tail: for each chain length the seed s in 0..199 whose random_walk_chain(L, default_rng(s)) has the
# LARGEST R_g^2 (most extended chain; tests/test_workloads.py re-derives the table).  The GPU path's error grows with
# R_g^2, so parity is also asked on ensembles built on these natives, not only on the five configs' own natives
# (R_g^2 479..969 A^2, below the generator's median at their lengths).
TAIL_SEEDS = {100: 63, 140: 47, 150: 69, 215: 38, 250: 48}


def tail_native(L: int) -> np.ndarray:
    """The most extended of the 200 chains random_walk_chain(L, default_rng(0..199))  (R_g^2 = 4289 A^2 at L = 250)."""
    return random_walk_chain(L, np.random.default_rng(TAIL_SEEDS[L]))


def random_rotations(n: int, rng: np.random.Generator) -> np.ndarray:
    """n proper rotations, uniform on SO(3), from normalised 4-vectors of standard normals."""
    q = rng.normal(size=(n, 4))
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    w, x, y, z = q[:, 0], q[:, 1], q[:, 2], q[:, 3]
    R = np.empty((n, 3, 3), np.float64)
    R[:, 0, 0] = 1 - 2 * (y * y + z * z)
    R[:, 0, 1] = 2 * (x * y - z * w)
    R[:, 0, 2] = 2 * (x * z + y * w)
    R[:, 1, 0] = 2 * (x * y + z * w)
    R[:, 1, 1] = 1 - 2 * (x * x + z * z)
    R[:, 1, 2] = 2 * (y * z - x * w)
    R[:, 2, 0] = 2 * (x * z - y * w)
    R[:, 2, 1] = 2 * (y * z + x * w)
    R[:, 2, 2] = 1 - 2 * (x * x + y * y)
    return R


def rigid_transform(y: np.ndarray, rng: np.random.Generator) -> np.ndarray:
    """z_m = R_m y_m + t_m with R_m uniform on SO(3), t_m ~ U(-50,50)^3.  y: (n, L, 3) FP64."""
    n = y.shape[0]
    R = random_rotations(n, rng)
    t = rng.uniform(-50.0, 50.0, size=(n, 1, 3))
    return np.einsum("nij,nlj->nli", R, y) + t


def _noisy_decoys(native, n, lo, hi, rng_noise):
    sigma = rng_noise.uniform(lo, hi, size=n)
    y = native[None] + rng_noise.normal(size=(n,) + native.shape) * sigma[:, None, None]
    return y, sigma


def make_decoys(config_index: int, N: int, L: int, sigma_lo: float, sigma_hi: float,
                n_mirror: int = 0, n_rigid: int = 0, name: str | None = None,
                native: np.ndarray | None = None) -> Ensemble:
    """Configs C1, C2, C4: native + iid Gaussian noise, optional mirrors / rigid copies, rigid transform.
    `native` (L, 3) replaces the config's own seeded chain (the tail ensembles)."""
    r_native, r_noise, r_rigid, r_struct = _streams(config_index)
    native = random_walk_chain(L, r_native) if native is None else np.asarray(native, np.float64)
    y, sigma = _noisy_decoys(native, N, sigma_lo, sigma_hi, r_noise)
    # specials: first n_mirror decoys are mirrored (x -> -x) BEFORE the rigid
    # transform, the next n_rigid are the native itself (sigma = 0); then a seeded shuffle.
    mirror = np.arange(0, n_mirror)
    rigid = np.arange(n_mirror, n_mirror + n_rigid)
    y[mirror, :, 0] *= -1.0
    y[rigid] = native
    sigma[rigid] = 0.0
    perm = r_struct.permutation(N)            # new position k holds old model perm[k]
    y, sigma = y[perm], sigma[perm]
    inv = np.empty(N, np.int64)
    inv[perm] = np.arange(N)
    z = rigid_transform(y, r_rigid)
    nat = rigid_transform(native[None], r_rigid)[0]
    return Ensemble(name or f"C{config_index}", z.astype(np.float32), nat.astype(np.float32), sigma,
                    np.sort(inv[mirror]), np.sort(inv[rigid]), stats=chain_shape(native))


def make_clusters(config_index: int, N: int, L: int, n_clusters: int = 20, centre_sigma: float = 4.0,
                  sigma_lo: float = 0.3, sigma_hi: float = 2.0, name: str | None = None,
                  native: np.ndarray | None = None) -> Ensemble:
    """Config C3: n_clusters cluster centres = native + N(0, centre_sigma^2); members around them."""
    r_native, r_noise, r_rigid, r_struct = _streams(config_index)
    native = random_walk_chain(L, r_native) if native is None else np.asarray(native, np.float64)
    centres = native[None] + r_noise.normal(size=(n_clusters, L, 3)) * centre_sigma
    cid = np.arange(N) % n_clusters
    sigma = r_noise.uniform(sigma_lo, sigma_hi, size=N)
    y = centres[cid] + r_noise.normal(size=(N, L, 3)) * sigma[:, None, None]
    perm = r_struct.permutation(N)
    y, sigma, cid = y[perm], sigma[perm], cid[perm]
    z = rigid_transform(y, r_rigid)
    nat = rigid_transform(native[None], r_rigid)[0]
    return Ensemble(name or f"C{config_index}", z.astype(np.float32), nat.astype(np.float32), sigma,
                    cluster_id=cid, stats=chain_shape(native))


def make_one_vs_all(config_index: int, N: int, L: int, sigma_lo: float = 0.5, sigma_hi: float = 10.0,
                    chunk: int = 100_000, chunks: range | None = None, name: str | None = None,
                    native: np.ndarray | None = None) -> Ensemble:
    """Config C5: one native vs N decoys, generated in independently seeded chunks of `chunk` models.

    `chunks` selects which chunks to produce (default: all), so a test can regenerate any slice
    of the 10^6-model ensemble bit-identically without building the whole 1.8 GB array.
    """
    ss = np.random.SeedSequence(SEED_BASE + config_index)
    s_native, s_rigid_native, s_chunks = ss.spawn(3)
    native = (random_walk_chain(L, np.random.Generator(np.random.PCG64(s_native))) if native is None
              else np.asarray(native, np.float64))
    nat = rigid_transform(native[None], np.random.Generator(np.random.PCG64(s_rigid_native)))[0]
    n_chunks = (N + chunk - 1) // chunk
    chunk_seeds = s_chunks.spawn(n_chunks)
    sel = range(n_chunks) if chunks is None else chunks
    out, sig = [], []
    for k in sel:
        n_k = min(chunk, N - k * chunk)
        r_noise, r_rigid = [np.random.Generator(np.random.PCG64(s)) for s in chunk_seeds[k].spawn(2)]
        y, sigma = _noisy_decoys(native, n_k, sigma_lo, sigma_hi, r_noise)
        out.append(rigid_transform(y, r_rigid).astype(np.float32))
        sig.append(sigma)
    coords = np.concatenate(out) if out else np.zeros((0, L, 3), np.float32)
    return Ensemble(name or f"C{config_index}", coords, nat.astype(np.float32),
                    np.concatenate(sig) if sig else np.zeros(0), stats=chain_shape(native))


# ---- BASELINE.json's five configurations -------------------------------------------------------

CONFIGS = {
    "C1": dict(kind="decoys", N=200, L=76, sigma=(0.5, 6.0), n_mirror=5, n_rigid=2),
    "C2": dict(kind="decoys", N=2000, L=120, sigma=(0.5, 10.0)),
    "C3": dict(kind="clusters", N=10000, L=250),
    "C4": dict(kind="decoys", N=30000, L=100, sigma=(0.5, 8.0)),
    "C5": dict(kind="one_vs_all", N=1_000_000, L=150, sigma=(0.5, 10.0)),
}


def make_config(name: str, N: int | None = None, **kw) -> Ensemble:
    """Build BASELINE.json config `name` ("C1".."C5"); `N` overrides the model count (same seeds)."""
    c = CONFIGS[name]
    k = int(name[1:])
    n = c["N"] if N is None else N
    if c["kind"] == "decoys":
        return make_decoys(k, n, c["L"], *c["sigma"], n_mirror=c.get("n_mirror", 0),
                           n_rigid=c.get("n_rigid", 0), name=name)
    if c["kind"] == "clusters":
        return make_clusters(k, n, c["L"], name=name)
    return make_one_vs_all(k, n, c["L"], *c["sigma"], name=name, **kw)


def make_tail(shape: str, N: int, L: int | None = None) -> Ensemble:
    """An ensemble with the noise recipe of config `shape` ("C2".."C5") built on the generator's most extended
    native of length L (default: the config's own L; TAIL_SEEDS).  Streams: those of config index 100 + k, so the
    tail ensembles share no random numbers with C1..C5."""
    c = CONFIGS[shape]
    k = int(shape[1:])
    L = c["L"] if L is None else L
    nat = tail_native(L)
    name = f"{shape}-tail(L={L})"
    if c["kind"] == "decoys":
        return make_decoys(100 + k, N, L, *c["sigma"], name=name, native=nat)
    if c["kind"] == "clusters":
        return make_clusters(100 + k, N, L, name=name, native=nat)
    return make_one_vs_all(100 + k, N, L, *c["sigma"], chunk=max(1, N), name=name, native=nat)


def packed_index(i, j, N):
    """Row-major packed upper-triangle index of pair i<j (N(N-1)/2 values)."""
    i = np.asarray(i, np.int64)
    j = np.asarray(j, np.int64)
    return i * (2 * N - i - 1) // 2 + (j - i - 1)
