"""Seeded synthetic inputs shared by the CUDA path's tests/bench and by the oracle's tests.

Holds NONE of the method's arithmetic: only point clouds and charges with the shapes and
distributions of the paper's workloads (uniform cube and sphere shell; the
non-uniform and thin-film shapes of BASELINE.json configs 3-4).  numpy only.  Recipe is
documented in DESIGN.md "Input recipe".  Positions/charges are generated in fp64 and, for
fp32 workloads, rounded ONCE to fp32; both the GPU library and the oracle receive the
rounded values.
"""
import numpy as np


def _round(a, dtype):
    a = np.ascontiguousarray(a, dtype=np.float64)
    if np.dtype(dtype) == np.float32:
        return a.astype(np.float32)
    return a


def uniform_cube(N, seed, dtype=np.float64):
    """r ~ U[0,1)^3, q ~ U[-1,1]  (configs 1, 2, 5)."""
    rng = np.random.default_rng(seed)
    pos = rng.random((N, 3))
    q = rng.uniform(-1.0, 1.0, N)
    return _round(pos, dtype), _round(q, dtype)


def sphere_surface(N, seed, dtype=np.float64):
    """Normalised Gaussian vectors on the unit sphere, q ~ U[-1,1]  (config 5)."""
    rng = np.random.default_rng(seed)
    v = rng.standard_normal((N, 3))
    v /= np.linalg.norm(v, axis=1, keepdims=True)
    q = rng.uniform(-1.0, 1.0, N)
    return _round(v, dtype), _round(q, dtype)


def gaussian_clusters(N, seed, dtype=np.float32, n_clusters=20, background_frac=0.1):
    """Config 3: n_clusters isotropic Gaussian clusters (sigma ~ U[0.01,0.05], centres ~ U[0,1)^3, not clipped)
    plus a uniform background of background_frac*N points; q ~ N(0,1); shuffled."""
    rng = np.random.default_rng(seed)
    n_bg = int(round(N * background_frac))
    n_cl = N - n_bg
    per = [n_cl // n_clusters + (1 if i < n_cl % n_clusters else 0) for i in range(n_clusters)]
    centres = rng.random((n_clusters, 3))
    sigmas = rng.uniform(0.01, 0.05, n_clusters)
    parts = [centres[i] + sigmas[i] * rng.standard_normal((per[i], 3)) for i in range(n_clusters)]
    parts.append(rng.random((n_bg, 3)))
    pos = np.concatenate(parts, axis=0)
    q = rng.standard_normal(N)
    sh = rng.permutation(N)
    return _round(pos[sh], dtype), _round(q[sh], dtype)


def thin_film(nx, ny, nz, seed, dtype=np.float32, n_waves=8):
    """Config 4 shape: cell centres (i+1/2, j+1/2, k+1/2) of an nx x ny x nz film; the magnetisation m(x,y) is the
    normalised sum of n_waves seeded plane waves per component (wavelengths 64-512 cells, no z dependence);
    q = central-difference divergence of m with m := 0 outside the film (film surfaces carry charge)."""
    rng = np.random.default_rng(seed)
    x = np.arange(nx)[:, None] + 0.5
    y = np.arange(ny)[None, :] + 0.5
    m = np.zeros((3, nx, ny))
    for c in range(3):
        for _ in range(n_waves):
            lam = rng.uniform(64.0, 512.0)
            ang = rng.uniform(0.0, 2.0 * np.pi)
            ph = rng.uniform(0.0, 2.0 * np.pi)
            amp = rng.uniform(0.5, 1.0)
            m[c] += amp * np.cos(2.0 * np.pi * (np.cos(ang) * x + np.sin(ang) * y) / lam + ph)
    m /= np.maximum(np.linalg.norm(m, axis=0, keepdims=True), 1e-300)
    mp = np.zeros((3, nx + 2, ny + 2))
    mp[:, 1:-1, 1:-1] = m
    div_xy = 0.5 * (mp[0, 2:, 1:-1] - mp[0, :-2, 1:-1]) + 0.5 * (mp[1, 1:-1, 2:] - mp[1, 1:-1, :-2])
    q = np.empty((nx, ny, nz))
    for k in range(nz):
        up = m[2] if k + 1 < nz else 0.0
        dn = m[2] if k - 1 >= 0 else 0.0
        q[:, :, k] = div_xy + 0.5 * (up - dn)
    ii, jj, kk = np.meshgrid(np.arange(nx), np.arange(ny), np.arange(nz), indexing="ij")
    pos = np.stack([ii + 0.5, jj + 0.5, kk + 0.5], axis=-1).reshape(-1, 3)
    return _round(pos, dtype), _round(q.reshape(-1), dtype)


# BASELINE.json configs -> (generator, kwargs, FMM parameters).  theta defaults to 0.77.
CONFIGS = {
    "cfg1_cube4096_f64": dict(gen="uniform_cube", N=4096, seed=1, dtype="f64", p=6, s=3, N_max=64, theta=0.77),
    "cfg2_cube1M_f32": dict(gen="uniform_cube", N=1_000_000, seed=2, dtype="f32", p=8, s=3, N_max=128, theta=0.77),
    "cfg3_clusters1M_f32_s3": dict(gen="gaussian_clusters", N=1_000_000, seed=3, dtype="f32", p=8, s=3, N_max=128, theta=0.77),
    "cfg3_clusters1M_f32_s1": dict(gen="gaussian_clusters", N=1_000_000, seed=3, dtype="f32", p=8, s=1, N_max=128, theta=0.77),
    "cfg4_film_f32": dict(gen="thin_film", nx=1024, ny=1024, nz=4, seed=4, dtype="f32", p=6, s=3, N_max=64, theta=0.77),
}


def config5(name):
    """BASELINE config 5 (scaling sweep): `cfg5_<cube|sphere>_<N>_<f32|f64>_p<p>_n<N_max>[_s<s>]`, e.g. cfg5_cube_1000000_f32_p8_n128.
    Seeds 50 + round(log10 N); theta = 0.77; s = 3 unless given (the paper's own sweep uses s = 2)."""
    t = name.split("_")
    if len(t) < 6 or t[0] != "cfg5" or t[1] not in ("cube", "sphere") or t[3] not in ("f32", "f64") or t[4][0] != "p" or t[5][0] != "n":
        raise KeyError(name)
    N = int(float(t[2]))
    s = int(t[6][1:]) if len(t) > 6 else 3
    return dict(gen="uniform_cube" if t[1] == "cube" else "sphere_surface", N=N, seed=50 + int(round(np.log10(N))), dtype=t[3],
                p=int(t[4][1:]), s=s, N_max=int(t[5][1:]), theta=0.77)


def make(name):
    """Return (pos, q, params) for a named BASELINE config (CONFIGS, or a config-5 sweep point, see config5)."""
    c = dict(CONFIGS[name]) if name in CONFIGS else config5(name)
    dt = np.float32 if c["dtype"] == "f32" else np.float64
    g = c["gen"]
    if g == "uniform_cube":
        pos, q = uniform_cube(c["N"], c["seed"], dt)
    elif g == "sphere_surface":
        pos, q = sphere_surface(c["N"], c["seed"], dt)
    elif g == "gaussian_clusters":
        pos, q = gaussian_clusters(c["N"], c["seed"], dt)
    elif g == "thin_film":
        pos, q = thin_film(c["nx"], c["ny"], c["nz"], c["seed"], dt)
    else:
        raise KeyError(g)
    return pos, q, c
