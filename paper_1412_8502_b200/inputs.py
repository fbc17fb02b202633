"""Seeded synthetic inputs shared by the oracle tests, the GPU parity tests and bench.py.

Holds none of the method's arithmetic (no potential, no integrator, no cell or cluster logic):
only the workload table of BASELINE.json and random-state recipes.
numpy only; importing it never loads the CUDA library.
"""
import numpy as np

MASS = 939.0  # MeV

# The five BASELINE.json configs.  scale_per_step = 4**(1/20000).
CONFIGS = {
    1: dict(N=2048, Y_P=0.30, density=0.05, T=1.0, r_c=17.0, thermostat_interval=0, scale_per_step=1.0,
            steps=20, dt=2.0),
    2: dict(N=51200, Y_P=0.40, density=0.08, T=1.0, r_c=20.0, thermostat_interval=10, scale_per_step=1.0,
            steps=1000, dt=2.0),
    3: dict(N=51200, Y_P=0.20, density=0.08, T=0.75, r_c=20.0, thermostat_interval=10,
            scale_per_step=4.0 ** (1.0 / 20000.0), steps=20000, dt=2.0, r_cl=3.0),
    4: dict(N=409600, Y_P=0.30, density=0.08, T=0.5, r_c=20.0, thermostat_interval=10, scale_per_step=1.0,
            steps=500, dt=2.0),
    5: dict(N=409600, Y_P=0.05, density=0.08, T=0.5, r_c=20.0, thermostat_interval=10,
            scale_per_step=4.0 ** (1.0 / 20000.0), steps=20000, dt=2.0, r_cl=3.0),
}


def n_protons(N, Y_P):
    """N_p = floor(Y_P N + 1/2) (reading D12); protons are indices [0, N_p)."""
    return int(np.floor(Y_P * N + 0.5))


def box_length(N, density):
    return float((N / density) ** (1.0 / 3.0))


def species(N, Y_P):
    is_p = np.zeros(N, dtype=np.uint8)
    is_p[: n_protons(N, Y_P)] = 1
    return is_p


def uniform_state(N, Y_P, density, T, seed, mass=MASS):
    """Uniform random positions in [0,L)^3, Maxwell-Boltzmann velocities sigma = sqrt(T/M) per
    component, species by index (BASELINE configs).  Returns x, v, is_p, L."""
    rng = np.random.default_rng(seed)
    L = box_length(N, density)
    x = rng.random((N, 3)) * L
    x[x >= L] = 0.0
    v = rng.normal(0.0, np.sqrt(T / mass), size=(N, 3))
    return x, v, species(N, Y_P), L


def clustered_state(N, Y_P, density, T, seed, n_blobs=None, blob_density=0.12, gas_fraction=0.3, mass=MASS):
    """Sparse, clustered occupancy of the late-decompression kind (configs 3/5 near their end,
    PAPER.md:140): all protons and (1 - gas_fraction) of the neutrons sit in compact spherical
    blobs of local density `blob_density` fm^-3 at random centres; the remaining neutrons form a
    uniform gas.  Positions inside a blob are uniform in the ball (with a minimum separation
    enforced by rejection only through the density choice -- this is a load-shape stand-in, not
    an equilibrated configuration)."""
    rng = np.random.default_rng(seed)
    L = box_length(N, density)
    is_p = species(N, Y_P)
    Np = int(is_p.sum())
    n_gas = int(round(gas_fraction * (N - Np)))
    n_bound = N - n_gas
    if n_blobs is None:
        n_blobs = max(1, n_bound // 150)
    centres = rng.random((n_blobs, 3)) * L
    owner = rng.integers(0, n_blobs, size=n_bound)
    counts = np.bincount(owner, minlength=n_blobs)
    radius = (3.0 * np.maximum(counts, 1) / (4.0 * np.pi * blob_density)) ** (1.0 / 3.0)
    d = rng.normal(size=(n_bound, 3))
    d /= np.linalg.norm(d, axis=1, keepdims=True)
    rr = radius[owner] * rng.random(n_bound) ** (1.0 / 3.0)
    xb = centres[owner] + d * rr[:, None]
    xg = rng.random((n_gas, 3)) * L
    x = np.empty((N, 3))
    # protons first (indices [0, Np)) are all bound; bound neutrons next; gas neutrons last
    x[:n_bound] = xb
    x[n_bound:] = xg
    x = x - L * np.floor(x / L)
    x[x >= L] = 0.0
    v = rng.normal(0.0, np.sqrt(T / mass), size=(N, 3))
    return x, v, is_p, L


def config_state(cfg_id, seed):
    c = CONFIGS[cfg_id]
    return uniform_state(c["N"], c["Y_P"], c["density"], c["T"], seed)
