"""Shared test helpers (no arithmetic of the method)."""
import numpy as np

from paper_2012_06144_b200 import inputs


def random_state(p: inputs.Params, seed: int):
    """Random but physical-looking state for one-step comparisons: smooth phi in (0,1),
    small u, positive h around phi*w, small g."""
    rng = np.random.Generator(np.random.PCG64(seed))
    z, y, x = np.meshgrid(np.arange(p.nz), np.arange(p.ny), np.arange(p.nx), indexing="ij")
    phi = 0.5 + 0.35 * np.sin(2 * np.pi * (x + 0.3) / p.nx) * np.cos(2 * np.pi * (y + 0.1) / p.ny) \
        + 0.1 * np.sin(2 * np.pi * (z + 0.7) / p.nz)
    u = rng.uniform(-0.02, 0.02, size=(3,) + p.shape)
    h = rng.uniform(0.2, 1.0, size=(p.stencil_phase,) + p.shape) * phi[None] / p.stencil_phase
    g = rng.uniform(-1e-3, 1e-3, size=(p.stencil_hydro,) + p.shape)
    return phi, u, h, g
