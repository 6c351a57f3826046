"""Seeded probe vectors for the per-band functional <z_k | (V_x c)_nk> stored by make_golden.py and re-evaluated by the GPU
parity tests.  A test functional only: it holds none of the method's arithmetic and is imported by neither oracle/ nor the
package."""
import numpy as np


def probe_vector(seed, ik, npw):
    """z_k: npw i.i.d. complex standard normals, unit 2-norm, from default_rng(seed + 7919 * (ik + 1))."""
    rng = np.random.default_rng(int(seed) + 7919 * (int(ik) + 1))
    z = rng.standard_normal(npw) + 1j * rng.standard_normal(npw)
    return z / np.linalg.norm(z)
