"""Writes the stored oracle values under tests/golden/.  Calls ONLY oracle/ (plus the seeded input generators).

    python tests/golden/make_golden.py C1 C2 C3          # full V_x: E_x (E1, E2), per-band energies, per-band norms, 2 rows
    python tests/golden/make_golden.py C4a C4b C5        # sampled rows only (parity pinned by sampling)

Outputs per config: exx_<name>.json (scalars, per-band values) and exx_<name>_rows.npz (the sampled V_x rows).
Nothing here is a paper value: the paper prints no E_x; these are oracle results for the seeded
synthetic inputs of DESIGN.md section 4, stored because the oracle needs minutes to hours for them.
"""
import json
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import exx_ref as R  # noqa: E402
from paper_1111_0716_b200 import workloads as W  # noqa: E402

HERE = os.path.dirname(os.path.abspath(__file__))
FULL = ("C1", "C2", "C3")


def sample_rows(w):
    """first/last band at first/last k; fewer for the largest grids."""
    rows = [(0, 0), (w.nk - 1, w.nbands - 1)]
    if w.name in ("C2",):
        rows += [(0, w.nbands - 1), (3, 7)]
    return rows


def main(names):
    for name in names:
        w = W.make(name)
        o = R.RefExx(w.grid, w.lattice, w.kfrac, w.kweight, w.ecut, w.kernel_kind, w.mu, w.scale, w.nbands)
        psi = w.coefficients(o.npw)
        rows = sample_rows(w)
        rec = {"config": name, "seed": w.seed, "grid": list(w.grid), "npw": o.npw, "nbands": w.nbands, "nk": w.nk,
               "oracle_threads": R.num_threads(), "rows": [list(r) for r in rows],
               "psi_first": [psi[0].real, psi[0].imag], "map0_sum": int(o.index_map(0).astype(np.int64).sum())}
        t0 = time.time()
        if name in FULL:
            out = o.apply(psi, w.occ)
            e1, per_band = o.energy(psi, w.occ, out)
            rec["t_apply_s"] = time.time() - t0
            t1 = time.time()
            rec["E_x_E1"] = e1
            rec["E_x_E2"] = o.energy_e2(psi, w.occ)
            rec["t_e2_s"] = time.time() - t1
            rec["per_band_energy"] = per_band.tolist()
            rec["per_band_norm"] = [float(np.linalg.norm(o.band(out, k, n))) for k in range(w.nk) for n in range(w.nbands)]
            row_data = [o.band(out, k, n).copy() for k, n in rows]
        else:
            row_data = o.apply_rows(psi, w.occ, rows)
            rec["t_rows_s"] = time.time() - t0
        rec["row_energy"] = [0.5 * w.kweight[k] * w.occ[k * w.nbands + n] * float(np.vdot(o.band(psi, k, n), r).real)
                             for (k, n), r in zip(rows, row_data)]
        rec["row_norm"] = [float(np.linalg.norm(r)) for r in row_data]
        with open(os.path.join(HERE, "exx_%s.json" % name), "w") as f:
            json.dump(rec, f, indent=1)
        np.savez_compressed(os.path.join(HERE, "exx_%s_rows.npz" % name), **{"row%d" % i: r for i, r in enumerate(row_data)})
        print(name, "done in %.1f s" % (time.time() - t0), flush=True)


if __name__ == "__main__":
    main(sys.argv[1:] or list(FULL))
