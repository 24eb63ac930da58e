"""Literal triple loop of Eq. (1) in Python complex128 -- for tiny grids only (pin P2).

TEST INFRASTRUCTURE ONLY.  Independent of pdm_oracle.c: written separately from the same
passages (Eq. (1); Alg. 1 :59-70; readings R3, R5, R6, R8, R11) so
that an indexing slip in either shows up as a disagreement.
"""
from __future__ import annotations

import numpy as np


def brute_force_migrate(cfg: dict) -> np.ndarray:
    nx, nz, nw = cfg["nx"], cfg["nz"], cfg["nw"]
    table = cfg["table"]
    ntab, ntaps = table.shape
    half = (ntaps - 1) // 2
    image = [[0.0 for _ in range(nx)] for _ in range(nz)]
    for iw in range(nw):                                   # "for each frequency"
        w32 = np.float32(cfg["omega"][iw])
        prev = [complex(c) for c in cfg["P0"][iw]]
        for iz in range(nz):                               # "for each depth level"
            nxt = []
            for i in range(nx):                            # "for each space"
                q32 = np.float32(np.float64(cfg["dz"]) /
                                 (np.float64(cfg["velocity"][iz, i]) * np.float64(cfg["du"])))
                j = int(np.rint(np.float32(w32 * q32)))    # look-up table (R3)
                j = min(max(j, 0), ntab - 1)
                total = 0j
                for n in range(-half, half + 1):           # Eq. (1): h[n] u(x_{i-n})
                    if 0 <= i - n < nx:
                        total += complex(table[j, half + n]) * prev[i - n]
                nxt.append(total)
            prev = nxt
            for i in range(nx):                            # depth row: sum over frequencies
                image[iz][i] += prev[i].real
    return np.array(image, dtype=np.float64)
