"""Writes the rest states quoted in paper_1309_1720_b200/workloads.py (REST) — calls only oracle/.

Rest state = the stable fixed point N[z] = 0 of each model as implemented (Q10), found
by Newton iteration with a central-difference Jacobian of oracle.reaction, polished until the
update stalls.  Run:  python -m oracle.rest_states
"""
import numpy as np
from . import oracle as O

STARTS = {0: (-0.659, -0.373), 1: (0.0, 0.0), 2: (0.0, 0.7457, 0.98474, 0.02155)}


def rest_state(model: int) -> np.ndarray:
    z = np.array(STARTS[model], dtype=np.float64)
    n = z.size
    for _ in range(60):
        f = O.reaction(model, z)
        J = np.empty((n, n))
        for c in range(n):
            h = 1e-6
            zp, zm = z.copy(), z.copy()
            zp[c] += h
            zm[c] -= h
            J[:, c] = (O.reaction(model, zp) - O.reaction(model, zm)) / (2 * h)
        try:
            dz = np.linalg.solve(J, -f)
        except np.linalg.LinAlgError:
            break
        z = z + dz
        if np.max(np.abs(dz)) < 1e-17:
            break
    return z


if __name__ == "__main__":
    for m, name in ((0, "FHN"), (1, "KARMA"), (2, "BOCF")):
        z = rest_state(m)
        print(f"    {name}: ({', '.join(repr(float(x)) for x in z)}),   # |N| = "
              f"{np.max(np.abs(O.reaction(m, z))):.2e}")
