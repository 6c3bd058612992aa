"""Star files: the paper's code can read "a file of microlens positions and masses"
(P:212); the format is not specified there.  Here: text, one star per line, `x1 x2 mass` in units of
theta_star and of the mean mass, separated by blanks or commas, `#` starts a comment -- or a NumPy `.npy` array of
shape (n, 3).  Input/output only: the arrays go to `Field.from_stars(...)` together with the region (R or c1, c2) and
kappa_star the caller states; `Field.info()["kappa_star_actual"]` reports what the stars themselves amount to (eq 9).
"""
import numpy as np


def read_star_file(path):
    """Returns (x, y, m) as float64 arrays."""
    if str(path).endswith(".npy"):
        a = np.load(path)
    else:
        with open(path) as fh:
            rows = [ln.split("#", 1)[0].replace(",", " ").split() for ln in fh]
        a = np.array([[float(v) for v in r[:3]] for r in rows if r], dtype=np.float64).reshape(-1, 3)
    a = np.asarray(a, dtype=np.float64)
    if a.ndim != 2 or a.shape[1] != 3:
        raise ValueError("a star file holds three columns: x1 x2 mass")
    if not np.all(np.isfinite(a)) or np.any(a[:, 2] <= 0):
        raise ValueError("star positions must be finite and masses positive")
    return np.ascontiguousarray(a[:, 0]), np.ascontiguousarray(a[:, 1]), np.ascontiguousarray(a[:, 2])


def write_star_file(path, x, y, m):
    a = np.column_stack([np.asarray(x, dtype=np.float64), np.asarray(y, dtype=np.float64), np.asarray(m, dtype=np.float64)])
    if str(path).endswith(".npy"):
        np.save(path, a)
    else:
        np.savetxt(path, a, fmt="%.17g", header="x1 x2 mass (theta_star, mean mass)")
