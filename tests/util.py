"""Helpers for the tests: global <-> block arrays on uniform grids, error norm."""
import numpy as np


def to_global(cfg, blocks, X):
    """[nB][8][8][8][8] block arrays of a UNIFORM level-0 grid -> [8][Nz][Ny][Nx]."""
    nx, ny, nz = cfg["n_root"]
    G = np.zeros((X.shape[1], 8 * nz, 8 * ny, 8 * nx))
    for b, (lev, I, J, K) in enumerate(blocks):
        assert lev == 0
        G[:, 8 * K:8 * K + 8, 8 * J:8 * J + 8, 8 * I:8 * I + 8] = X[b]
    return G


def from_global(cfg, blocks, G):
    X = np.zeros((len(blocks), G.shape[0], 8, 8, 8))
    for b, (lev, I, J, K) in enumerate(blocks):
        X[b] = G[:, 8 * K:8 * K + 8, 8 * J:8 * J + 8, 8 * I:8 * I + 8]
    return X


def rel_err_O9(x, ref):
    """SURVEY.md 8(c) O-9 / DESIGN.md: per variable group g in {rho, |rho u|, |B|, e}:
    max_cells |x - ref| / max_cells |ref|_g, vector components scaled by the group's
    max vector magnitude.  x, ref: [nB][8][...]."""
    out = []
    for sl in (slice(0, 1), slice(1, 4), slice(4, 7), slice(7, 8)):
        mag = np.sqrt((ref[:, sl] ** 2).sum(axis=1)).max()
        out.append(np.abs(x[:, sl] - ref[:, sl]).max() / max(mag, 1e-300))
    return max(out)


def rel_err_per_block(x, ref, floor=1e-4):
    """The O-9 norm taken block by block: per group g, max over blocks of
    max_cells |x - ref| / max(max_cells |ref|_g of the SAME block, floor * global max).  On a grid that
    spans several refinement levels and a large contrast (config 5) a block far below the global
    maximum cannot hide behind it: one 10^4 times smaller is still held to 1e-11 of its own size.  The
    floor keeps blocks whose group is zero up to round-off (momentum in gas at rest) from dividing
    noise by noise.  Returns {group: value}."""
    out = {}
    nB = ref.shape[0]
    for name, sl in (("rho", slice(0, 1)), ("mom", slice(1, 4)), ("B", slice(4, 7)), ("e", slice(7, 8))):
        mag = np.sqrt((ref[:, sl] ** 2).sum(axis=1)).reshape(nB, -1).max(axis=1)
        err = np.abs(x[:, sl] - ref[:, sl]).reshape(nB, -1).max(axis=1)
        out[name] = float((err / np.maximum(np.maximum(mag, floor * mag.max()), 1e-300)).max())
    return out


def golden():
    """Values the paper prints (tests/golden/paper_values.txt): {key: float or tuple of floats}."""
    import os
    out = {}
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "paper_values.txt")
    for line in open(path):
        line = line.split("#", 1)[0].strip()
        if not line:
            continue
        key, val = (x.strip() for x in line.split("=", 1))
        nums = tuple(float(x) for x in val.split())
        out[key] = nums[0] if len(nums) == 1 else nums
    return out
