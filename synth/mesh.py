"""Hex8 meshes.  Node order per element: xi-signs
(-,-,-),(+,-,-),(+,+,-),(-,+,-),(-,-,+),(+,-,+),(+,+,+),(-,+,+).
Nodes lexicographic (x fastest), elements lexicographic."""
import numpy as np
from . import rng

_OFF = np.array([[0, 0, 0], [1, 0, 0], [1, 1, 0], [0, 1, 0],
                 [0, 0, 1], [1, 0, 1], [1, 1, 1], [0, 1, 1]], dtype=np.int64)


def structured_hex_mesh(nx, ny, nz, lx=1.0, ly=1.0, lz=1.0):
    xs = np.linspace(0.0, lx, nx + 1)
    ys = np.linspace(0.0, ly, ny + 1)
    zs = np.linspace(0.0, lz, nz + 1)
    Z, Y, X = np.meshgrid(zs, ys, xs, indexing="ij")
    coords = np.stack([X.ravel(), Y.ravel(), Z.ravel()], axis=1).astype(np.float64)
    ez, ey, ex = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    ex, ey, ez = ex.ravel(), ey.ravel(), ez.ravel()
    conn = np.empty((ex.size, 8), dtype=np.int32)
    for a in range(8):
        i, j, k = ex + _OFF[a, 0], ey + _OFF[a, 1], ez + _OFF[a, 2]
        conn[:, a] = (i + (nx + 1) * (j + (ny + 1) * k)).astype(np.int32)
    return coords, conn


def distort(coords, seed, amp):
    """Move every node by amp*U[-1,1) per component (used by oracle pins only)."""
    n = coords.shape[0]
    idx = np.arange(3 * n, dtype=np.uint64)
    d = (2.0 * rng.uniform(seed, rng.STREAM["aux"], idx) - 1.0).reshape(n, 3)
    return coords + amp * d


def void_mask_mesh(nx, ny, nz, seed, void_frac=0.30, shuffle=True):
    """Structured cube minus a smooth-field void mask (config 4): element
    removed iff v(centroid) < quantile(void_frac); unreferenced nodes deleted,
    remaining nodes renumbered in lexicographic order; element order shuffled."""
    coords, conn = structured_hex_mesh(nx, ny, nz)
    cen = coords[conn.astype(np.int64)].mean(axis=1)
    v = np.zeros(cen.shape[0])
    for k in range(6):
        kk = 1 + np.floor(3 * rng.uniform(seed, rng.STREAM["void"], np.arange(3) + 10 * k)).astype(int)
        ph = 2 * np.pi * rng.uniform(seed, rng.STREAM["void"], np.arange(3) + 10 * k + 5)
        v += np.cos(2 * np.pi * kk[0] * cen[:, 0] + ph[0]) * np.cos(2 * np.pi * kk[1] * cen[:, 1] + ph[1]) \
            * np.cos(2 * np.pi * kk[2] * cen[:, 2] + ph[2])
    keep = v >= np.quantile(v, void_frac)
    conn = conn[keep]
    used = np.zeros(coords.shape[0], dtype=bool)
    used[conn.ravel()] = True
    new_id = np.cumsum(used) - 1
    coords = coords[used]
    conn = new_id[conn.astype(np.int64)].astype(np.int32)
    if shuffle:
        p = rng.permutation(seed, rng.STREAM["shuffle"], conn.shape[0])
        conn = conn[p]
    return np.ascontiguousarray(coords), np.ascontiguousarray(conn)
