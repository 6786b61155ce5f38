"""Test-side helpers: tiny octrees and an INDEPENDENT geometric description of a hierarchy.

Nothing here is imported by the product or by the oracle.  `Geometry` re-derives leaf boxes from the
(child, n_cells) arrays alone (top-down from the root), so it can check walks produced by either side.
"""
from __future__ import annotations

import numpy as np


def random_octree(root_shape, n_levels, p_refine, seed, rho_lo=0.2, rho_hi=3.0, p_empty=0.0):
    """Random hierarchy in the paper's cell-vector order.  Returns (n_cells, rho, child)."""
    rng = np.random.default_rng(seed)
    nx, ny, nz = root_shape
    n = nx * ny * nz
    n_cells, rhos, childs = [], [], []
    for lev in range(n_levels):
        refine = (rng.random(n) < p_refine) if lev < n_levels - 1 else np.zeros(n, dtype=bool)
        child = np.full(n, -1, dtype=np.int32)
        child[refine] = 8 * np.arange(int(refine.sum()), dtype=np.int32)
        rho = rng.uniform(rho_lo, rho_hi, n).astype(np.float32)
        if p_empty > 0:
            rho[rng.random(n) < p_empty] = 0.0
        rho[refine] = 0.0
        n_cells.append(n); rhos.append(rho); childs.append(child)
        n = 8 * int(refine.sum())
        if n == 0:
            break
    return np.asarray(n_cells, dtype=np.int64), np.concatenate(rhos), np.concatenate(childs)


def fully_refined(rho2n):
    """Hierarchy whose every root cell is refined once and whose leaves are the cells of the regular
    (2N)^3 array rho2n[z][y][x].  Returns (n_cells, rho, child, leaf_gid_of[z][y][x])."""
    n2 = rho2n.shape[0]
    n = n2 // 2
    n_root = n ** 3
    child = np.concatenate([8 * np.arange(n_root, dtype=np.int32), np.full(8 * n_root, -1, dtype=np.int32)])
    rho = np.zeros(9 * n_root, dtype=np.float32)
    gid_of = np.zeros((n2, n2, n2), dtype=np.int64)
    iz, iy, ix = np.meshgrid(np.arange(n2), np.arange(n2), np.arange(n2), indexing="ij")
    root = (ix // 2) + n * ((iy // 2) + n * (iz // 2))
    slot = (ix & 1) + 2 * (iy & 1) + 4 * (iz & 1)
    gid = n_root + 8 * root + slot
    rho[gid.ravel()] = rho2n.ravel()
    gid_of[...] = gid
    return np.array([n_root, 8 * n_root], dtype=np.int64), rho, child, gid_of


class Geometry:
    """Leaf boxes of a hierarchy, derived top-down from (root shape, n_cells, child)."""

    def __init__(self, root_shape, n_cells, child):
        self.nx, self.ny, self.nz = root_shape
        self.n_cells = np.asarray(n_cells, dtype=np.int64)
        self.off = np.concatenate([[0], np.cumsum(self.n_cells)])
        self.child = None if child is None else np.asarray(child)

    def is_leaf(self, gid):
        return self.child is None or self.child[gid] < 0

    def locate(self, x, y, z):
        """Leaf (gid, level, origin[3], edge) that contains the point (half-open boxes)."""
        ix, iy, iz = int(np.floor(x)), int(np.floor(y)), int(np.floor(z))
        ix = min(max(ix, 0), self.nx - 1); iy = min(max(iy, 0), self.ny - 1); iz = min(max(iz, 0), self.nz - 1)
        level, c = 1, ix + self.nx * (iy + self.ny * iz)
        org = np.array([ix, iy, iz], dtype=np.float64)
        h = 1.0
        while True:
            gid = int(self.off[level - 1] + c)
            if self.is_leaf(gid):
                return gid, level, org, h
            h *= 0.5
            bx, by, bz = int(x >= org[0] + h), int(y >= org[1] + h), int(z >= org[2] + h)
            org = org + h * np.array([bx, by, bz])
            c = int(self.child[gid]) + bx + 2 * by + 4 * bz
            level += 1

    def leaf_boxes(self):
        """All leaves: arrays gid, level, origin[n,3], edge."""
        out = []
        n_root = self.nx * self.ny * self.nz
        c = np.arange(n_root)
        org = np.stack([c % self.nx, (c // self.nx) % self.ny, c // (self.nx * self.ny)], axis=1).astype(np.float64)
        cells = c
        h = 1.0
        for level in range(1, len(self.n_cells) + 1):
            gid = self.off[level - 1] + cells
            ch = np.full(len(cells), -1) if self.child is None else self.child[gid]
            leaf = ch < 0
            out.append((gid[leaf], np.full(int(leaf.sum()), level), org[leaf], np.full(int(leaf.sum()), h)))
            if leaf.all():
                break
            par_org, par_ch = org[~leaf], ch[~leaf]
            h *= 0.5
            s = np.arange(8)
            off = np.stack([s & 1, (s >> 1) & 1, (s >> 2) & 1], axis=1) * h
            org = (par_org[:, None, :] + off[None, :, :]).reshape(-1, 3)
            cells = (par_ch[:, None] + s[None, :]).reshape(-1)
        return (np.concatenate([o[0] for o in out]), np.concatenate([o[1] for o in out]),
                np.concatenate([o[2] for o in out]), np.concatenate([o[3] for o in out]))

    def interior_interface_area(self):
        """Total area of the faces shared by two different leaves (root-cell units), brute force on the
        finest lattice."""
        gid, level, org, h = self.leaf_boxes()
        m = 2 ** (int(level.max()) - 1)
        lab = np.zeros((self.nz * m, self.ny * m, self.nx * m), dtype=np.int64)
        for g, o, e in zip(gid, org, h):
            x0, y0, z0 = (o * m).astype(int)
            k = int(round(e * m))
            lab[z0:z0 + k, y0:y0 + k, x0:x0 + k] = g
        cnt = 0
        cnt += int((lab[1:, :, :] != lab[:-1, :, :]).sum())
        cnt += int((lab[:, 1:, :] != lab[:, :-1, :]).sum())
        cnt += int((lab[:, :, 1:] != lab[:, :, :-1]).sum())
        return cnt / float(m * m)
