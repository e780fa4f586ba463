"""Synthetic tetrahedral box meshes (stand-ins for the paper's unstructured meshes, which are not
available: PAPER.md:413-422 validation meshes, PAPER.md:454 salt-dome mesh).

A box of nx*ny*nz hexahedra, each hexahedron cut into 6 tetrahedra around its main diagonal (Kuhn
split).  The same split is used in every hexahedron, so the mesh is conforming.  Interior vertices
may be jittered; boundary vertices stay put so the box stays a box.

Outputs are plain arrays only: EToV int32 [K,4] (0-based vertex ids, positive orientation),
VX float64 [Nv,3].
"""
from itertools import permutations

import numpy as np


def _perm_sign(p):
    sign = 1
    p = list(p)
    for i in range(len(p)):
        while p[i] != i:
            j = p[i]
            p[i], p[j] = p[j], p[i]
            sign = -sign
    return sign


def _lattice_vertices(nx, ny, nz, lengths):
    lx, ly, lz = lengths
    xs = np.linspace(0.0, lx, nx + 1)
    ys = np.linspace(0.0, ly, ny + 1)
    zs = np.linspace(0.0, lz, nz + 1)
    # vertex id = i + (nx+1)*(j + (ny+1)*k)
    Z, Y, X = np.meshgrid(zs, ys, xs, indexing="ij")
    return np.stack([X.ravel(), Y.ravel(), Z.ravel()], axis=1)


def _kuhn_tets(nx, ny, nz):
    """EToV for the Kuhn split, hex-major (6 consecutive tets per hex, hexes x fastest)."""
    def vid(i, j, k):
        return i + (nx + 1) * (j + (ny + 1) * k)

    k_idx, j_idx, i_idx = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    i_idx = i_idx.ravel()
    j_idx = j_idx.ravel()
    k_idx = k_idx.ravel()
    nhex = i_idx.size
    etov = np.empty((nhex, 6, 4), dtype=np.int64)
    unit = np.eye(3, dtype=np.int64)
    for t, perm in enumerate(permutations(range(3))):
        off0 = np.zeros(3, dtype=np.int64)
        off1 = off0 + unit[perm[0]]
        off2 = off1 + unit[perm[1]]
        off3 = np.ones(3, dtype=np.int64)
        offs = [off0, off1, off2, off3]
        if _perm_sign(perm) < 0:
            offs[2], offs[3] = offs[3], offs[2]
        for v, off in enumerate(offs):
            etov[:, t, v] = vid(i_idx + off[0], j_idx + off[1], k_idx + off[2])
    return etov.reshape(nhex * 6, 4).astype(np.int32)


def box_tet_mesh(nx, ny, nz, lengths=(1.0, 1.0, 1.0), jitter=0.0, seed=None):
    """Kuhn-split box mesh.  `jitter` is the fraction of the hex size h by which each coordinate
    of each INTERIOR vertex is moved, uniformly in [-jitter*h, +jitter*h] (seeded)."""
    vx = _lattice_vertices(nx, ny, nz, lengths)
    etov = _kuhn_tets(nx, ny, nz)
    if jitter > 0.0:
        rng = np.random.default_rng(seed)
        h = np.array([lengths[0] / nx, lengths[1] / ny, lengths[2] / nz])
        delta = rng.uniform(-jitter, jitter, size=vx.shape) * h
        interior = np.ones(vx.shape[0], dtype=bool)
        for d in range(3):
            interior &= (vx[:, d] > 1e-12 * lengths[d]) & (vx[:, d] < lengths[d] * (1 - 1e-12))
        vx = vx + delta * interior[:, None]
    return etov, vx


def graded_box_tet_mesh(nx, ny, nz, lengths, band_center, band_width, max_ratio, seed,
                        blob_sigma_cells=4.0):
    """Conforming *graded* box mesh (stand-in for the 4x local refinement of BASELINE.json config 3):
    inside a horizontal band of thickness `band_width` around depth `band_center` the layer
    thickness is shrunk by a factor that varies smoothly in (x, y) between 1 and `max_ratio`
    (seeded Gaussian-filtered noise, thresholded into blobs).  Only z coordinates move, the top and
    bottom of the box stay planar."""
    from scipy.ndimage import gaussian_filter

    lx, ly, lz = lengths
    rng = np.random.default_rng(seed)
    noise = rng.standard_normal((ny + 1, nx + 1))
    smooth = gaussian_filter(noise, sigma=blob_sigma_cells, mode="reflect")
    smooth = (smooth - smooth.min()) / (smooth.max() - smooth.min())
    # blobs: ramp from 1 to max_ratio over the upper 40 % of the filtered-noise range
    ramp = np.clip((smooth - 0.6) / 0.25, 0.0, 1.0)
    shrink = 1.0 + (max_ratio - 1.0) * ramp                    # [ny+1, nx+1], in [1, max_ratio]
    zc = (np.arange(nz) + 0.5) * (lz / nz)                     # nominal layer centres
    in_band = np.abs(zc - band_center) <= 0.5 * band_width     # [nz]
    weight = np.ones((nz, ny + 1, nx + 1))
    weight[in_band] = 1.0 / shrink[None, :, :]
    cum = np.concatenate([np.zeros((1, ny + 1, nx + 1)), np.cumsum(weight, axis=0)], axis=0)
    zcol = lz * cum / cum[-1][None, :, :]                      # [nz+1, ny+1, nx+1]
    vx = _lattice_vertices(nx, ny, nz, lengths)
    vx[:, 2] = zcol.ravel()
    etov = _kuhn_tets(nx, ny, nz)
    return etov, vx


def permute_elements(etov, seed):
    """Seeded random element permutation (mimics the arbitrary element order of an unstructured
    mesh).  Returns (etov_permuted, perm) with etov_permuted[i] = etov[perm[i]]."""
    rng = np.random.default_rng(seed)
    perm = rng.permutation(etov.shape[0])
    return np.ascontiguousarray(etov[perm]), perm


def box_side_bc(etov, vx, lengths, top=1, bottom=3, sides=2):
    """face_bc[K][4] (int8) of a box mesh by box side: faces on z = 0 get `top`, on z = Lz `bottom`, all others `sides`
    (1 free surface, 2 absorbing, 3 rigid, 4 prescribed; only the entries of boundary faces are read by the solvers).
    A face is assigned by the position of its centroid; local face f holds the vertices below (reference-element
    convention shared by all users: F0 = {0,1,2}, F1 = {0,1,3}, F2 = {1,2,3}, F3 = {0,2,3})."""
    faces = ((0, 1, 2), (0, 1, 3), (1, 2, 3), (0, 2, 3))
    bc = np.full((etov.shape[0], 4), sides, dtype=np.int8)
    for f, fv in enumerate(faces):
        zc = vx[etov[:, fv]].mean(axis=1)[:, 2]
        bc[zc < 1e-9 * lengths[2], f] = top
        bc[zc > lengths[2] * (1 - 1e-9), f] = bottom
    return bc
