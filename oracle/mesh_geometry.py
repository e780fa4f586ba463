"""ORACLE (test infrastructure, fp64, plain numpy) - per-element geometry and connectivity.

Geometry: affine map Psi_k from the reference tet (App. A).  The volume factors
are read as the INVERSE Jacobian g^vol_{k,i,j} = d r_j / d x_i (reading Q3: PAPER.md:610,
622 print dPsi_i/dr_j, which is dimensionally wrong for the chain rule).  Surface factor
g^sur_{k,f} = J_{k,f}/J_k with J_{k,f} = (face area)/2 (reference triangle of area 2).

Connectivity: two faces are the same face iff their sorted vertex-id triples are equal; face-node
matching by nearest physical node (reading O3).
"""
import numpy as np

from .reference_element import FACE_VERTICES


def element_geometry(EToV, VX):
    """Returns dict with J [K], ginv [K,3,3] (ginv[k,i,j] = d r_j/d x_i), normals [K,4,3] (outward,
    unit), gsur [K,4] (= J_{k,f}/J_k), area [K,4], volume [K], ell [K] (smallest face-to-opposite-
    vertex distance)."""
    v = VX[EToV]                                   # [K,4,3]
    # x(r,s,t) = (-(1+r+s+t) v0 + (1+r) v1 + (1+s) v2 + (1+t) v3)/2
    xr = 0.5 * (v[:, 1] - v[:, 0])
    xs = 0.5 * (v[:, 2] - v[:, 0])
    xt = 0.5 * (v[:, 3] - v[:, 0])
    jac = np.stack([xr, xs, xt], axis=2)           # jac[k,i,j] = d x_i / d r_j
    J = np.linalg.det(jac)
    inv = np.linalg.inv(jac)                       # inv[k,j,i] = d r_j / d x_i
    ginv = np.transpose(inv, (0, 2, 1))            # ginv[k,i,j] = d r_j / d x_i
    grad_r, grad_s, grad_t = ginv[:, :, 0], ginv[:, :, 1], ginv[:, :, 2]
    # outward normals of F0 (t=-1), F1 (s=-1), F2 (r+s+t=-1), F3 (r=-1): -grad t, -grad s,
    # grad(r+s+t), -grad r
    nvec = np.stack([-grad_t, -grad_s, grad_r + grad_s + grad_t, -grad_r], axis=1)   # [K,4,3]
    gsur = np.linalg.norm(nvec, axis=2)            # |grad xi_f| = J_{k,f}/J_k
    normals = nvec / gsur[:, :, None]
    volume = J * (4.0 / 3.0)
    area = 2.0 * gsur * J[:, None]
    ell = (3.0 * volume[:, None] / area).min(axis=1)
    return dict(J=J, ginv=ginv, normals=normals, gsur=gsur, area=area, volume=volume, ell=ell)


def node_coordinates(ref, EToV, VX):
    """Physical coordinates of all nodes, [K,Np,3]."""
    lam = np.stack([-(1 + ref.r + ref.s + ref.t) / 2, (1 + ref.r) / 2, (1 + ref.s) / 2,
                    (1 + ref.t) / 2], axis=1)      # [Np,4]
    return np.einsum("nv,kvd->knd", lam, VX[EToV])


def face_vertex_keys(EToV):
    """Sorted global vertex triple of every (element, local face): [K,4,3]."""
    K = EToV.shape[0]
    keys = np.empty((K, 4, 3), dtype=np.int64)
    for f, fv in enumerate(FACE_VERTICES):
        keys[:, f, :] = np.sort(EToV[:, list(fv)], axis=1)
    return keys


def connect_faces(EToV):
    """EToE, EToF [K,4] int32, -1 on boundary faces (sort-based matching)."""
    K = EToV.shape[0]
    keys = face_vertex_keys(EToV).reshape(K * 4, 3)
    order = np.lexsort((keys[:, 2], keys[:, 1], keys[:, 0]))
    sk = keys[order]
    same = np.all(sk[1:] == sk[:-1], axis=1)
    if np.any(same[1:] & same[:-1]):
        raise ValueError("non-conforming mesh: a face is shared by more than two elements")
    EToE = np.full(K * 4, -1, dtype=np.int32)
    EToF = np.full(K * 4, -1, dtype=np.int32)
    a = order[:-1][same]
    b = order[1:][same]
    EToE[a], EToF[a] = b // 4, b % 4
    EToE[b], EToF[b] = a // 4, a % 4
    return EToE.reshape(K, 4), EToF.reshape(K, 4)


def connect_faces_bruteforce(EToV):
    """O(K^2) reference implementation for tiny meshes (pin for connect_faces)."""
    K = EToV.shape[0]
    keys = face_vertex_keys(EToV)
    EToE = np.full((K, 4), -1, dtype=np.int32)
    EToF = np.full((K, 4), -1, dtype=np.int32)
    for k in range(K):
        for f in range(4):
            for k2 in range(K):
                if k2 == k:
                    continue
                for f2 in range(4):
                    if tuple(keys[k, f]) == tuple(keys[k2, f2]):
                        assert EToE[k, f] == -1
                        EToE[k, f], EToF[k, f] = k2, f2
    return EToE, EToF


def match_face_nodes(ref, EToV, VX, EToE, EToF, chunk=20000):
    """mapP [K,4,Nfp] int32: face-node index i' on the neighbour face whose physical node coincides
    with face node i of (k,f); the identity on boundary faces."""
    K = EToV.shape[0]
    Nfp = ref.Nfp
    geo_ell = element_geometry(EToV, VX)["ell"]
    mapP = np.tile(np.arange(Nfp, dtype=np.int32), (K, 4, 1))
    for k0 in range(0, K, chunk):
        ks = np.arange(k0, min(K, k0 + chunk))
        X = node_coordinates(ref, EToV[ks], VX)                     # [kc,Np,3]
        for f in range(4):
            nb = EToE[ks, f]
            inter = nb >= 0
            if not np.any(inter):
                continue
            kk = ks[inter]
            own = X[inter][:, ref.Fmask[f], :]                       # [m,Nfp,3]
            nbX = node_coordinates(ref, EToV[nb[inter]], VX)         # [m,Np,3]
            fm = ref.Fmask[EToF[kk, f]]                              # [m,Nfp]
            other = np.take_along_axis(nbX, fm[:, :, None], axis=1)  # [m,Nfp,3]
            d = np.linalg.norm(own[:, :, None, :] - other[:, None, :, :], axis=3)
            idx = d.argmin(axis=2)
            dmin = d.min(axis=2)
            if np.any(dmin > 1e-9 * geo_ell[kk][:, None]):
                raise ValueError("face nodes of neighbouring elements do not coincide")
            if np.any(np.sort(idx, axis=1) != np.arange(Nfp)[None, :]):
                raise ValueError("face-node matching is not a bijection")
            mapP[kk, f, :] = idx
    return mapP
