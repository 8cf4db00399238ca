"""Face connectivity and trace node maps (oracle; test infrastructure only).

PAPER.md:L75 defines q- (own trace) and q+ (neighbouring trace); L196 "trace data of the element and all its
neighbor node data"; L73: topology fixed for the whole run, all elements positively oriented.

Faces are matched through vertex ids (periodic images identified through ``vertex_equiv``); face nodes are matched
through the vertex permutation, never through coordinates: node n of element e has integer barycentric
weights attached to e's vertices; its partner in the neighbour is the node that attaches the same weights to the same
(equivalence classes of) vertices.  This exists because the node set is symmetric under vertex permutations.
"""
import numpy as np


class MeshError(ValueError):
    pass


def connect(ref, EToV, vertex_equiv=None, EToB=None):
    """Returns dict(EToE[K,Nfaces], EToF[K,Nfaces], vmapM[K,Nfaces,Nfp], vmapP[K,Nfaces,Nfp]).

    vmapM / vmapP index the flattened [K, Np] node array: vmap = e*Np + n.  Boundary faces (no partner) point to
    themselves (EToE = e, EToF = f, vmapP = vmapM) and must carry a non-zero tag in EToB.
    """
    EToV = np.asarray(EToV, dtype=np.int64)
    K, nv = EToV.shape
    dim = ref.dim
    assert nv == dim + 1
    ids = EToV if vertex_equiv is None else np.asarray(vertex_equiv, dtype=np.int64)[EToV]
    if np.any(np.sort(ids, axis=1)[:, 1:] == np.sort(ids, axis=1)[:, :-1]):
        raise MeshError("an element touches the same (periodic class of a) vertex twice: "
                        "a periodic direction needs at least 3 cells")
    Nfaces, Nfp, Np = ref.Nfaces, ref.Nfp, ref.Np
    fv = ref.face_verts                                     # [Nfaces, dim]
    faceids = ids[:, fv]                                    # [K, Nfaces, dim] ids of the face's vertices, local order
    key = np.sort(faceids, axis=2).reshape(K * Nfaces, dim)
    order = np.lexsort(key.T[::-1])
    ks = key[order]
    same = np.all(ks[1:] == ks[:-1], axis=1)
    # a face key may appear once (boundary) or twice (interior); three times means a non-manifold / too-short period
    if np.any(same[1:] & same[:-1]):
        raise MeshError("a face is shared by more than two elements (non-conforming or periodic direction < 3 cells)")
    EToE = np.repeat(np.arange(K)[:, None], Nfaces, axis=1)
    EToF = np.repeat(np.arange(Nfaces)[None, :], K, axis=0)
    a = order[:-1][same]
    b = order[1:][same]
    ea, fa = a // Nfaces, a % Nfaces
    eb, fb = b // Nfaces, b % Nfaces
    EToE[ea, fa], EToF[ea, fa] = eb, fb
    EToE[eb, fb], EToF[eb, fb] = ea, fa

    vmapM = (np.arange(K)[:, None, None] * Np + ref.fmask[None, :, :]).astype(np.int64)
    vmapP = vmapM.copy()
    interior = np.zeros((K, Nfaces), dtype=bool)
    interior[ea, fa] = True
    interior[eb, fb] = True
    if EToB is not None:
        EToB = np.asarray(EToB)
        if np.any((EToB != 0) & interior) or np.any((EToB == 0) & ~interior):
            raise MeshError("EToB tags do not match the unmatched faces")
    elif not interior.all():
        raise MeshError("unmatched faces but no EToB")

    # node matching, grouped by (own face, where each own-face vertex sits in the neighbour)
    E, F = np.nonzero(interior)
    En = EToE[E, F]
    own_ids = faceids[E, F]                                               # [n, dim]
    nbr_local = np.argmax(ids[En][:, None, :] == own_ids[:, :, None], axis=2)   # [n, dim] local vertex no. in nbr
    code = F.copy()
    for m in range(dim):
        code = code * (dim + 1) + nbr_local[:, m]
    for c in np.unique(code):
        sel = np.nonzero(code == c)[0]
        f = F[sel[0]]
        loc = nbr_local[sel[0]]
        partner = np.empty(Nfp, dtype=np.int64)
        for m, n in enumerate(ref.fmask[f]):
            w = ref.lattice[n]                                            # weights on own local vertices
            wn = [0] * (dim + 1)
            for j, v in enumerate(fv[f]):
                wn[loc[j]] = int(w[v])
            partner[m] = ref.node_of[tuple(wn)]
        vmapP[E[sel], f, :] = En[sel, None] * Np + partner[None, :]
    return dict(EToE=EToE, EToF=EToF, vmapM=vmapM, vmapP=vmapP)
