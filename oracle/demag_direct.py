"""Direct real-space demagnetizing field (oracle, test infrastructure).

This is the definition, PAPER.md:L323 (Table 1), equal to Eq. 4
with a single mesh:

    H_a(t) = - sum_{s in mesh} sum_b N_ab(r_t - r_s) M_b(s),   a, b in {x, y, z}

with the self term s = t included, N symmetric, everything in fp64, M the
float32 input upcast to fp64.  The argument order (PAPER.md writes N(r - r0)
in Table 1 and N(r' - r) in Eq. 4) is immaterial because N_ab(-R) = N_ab(R)
for equal cells (reading R2); target - source is used.

Arrays: M, H are [3][nz][ny][nx] (x fastest).  The tensor table comes from
``oracle.newell.newell_tensor_octant`` (non-negative displacements) and is
extended to negative displacements by parity.
"""
import numpy as np

from .newell import PARITY, SYM_INDEX, newell_tensor_octant


def _components_needed(nz):
    # reading R7: at nz == 1 every displacement has Z = 0, where Nxz = Nyz = 0
    # (odd in z), so they need not be evaluated.
    return (0, 1, 2, 3) if nz == 1 else (0, 1, 2, 3, 4, 5)


def tensor_table(shape, h):
    """fp64 octant table [6][nz][ny][nx] for a mesh of `shape` = (nz, ny, nx)."""
    nz, ny, nx = shape
    return newell_tensor_octant(nx, ny, nz, h[0], h[1], h[2],
                                components=_components_needed(nz))


def demag_at(M, h, targets, table=None):
    """H at the listed target cells, by the plain sum over all source cells.

    M: [3][nz][ny][nx] (any float dtype; upcast to fp64).  h = (hx, hy, hz).
    targets: iterable of (k, j, i) = (z, y, x) cell indices.
    Returns fp64 array [len(targets)][3].
    """
    M = np.asarray(M, np.float64)
    _, nz, ny, nx = M.shape
    if table is None:
        table = tensor_table((nz, ny, nx), h)
    ks, js, is_ = np.arange(nz), np.arange(ny), np.arange(nx)
    out = np.zeros((len(targets), 3), np.float64)
    for n, (kt, jt, it) in enumerate(targets):
        dk, dj, di = kt - ks, jt - js, it - is_          # target - source
        idx = np.ix_(np.abs(dk), np.abs(dj), np.abs(di))
        sk = np.sign(dk)[:, None, None]
        sj = np.sign(dj)[None, :, None]
        si = np.sign(di)[None, None, :]
        # N_c(dk, dj, di) = table_c(|dk|,|dj|,|di|) * (parity sign per negative
        # coordinate); sign(0) = 0 is harmless: odd components vanish there.
        Nc = []
        for c in range(6):
            W = table[c][idx]
            px, py, pz = PARITY[c]
            if px < 0:
                W = W * si
            if py < 0:
                W = W * sj
            if pz < 0:
                W = W * sk
            Nc.append(W)
        for a in range(3):
            acc = 0.0
            for b in range(3):
                acc += np.sum(Nc[SYM_INDEX[a, b]] * M[b])   # numpy pairwise sum
            out[n, a] = -acc
    return out


def demag_direct(M, h, table=None):
    """H on the whole mesh by the plain double sum (small meshes only: O(N^2))."""
    M = np.asarray(M, np.float64)
    _, nz, ny, nx = M.shape
    targets = [(k, j, i) for k in range(nz) for j in range(ny) for i in range(nx)]
    Ht = demag_at(M, h, targets, table=table)
    return np.ascontiguousarray(Ht.T.reshape(3, nz, ny, nx))
