"""Test-side mathematics used to PIN the oracle (and, on the GPU box, the CUDA path) to something other than
itself: closed forms, brute force, library routines.  Nothing here is imported by the oracle or the product."""
from __future__ import annotations

import zlib

import numpy as np


def crc(a: np.ndarray) -> str:
    return "%08x" % zlib.crc32(np.ascontiguousarray(a).tobytes())


def lattice_shape(L, d):
    return (L,) * d          # numpy index order [z][y][x]; site i = x + L*y + L*L*z  ==  C-order ravel


def axis_of(mu, d):
    return d - 1 - mu        # direction mu (0 = x) -> numpy axis


def energy_bruteforce(J, s, L, d):
    """E = -sum_mu sum_i J[mu][i] s_i s_{i+e_mu} via np.roll (Eq. (1)).  J [d][N], s [N]."""
    sg = s.reshape(lattice_shape(L, d)).astype(np.int64)
    e = 0
    for mu in range(d):
        Jg = J[mu].reshape(lattice_shape(L, d)).astype(np.int64)
        e -= int((Jg * sg * np.roll(sg, -1, axis=axis_of(mu, d))).sum())
    return e


def neighbour_list(L, d):
    """Explicit neighbour table nbr[i][2mu] = i+e_mu, nbr[i][2mu+1] = i-e_mu, built from coordinates."""
    N = L ** d
    idx = np.arange(N).reshape(lattice_shape(L, d))
    out = np.zeros((N, 2 * d), dtype=np.int64)
    for mu in range(d):
        out[:, 2 * mu] = np.roll(idx, -1, axis=axis_of(mu, d)).ravel()
        out[:, 2 * mu + 1] = np.roll(idx, +1, axis=axis_of(mu, d)).ravel()
    return out


def colours(L, d):
    g = np.indices(lattice_shape(L, d)).sum(axis=0) & 1
    return g.ravel()


def overlap_bruteforce(A, B, L, d):
    q = (A.astype(np.int64) * B.astype(np.int64)).reshape(lattice_shape(L, d))
    Q = int(q.sum())
    QL = sum(int((q * np.roll(q, -1, axis=axis_of(mu, d))).sum()) for mu in range(d))
    return Q, QL


def component_of(negmask, i0, L, d):
    """Connected component of i0 among sites with negmask True, nearest-neighbour periodic edges, using
    scipy's connected_components (a library routine independent of the oracle's BFS)."""
    from scipy.sparse import coo_matrix
    from scipy.sparse.csgraph import connected_components

    N = L ** d
    nbr = neighbour_list(L, d)
    rows, cols = [], []
    for k in range(2 * d):
        ok = negmask & negmask[nbr[:, k]]
        rows.append(np.nonzero(ok)[0])
        cols.append(nbr[ok, k])
    rows, cols = np.concatenate(rows), np.concatenate(cols)
    g = coo_matrix((np.ones(len(rows), dtype=np.int8), (rows, cols)), shape=(N, N))
    _, lab = connected_components(g, directed=False)
    return (lab == lab[i0]) & negmask


def enumerate_2d_L4(J, betas):
    """Exact canonical averages for one 2D L=4 sample by enumerating 2^16 states.
    Returns (<E>_beta [T], <q^2>_beta [T]) with <q^2> = N^-2 sum_ij <s_i s_j>^2 (two independent chains)."""
    return _enumerate(J, betas, 4, 2)


def _enumerate(J, betas, L, d):
    N = L ** d
    states = ((np.arange(1 << N)[:, None] >> np.arange(N)[None, :]) & 1).astype(np.int8) * 2 - 1
    nbr = neighbour_list(L, d)
    Jt = np.asarray(J)
    acc = np.float64 if np.issubdtype(Jt.dtype, np.floating) else np.int64      # real couplings: NEXT-3
    E = np.zeros(1 << N, dtype=acc)
    for mu in range(d):
        E -= (Jt[mu][None, :].astype(acc) * states * states[:, nbr[:, 2 * mu]]).sum(axis=1)
    Em, q2 = [], []
    sf = states.astype(np.float64)
    for b in betas:
        w = np.exp(-b * (E - E.min()))
        w /= w.sum()
        Em.append(float((w * E).sum()))
        corr = (sf * w[:, None]).T @ sf
        q2.append(float((corr ** 2).sum()) / N ** 2)
    return np.array(Em), np.array(q2), E


def enumerate_any(J, betas, L, d):
    return _enumerate(J, betas, L, d)


def binned_mean_err(x, nbins=40):
    x = np.asarray(x, dtype=np.float64)
    n = (len(x) // nbins) * nbins
    b = x[:n].reshape(nbins, -1).mean(axis=1)
    return b.mean(), b.std(ddof=1) / np.sqrt(nbins)


# ---- an independent, vectorised numpy Philox4x32-10 (test-side; uint64 arithmetic) ----

def philox_np(key, ctr):
    """key (2,), ctr (..., 4) uint32 -> (..., 4) uint32."""
    M0, M1 = np.uint64(0xD2511F53), np.uint64(0xCD9E8D57)
    c = [np.asarray(ctr)[..., k].astype(np.uint64) for k in range(4)]
    k0, k1 = np.uint64(key[0]), np.uint64(key[1])
    mask = np.uint64(0xFFFFFFFF)
    for _ in range(10):
        p0, p1 = M0 * c[0], M1 * c[2]
        c = [(p1 >> np.uint64(32)) ^ c[1] ^ k0, p1 & mask, (p0 >> np.uint64(32)) ^ c[3] ^ k1, p0 & mask]
        k0 = (k0 + np.uint64(0x9E3779B9)) & mask
        k1 = (k1 + np.uint64(0xBB67AE85)) & mask
    return np.stack(c, axis=-1).astype(np.uint32)
