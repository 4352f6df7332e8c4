"""Triangle-soup analysis used by the MC pins (pure numpy; no method code)."""
import numpy as np


def weld(tris):
    """tris (T,3,3) float32 -> (vertex ids (T,3), n_vertices) by BITWISE vertex equality (D:A-EDGE)."""
    flat = np.ascontiguousarray(tris.reshape(-1, 3), dtype=np.float32)
    flat = flat + np.float32(0.0)  # -0.0 -> +0.0 so that equal values have equal bits
    keys = flat.view(np.uint32).reshape(-1, 3)
    _, inv = np.unique(keys, axis=0, return_inverse=True)
    inv = inv.reshape(-1)
    return inv.reshape(-1, 3), int(inv.max()) + 1 if inv.size else 0


def edge_stats(ids):
    """Directed-edge census: returns (n_undirected_edges, all_edges_twice_opposite: bool, n_degenerate)."""
    a = ids[:, [0, 1, 2]].reshape(-1)
    b = ids[:, [1, 2, 0]].reshape(-1)
    degenerate = int(np.sum(a == b))
    directed = np.stack([a, b], 1)
    und = np.sort(directed, axis=1)
    uniq, counts = np.unique(und, axis=0, return_counts=True)
    ok = bool(np.all(counts == 2))
    # orientation: each directed edge must appear exactly once (its reverse is the partner)
    _, dc = np.unique(directed, axis=0, return_counts=True)
    ok = ok and bool(np.all(dc == 1))
    return len(uniq), ok, degenerate


def area_volume(tris):
    t = tris.astype(np.float64)
    a, b, c = t[:, 0], t[:, 1], t[:, 2]
    n = np.cross(b - a, c - a)
    area = 0.5 * np.linalg.norm(n, axis=1).sum()
    vol = np.einsum("ij,ij->i", a, np.cross(b, c)).sum() / 6.0
    return area, vol, n
