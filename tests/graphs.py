"""Test helpers: seeded synthetic inputs, golden-file readers and brute-force checkers.

Nothing here implements the method under test (no union-find, no atomicMin chains): the checkers are textbook
breadth-first searches, used to pin the oracle to something other than itself.
"""
import os
from collections import deque

import numpy as np

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


# ---------------------------------------------------------------- golden files
def read_fig1_nn_list():
    nn = {}
    with open(os.path.join(GOLDEN, "e0_fig1_nn_list.txt")) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            site, rest = line.split(":")
            nn[int(site)] = [int(t) for t in rest.split()]
    return [nn[i] for i in range(len(nn))]


def read_e0_labels():
    out, residual = {}, {}
    with open(os.path.join(GOLDEN, "e0_labels.txt")) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            name, rest = line.split(":")
            if name.startswith("residual"):
                residual[int(name.split()[1])] = [int(t) for t in rest.split()]
            else:
                out[name] = [int(t) for t in rest.split()]
    return out, residual


def bonds_from_nn_list(nn):
    """Each undirected bond once, as (lower, higher), sorted."""
    bonds = sorted({(min(i, j), max(i, j)) for i, row in enumerate(nn) for j in row})
    src = np.array([b[0] for b in bonds], dtype=np.int32)
    dst = np.array([b[1] for b in bonds], dtype=np.int32)
    return src, dst


def read_philox_kat():
    rows = []
    with open(os.path.join(GOLDEN, "philox4x32_10_kat.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            w = [int(t, 16) for t in line.split()]
            rows.append((w[0:4], w[4:6], w[6:10]))
    return rows


# ---------------------------------------------------------------- brute force
def bfs_min_labels(n_sites, src, dst, occupied=None):
    """labels[i] = min site of i's component, by breadth-first search from every unvisited site in ascending order."""
    adj = [[] for _ in range(n_sites)]
    for b in range(len(src)):
        if occupied is not None and not occupied[b]:
            continue
        u, v = int(src[b]), int(dst[b])
        adj[u].append(v)
        adj[v].append(u)
    labels = [-1] * n_sites
    for s in range(n_sites):
        if labels[s] >= 0:
            continue
        labels[s] = s                    # ascending start order => s is the minimum of its component
        q = deque([s])
        while q:
            x = q.popleft()
            for y in adj[x]:
                if labels[y] < 0:
                    labels[y] = s
                    q.append(y)
    return np.array(labels, dtype=np.int32)


def bfs_winding(n_sites, src, dst, dx, dy, occupied=None):
    """(wrap_x, wrap_y) by BFS on the unwrapped cover: walk each component assigning unwrapped positions; an occupied
    bond whose ends are both placed and disagree with the bond's displacement closes a winding cycle."""
    adj = [[] for _ in range(n_sites)]
    for b in range(len(src)):
        if occupied is not None and not occupied[b]:
            continue
        u, v = int(src[b]), int(dst[b])
        adj[u].append((v, int(dx[b]), int(dy[b])))
        adj[v].append((u, -int(dx[b]), -int(dy[b])))
    pos = [None] * n_sites
    wx = wy = False
    for s in range(n_sites):
        if pos[s] is not None:
            continue
        pos[s] = (0, 0)
        q = deque([s])
        while q:
            x = q.popleft()
            for (y, ddx, ddy) in adj[x]:
                want = (pos[x][0] + ddx, pos[x][1] + ddy)
                if pos[y] is None:
                    pos[y] = want
                    q.append(y)
                else:
                    if pos[y][0] != want[0]:
                        wx = True
                    if pos[y][1] != want[1]:
                        wy = True
    return wx, wy


# ---------------------------------------------------------------- seeded synthetic inputs (no method arithmetic)
def random_graph(rng, n_sites, n_bonds, self_loops=True):
    """Uniform random endpoints (duplicates and, optionally, self-loops allowed)."""
    src = rng.integers(0, n_sites, size=n_bonds, dtype=np.int32)
    dst = rng.integers(0, n_sites, size=n_bonds, dtype=np.int32)
    if not self_loops and n_sites > 1:
        same = src == dst
        dst[same] = (dst[same] + 1) % n_sites
    return src, dst


def path_graph(n_sites, order="ascending", rng=None):
    """A path through all sites; numbering along the path ascending, descending or shuffled."""
    if order == "ascending":
        ids = np.arange(n_sites, dtype=np.int32)
    elif order == "descending":
        ids = np.arange(n_sites - 1, -1, -1, dtype=np.int32)
    else:
        ids = rng.permutation(n_sites).astype(np.int32)
    return ids[:-1].copy(), ids[1:].copy()


def pack_bits(mask):
    """uint8 mask -> uint32 words, bond b = bit (b & 31) of word (b >> 5)."""
    mask = np.asarray(mask, dtype=np.uint8)
    pad = (-mask.size) % 32
    m = np.concatenate([mask, np.zeros(pad, dtype=np.uint8)]).reshape(-1, 32).astype(np.uint32)
    return (m << np.arange(32, dtype=np.uint32)).sum(axis=1, dtype=np.uint64).astype(np.uint32)


def same_partition(a, b):
    """Do two label arrays describe the same partition of the sites?"""
    a = np.asarray(a)
    b = np.asarray(b)
    fwd, bwd = {}, {}
    for x, y in zip(a.tolist(), b.tolist()):
        if fwd.setdefault(x, y) != y or bwd.setdefault(y, x) != x:
            return False
    return True


def nn_list_from_bonds(n_sites, src, dst, occupied=None, both_sides=True, rng=None):
    """Dense z_max x n_sites nearest-neighbour list (structure of arrays, -1 padding) of the occupied bonds.
    both_sides: True = each bond is listed at both of its ends (the paper's form); False or "higher" = only at its
    higher-numbered end; "lower" = only at its lower-numbered end; "random" = at one end chosen by rng per bond."""
    keep = np.ones(len(src), dtype=bool) if occupied is None else np.asarray(occupied) != 0
    u = np.asarray(src)[keep].astype(np.int64)
    v = np.asarray(dst)[keep].astype(np.int64)
    if both_sides is True:
        a, b = np.concatenate([u, v]), np.concatenate([v, u])
    elif both_sides == "lower":
        a, b = np.minimum(u, v), np.maximum(u, v)
    elif both_sides == "random":
        flip = rng.random(u.size) < 0.5
        a, b = np.where(flip, u, v), np.where(flip, v, u)
    else:
        a, b = np.maximum(u, v), np.minimum(u, v)
    order = np.argsort(a, kind="stable")
    a, b = a[order], b[order]
    deg = np.bincount(a, minlength=n_sites) if a.size else np.zeros(n_sites, dtype=np.int64)
    z_max = int(deg.max()) if n_sites and a.size else 0
    nn = np.full((z_max, n_sites), -1, dtype=np.int32)
    start = np.concatenate([[0], np.cumsum(deg)[:-1]]) if n_sites else np.zeros(0, dtype=np.int64)
    slot = np.arange(a.size) - start[a] if a.size else np.zeros(0, dtype=np.int64)
    nn[slot, a] = b
    return nn
