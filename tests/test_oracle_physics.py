"""Physics pins for the oracle: the exact thresholds the paper's lattices fix (p_c^tr = 2 sin(pi/18),
p_c^hc = 1 - 2 sin(pi/18); Bethe p_c = 1/(z-1)) and closed forms of percolation theory.

The paper's own correctness evidence is exactly this kind of test: 'all curves intersect at one point' and the crossing
gives p_c^hc = 0.6527 +- 0.0002, p_c^tr = 0.3472 +- 0.0002.  A labeling mistake (a dropped bond class,
a wrong neighbour in a generator, a biased mask) moves these numbers far outside the tolerances used here.
"""
import math

import numpy as np
import pytest

from oracle import oracle

PC_TR = 2.0 * math.sin(math.pi / 18.0)
PC_HC = 1.0 - PC_TR


def _sweep(gen, spc, L, ps, n_real, seed):
    src, dst, dx, dy = gen(L, with_disp=True)
    n = spc * L * L
    wrap = np.zeros(len(ps))
    smax = np.zeros(len(ps))
    ncl = np.zeros(len(ps))
    for r in range(n_real):
        for k, p in enumerate(ps):
            mask, _ = oracle.gen_occupancy(src.size, p, seed, realization=r)      # same (seed, r): nested in p
            labels = oracle.label(n, src, dst, mask)
            wx, wy = oracle.wrap(n, src, dst, dx, dy, mask)
            wrap[k] += wx or wy
            smax[k] += np.bincount(labels).max()
            ncl[k] += (labels == np.arange(n)).sum()
    return wrap / n_real, smax / n_real, ncl / n_real / n


@pytest.mark.parametrize("gen,spc,pc", [(oracle.gen_triangular, 1, PC_TR), (oracle.gen_honeycomb, 2, PC_HC)])
def test_wrapping_and_largest_cluster_curves_cross_at_pc(gen, spc, pc):
    delta = 0.008
    ps = [pc - delta, pc, pc + delta]
    n_real = 1000
    Ls = (24, 96)
    R, S = {}, {}
    for L in Ls:
        R[L], s, _ = _sweep(gen, spc, L, ps, n_real, seed=oracle.seed_for(100 + L))
        S[L] = s * float(L) ** (-91.0 / 48.0)                     # 2-D percolation: s_max ~ L^(91/48) at p_c
    a, b = Ls
    # below p_c the larger lattice wraps less often, above p_c more often; at p_c the curves meet
    assert R[b][0] < R[a][0] - 0.1 and R[b][2] > R[a][2] + 0.05
    assert R[a][0] < R[a][1] < R[a][2] and R[b][0] < R[b][1] < R[b][2]
    assert abs(R[b][1] - R[a][1]) < 0.08
    assert 0.55 < R[a][1] < 0.8 and 0.55 < R[b][1] < 0.8          # SURVEY probe: R_either(p_c) ~ 0.68-0.69
    # crossing point of the two curves: piecewise-linear interpolation of their difference through the three points
    d = R[b] - R[a]
    k = 0 if d[1] >= 0 else 1                                     # the sign change lies in [ps[k], ps[k+1]]
    p_cross = ps[k] + (ps[k + 1] - ps[k]) * (-d[k]) / (d[k + 1] - d[k])
    assert abs(p_cross - pc) < 0.003, p_cross
    # largest-cluster scaling curves cross at p_c too
    assert S[b][0] < S[a][0] and S[b][2] > S[a][2]
    assert abs(S[b][1] / S[a][1] - 1.0) < 0.08


@pytest.mark.parametrize("gen,spc,pc,per_site", [
    (oracle.gen_triangular, 1, PC_TR, 35.0 / 4.0 - 3.0 / PC_TR),          # clusters per site at p_c, triangular bond
    (oracle.gen_honeycomb, 2, PC_HC, None),                               # dual lattice, by Euler's relation (below)
])
def test_cluster_density_at_pc(gen, spc, pc, per_site):
    """Exact critical cluster densities: triangular bond percolation has 35/4 - 3/p_c = 0.1118443 clusters per site;
    the honeycomb value follows from duality + Euler: C_hc = V - E_occ + C_tr(dual) => n_hc = (n_tr - 1 + 3 p_c^tr) / 2 per honeycomb site
    = 0.0768667."""
    if per_site is None:
        n_tr = 35.0 / 4.0 - 3.0 / PC_TR
        per_site = (n_tr - 1.0 + 3.0 * PC_TR) / 2.0
        assert abs(per_site - 0.0768667) < 1e-6
    else:
        assert abs(per_site - 0.1118443) < 1e-6
    L = 128
    _, _, dens = _sweep(gen, spc, L, [pc], 120, seed=oracle.seed_for(200 + spc))
    assert abs(dens[0] - per_site) < 6e-4, dens[0]


@pytest.mark.parametrize("z,p", [(3, 0.75), (4, 0.45), (3, 0.6)])
def test_giant_component_fraction_on_regular_graphs(z, p):
    """Tree-like random z-regular graph: giant fraction = 1 - u^z, u = smallest root of u = 1 - p + p u^(z-1)."""
    u = 0.5
    for _ in range(10000):
        u = 1.0 - p + p * u ** (z - 1)
    if z == 3:
        assert abs(u - (1 - p) / p) < 1e-9
    want = 1.0 - u ** z
    if (z, p) == (3, 0.75):
        assert abs(want - 26.0 / 27.0) < 1e-12
    if (z, p) == (4, 0.45):
        assert abs(want - 0.741051) < 1e-5
    n = 1 << 18
    src, dst, _ = oracle.gen_regular(n, z, seed=oracle.seed_for(300 + z))
    mask, _ = oracle.gen_occupancy(src.size, p, seed=oracle.seed_for(301), realization=0)
    labels = oracle.label(n, src, dst, mask)
    st, _, _ = oracle.stats(labels)
    assert abs(st["largest"] / n - want) < 0.006, st["largest"] / n
    assert st["largest_label"] < 64                      # the giant cluster's minimum site is a very small index


@pytest.mark.parametrize("z", [3, 4])
def test_regular_graph_threshold_is_one_over_z_minus_1(z):
    """s_max * N^(-2/3) curves for two sizes cross at p_c = 1/(z-1) (mean-field scaling); well below p_c the largest
    cluster is O(log N)."""
    pc = 1.0 / (z - 1)
    sizes = (1 << 13, 1 << 17)
    S = {}
    for n in sizes:
        src, dst, _ = oracle.gen_regular(n, z, seed=oracle.seed_for(400 + z))
        acc = np.zeros(3)
        n_real = 12
        for r in range(n_real):
            for k, p in enumerate((0.8 * pc, pc, 1.2 * pc)):
                mask, _ = oracle.gen_occupancy(src.size, p, seed=oracle.seed_for(401), realization=r)
                acc[k] += np.bincount(oracle.label(n, src, dst, mask)).max()
        S[n] = acc / n_real * float(n) ** (-2.0 / 3.0)
        if n == sizes[1]:
            mask, _ = oracle.gen_occupancy(src.size, 0.5 * pc, seed=oracle.seed_for(402))
            assert np.bincount(oracle.label(n, src, dst, mask)).max() < 12 * math.log(n)
    a, b = sizes
    assert S[b][0] < 0.7 * S[a][0] and S[b][2] > 1.5 * S[a][2]
    assert 0.6 < S[b][1] / S[a][1] < 1.6


@pytest.mark.parametrize("z,p", [(3, 0.5), (4, 0.25), (4, 1.0 / 3.0), (4, 0.45)])
def test_small_cluster_histogram_on_regular_graphs(z, p):
    """Expected number of size-s tree clusters on a locally tree-like z-regular graph:
    N * z * ((z-1)s)! / (s! * ((z-2)s+2)!) * p^(s-1) * (1-p)^((z-2)s+2)."""
    n = 1 << 18
    src, dst, _ = oracle.gen_regular(n, z, seed=oracle.seed_for(500 + z))
    mask, _ = oracle.gen_occupancy(src.size, p, seed=oracle.seed_for(501))
    labels = oracle.label(n, src, dst, mask)
    _, hd, _ = oracle.stats(labels, n_dense=8)
    for s in (1, 2, 3, 5, 8):
        expect = (n * z * math.factorial((z - 1) * s) / (math.factorial(s) * math.factorial((z - 2) * s + 2))
                  * p ** (s - 1) * (1 - p) ** ((z - 2) * s + 2))
        assert abs(hd[s] - expect) < 6.0 * math.sqrt(expect) + 0.01 * expect, (s, hd[s], expect)
