"""Pins for the oracle's cell grid (O3) and friends-of-friends labeller (O4)."""
import numpy as np
import pytest

from paper_1412_8502_b200 import inputs


def test_p13_cells_invariants(orc):
    """Sum of counts = N; c w <= x < (c+1) w; cell_start monotone; id = (cz nc + cy) nc + cx."""
    c = inputs.CONFIGS[1]
    x, v, is_p, L = inputs.uniform_state(c["N"], c["Y_P"], c["density"], c["T"], seed=2)
    for k, expect_nc in ((1, 2), (2, 4), (3, 6)):  # cfg1 2/4/6 cells per side
        nc = orc.ncell(L, c["r_c"], k)
        assert nc == expect_nc
        cid, start = orc.cells(x, L, nc)
        assert start[0] == 0 and start[-1] == c["N"] and (np.diff(start) >= 0).all()
        assert np.array_equal(np.bincount(cid, minlength=nc ** 3), np.diff(start))
        w = L / nc
        cx, cy, cz = cid % nc, (cid // nc) % nc, cid // (nc * nc)
        for a, ca in enumerate((cx, cy, cz)):
            assert (ca * w <= x[:, a] + 1e-12).all() and (x[:, a] < (ca + 1) * w + 1e-12).all()
            assert np.array_equal(ca, np.minimum(nc - 1, np.floor(x[:, a] * (nc / L)).astype(np.int64)))


def test_cells_grid_sizes_of_the_configs(orc):
    """Cells per side at width >= r_c/k: cfg2 4/8/12, cfg4 8/17/25, ends 17, 34."""
    for L, expect in ((86.1774, (4, 8, 12)), (172.3548, (8, 17, 25)), (344.7096, (17, 34, 51)),
                      (689.4191, (34, 68, 103))):
        assert tuple(orc.ncell(L, 20.0, k) for k in (1, 2, 3)) == expect


def test_cells_faces_and_clamp(orc):
    L, nc = 12.0, 4
    x = np.array([[0.0, 3.0, 6.0], [9.0, 11.999999999999998, 2.9999999999999996], [3.0, 3.0, 3.0]])
    cid, start = orc.cells(x, L, nc)
    assert list(cid) == [(2 * 4 + 1) * 4 + 0, (0 * 4 + 3) * 4 + 3, (1 * 4 + 1) * 4 + 1]
    assert orc.ncell(5.0, 20.0, 1) == 1  # max(1, .)


def test_cell_coords_per_axis_is_the_o3_statement(orc):
    """orc.cell_coords (O3 per axis, used to check the force path's anisotropic grids) against what pins O3
    itself: the ids of orc.cells decoded axis by axis, the face/clamp hand cases above, and the interval property."""
    x, v, is_p, L = inputs.uniform_state(3000, 0.3, 0.05, 1.0, seed=4)
    for nc in (1, 2, 5, 13):
        cid, _ = orc.cells(x, L, nc)
        c = orc.cell_coords(x, L, nc)
        assert c.shape == x.shape and c.dtype == np.int32
        assert np.array_equal(c[:, 0], cid % nc) and np.array_equal(c[:, 1], (cid // nc) % nc)
        assert np.array_equal(c[:, 2], cid // (nc * nc))
    hand = np.array([[0.0, 3.0, 6.0], [9.0, 11.999999999999998, 2.9999999999999996], [3.0, 3.0, 3.0]])
    assert orc.cell_coords(hand, 12.0, 4).tolist() == [[0, 1, 2], [3, 3, 0], [1, 1, 1]]
    # a different cell count for one axis (thin cells along x): intervals [c w, (c+1) w) with w = L / n
    n = 37
    c = orc.cell_coords(x[:, 0], L, n)
    w = L / n
    assert c.min() == 0 and c.max() == n - 1
    assert (c * w <= x[:, 0] + 1e-12).all() and (x[:, 0] < (c + 1) * w + 1e-12).all()
    assert orc.cell_coords(np.array([L * (1 - 1e-17), -0.0]), L, n).tolist() == [n - 1, 0]  # clamp, as orc_cells


def _chain(n, spacing, start, axis=0):
    x = np.tile(np.asarray(start, dtype=float), (n, 1))
    x[:, axis] += spacing * np.arange(n)
    return x


def test_p14_chains_and_singletons(orc):
    """Hand-built cases (within the cut-off distance of at least one member)."""
    L = 60.0
    is_p = np.array([1, 0, 0, 1, 0, 0], dtype=np.uint8)
    lab, A, Z, n = orc.clusters(_chain(6, 2.9, [5, 5, 5]), is_p, L, 3.0)
    assert list(lab) == [0] * 6 and n == 1 and A[0] == 6 and Z[0] == 2 and A[1:].sum() == 0
    lab, A, Z, n = orc.clusters(_chain(6, 3.1, [5, 5, 5]), is_p, L, 3.0)
    assert list(lab) == list(range(6)) and n == 6 and list(A) == [1] * 6 and list(Z) == [1, 0, 0, 1, 0, 0]
    # exactly at the linking length: r^2 <= r_cl^2 links (D13)
    lab, _, _, n = orc.clusters(np.array([[1.0, 1, 1], [4.0, 1, 1]]), [0, 0], L, 3.0)
    assert n == 1
    # a chain through the periodic face, along each axis
    for axis in range(3):
        x = orc.wrap(_chain(5, 2.5, [L - 4.0 if a == axis else 7.0 for a in range(3)], axis), L)
        lab, A, Z, n = orc.clusters(x, [0] * 5, L, 3.0)
        assert n == 1 and list(lab) == [0] * 5
    # two separate groups; label = minimum member index regardless of input order
    x = np.vstack([_chain(3, 2.0, [40, 40, 40]), _chain(3, 2.0, [10, 10, 10])])
    order = [3, 0, 4, 1, 5, 2]
    lab, A, Z, n = orc.clusters(x[order], np.array([1, 0, 0, 0, 0, 1], dtype=np.uint8)[order], L, 3.0)
    assert n == 2 and list(lab) == [0, 1, 0, 1, 0, 1]
    assert A[0] == 3 and A[1] == 3 and Z[0] + Z[1] == 2


def test_p14_invariants_and_brute_vs_cells(orc):
    """Sum A = N, Sum Z = N_p; raising r_cl only merges; an index permutation maps labels
    consistently; brute force == independent cell-grid enumeration."""
    N = 3000
    x, v, is_p, L = inputs.clustered_state(N, 0.2, 0.004, 0.75, seed=6)
    prev_n = None
    prev_lab = None
    for r_cl in (1.5, 3.0, 4.5):
        lab, A, Z, n = orc.clusters(x, is_p, L, r_cl)
        lab2, A2, Z2, n2 = orc.clusters_cells(x, is_p, L, r_cl)
        assert np.array_equal(lab, lab2) and np.array_equal(A, A2) and np.array_equal(Z, Z2) and n == n2
        assert A.sum() == N and Z.sum() == is_p.sum() and n == (A > 0).sum()
        assert (lab <= np.arange(N)).all() and (lab[lab] == lab).all()
        assert np.array_equal(A[lab == np.arange(N)], np.bincount(lab, minlength=N)[lab == np.arange(N)])
        if prev_n is not None:
            assert n <= prev_n
            # same old label => same new label (merging only)
            assert (lab[prev_lab] == lab).all()
        prev_n, prev_lab = n, lab
    rng = np.random.default_rng(1)
    perm = rng.permutation(N)
    lab, A, Z, n = orc.clusters(x, is_p, L, 3.0)
    labp, Ap, Zp, np_ = orc.clusters(x[perm], is_p[perm], L, 3.0)
    assert np_ == n
    # partitions agree: i ~ j in the original  <=>  perm^-1(i) ~ perm^-1(j) in the permuted
    assert np.array_equal(np.unique(lab[perm], return_inverse=True)[1].shape, labp.shape)
    a = lab[perm]
    pairs = set(zip(a.tolist(), labp.tolist()))
    assert len(pairs) == n
    assert sorted(Ap[Ap > 0].tolist()) == sorted(A[A > 0].tolist())


def test_composition_summary(orc):
    """free-neutron fraction = #(A=1,Z=0)/N; mean/sigma over A >= 12."""
    A = np.array([1, 1, 0, 12, 0, 20, 11, 1], dtype=np.int32)
    Z = np.array([0, 1, 0, 4, 0, 8, 5, 0], dtype=np.int32)
    c = orc.composition(A, Z, 12)
    assert c["free_n_fraction"] == pytest.approx(2 / 8)
    assert c["n_heavy"] == 2 and c["mean_A"] == 16 and c["sigma_A"] == 4 and c["mean_Z"] == 6 and c["sigma_Z"] == 2


def test_mst_clusters_of_the_paper(orc):
    """PAPER.md:154-158 (reading D24).  Hand-built: two protons 4.4 fm apart form one cluster, a third 4.6 fm further
    is its own; a neutron 2.9 fm from a proton joins it, one 3.1 fm away is free; neutrons never link neutrons (a
    chain of neutrons hanging off a proton attaches only its first member); a neutron within r_np of protons of
    two clusters goes to the nearer one; the periodic image counts.  Invariants on a random state: sum A = N,
    sum Z = N_p, every cluster with A > 1 has Z >= 1, and with no neutrons the result equals friends-of-friends
    at r_cl = r_pp."""
    L = 100.0
    x = np.array([[10, 10, 10], [14.4, 10, 10], [19.0, 10, 10],      # protons 0, 1 (cluster 0), 2 (own)
                  [10, 12.9, 10], [10, 13.1 + 2.9, 10],               # neutron 3 joins 0; neutron 4 is 2.9 from 3, 6 from 0: free
                  [16.6, 10, 10],                                     # neutron 5: 2.2 from proton 1, 2.4 from proton 2 -> cluster 0
                  [99.0, 10, 10], [1.5, 10, 10]], dtype=float)        # proton 6 and neutron 7 across the face (2.5 fm)
    is_p = np.array([1, 1, 1, 0, 0, 0, 1, 0], dtype=np.uint8)
    label, A, Z, n = orc.clusters_mst(x, is_p, L)
    assert label.tolist() == [0, 0, 2, 0, 4, 0, 6, 6] and n == 4
    assert (A[0], Z[0]) == (4, 2) and (A[2], Z[2]) == (1, 1) and (A[4], Z[4]) == (1, 0) and (A[6], Z[6]) == (2, 1)
    x2, _, p2, L2 = inputs.uniform_state(1500, 0.3, 0.01, 1.0, seed=8)
    label, A, Z, n = orc.clusters_mst(x2, p2, L2)
    assert A.sum() == 1500 and Z.sum() == p2.sum() and np.all(Z[A > 1] >= 1) and n == np.count_nonzero(A)
    assert np.all(label[p2 == 1] < p2.sum())                          # clusters are named after protons
    xp = x2[p2 == 1]
    lf, Af, Zf, nf = orc.clusters(xp, np.ones(len(xp), np.uint8), L2, 4.5)
    lm, Am, Zm, nm = orc.clusters_mst(xp, np.ones(len(xp), np.uint8), L2, 4.5, 3.0)
    assert np.array_equal(lf, lm) and nf == nm
